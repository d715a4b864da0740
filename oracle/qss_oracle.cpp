// CPU ORACLE -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see qss_oracle.h).
//
// Written from the paper (PAPER.md = arXiv 2405.05974) and the standard CHEMKIN / NASA-7 forms the
// paper leaves implicit. Every routine is the plain definition, written out:
// dense loops, no sparsity, no rank-1 tricks, no blocking, one full-size elimination.
//
//   steps 1-5 (eval_wdot<S>)  : PAPER.md Eq. 2-3 (L59-64), Eq. 4 (L71), Eq. 6 (L150-157)
//   step 6   (eval_jac<S>)    : PAPER.md Eq. 7 (L185), Eq. 9 (L224) with k running over ALL species
//                               (reading G3), implicit-function theorem for dC_QSS/dx
//   templated scalar S        : double, __float128 (referee), Dual (forward-mode AD), std::complex
//                               (complex step) -- the last two differentiate eval_wdot mechanically, so
//                               they pin the hand-derived formulas of eval_jac.
//
// Pins (tests/test_oracle_*.py): toy closed forms, Kc closed form, Lindemann / high-pressure Troe limits,
// mass + element conservation, detailed-balance equilibrium, closure residual, dual / complex-step /
// float128 agreement, element null-space of every Jacobian column, N_q = 0 textbook Jacobian,
// first-order FD convergence (App. C).
//
// Parity status: every function below is pinned by at least one of those.  The Troe blending function at
// intermediate Pr is pinned by hand-derived points (f1 = 0, +1, -1 and the pole of f1, each at two hand-computed
// values of Fcent: tests/test_oracle_pins.py::test_troe_blending_hand_derived_points; every one of its five
// constants and the roles of alpha, T***, T*, T** are separated: a mutation of any of them fails that test).
#include "qss_oracle.h"

#include <cmath>
#include <complex>
#include <cstdlib>
#include <vector>
#include <quadmath.h>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double R_GAS = 8.31446261815324;   // J/(mol K)
const double P_REF = 101325.0;           // Pa
const double LN10 = 2.302585092994045684017991454684;

// ------------------------------------------------------------------------------------------------
// scalar types
// ------------------------------------------------------------------------------------------------
struct Dual {                      // value + tangent vector (empty tangent == zero)
    double v;
    std::vector<double> d;
    Dual(double x = 0.0) : v(x) {}
};
inline size_t dn(const Dual &a, const Dual &b) { return a.d.size() > b.d.size() ? a.d.size() : b.d.size(); }
inline double dg(const Dual &a, size_t i) { return a.d.empty() ? 0.0 : a.d[i]; }
inline Dual operator+(const Dual &a, const Dual &b) {
    Dual r(a.v + b.v); size_t n = dn(a, b); r.d.resize(n);
    for (size_t i = 0; i < n; ++i) r.d[i] = dg(a, i) + dg(b, i);
    return r;
}
inline Dual operator-(const Dual &a, const Dual &b) {
    Dual r(a.v - b.v); size_t n = dn(a, b); r.d.resize(n);
    for (size_t i = 0; i < n; ++i) r.d[i] = dg(a, i) - dg(b, i);
    return r;
}
inline Dual operator-(const Dual &a) { Dual r(-a.v); r.d.resize(a.d.size()); for (size_t i = 0; i < a.d.size(); ++i) r.d[i] = -a.d[i]; return r; }
inline Dual operator*(const Dual &a, const Dual &b) {
    Dual r(a.v * b.v); size_t n = dn(a, b); r.d.resize(n);
    for (size_t i = 0; i < n; ++i) r.d[i] = dg(a, i) * b.v + a.v * dg(b, i);
    return r;
}
inline Dual operator/(const Dual &a, const Dual &b) {
    Dual r(a.v / b.v); size_t n = dn(a, b); r.d.resize(n);
    for (size_t i = 0; i < n; ++i) r.d[i] = (dg(a, i) - r.v * dg(b, i)) / b.v;
    return r;
}
inline Dual &operator+=(Dual &a, const Dual &b) { a = a + b; return a; }
inline Dual &operator-=(Dual &a, const Dual &b) { a = a - b; return a; }
inline Dual chain(const Dual &a, double f, double df) { Dual r(f); r.d.resize(a.d.size()); for (size_t i = 0; i < a.d.size(); ++i) r.d[i] = df * a.d[i]; return r; }

typedef std::complex<double> Cplx;
typedef __float128 Quad;

inline double s_exp(double x) { return std::exp(x); }
inline double s_log(double x) { return std::log(x); }
inline double s_log10(double x) { return std::log10(x); }
inline double s_pow(double x, double p) { return std::pow(x, p); }
inline double s_re(double x) { return x; }
inline double s_abs(double x) { return std::fabs(x); }

inline Quad s_exp(Quad x) { return expq(x); }
inline Quad s_log(Quad x) { return logq(x); }
inline Quad s_log10(Quad x) { return log10q(x); }
inline Quad s_pow(Quad x, double p) { return powq(x, (Quad)p); }
inline double s_re(Quad x) { return (double)x; }
inline Quad s_abs(Quad x) { return fabsq(x); }

inline Cplx s_exp(Cplx x) { return std::exp(x); }
inline Cplx s_log(Cplx x) { return std::log(x); }
inline Cplx s_log10(Cplx x) { return std::log(x) / LN10; }
inline Cplx s_pow(Cplx x, double p) { return std::exp(p * std::log(x)); }
inline double s_re(Cplx x) { return x.real(); }
inline Cplx s_abs(Cplx x) { return x; }      // scales are not meaningful in complex-step mode

inline Dual s_exp(const Dual &x) { double e = std::exp(x.v); return chain(x, e, e); }
inline Dual s_log(const Dual &x) { return chain(x, std::log(x.v), 1.0 / x.v); }
inline Dual s_log10(const Dual &x) { return chain(x, std::log10(x.v), 1.0 / (x.v * LN10)); }
inline Dual s_pow(const Dual &x, double p) { double f = std::pow(x.v, p); return chain(x, f, p * f / x.v); }
inline double s_re(const Dual &x) { return x.v; }
inline Dual s_abs(const Dual &x) { return x.v < 0 ? -x : x; }

template <class S> inline S ipow(const S &c, int nu) {   // integer power by repeated multiplication
    S r = c;
    for (int i = 1; i < nu; ++i) r = r * c;
    return r;
}

// ------------------------------------------------------------------------------------------------
// one direction of one reaction
// ------------------------------------------------------------------------------------------------
struct Side { const int32_t *sp; const int32_t *nu; int n; };
inline Side reactants(const oracle_mech_t *m, int j) { int a = m->reac_ptr[j]; return Side{m->reac_sp + a, m->reac_nu + a, m->reac_ptr[j + 1] - a}; }
inline Side products(const oracle_mech_t *m, int j) { int a = m->prod_ptr[j]; return Side{m->prod_sp + a, m->prod_nu + a, m->prod_ptr[j + 1] - a}; }
inline int qss_of(const oracle_mech_t *m, const Side &s) {   // local QSS index on this side, -1 if none, -2 if invalid
    int q = -1;
    for (int i = 0; i < s.n; ++i)
        if (s.sp[i] >= m->n_nqss) { if (q != -1 || s.nu[i] != 1) return -2; q = s.sp[i] - m->n_nqss; }
    return q;
}

// ------------------------------------------------------------------------------------------------
// steps 1-3: thermo and rate constants (standard forms; reading G4)
// ------------------------------------------------------------------------------------------------
template <class S> struct Rates {
    std::vector<S> h_RT, g_RT;          // per species
    std::vector<S> kf, kb;              // effective k (incl. third-body / fall-off), kb = k / Kc
    std::vector<S> dlnkf_dT, dlnKc_dT;  // d ln k / dT at fixed M ; d ln Kc / dT
    std::vector<S> dkf_dM, dkb_dM;      // d k / d M and d kb / d M = (d k / d M) / Kc  (types 1, 2)
    std::vector<S> alpha;               // scratch: third-body efficiencies of the current reaction
};

template <class S> void eval_rates(const oracle_mech_t *m, const S *C, const S &T, Rates<S> &r) {
    const int N = m->n_nqss, nsp = m->n_nqss + m->n_qss, M = m->n_reac;
    r.h_RT.assign(nsp, S(0.0)); r.g_RT.assign(nsp, S(0.0));
    r.kf.assign(M, S(0.0)); r.kb.assign(M, S(0.0));
    r.dlnkf_dT.assign(M, S(0.0)); r.dlnKc_dT.assign(M, S(0.0)); r.dkf_dM.assign(M, S(0.0)); r.dkb_dM.assign(M, S(0.0));
    const S lnT = s_log(T);
    const S T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    for (int s = 0; s < nsp; ++s) {      // NASA-7; low set for T < Tmid, else high (reading G9)
        const double *a = (s_re(T) < m->nasa_T[3 * s + 1]) ? m->nasa_lo + 7 * s : m->nasa_hi + 7 * s;
        S h = S(a[0]) + S(a[1] / 2.0) * T + S(a[2] / 3.0) * T2 + S(a[3] / 4.0) * T3 + S(a[4] / 5.0) * T4 + S(a[5]) / T;
        S sR = S(a[0]) * lnT + S(a[1]) * T + S(a[2] / 2.0) * T2 + S(a[3] / 3.0) * T3 + S(a[4] / 4.0) * T4 + S(a[6]);
        r.h_RT[s] = h; r.g_RT[s] = h - sR;
    }
    const S lnP0RT = s_log(S(P_REF) / (S(R_GAS) * T));
    for (int j = 0; j < M; ++j) {
        const double A = m->arr[3 * j], beta = m->arr[3 * j + 1], Ea = m->arr[3 * j + 2];
        const S kinf = S(A) * s_pow(T, beta) * s_exp(S(-Ea) / (S(R_GAS) * T));
        const S dlnkinf = (S(beta) + S(Ea) / (S(R_GAS) * T)) / T;
        S k = kinf, dlnk = dlnkinf, dkdM = S(0.0);
        const int type = m->rtype[j];
        if (type >= 1) {
            r.alpha.assign(N, S(1.0));
            for (int e = m->eff_ptr[j]; e < m->eff_ptr[j + 1]; ++e) r.alpha[m->eff_sp[e]] = S(m->eff_val[e]);
            S Mc = S(0.0);                  // transported species only (reading G7)
            for (int i = 0; i < N; ++i) Mc = Mc + r.alpha[i] * C[i];
            if (type == 1) {
                k = kinf * Mc; dkdM = kinf;
            } else {
                const double A0 = m->arr_low[3 * j], b0 = m->arr_low[3 * j + 1], E0 = m->arr_low[3 * j + 2];
                const double ta = m->troe[4 * j], T3s = m->troe[4 * j + 1], T1s = m->troe[4 * j + 2], T2s = m->troe[4 * j + 3];
                const S k0 = S(A0) * s_pow(T, b0) * s_exp(S(-E0) / (S(R_GAS) * T));
                const S dlnk0 = (S(b0) + S(E0) / (S(R_GAS) * T)) / T;
                const S Pr = k0 * Mc / kinf;
                const S e3 = s_exp(-T / S(T3s)), e1 = s_exp(-T / S(T1s)), e2 = s_exp(S(-T2s) / T);
                const S Fc = S(1.0 - ta) * e3 + S(ta) * e1 + e2;
                const S dFc = S(-(1.0 - ta) / T3s) * e3 - S(ta / T1s) * e1 + S(T2s) / (T * T) * e2;
                const S L = s_log10(Pr), Lc = s_log10(Fc);
                const S c = S(-0.4) - S(0.67) * Lc, n = S(0.75) - S(1.27) * Lc;
                const S num = L + c, den = n - S(0.14) * num;
                const S f1 = num / den;
                const S one_f = S(1.0) + f1 * f1;
                const S log10F = Lc / one_f;
                const S F = s_exp(S(LN10) * log10F);
                k = kinf * (Pr / (S(1.0) + Pr)) * F;
                const S df1_dL = n / (den * den);
                const S dlF_dL = S(-2.0) * Lc * f1 * df1_dL / (one_f * one_f);
                const S df1_dLc = (S(-0.67) * den - num * S(-1.27 + 0.14 * 0.67)) / (den * den);
                const S dlF_dLc = S(1.0) / one_f - S(2.0) * Lc * f1 * df1_dLc / (one_f * one_f);
                dkdM = k * (S(1.0) / (S(1.0) + Pr) + dlF_dL) / Mc;
                const S delta = dlnk0 - dlnkinf;
                dlnk = dlnkinf + delta / (S(1.0) + Pr) + dlF_dL * delta + dlF_dLc * dFc / Fc;
            }
        }
        r.kf[j] = (m->dir_mask[j] & 1) ? k : S(0.0);
        r.dlnkf_dT[j] = dlnk; r.dkf_dM[j] = dkdM;
        if (m->dir_mask[j] & 2) {            // reverse from the equilibrium constant (reading G10: only if enabled)
            const Side re = reactants(m, j), pr = products(m, j);
            S dG = S(0.0), dH = S(0.0); int dnu = 0;
            for (int i = 0; i < pr.n; ++i) { dG = dG + S((double)pr.nu[i]) * r.g_RT[pr.sp[i]]; dH = dH + S((double)pr.nu[i]) * r.h_RT[pr.sp[i]]; dnu += pr.nu[i]; }
            for (int i = 0; i < re.n; ++i) { dG = dG - S((double)re.nu[i]) * r.g_RT[re.sp[i]]; dH = dH - S((double)re.nu[i]) * r.h_RT[re.sp[i]]; dnu -= re.nu[i]; }
            const S lnKc = -dG + S((double)dnu) * lnP0RT;
            const S Kc = s_exp(lnKc);
            r.kb[j] = k / Kc;                 // also when the forward direction is disabled
            r.dkb_dM[j] = dkdM / Kc;
            r.dlnKc_dT[j] = (dH - S((double)dnu)) / T;
        }
    }
}

// ------------------------------------------------------------------------------------------------
// steps 4-5: QSS closure (subtraction-free elimination, natural order, full size) and wdot
// ------------------------------------------------------------------------------------------------
template <class S> struct Closure {
    int nq;
    std::vector<S> P, leak, p0, D, y;     // P[m*nq + n]: production of m from n. After solve(): factors.
    void init(int n) { nq = n; P.assign((size_t)n * n, S(0.0)); leak.assign(n, S(0.0)); p0.assign(n, S(0.0)); D.assign(n, S(0.0)); y.assign(n, S(0.0)); }
    void eliminate() {                    // SURVEY.md 8(c)-4; no subtraction anywhere
        const int g = nq;
        for (int k = g - 1; k >= 1; --k) {
            S Dk = leak[k];
            for (int mm = 0; mm < k; ++mm) Dk = Dk + P[mm * g + k];
            D[k] = Dk;
            for (int j = 0; j < k; ++j) {
                const S f = P[k * g + j] / Dk;
                leak[j] = leak[j] + f * leak[k];
                for (int mm = 0; mm < k; ++mm)
                    if (mm != j) P[mm * g + j] = P[mm * g + j] + P[mm * g + k] * f;
            }
        }
        if (g > 0) D[0] = leak[0];
    }
    // solve (diag D - P) x = rhs with the stored factors; rhs may have any sign. In place.
    void solve(S *rhs) const {
        const int g = nq;
        for (int k = g - 1; k >= 1; --k) {
            const S t = rhs[k] / D[k];
            for (int mm = 0; mm < k; ++mm) rhs[mm] = rhs[mm] + P[mm * g + k] * t;
        }
        for (int k = 0; k < g; ++k) {
            S acc = rhs[k];
            for (int j = 0; j < k; ++j) acc = acc + P[k * g + j] * rhs[j];
            rhs[k] = acc / D[k];
        }
    }
};

template <class S> struct WdotOut { std::vector<S> wdot, Sscale; };

// kappa_d = k_d * prod of TRANSPORTED reactant concentrations of direction d
template <class S> S kappa_of(const oracle_mech_t *m, const Side &re, const S &kd, const S *C) {
    S kap = kd;
    for (int i = 0; i < re.n; ++i)
        if (re.sp[i] < m->n_nqss) kap = kap * ipow(C[re.sp[i]], re.nu[i]);
    return kap;
}

template <class S>
int eval_wdot(const oracle_mech_t *m, const S *C, const S &T, Rates<S> &rt, Closure<S> &cl, WdotOut<S> &out) {
    const int N = m->n_nqss, Nq = m->n_qss, M = m->n_reac;
    eval_rates(m, C, T, rt);
    cl.init(Nq);
    for (int j = 0; j < M; ++j)
        for (int dir = 0; dir < 2; ++dir) {
            if (!(m->dir_mask[j] & (1 << dir))) continue;
            const Side re = dir == 0 ? reactants(m, j) : products(m, j);
            const Side pr = dir == 0 ? products(m, j) : reactants(m, j);
            const int qn = qss_of(m, re), qm = qss_of(m, pr);
            if (qn == -2 || qm == -2) return -1;           // quadratic coupling: not linearised
            const S kap = kappa_of(m, re, dir == 0 ? rt.kf[j] : rt.kb[j], C);
            if (qn >= 0) {
                if (qm >= 0 && qm != qn) cl.P[qm * Nq + qn] = cl.P[qm * Nq + qn] + kap;
                else if (qm < 0) cl.leak[qn] = cl.leak[qn] + kap;
                /* qm == qn: the species is consumed and re-formed; no net contribution */
            } else if (qm >= 0) {
                cl.p0[qm] = cl.p0[qm] + kap;
            }
        }
    cl.eliminate();
    for (int i = 0; i < Nq; ++i) cl.y[i] = cl.p0[i];
    cl.solve(cl.y.data());
    out.wdot.assign(N, S(0.0)); out.Sscale.assign(N, S(0.0));
    for (int j = 0; j < M; ++j) {
        S rate[2] = {S(0.0), S(0.0)};
        for (int dir = 0; dir < 2; ++dir) {
            if (!(m->dir_mask[j] & (1 << dir))) continue;
            const Side re = dir == 0 ? reactants(m, j) : products(m, j);
            const int qn = qss_of(m, re);
            S r = kappa_of(m, re, dir == 0 ? rt.kf[j] : rt.kb[j], C);
            if (qn >= 0) r = r * cl.y[qn];
            rate[dir] = r;
        }
        const S Q = rate[0] - rate[1], Sabs = rate[0] + rate[1];
        const Side re = reactants(m, j), pr = products(m, j);
        // Eq. 3: wdot_i = sum_j nu_ij Q_j with the NET coefficient nu_ij = nu'' - nu'; a species that stands on
        // both sides of a reaction with the same coefficient (a collision partner written out) gets no term at all.  The scale
        // S_i = sum_j |nu_ij| (r_f + r_r) uses the same coefficient.
        for (int s = 0; s < N; ++s) {
            int net = 0;
            for (int i = 0; i < pr.n; ++i) if (pr.sp[i] == s) net += pr.nu[i];
            for (int i = 0; i < re.n; ++i) if (re.sp[i] == s) net -= re.nu[i];
            if (net != 0) {
                out.wdot[s] = out.wdot[s] + S((double)net) * Q;
                out.Sscale[s] = out.Sscale[s] + S((double)std::abs(net)) * Sabs;
            }
        }
    }
    return 0;
}

// ------------------------------------------------------------------------------------------------
// step 6: explicit analytical Jacobian, dense. J = W_x + W_y * Y_x, (diag D - P) Y_x = G_x
// ------------------------------------------------------------------------------------------------
template <class S> struct JacWork {
    std::vector<S> E, Eabs;      // [(N+Nq) x (N+1)]  rows < N: W_x, rows >= N: G_x   (d w_s / d x_k at fixed y)
    std::vector<S> Wy, Wyabs;    // [N x Nq]
    std::vector<S> col, c, alpha;
    std::vector<int> net;
};

template <class S>
int eval_jac(const oracle_mech_t *m, const S *C, const S &T, Rates<S> &rt, Closure<S> &cl, WdotOut<S> &wo,
             JacWork<S> &w, S *J /* [N*(N+1)] row-major */, S *Jscale /* may be null */, bool drop_chain, bool zero_qss = false) {
    const int N = m->n_nqss, Nq = m->n_qss, M = m->n_reac, nsp = N + Nq, NC = N + 1;
    if (eval_wdot(m, C, T, rt, cl, wo) != 0) return -1;
    w.E.assign((size_t)nsp * NC, S(0.0)); w.Eabs.assign((size_t)nsp * NC, S(0.0));
    w.Wy.assign((size_t)N * Nq, S(0.0)); w.Wyabs.assign((size_t)N * Nq, S(0.0));
    w.c.resize(nsp);
    for (int s = 0; s < N; ++s) w.c[s] = C[s];
    for (int q = 0; q < Nq; ++q) w.c[N + q] = zero_qss ? S(0.0) : cl.y[q];      // zero-QSS AJ: C_QSS := 0 in the partials
    w.net.assign(nsp, 0);
    for (int j = 0; j < M; ++j) {
        const Side rs = reactants(m, j), ps = products(m, j);
        for (int s = 0; s < nsp; ++s) w.net[s] = 0;
        for (int i = 0; i < ps.n; ++i) w.net[ps.sp[i]] += ps.nu[i];
        for (int i = 0; i < rs.n; ++i) w.net[rs.sp[i]] -= rs.nu[i];
        const int type = m->rtype[j];
        if (type >= 1) {
            w.alpha.assign(N, S(1.0));
            for (int e = m->eff_ptr[j]; e < m->eff_ptr[j + 1]; ++e) w.alpha[m->eff_sp[e]] = S(m->eff_val[e]);
        }
        for (int dir = 0; dir < 2; ++dir) {
            if (!(m->dir_mask[j] & (1 << dir))) continue;
            const Side re = dir == 0 ? rs : ps;
            const double sg = dir == 0 ? 1.0 : -1.0;
            // k_d, d ln k_d / dT, d k_d / dM  (kb = k / Kc with Kc a function of T only)
            const S kd = dir == 0 ? rt.kf[j] : rt.kb[j];
            const S dlnk = dir == 0 ? rt.dlnkf_dT[j] : rt.dlnkf_dT[j] - rt.dlnKc_dT[j];
            const S dlnk_abs = dir == 0 ? s_abs(rt.dlnkf_dT[j]) : s_abs(rt.dlnkf_dT[j]) + s_abs(rt.dlnKc_dT[j]);
            const S dkdM = dir == 0 ? rt.dkf_dM[j] : rt.dkb_dM[j];
            // product over all reactants of the direction (transported and QSS)
            S prod_all = S(1.0);
            for (int i = 0; i < re.n; ++i) prod_all = prod_all * ipow(w.c[re.sp[i]], re.nu[i]);
            const S r_d = kd * prod_all;
            // explicit dependence on each reactant concentration: product of the others (valid at C = 0)
            for (int a = 0; a < re.n; ++a) {
                S part = kd * S((double)re.nu[a]);
                if (re.nu[a] > 1) part = part * ipow(w.c[re.sp[a]], re.nu[a] - 1);
                for (int b = 0; b < re.n; ++b) if (b != a) part = part * ipow(w.c[re.sp[b]], re.nu[b]);
                const int v = re.sp[a];
                if (v < N) {
                    for (int s = 0; s < nsp; ++s) if (w.net[s] != 0) {
                        w.E[(size_t)s * NC + v] = w.E[(size_t)s * NC + v] + S(sg * w.net[s]) * part;
                        w.Eabs[(size_t)s * NC + v] = w.Eabs[(size_t)s * NC + v] + S((double)std::abs(w.net[s])) * s_abs(part);
                    }
                } else {
                    const int q = v - N;      // d r_d / d y_q = kappa_d
                    for (int s = 0; s < N; ++s) if (w.net[s] != 0) {
                        w.Wy[(size_t)s * Nq + q] = w.Wy[(size_t)s * Nq + q] + S(sg * w.net[s]) * part;
                        w.Wyabs[(size_t)s * Nq + q] = w.Wyabs[(size_t)s * Nq + q] + S((double)std::abs(w.net[s])) * s_abs(part);
                    }
                }
            }
            // dependence through the third-body concentration M (every transported species)
            if (type >= 1) {
                for (int v = 0; v < N; ++v) {
                    const S part = dkdM * w.alpha[v] * prod_all;
                    for (int s = 0; s < nsp; ++s) if (w.net[s] != 0) {
                        w.E[(size_t)s * NC + v] = w.E[(size_t)s * NC + v] + S(sg * w.net[s]) * part;
                        w.Eabs[(size_t)s * NC + v] = w.Eabs[(size_t)s * NC + v] + S((double)std::abs(w.net[s])) * s_abs(part);
                    }
                }
            }
            // temperature
            for (int s = 0; s < nsp; ++s) if (w.net[s] != 0) {
                w.E[(size_t)s * NC + N] = w.E[(size_t)s * NC + N] + S(sg * w.net[s]) * r_d * dlnk;
                w.Eabs[(size_t)s * NC + N] = w.Eabs[(size_t)s * NC + N] + S((double)std::abs(w.net[s])) * s_abs(r_d) * dlnk_abs;
            }
        }
    }
    // chain rule through the closure: columns of Y_x = dy/dx, then J = W_x + W_y Y_x
    w.col.resize(Nq);
    for (int pass = 0; pass < (Jscale ? 2 : 1); ++pass) {
        const std::vector<S> &EE = pass == 0 ? w.E : w.Eabs;
        const std::vector<S> &WW = pass == 0 ? w.Wy : w.Wyabs;
        S *out = pass == 0 ? J : Jscale;
        for (int k = 0; k < NC; ++k) {
            for (int q = 0; q < Nq; ++q) w.col[q] = EE[(size_t)(N + q) * NC + k];
            if (Nq > 0) cl.solve(w.col.data());
            for (int i = 0; i < N; ++i) {
                S acc = EE[(size_t)i * NC + k];
                if (!(drop_chain && pass == 0))
                    for (int q = 0; q < Nq; ++q) acc = acc + WW[(size_t)i * Nq + q] * w.col[q];
                out[(size_t)i * NC + k] = acc;
            }
        }
    }
    return 0;
}

template <class S> struct Work { Rates<S> rt; Closure<S> cl; WdotOut<S> wo; JacWork<S> jw; std::vector<S> C, J, Js; };

template <class S>
int run_explicit(const oracle_mech_t *m, int64_t c, int64_t ld, const double *C, const double *T, double *wdot,
                 double *cqss, double *Sc, double *jac, double *jscale, bool drop_chain, Work<S> &w, bool zero_qss = false) {
    const int N = m->n_nqss, Nq = m->n_qss, NC = N + 1;
    w.C.resize(N);
    for (int k = 0; k < N; ++k) w.C[k] = S(C[(size_t)k * ld + c]);
    const S Tc = S(T[c]);
    int rc;
    if (jac || jscale) {
        w.J.resize((size_t)N * NC); w.Js.resize((size_t)N * NC);
        rc = eval_jac(m, w.C.data(), Tc, w.rt, w.cl, w.wo, w.jw, w.J.data(), jscale ? w.Js.data() : (S *)0, drop_chain, zero_qss);
        if (rc) return rc;
        for (int e = 0; e < N * NC; ++e) {
            if (jac) jac[(size_t)e * ld + c] = s_re(w.J[e]);
            if (jscale) jscale[(size_t)e * ld + c] = s_re(w.Js[e]);
        }
    } else {
        rc = eval_wdot(m, w.C.data(), Tc, w.rt, w.cl, w.wo);
        if (rc) return rc;
    }
    for (int i = 0; i < N; ++i) {
        if (wdot) wdot[(size_t)i * ld + c] = s_re(w.wo.wdot[i]);
        if (Sc) Sc[(size_t)i * ld + c] = s_re(w.wo.Sscale[i]);
    }
    if (cqss) for (int q = 0; q < Nq; ++q) cqss[(size_t)q * ld + c] = s_re(w.cl.y[q]);
    return 0;
}

// ------------------------------------------------------------------------------------------------
// NEXT-1: temperature right-hand side and the energy row of the (N+1) x (N+1) Jacobian (Eq. 7: "the
// contribution of the heat release rate can be simply obtained from the species production rates").
// Reading G17: adiabatic CONSTANT-VOLUME reactor, thermodynamic sums over the transported
// species only (the QSS species carry no inventory: dC_q/dt = 0, L69-73):
//     sum_i C_i cv_i dT/dt = - sum_i u_i wdot_i,   u_i = h_i - R T,  cv_i = cp_i - R      (molar, NASA-7)
//  => Tdot = - T E / Cv,   E = sum_i (h_i/RT - 1) wdot_i,   Cv = sum_i C_i (cp_i/R - 1).
// ------------------------------------------------------------------------------------------------
template <class S> struct Thermo1 { S hRT, cpR, dcpR_dT; };
template <class S> Thermo1<S> nasa_species(const oracle_mech_t *m, int s, const S &T) {     // low set for T < Tmid, else high (G9)
    const double *a = (s_re(T) < m->nasa_T[3 * s + 1]) ? m->nasa_lo + 7 * s : m->nasa_hi + 7 * s;
    const S T2 = T * T, T3 = T2 * T, T4 = T3 * T;
    Thermo1<S> t;
    t.hRT = S(a[0]) + S(a[1] / 2.0) * T + S(a[2] / 3.0) * T2 + S(a[3] / 4.0) * T3 + S(a[4] / 5.0) * T4 + S(a[5]) / T;
    t.cpR = S(a[0]) + S(a[1]) * T + S(a[2]) * T2 + S(a[3]) * T3 + S(a[4]) * T4;
    t.dcpR_dT = S(a[1]) + S(2.0 * a[2]) * T + S(3.0 * a[3]) * T2 + S(4.0 * a[4]) * T3;
    return t;
}

// the right-hand side itself, templated: its dual-number / complex-step instantiations differentiate it mechanically
template <class S> int eval_tdot(const oracle_mech_t *m, const S *C, const S &T, Rates<S> &rt, Closure<S> &cl, WdotOut<S> &wo, S &Tdot) {
    if (eval_wdot(m, C, T, rt, cl, wo) != 0) return -1;
    S E = S(0.0), Cv = S(0.0);
    for (int i = 0; i < m->n_nqss; ++i) {
        const Thermo1<S> t = nasa_species(m, i, T);
        E = E + (t.hRT - S(1.0)) * wo.wdot[i];
        Cv = Cv + C[i] * (t.cpR - S(1.0));
    }
    Tdot = S(0.0) - T * E / Cv;
    return 0;
}

// explicit energy row from the species block J [N x (N+1)] and wdot (the plain differentiation of Tdot = -T E / Cv):
//   d Tdot / d C_k = -(T / Cv) sum_i u_i J_ik - Tdot (cp_k/R - 1) / Cv                                     u_i = h_i/RT - 1
//   d Tdot / d T   = Tdot / T - (T / Cv) sum_i (u_i J_iT + wdot_i (cp_i/R - h_i/RT) / T) - Tdot sum_i C_i d(cp_i/R)/dT / Cv
// `scale` (may be null): the same sums with every term replaced by its absolute value (running-error scale for the gates).
template <class S>
void energy_row(const oracle_mech_t *m, const S *C, const S &T, const S *wdot, const S *J, const S *Jscale, S &Tdot, S *row, S *scale) {
    const int N = m->n_nqss, NC = N + 1;
    std::vector<Thermo1<S>> th(N);
    S E = S(0.0), Eabs = S(0.0), Cv = S(0.0), dCv = S(0.0), dCvabs = S(0.0);
    for (int i = 0; i < N; ++i) {
        th[i] = nasa_species(m, i, T);
        E = E + (th[i].hRT - S(1.0)) * wdot[i];
        Eabs = Eabs + s_abs((th[i].hRT - S(1.0)) * wdot[i]);
        Cv = Cv + C[i] * (th[i].cpR - S(1.0));
        dCv = dCv + C[i] * th[i].dcpR_dT;
        dCvabs = dCvabs + s_abs(C[i] * th[i].dcpR_dT);
    }
    Tdot = S(0.0) - T * E / Cv;
    const S g = T / Cv;
    for (int k = 0; k < NC; ++k) {
        S e = S(0.0), ea = S(0.0);
        for (int i = 0; i < N; ++i) {
            e = e + (th[i].hRT - S(1.0)) * J[(size_t)i * NC + k];
            if (scale) ea = ea + s_abs(th[i].hRT - S(1.0)) * Jscale[(size_t)i * NC + k];
            if (k == N) {
                const S dh = (th[i].cpR - th[i].hRT) / T * wdot[i];
                e = e + dh; ea = ea + s_abs(dh);
            }
        }
        if (k < N) {
            row[k] = S(0.0) - g * e - Tdot * (th[k].cpR - S(1.0)) / Cv;
            if (scale) scale[k] = s_abs(g) * ea + s_abs(g * Eabs / Cv * (th[k].cpR - S(1.0)));
        } else {
            row[k] = Tdot / T - g * e - Tdot * dCv / Cv;
            if (scale) scale[k] = s_abs(Eabs / Cv) + s_abs(g) * ea + s_abs(g * Eabs / Cv) * dCvabs / s_abs(Cv);
        }
    }
}

template <class S>
int run_energy(const oracle_mech_t *m, int64_t c, int64_t ld, const double *C, const double *T, double *tdot, double *erow, double *escale, Work<S> &w) {
    const int N = m->n_nqss, NC = N + 1;
    w.C.resize(N);
    for (int k = 0; k < N; ++k) w.C[k] = S(C[(size_t)k * ld + c]);
    const S Tc = S(T[c]);
    w.J.resize((size_t)N * NC); w.Js.resize((size_t)N * NC);
    if (eval_jac(m, w.C.data(), Tc, w.rt, w.cl, w.wo, w.jw, w.J.data(), w.Js.data(), false)) return -1;
    std::vector<S> row(NC), sc(NC);
    S Td;
    energy_row(m, w.C.data(), Tc, w.wo.wdot.data(), w.J.data(), w.Js.data(), Td, row.data(), sc.data());
    if (tdot) tdot[c] = s_re(Td);
    for (int k = 0; k < NC; ++k) { if (erow) erow[(size_t)k * ld + c] = s_re(row[k]); if (escale) escale[(size_t)k * ld + c] = s_re(sc[k]); }
    return 0;
}

}  // namespace

// Temperature right-hand side tdot[c] and energy row erow[k*ld + c] (k < N: d Tdot/d C_k, k = N: d Tdot/d T); escale: the
// running-error scale of the row.  mode: ORACLE_EXPLICIT_F64 / _F128 (explicit formulas), ORACLE_JAC_DUAL / _CSTEP (the row by
// differentiating the right-hand side mechanically; tdot from the plain double routine, escale not written).
extern "C" int oracle_eval_energy(const oracle_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T,
                                  double *tdot, double *erow, double *escale, int mode, int nthreads) {
    if (!m || !C || !T || ncells < 0 || ld < ncells || mode < 0 || mode > 3) return -1;
    const int N = m->n_nqss, NC = N + 1;
    if (nthreads <= 0) nthreads = oracle_max_threads();
    int err = 0;
#pragma omp parallel num_threads(nthreads)
    {
        Work<double> wd; Work<Quad> wq; Work<Dual> wdu; Work<Cplx> wc;
#pragma omp for schedule(dynamic, 8)
        for (int64_t c = 0; c < ncells; ++c) {
            int rc = 0;
            if (mode == ORACLE_EXPLICIT_F64) rc = run_energy<double>(m, c, ld, C, T, tdot, erow, escale, wd);
            else if (mode == ORACLE_EXPLICIT_F128) rc = run_energy<Quad>(m, c, ld, C, T, tdot, erow, escale, wq);
            else {
                rc = run_energy<double>(m, c, ld, C, T, tdot, (double *)0, (double *)0, wd);
                if (!rc && erow && mode == ORACLE_JAC_DUAL) {
                    wdu.C.resize(N);
                    for (int k = 0; k < N; ++k) { wdu.C[k] = Dual(C[(size_t)k * ld + c]); wdu.C[k].d.assign(NC, 0.0); wdu.C[k].d[k] = 1.0; }
                    Dual Td(T[c]); Td.d.assign(NC, 0.0); Td.d[N] = 1.0;
                    Dual out;
                    rc = eval_tdot(m, wdu.C.data(), Td, wdu.rt, wdu.cl, wdu.wo, out);
                    if (!rc) for (int k = 0; k < NC; ++k) erow[(size_t)k * ld + c] = dg(out, k);
                } else if (!rc && erow) {
                    const double h = 1e-30;
                    wc.C.resize(N);
                    for (int k = 0; k < NC && !rc; ++k) {
                        for (int s = 0; s < N; ++s) wc.C[s] = Cplx(C[(size_t)s * ld + c], s == k ? h : 0.0);
                        Cplx Tc(T[c], k == N ? h : 0.0), out;
                        rc = eval_tdot(m, wc.C.data(), Tc, wc.rt, wc.cl, wc.wo, out);
                        if (!rc) erow[(size_t)k * ld + c] = out.imag() / h;
                    }
                }
            }
            if (rc) {
#pragma omp atomic write
                err = rc;
            }
        }
    }
    return err;
}

extern "C" int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

extern "C" int oracle_eval(const oracle_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T,
                           double *wdot, double *cqss, double *Sc, double *jac, double *jscale, int mode, int nthreads) {
    if (!m || !C || !T || ncells < 0 || ld < ncells || mode < 0 || mode > 5) return -1;
    const int N = m->n_nqss, NC = N + 1;
    if (nthreads <= 0) nthreads = oracle_max_threads();
    int err = 0;
#pragma omp parallel num_threads(nthreads)
    {
        Work<double> wd; Work<Quad> wq; Work<Dual> wdu; Work<Cplx> wc;
#pragma omp for schedule(dynamic, 8)
        for (int64_t c = 0; c < ncells; ++c) {
            int rc = 0;
            if (mode == ORACLE_EXPLICIT_F64 || mode == ORACLE_JAC_CONST_QSS || mode == ORACLE_JAC_ZERO_QSS) {
                rc = run_explicit<double>(m, c, ld, C, T, wdot, cqss, Sc, jac, jscale, mode != ORACLE_EXPLICIT_F64, wd, mode == ORACLE_JAC_ZERO_QSS);
            } else if (mode == ORACLE_EXPLICIT_F128) {
                rc = run_explicit<Quad>(m, c, ld, C, T, wdot, cqss, Sc, jac, jscale, false, wq);
            } else {
                // wdot / cqss / S from the plain double routine; Jacobian by differentiating eval_wdot mechanically
                rc = run_explicit<double>(m, c, ld, C, T, wdot, cqss, Sc, (double *)0, (double *)0, false, wd);
                if (!rc && jac && mode == ORACLE_JAC_DUAL) {
                    wdu.C.resize(N);
                    for (int k = 0; k < N; ++k) { wdu.C[k] = Dual(C[(size_t)k * ld + c]); wdu.C[k].d.assign(NC, 0.0); wdu.C[k].d[k] = 1.0; }
                    Dual Td(T[c]); Td.d.assign(NC, 0.0); Td.d[N] = 1.0;
                    rc = eval_wdot(m, wdu.C.data(), Td, wdu.rt, wdu.cl, wdu.wo);
                    if (!rc) for (int i = 0; i < N; ++i) for (int k = 0; k < NC; ++k)
                        jac[((size_t)i * NC + k) * ld + c] = dg(wdu.wo.wdot[i], k);
                } else if (!rc && jac && mode == ORACLE_JAC_CSTEP) {
                    const double h = 1e-30;
                    wc.C.resize(N);
                    for (int k = 0; k < NC && !rc; ++k) {
                        for (int s = 0; s < N; ++s) wc.C[s] = Cplx(C[(size_t)s * ld + c], s == k ? h : 0.0);
                        Cplx Tc(T[c], k == N ? h : 0.0);
                        rc = eval_wdot(m, wc.C.data(), Tc, wc.rt, wc.cl, wc.wo);
                        if (!rc) for (int i = 0; i < N; ++i) jac[((size_t)i * NC + k) * ld + c] = wc.wo.wdot[i].imag() / h;
                    }
                }
            }
            if (rc) {
#pragma omp atomic write
                err = rc;
            }
        }
    }
    return err;
}

extern "C" int oracle_rate_constants(const oracle_mech_t *m, const double *C, double T, double *kf, double *kb) {
    if (!m || !C || !kf || !kb) return -1;
    Rates<double> rt;
    eval_rates<double>(m, C, T, rt);
    for (int j = 0; j < m->n_reac; ++j) { kf[j] = rt.kf[j]; kb[j] = rt.kb[j]; }
    return 0;
}

extern "C" int oracle_closure_check(const oracle_mech_t *m, const double *C, double T, double *y, double *res, double *res_scale) {
    if (!m || !C || !y || !res || !res_scale) return -1;
    const int Nq = m->n_qss;
    Rates<double> rt; Closure<double> cl; WdotOut<double> wo;
    if (eval_wdot<double>(m, C, T, rt, cl, wo)) return -1;
    for (int q = 0; q < Nq; ++q) { y[q] = cl.y[q]; res[q] = 0.0; res_scale[q] = 0.0; }
    // net production rate of every QSS species from the definition (Eq. 4): must vanish
    for (int j = 0; j < m->n_reac; ++j)
        for (int dir = 0; dir < 2; ++dir) {
            if (!(m->dir_mask[j] & (1 << dir))) continue;
            const Side re = dir == 0 ? reactants(m, j) : products(m, j);
            const Side pr = dir == 0 ? products(m, j) : reactants(m, j);
            const int qn = qss_of(m, re);
            double r = kappa_of<double>(m, re, dir == 0 ? rt.kf[j] : rt.kb[j], C);
            if (qn >= 0) r *= cl.y[qn];
            for (int i = 0; i < pr.n; ++i) if (pr.sp[i] >= m->n_nqss) { res[pr.sp[i] - m->n_nqss] += pr.nu[i] * r; res_scale[pr.sp[i] - m->n_nqss] += pr.nu[i] * r; }
            for (int i = 0; i < re.n; ++i) if (re.sp[i] >= m->n_nqss) { res[re.sp[i] - m->n_nqss] -= re.nu[i] * r; res_scale[re.sp[i] - m->n_nqss] += re.nu[i] * r; }
        }
    return 0;
}
