// Kernel variant 3 for sm_100a: per-cell QSS chemistry -- rate constants -> QSS closure -> wdot -> analytical Jacobian with
// the chain rule through the closure (Eq. 2-4, 6, 7, 9).  This source is compiled ONLY at run time (NVRTC, by
// qss_jit.cpp) together with the header `qss_gen3.h` that qss_gen3.cpp generates for one mechanism: every size, row and
// offset below (G_*, R_*, S_*) is a compile-time constant of that mechanism.
//
// One persistent block of G_NW warps per SM; a slab = 32 consecutive cells; per-cell state in shared memory as rows of 33
// doubles (pitch G_PITCH = 264 bytes), free of bank conflicts both for "lane = cell" (one row per warp access) and for
// "lane = item" (32 consecutive rows, one cell).  Phases (block barrier between them):
//   P0  inputs -> V rows; T, ln T, 1/T, sum C                                            lane = cell
//   P2  rate constants k_f, k_b, d ln k/dM, d ln k/dT, d ln Kc/dT                        lane = REACTION (tasks)
//   P2c kappa_d = k_d prod C in place; k_d -> scratch slab                               lane = cell
//   P3  closure slots = signed sums of kappa_d (generated)                               lane = cell
//   P4  closure solve, group by group in DAG order (generated, matrices in registers)    lane = cell
//   P5  Q_j, dQ_j/dT, dQ_j/dM                                                            lane = REACTION (tasks)
//   P6  species sums: wdot, T-column vector, third-body vector                           lane = cell
//   P8  Jacobian columns: [W_x; G_x][:, k] in registers, dy/dx solve, W_y dy/dx (generated)   lane = cell, warp = column
#include "qss_stdint.h"
__device__ __forceinline__ double lds(unsigned a);
#define QSS_EXP_TAB_LOAD(tab, j) lds((tab) + (unsigned)(j) * 8u)      // the table of qss_exp_tab stands in shared memory (tab: its shared-window address)
#include "qss_math.h"
#include "qss_v3.h"

extern __shared__ double qss_smem[];

__device__ __forceinline__ double lds(unsigned a) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
template <int O> __device__ __forceinline__ double lS(unsigned b) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(b), "n"(O) : "memory");
    return v;
}
template <int O> __device__ __forceinline__ double2 lS2(unsigned b) {          // 16-byte read of a lane's pair
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(v.x), "=d"(v.y) : "r"(b), "n"(O) : "memory");
    return v;
}
template <int O> __device__ __forceinline__ void sS(unsigned b, double v) { asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(b), "n"(O), "d"(v) : "memory"); }
template <int O> __device__ __forceinline__ double lG(const double *b) {
    double v;
    asm volatile("ld.global.f64 %0, [%1+%2];" : "=d"(v) : "l"(b), "n"(O) : "memory");
    return v;
}
__device__ __forceinline__ double ldg_pin(const double *q) {
    double v;
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(v) : "l"(q) : "memory");
    return v;
}
__device__ __forceinline__ double ldg_nc(const double *q) {          // read-only parameter, pinned where it is written (prefetch)
    double v;
    asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(q));
    return v;
}
__device__ __forceinline__ int ldg_nc(const int32_t *q) {
    int v;
    asm volatile("ld.global.nc.s32 %0, [%1];" : "=r"(v) : "l"(q));
    return v;
}

// pinned arithmetic (volatile: keeps its place among the pinned loads, so that loads issued ahead stay ahead)
__device__ __forceinline__ void vfma(double &c, double a, double b) { asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(c) : "d"(a), "d"(b)); }
__device__ __forceinline__ void vfnma(double &c, double a, double b) { asm volatile("{\n\t.reg .f64 n;\n\tneg.f64 n, %1;\n\tfma.rn.f64 %0, n, %2, %0;\n\t}" : "+d"(c) : "d"(a), "d"(b)); }
__device__ __forceinline__ double vmul(double a, double b) { double r; asm volatile("mul.f64 %0, %1, %2;" : "=d"(r) : "d"(a), "d"(b)); return r; }
__device__ __forceinline__ double vfms(double a, double b, double c) {      // a b - c
    double r;
    asm volatile("{\n\t.reg .f64 n;\n\tneg.f64 n, %3;\n\tfma.rn.f64 %0, %1, %2, n;\n\t}" : "=d"(r) : "d"(a), "d"(b), "d"(c));
    return r;
}

#include "qss_gen3.h"

#ifndef QSS3_JAC
#define QSS3_JAC 1
#endif
// phase timing (only in images built with -DQSS3_TIMING=1, i.e. when QSS_TIMING is set at qss_mech_create): thread 0 of
// block 0 accumulates the cycles between the phase boundaries
#if QSS3_TIMING
#define QSS_TICK(ph) do { if (p.timing && blockIdx.x == 0 && threadIdx.x == 0) { const long long t_ = clock64(); p.timing[ph] += t_ - tick_; tick_ = t_; } } while (0)
#else
#define QSS_TICK(ph) do { } while (0)
#endif

#ifndef QSS3_X
#define QSS3_X 66                // bit 1: Estrin form of qss_exp where it is still used; bit 6: table form of the exponential in the rate phases
#endif
#if QSS3_X & 2
#define qss_exp qss_exp_e        // (its constants as operands from the constant bank instead of literals: measured, no gain)
#endif
constexpr double kLn10 = 2.302585092994045684017991454684;
constexpr double kInvLn10 = 0.434294481903251827651128918916605;

// interpreter tables (a few KB: task lists, kappa pass, species sums), staged once per block behind the per-cell rows
__device__ __forceinline__ int tab(const unsigned sm0, const int i) {
    int v;
    asm volatile("ld.shared.s32 %0, [%1];" : "=r"(v) : "r"(sm0 + R_TAB * G_PITCH + i * 4) : "memory");
    return v;
}

__device__ __forceinline__ int4 tab4(const unsigned sm0, const int i) {          // i: a multiple of 4
    int4 v;
    asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(sm0 + R_TAB * G_PITCH + i * 4) : "memory");
    return v;
}

// four terms of a species list: two words of two 16-bit row numbers -> byte offsets (x: a multiple of 4 terms)
__device__ __forceinline__ int4 tab_rows4(const unsigned sm0, const int x) {
    int a, b;
    asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(a), "=r"(b) : "r"(sm0 + R_TAB * G_PITCH + (T_SS + (x >> 1)) * 4) : "memory");
    return make_int4((a & 0xffff) * G_PITCH, (int)((unsigned)a >> 16) * G_PITCH, (b & 0xffff) * G_PITCH, (int)((unsigned)b >> 16) * G_PITCH);
}

// Per-lane parameters of one reaction (lane = reaction): what every reaction type needs.  Loaded with pinned read-only
// loads so that the first task of a slab can be fetched before the input phase (the L2 latency hides behind it).
struct RateCommon {
    double lnA, beta, EaR, tmid, elo[7], ehi[7];
    int flags, kap, tb;
#if G_HAS_CORR
    double tmax;                 // species with their own NASA-7 mid temperatures: [tmid, tmax) has one coefficient set per interval
    int ncorr;
    const double *corr;          // p.dP + QSS3_D_CORR rows of this lane's slot
#endif
};
__device__ __forceinline__ void qss3_load_common(RateCommon &r, const QssV3 &p, const int slot) {
    const double *dP = p.dP + slot;
    const int32_t *iP = p.iP + slot;
    r.flags = ldg_nc(iP + (size_t)QSS3_I_FLAGS * G_NSLOT); r.kap = ldg_nc(iP + (size_t)QSS3_I_KAP * G_NSLOT); r.tb = ldg_nc(iP + (size_t)QSS3_I_TB * G_NSLOT);
    r.lnA = ldg_nc(dP + (size_t)QSS3_D_LNA * G_NSLOT); r.beta = ldg_nc(dP + (size_t)QSS3_D_BETA * G_NSLOT);
    r.EaR = ldg_nc(dP + (size_t)QSS3_D_EAR * G_NSLOT); r.tmid = ldg_nc(dP + (size_t)QSS3_D_TMID * G_NSLOT);
#pragma unroll
    for (int i = 0; i < 7; ++i) { r.elo[i] = ldg_nc(dP + (size_t)(QSS3_D_ELO + i) * G_NSLOT); r.ehi[i] = ldg_nc(dP + (size_t)(QSS3_D_EHI + i) * G_NSLOT); }
#if G_HAS_CORR
    r.tmax = ldg_nc(dP + (size_t)QSS3_D_TMAX * G_NSLOT); r.ncorr = ldg_nc(iP + (size_t)QSS3_I_NCORR * G_NSLOT);
    r.corr = dP + (size_t)QSS3_D_CORR * G_NSLOT;
#endif
}
struct RateTyped {
    double lnA0, beta0, E0R, alpha, i3, i1, T2s, effv[QSS3_MAX_EFF];
    int effs[QSS3_MAX_EFF];
};

// Rate constants of one reaction for ONE cell.  smc = shared-window address of cell c in row 0.
//   dlnk = d ln k/dT at fixed M, dlnKc = d ln Kc/dT, dlm = d ln k/dM
#if QSS3_X & 64
#define QEXP(x) qss_exp_tab((x), smx)                                    // table form: 12 instead of 22 fp64 operations (qss_math.h)
#define QEXP_SAT(x) qss_exp_tab(qss3_clamp_exp_arg(x), smx)
#else
#define QEXP(x) qss_exp(x)
#define QEXP_SAT(x) qss_exp_sat(x)
#endif
__device__ __forceinline__ double qss3_clamp_exp_arg(double x) { return x < -746.0 ? -746.0 : (x > 710.0 ? 710.0 : x); }      // as qss_exp_sat: NaN stays NaN
template <int TYPE>
__device__ __forceinline__ void qss3_rate_cell(const RateCommon &r, const RateTyped &y, const double (&flo)[3], const double (&fhi)[3], const unsigned smc,
                                               const unsigned smx, double &kf, double &kb, double &dlm, double &dlnk, double &dlnKc) {
    const double T = lds(smc + R_T * G_PITCH), lnT = lds(smc + R_LNT * G_PITCH), invT = lds(smc + R_INVT * G_PITCH);
    const double lnkinf = fma(-r.EaR, invT, fma(r.beta, lnT, r.lnA));
    const bool lo = T < r.tmid;                                  // NASA-7 range (reading G9: T < Tmid low, else high)
#if G_HAS_CORR
    double e0 = lo ? r.elo[0] : r.ehi[0], e1 = lo ? r.elo[1] : r.ehi[1], e2 = lo ? r.elo[2] : r.ehi[2], e3 = lo ? r.elo[3] : r.ehi[3];
    double e4 = lo ? r.elo[4] : r.ehi[4], e5 = lo ? r.elo[5] : r.ehi[5], e6 = lo ? r.elo[6] : r.ehi[6];
    const bool between = !lo && T < r.tmax;                      // some species of the reaction are in their high range, some are not
    if (between) {                                               // (a band of a few hundred K; the lanes of the other reactions wait)
        int iv = 0;                                              // inner breakpoints at or below T: all loads independent
#pragma unroll
        for (int i = 0; i < QSS3_MAX_CORR - 2; ++i) if (i < r.ncorr) iv += T < __ldg(r.corr + (size_t)i * G_NSLOT) ? 0 : 1;
        const double *cp = r.corr + (size_t)(8 + 7 * iv) * G_NSLOT;
        e0 = __ldg(cp); e1 = __ldg(cp + (size_t)1 * G_NSLOT); e2 = __ldg(cp + (size_t)2 * G_NSLOT); e3 = __ldg(cp + (size_t)3 * G_NSLOT);
        e4 = __ldg(cp + (size_t)4 * G_NSLOT); e5 = __ldg(cp + (size_t)5 * G_NSLOT); e6 = __ldg(cp + (size_t)6 * G_NSLOT);
    }
#else
    const double e0 = lo ? r.elo[0] : r.ehi[0], e1 = lo ? r.elo[1] : r.ehi[1], e2 = lo ? r.elo[2] : r.ehi[2], e3 = lo ? r.elo[3] : r.ehi[3];
    const double e4 = lo ? r.elo[4] : r.ehi[4], e5 = lo ? r.elo[5] : r.ehi[5], e6 = lo ? r.elo[6] : r.ehi[6];
#endif
    const double lniKc = fma(e6, invT, fma(e1, lnT, fma(T, fma(T, fma(T, fma(T, e5, e4), e3), e2), e0)));     // -ln Kc
    double k = QEXP(lnkinf);
    const double iKc = QEXP(lniKc);
#if QSS3_JAC
    // T d ln Kc/dT = sum nu h/RT - dnu = e6/T - e1 - T (e2 + T (2 e3 + T (3 e4 + 4 e5 T)))   (e: coefficients of -ln Kc)
#if G_HAS_CORR
    const double f3 = between ? 2.0 * e3 : lo ? flo[0] : fhi[0], f4 = between ? 3.0 * e4 : lo ? flo[1] : fhi[1], f5 = between ? 4.0 * e5 : lo ? flo[2] : fhi[2];
#else
    const double f3 = lo ? flo[0] : fhi[0], f4 = lo ? flo[1] : fhi[1], f5 = lo ? flo[2] : fhi[2];
#endif
    const double w = fma(T, fma(T, fma(T, f5, f4), f3), e2);
    dlnKc = (r.flags & 2) ? (fma(e6, invT, -e1) - T * w) * invT : 0.0;
    dlnk = (r.beta + r.EaR * invT) * invT;
#endif
    dlm = 0.0;
    if (TYPE >= 1) {
        double Mc = lds(smc + R_CT * G_PITCH);                   // M = sum_k alpha_k C_k, transported species only (G7)
        const int ne = (r.flags >> 8) & 15;
#pragma unroll
        for (int e = 0; e < QSS3_MAX_EFF; ++e) if (e < ne) Mc = fma(y.effv[e], lds(smc + y.effs[e]), Mc);
        if (TYPE == 1) {
            k *= Mc;
            dlm = qss_rcp(Mc);
        } else {                                                 // Troe fall-off
            const double dlnkinf = (r.beta + r.EaR * invT) * invT;
            const double lnk0 = fma(-y.E0R, invT, fma(y.beta0, lnT, y.lnA0));
            const double dlnk0 = (y.beta0 + y.E0R * invT) * invT;
            const double Pr = QEXP(lnk0 - lnkinf) * Mc;
            const double al = y.alpha;
            const double x3 = QEXP_SAT(-T * y.i3), x1 = QEXP_SAT(-T * y.i1), x2 = QEXP_SAT(-y.T2s * invT);
            const double Fc = (1.0 - al) * x3 + al * x1 + x2;
            const double L = log(Pr) * kInvLn10, Lc = log(Fc) * kInvLn10;
            const double cc = -0.4 - 0.67 * Lc, n = 0.75 - 1.27 * Lc;
            const double num = L + cc, den = n - 0.14 * num;
            const double iden = qss_rcp(den);
            const double f1 = num * iden;
            const double ione_f = qss_rcp(1.0 + f1 * f1);
            const double F = QEXP(kLn10 * Lc * ione_f);
            const double i1pr = qss_rcp(1.0 + Pr);
            k = k * (Pr * i1pr) * F;
            const double df1_dL = n * iden * iden;
            const double dlF_dL = -2.0 * Lc * f1 * df1_dL * ione_f * ione_f;
            dlm = (i1pr + dlF_dL) * qss_rcp(Mc);
            const double dFc = -(1.0 - al) * y.i3 * x3 - al * y.i1 * x1 + y.T2s * invT * invT * x2;
            const double df1_dLc = (-0.67 * den - num * (-1.27 + 0.14 * 0.67)) * iden * iden;
            const double dlF_dLc = ione_f - 2.0 * Lc * f1 * df1_dLc * ione_f * ione_f;
            const double delta = dlnk0 - dlnkinf;
            dlnk = dlnkinf + delta * i1pr + dlF_dL * delta + dlF_dLc * dFc * qss_rcp(Fc);
        }
    }
    // reverse rate from the equilibrium constant; a disabled direction contributes nothing (G10)
    kf = (r.flags & 1) ? k : 0.0;
    kb = (r.flags & 2) ? k * iKc : 0.0;
}

// One rate task: the 32 reactions of slots slot0 .. slot0+31 (lane = reaction) for the cells c0 .. c1-1 of the slab.
// k_f and k_b go to the reaction's two rows (32 consecutive rows per task: no bank conflict), d ln k/dM to its DLM row;
// d ln k/dT and d ln Kc/dT are consumed by the net-rate tasks with the same lanes and therefore stored [cell][slot].
template <int TYPE>
__device__ __forceinline__ void qss3_rate_task(const RateCommon &r, const int slot0, const int c0, const int c1, const unsigned sm0, double *scb, const QssV3 &p) {
    const int slot = slot0 + (threadIdx.x & 31);
    RateTyped y;
    if (TYPE >= 1) {
#pragma unroll
        for (int e = 0; e < QSS3_MAX_EFF; ++e) { y.effv[e] = ldg_nc(p.dP + (size_t)(QSS3_D_EFFV + e) * G_NSLOT + slot); y.effs[e] = ldg_nc(p.iP + (size_t)(QSS3_I_EFFS + e) * G_NSLOT + slot); }
    }
    if (TYPE == 2) {
        y.lnA0 = ldg_nc(p.dP + (size_t)QSS3_D_LNA0 * G_NSLOT + slot); y.beta0 = ldg_nc(p.dP + (size_t)QSS3_D_BETA0 * G_NSLOT + slot);
        y.E0R = ldg_nc(p.dP + (size_t)QSS3_D_E0R * G_NSLOT + slot); y.alpha = ldg_nc(p.dP + (size_t)QSS3_D_ALPHA * G_NSLOT + slot);
        y.i3 = ldg_nc(p.dP + (size_t)QSS3_D_I3 * G_NSLOT + slot); y.i1 = ldg_nc(p.dP + (size_t)QSS3_D_I1 * G_NSLOT + slot);
        y.T2s = ldg_nc(p.dP + (size_t)QSS3_D_T2S * G_NSLOT + slot);
    }
    const double flo[3] = {2.0 * r.elo[3], 3.0 * r.elo[4], 4.0 * r.elo[5]}, fhi[3] = {2.0 * r.ehi[3], 3.0 * r.ehi[4], 4.0 * r.ehi[5]};
    const bool valid = (r.flags >> 4) & 1;
    const unsigned kap = sm0 + r.kap;
    constexpr int STEP = (TYPE == 2 || !(QSS3_X & 1)) ? 1 : 2;     // two cells per step: four independent exponential chains
#pragma unroll 1
    for (int c = c0; c < c1; c += STEP) {
        double kf[STEP], kb[STEP], dm[STEP], dk[STEP], dz[STEP];
#pragma unroll
        for (int u = 0; u < STEP; ++u) qss3_rate_cell<TYPE>(r, y, flo, fhi, sm0 + (c + u) * 8, sm0 + R_TAB * G_PITCH + T_EXP * 4, kf[u], kb[u], dm[u], dk[u], dz[u]);
        if (valid) {
#pragma unroll
            for (int u = 0; u < STEP; ++u) {
                sts(kap + (c + u) * 8, kf[u]);
                sts(kap + G_MS * G_PITCH + (c + u) * 8, kb[u]);
#if QSS3_JAC
                if (TYPE >= 1) sts(sm0 + (R_DLM + r.tb) * G_PITCH + (c + u) * 8, dm[u]);
                double *dt = scb + (size_t)S_DT * 32 + (size_t)(c + u) * (2 * G_NSLOT) + slot;
                dt[0] = dk[u]; dt[G_NSLOT] = dz[u];
#endif
            }
        }
    }
}

// One net-rate task (after the closure): Q_j, dQ_j/dT at fixed y and M, dQ_j/dM for 32 reactions (lane = reaction) and the
// cells c0 .. c1-1 (a multiple of 4), four cells per step, all loads of a step first.
struct NetParams { int flags, kap, qf, qb, tb; };
__device__ __forceinline__ void qss3_load_net(NetParams &n, const QssV3 &p, const int slot) {
    const int32_t *iP = p.iP + slot;
    n.flags = ldg_nc(iP + (size_t)QSS3_I_FLAGS * G_NSLOT); n.kap = ldg_nc(iP + (size_t)QSS3_I_KAP * G_NSLOT);
    n.qf = ldg_nc(iP + (size_t)QSS3_I_QF * G_NSLOT); n.qb = ldg_nc(iP + (size_t)QSS3_I_QB * G_NSLOT); n.tb = ldg_nc(iP + (size_t)QSS3_I_TB * G_NSLOT);
}
__device__ __forceinline__ void qss3_net_task(const NetParams &n, const int slot0, const int c0, const int c1, const unsigned sm0, const double *scb) {
    const int slot = slot0 + (threadIdx.x & 31);
    const unsigned kap = sm0 + n.kap, qf = sm0 + n.qf, qb = sm0 + n.qb;
    const bool valid = (n.flags >> 4) & 1;
#if QSS3_JAC
    // d ln k/dT and d ln Kc/dT are L2 reads: those of step i + 1 are in flight while step i is computed
    double dkn[4], dzn[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
        const double *dt = scb + (size_t)S_DT * 32 + (size_t)(c0 + u) * (2 * G_NSLOT) + slot;
        dkn[u] = ldg_pin(dt); dzn[u] = ldg_pin(dt + G_NSLOT);
    }
#endif
#pragma unroll 1
    for (int cb = c0; cb < c1; cb += 4) {
        double kf[4], kb[4], yf[4], yb[4];
#if QSS3_JAC
        double dk[4], dz[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) { dk[u] = dkn[u]; dz[u] = dzn[u]; }
        const int cn = cb + 4 < c1 ? cb + 4 : cb;
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const double *dt = scb + (size_t)S_DT * 32 + (size_t)(cn + u) * (2 * G_NSLOT) + slot;
            dkn[u] = ldg_pin(dt); dzn[u] = ldg_pin(dt + G_NSLOT);
        }
#endif
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int c = cb + u;
            kf[u] = lds(kap + c * 8); kb[u] = lds(kap + G_MS * G_PITCH + c * 8);
            yf[u] = lds(qf + c * 8); yb[u] = lds(qb + c * 8);
        }
        if (valid) {
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int c = cb + u;
                const double rf = kf[u] * yf[u], rb = kb[u] * yb[u];
                const double Q = rf - rb;
                sts(kap + c * 8, Q);
#if QSS3_JAC
                sts(kap + G_MS * G_PITCH + c * 8, fma(Q, dk[u], rb * dz[u]));
                if (n.tb >= 0) { const unsigned a = sm0 + (R_DLM + n.tb) * G_PITCH + c * 8; sts(a, lds(a) * Q); }
#endif
            }
        }
    }
}

// Signed sum over a species' term lists (table words = byte offsets of rows; [xa, xb) added, [xb, xc) subtracted, both padded to
// multiples of four with the row that stays zero), four terms per step; with TWO also the same sum over the rows G_MS further.
// (A hand-pipelined version -- table words two steps and values one step ahead -- measured slower: 14.06 vs 13.72 ms.)
template <bool TWO>
__device__ __forceinline__ void qss3_sum_lists(const unsigned sm0, const unsigned sml, const int xa, const int xb, const int xc, double &s1, double &s2) {
    double p1 = 0.0, m1 = 0.0, p2 = 0.0, m2 = 0.0;
#pragma unroll 1
    for (int x = xa; x < xc; x += 4) {
        const int4 o = tab_rows4(sm0, x);
        const double qs = (lds(sml + o.x) + lds(sml + o.y)) + (lds(sml + o.z) + lds(sml + o.w));
        if (x < xb) p1 += qs; else m1 += qs;
        if (TWO) {
            const double ts = (lds(sml + o.x + G_MS * G_PITCH) + lds(sml + o.y + G_MS * G_PITCH)) + (lds(sml + o.z + G_MS * G_PITCH) + lds(sml + o.w + G_MS * G_PITCH));
            if (x < xb) p2 += ts; else m2 += ts;
        }
    }
    s1 = p1 - m1; s2 = p2 - m2;
}

extern "C" __global__ void __launch_bounds__(G_NW * 32, 1)
#if QSS3_JAC
qss_v3_jac(const __grid_constant__ QssV3 p) {
#else
qss_v3_wdot(const __grid_constant__ QssV3 p) {
#endif
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int64_t ld = p.ld;
    const int64_t nslab = (p.ncells + 31) / 32;
    double *scb = p.scratch + (size_t)blockIdx.x * p.scratch_stride;     // this block's scratch slab
    double *sc = scb + lane;
    const unsigned sm0 = (unsigned)__cvta_generic_to_shared(qss_smem);
    const unsigned sml = sm0 + lane * 8;                         // this lane's (= cell's) column of the rows

    // interpreter tables -> shared memory, once per block (the block is persistent over slabs)
    for (int i = threadIdx.x; i < G_NTAB; i += G_NW * 32)
        asm volatile("st.shared.s32 [%0], %1;" ::"r"(sm0 + R_TAB * G_PITCH + i * 4), "r"(ldg_nc(p.iP + (size_t)QSS3_NIP * G_NSLOT + i)) : "memory");
    __syncthreads();
    const int rt0 = tab(sm0, T_RT_PTR + warp), rt1 = tab(sm0, T_RT_PTR + warp + 1);
    const int nt0 = tab(sm0, T_NT_PTR + warp), nt1 = tab(sm0, T_NT_PTR + warp + 1);

#if QSS3_TIMING
    long long tick_ = clock64();
#endif
    for (int64_t slab = blockIdx.x; slab < nslab; slab += gridDim.x) {
        const int64_t cell = slab * 32 + lane;
        const bool active = cell < p.ncells;
        const int64_t cc = active ? cell : p.ncells - 1;          // idle lanes of a ragged tail shadow the last cell
        // the parameters of the warp's first rate task are fetched now (independent of the cells; L2 latency)
        RateCommon rc;
#if QSS3_X & 4
        if (rt0 < rt1) qss3_load_common(rc, p, tab(sm0, T_RT + 4 * rt0 + 1) + lane);
#endif
        // ---- P0: inputs.  Every slab but the block's first was fetched into the staging rows during the previous slab's
        //      column sweep (cp.async below); every warp waits for and moves the rows it fetched itself.
#if QSS3_JAC
        if (slab != blockIdx.x) {
            asm volatile("cp.async.wait_all;" ::: "memory");
            for (int s = warp; s < G_N; s += G_NW) sts(sml + (R_V + s) * G_PITCH, lds(sml + (R_STAGE + s) * G_PITCH));
            if (warp == 0) sts(sml + R_T * G_PITCH, lds(sml + (R_STAGE + G_N) * G_PITCH));
        } else
#endif
        {
            for (int s = warp; s < G_N; s += G_NW) sts(sml + (R_V + s) * G_PITCH, p.C[(size_t)s * ld + cc]);
            if (warp == 0) sts(sml + R_T * G_PITCH, p.T[cc]);
        }
        if (warp == 0) {
            const double T = lds(sml + R_T * G_PITCH);
            sts(sml + R_LNT * G_PITCH, log(T));
            sts(sml + R_INVT * G_PITCH, 1.0 / T);
            sts(sml + R_ONE * G_PITCH, 1.0);
        }
        __syncthreads();
        // (the two rows that pad the species-sum lists are zeroed every slab, after the staged inputs have been moved: in a small
        //  mechanism the kappa_d pairs and the staging rows of the previous sweep cover them)
        if (warp == 0) { sts(sml + (R_KAP + G_M) * G_PITCH, 0.0); sts(sml + (R_KAP + G_MS + G_M) * G_PITCH, 0.0); }
        if (warp == G_NW - 1) {
            double ct = 0.0;
#pragma unroll 5
            for (int k = 0; k < G_N; ++k) ct += lds(sml + (R_V + k) * G_PITCH);
            sts(sml + R_CT * G_PITCH, ct);
        }
        __syncthreads();
        QSS_TICK(0);
#if QSS3_TIMING
        const long long tick_w = clock64();
#endif
        // ---- P2: rate constants (Eq. 2), lane = reaction
        for (int t = rt0; t < rt1; ++t) {
            const int type = tab(sm0, T_RT + 4 * t), slot0 = tab(sm0, T_RT + 4 * t + 1), c0 = tab(sm0, T_RT + 4 * t + 2), c1 = tab(sm0, T_RT + 4 * t + 3);
#if QSS3_X & 4
            const RateCommon cur = rc;
            if (t + 1 < rt1) qss3_load_common(rc, p, tab(sm0, T_RT + 4 * t + 5) + lane);      // the next task's parameters, under this one
#else
            qss3_load_common(rc, p, slot0 + lane);                // (128 registers per thread: no room for a second parameter set)
            const RateCommon &cur = rc;
#endif
            if (type == 0) qss3_rate_task<0>(cur, slot0, c0, c1, sm0, scb, p);
            else if (type == 1) qss3_rate_task<1>(cur, slot0, c0, c1, sm0, scb, p);
            else qss3_rate_task<2>(cur, slot0, c0, c1, sm0, scb, p);
        }
        QSS_TICK(1);
#if QSS3_TIMING
        if (p.timing && blockIdx.x == 0 && lane == 0) p.timing[16 + warp] += clock64() - tick_w;
#endif
        __syncthreads();
        QSS_TICK(2);
        // ---- P2c: kappa_d = k_d times the transported reactant molecules (Eq. 6), in place, four directions per step; k_d
        //      itself leaves for the scratch slab (the column records read it), kappa_d of the QSS-consuming directions too
        //      (their rows are reused for Q_j).  Table word: V rows of the three molecules (6 bits each) | (kq row + 1) << 18.
#if QSS3_X & 8
        qss_gen_kappa(warp, sml, sc);
#else
        for (int e = warp * 4; e < 2 * G_MS; e += G_NW * 4) {
            const int4 wa = tab4(sm0, T_KAP + e);
            const int w[4] = {wa.x, wa.y, wa.z, wa.w};
            double k[4], x0[4], x1[4], x2[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                k[u] = lds(sml + (R_KAP + min(e + u, 2 * G_MS - 1)) * G_PITCH);
                x0[u] = lds(sml + (w[u] & 63) * G_PITCH); x1[u] = lds(sml + ((w[u] >> 6) & 63) * G_PITCH); x2[u] = lds(sml + ((w[u] >> 12) & 63) * G_PITCH);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) if (e + u < 2 * G_MS) {
                const double kp = k[u] * x0[u] * x1[u] * x2[u];
                sts(sml + (R_KAP + e + u) * G_PITCH, kp);
#if QSS3_JAC
                sc[(size_t)(S_K + e + u) * 32] = k[u];
                if (w[u] >> 18) sc[(size_t)(S_KQ + (w[u] >> 18) - 1) * 32] = kp;
#endif
            }
        }
#endif
        __syncthreads();
        QSS_TICK(10);
        NetParams np;        // (the first net-rate task's parameters: fetched under the closure phases)
        if (nt0 < nt1) qss3_load_net(np, p, tab(sm0, T_NT + 4 * nt0) + lane);
        // ---- P3: closure slots (Eq. 6), P4: closure solve (block barrier after every level inside)
        qss_gen_gather(warp, sml);
        __syncthreads();
        QSS_TICK(3);
        qss_gen_closure(warp, sml);
#if QSS3_JAC
        if (p.mode == 2) {      // zero-QSS AJ: the QSS concentrations are nullified in every partial derivative
            for (int q = warp; q < G_NQ; q += G_NW) sts(sml + (R_Y + q) * G_PITCH, 0.0);
            __syncthreads();
        }
#endif
        QSS_TICK(4);
        // ---- P5: net rates of progress Q_j (Eq. 2), dQ_j/dT, dQ_j/dM; they replace kappa_f, kappa_b, d ln k/dM in place
        for (int t = nt0; t < nt1; ++t) {
            const NetParams cur = np;
            if (t + 1 < nt1) qss3_load_net(np, p, tab(sm0, T_NT + 4 * t + 4) + lane);
            qss3_net_task(cur, tab(sm0, T_NT + 4 * t), tab(sm0, T_NT + 4 * t + 1), tab(sm0, T_NT + 4 * t + 2), sm0, scb);
        }
        __syncthreads();
        QSS_TICK(5);
        // ---- P6: species sums: wdot (Eq. 3); for the Jacobian the T-column vector and the third-body vector.
        //      One table word per unit of |nu|: the sign bit of the word flips the sign bit of the value.
#if QSS3_JAC
        // (kappa_d of the QSS-consuming directions comes back from the scratch slab for the column sweep: the reads are issued
        //  here, the values are held in registers over the sums and stored once the Q_j rows are free)
        double kq[G_KQ_PER_WARP];
#pragma unroll
        for (int u = 0; u < G_KQ_PER_WARP; ++u) kq[u] = ldg_pin(sc + (size_t)(S_KQ + min(warp * G_KQ_PER_WARP + u, G_NKQ - 1)) * 32);
#endif
#if QSS3_X & 16
        qss_gen_sums(warp, sml, sc, p.wdot ? p.wdot + cell : nullptr, ld, active);
#else
        for (int u = tab(sm0, T_SSW_PTR + warp); u < tab(sm0, T_SSW_PTR + warp + 1); ++u) {
            const int s = tab(sm0, T_SSW + u);
            double w, et, tv, unused;
            qss3_sum_lists<QSS3_JAC != 0>(sm0, sml, tab(sm0, T_SS_PTR + 2 * s), tab(sm0, T_SS_PTR + 2 * s + 1), tab(sm0, T_SS_PTR + 2 * s + 2), w, et);
            if (s < G_N && p.wdot && active) p.wdot[(size_t)s * ld + cell] = w;
#if QSS3_JAC
            qss3_sum_lists<false>(sm0, sml, tab(sm0, T_ST_PTR + 2 * s), tab(sm0, T_ST_PTR + 2 * s + 1), tab(sm0, T_ST_PTR + 2 * s + 2), tv, unused);
            sts(sml + (R_TV + s) * G_PITCH, tv);
            sc[(size_t)(S_ET + s) * 32] = et;
#endif
        }
#endif
        if (p.cqss && active)
            for (int q = warp; q < G_NQ; q += G_NW) p.cqss[(size_t)q * ld + cell] = lds(sml + (R_Y + q) * G_PITCH);
#if QSS3_JAC
        __syncthreads();
        QSS_TICK(6);
        // ---- P8: kappa_d of the QSS-consuming directions -> the (now free) kappa region; then each warp takes its columns one
        //      after the other, everything in registers, no barrier between
#pragma unroll
        for (int u = 0; u < G_KQ_PER_WARP; ++u) {          // pair layout [pair][lane][2] (the columns read 16 bytes at a time)
            const int e = warp * G_KQ_PER_WARP + u;
            if (e < G_NKQ) sts(sm0 + KQ_BASE + (e >> 1) * 528 + lane * 16 + (e & 1) * 8, kq[u]);
        }
        __syncthreads();
        QSS_TICK(7);
        if (slab + gridDim.x < nslab) {      // inputs of the block's next slab -> staging rows behind kappa_d, under the sweep
            const int64_t cell2 = (slab + gridDim.x) * 32 + lane;
            const int64_t cc2 = cell2 < p.ncells ? cell2 : p.ncells - 1;
            for (int s = warp; s < G_N; s += G_NW)
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sml + (R_STAGE + s) * G_PITCH), "l"(p.C + (size_t)s * ld + cc2) : "memory");
            if (warp == 0) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sml + (R_STAGE + G_N) * G_PITCH), "l"(p.T + cc2) : "memory");
        }
#if G_NW > G_NWC
        // More warps than columns in flight (a column needs ~160 registers, the other phases run G_NW warps at 128): the extra
        // warp group hands its registers to the column warps for the sweep (setmaxnreg) and waits at the end-of-slab barrier.
        if (warp < G_NWC) {
            asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(G_REG_COL));
            for (int dd = 0; dd < QSS_GEN_DEPTH; ++dd) {
                const int k = qss_gen_cols[warp * QSS_GEN_DEPTH + dd];
                if (k >= 0) qss_gen_column(k, p.mode, sml, sm0 + lane * 16, sc, p.jac + (size_t)(unsigned)k * (size_t)ld + cell, (long long)(G_N + 1) * ld, active);
            }
            asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(G_REG_BASE));
            asm volatile("bar.arrive 1, %0;" ::"n"(G_NW * 32));
        } else {
            asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(G_REG_IDLE));
            asm volatile("bar.sync 1, %0;" ::"n"(G_NW * 32));            // until the column warps have released their registers
            asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(G_REG_BASE));
        }
#else
        for (int dd = 0; dd < QSS_GEN_DEPTH; ++dd) {
            const int k = qss_gen_cols[warp * QSS_GEN_DEPTH + dd];
#if QSS3_X & 32      // (timing experiment, WRONG results: every column of a warp runs the code of the warp's first column -> a third of the once-per-slab code)
            if (k >= 0) qss_gen_column(qss_gen_cols[warp * QSS_GEN_DEPTH], p.mode, sml, sm0 + lane * 16, sc, p.jac + (size_t)(unsigned)k * (size_t)ld + cell, (long long)(G_N + 1) * ld, active);
#else
            if (k >= 0) qss_gen_column(k, p.mode, sml, sm0 + lane * 16, sc, p.jac + (size_t)(unsigned)k * (size_t)ld + cell, (long long)(G_N + 1) * ld, active);
#endif
        }
#endif
        QSS_TICK(8);
#endif
        __syncthreads();      // shared memory and the scratch slab are reused by the next cell slab
        QSS_TICK(9);
    }
}
