// CUDA kernels (sm_100a) for per-cell QSS chemistry: rate constants -> QSS closure -> wdot -> analytical
// Jacobian with the chain rule through the closure (Eq. 2-4, 6, 7, 9).  Table-driven: the kernels
// interpret the tables built by qss_compile.cpp; nothing is generated per mechanism.
//
// Kernel "slab" (variant 0, general): a thread block owns a slab of 32 consecutive cells.  Lane l of every
// warp works on cell l of the slab, so every table read is warp-uniform and every per-cell array access
// ws[(offset + item) * 32 + lane] is a fully coalesced 256-byte transaction; the warps of the block split
// the ITEMS of each phase (species, reactions, closure entries, QSS groups, Jacobian columns) and meet at
// block barriers between phases.  Per-cell temporaries live in a per-block workspace slab that is reused
// for every slab the (persistent) block processes, so it stays resident in L2.
#include <cuda_runtime.h>
#include <stdint.h>

#include "qss_math.h"
#include "qss_tables.h"

namespace {

constexpr double kLn10 = 2.302585092994045684017991454684;
constexpr double kInvLn10 = 0.434294481903251827651128918916605;
constexpr double kRgas = 8.31446261815324;
constexpr double kPref = 101325.0;

__device__ __forceinline__ double ipow_d(double c, int nu) {   // integer power by multiplication
    double r = c;
    for (int i = 1; i < nu; ++i) r *= c;
    return r;
}

struct CellCtx {
    double T, lnT, invT, lnP0RT, Ctot;
    const double *Cg;     // &C[cell], stride ld between species
    int64_t ld;
    double *ws;           // workspace slab + lane
};

#define WS(off, i) cx.ws[(size_t)((off) + (i)) * 32]

// concentration of species s: transported from the input, QSS from the closure
__device__ __forceinline__ double conc(const QssTab &t, const CellCtx &cx, int s) {
    return s < t.N ? cx.Cg[(size_t)s * cx.ld] : WS(t.w_Y, s - t.N);
}

// steps 2: NASA-7 h/RT and g/RT of species s (reading G4, G9)
__device__ __forceinline__ void thermo(const QssTab &t, const CellCtx &cx, int s) {
    const double *th = t.D + t.d_thermo + s * QSS_TH_STRIDE;
    const double *a = th + 1 + (cx.T < th[0] ? 0 : 11);
    const double T = cx.T;
    const double h = a[0] + T * (a[1] + T * (a[2] + T * (a[3] + T * a[4]))) + a[5] * cx.invT;
    const double sR = a[0] * cx.lnT + T * (a[6] + T * (a[7] + T * (a[8] + T * a[9]))) + a[10];
    WS(t.w_H, s) = h;
    WS(t.w_G, s) = h - sR;
}

// step 3-4: rate constants of reaction j and the direction coefficients kappa_d
template <bool JAC>
__device__ __forceinline__ void rates(const QssTab &t, const CellCtx &cx, int j) {
    const double *rd = t.D + t.d_rate + j * QSS_RD_STRIDE;
    const int32_t *ri = t.I + t.i_reac + j * QSS_RI_STRIDE;
    const int type = ri[0], mask = ri[1], tb = ri[2];
    const double T = cx.T, invT = cx.invT;
    const double lnkinf = rd[0] + rd[1] * cx.lnT - rd[2] * invT;
    const double dlnkinf = (rd[1] + rd[2] * invT) * invT;
    double k = qss_exp(lnkinf), dlnk = dlnkinf, dlm = 0.0;
    if (type >= 1) {
        double Mc = cx.Ctot;                                   // M = sum_k alpha_k C_k, transported only (G7)
        const int e0 = t.I[t.i_eff_ptr + j], e1 = t.I[t.i_eff_ptr + j + 1];
        for (int e = e0; e < e1; ++e) Mc += t.D[t.d_effm1 + e] * cx.Cg[(size_t)t.I[t.i_eff_sp + e] * cx.ld];
        if (type == 1) {
            k *= Mc;
            dlm = 1.0 / Mc;
        } else {                                               // Troe fall-off
            const double lnk0 = rd[3] + rd[4] * cx.lnT - rd[5] * invT;
            const double dlnk0 = (rd[4] + rd[5] * invT) * invT;
            const double Pr = qss_exp(lnk0 - lnkinf) * Mc;
            const double al = rd[6], i3 = rd[7], i1 = rd[8], T2s = rd[9];
            const double e3 = qss_exp_sat(-T * i3), e1x = qss_exp_sat(-T * i1), e2 = qss_exp_sat(-T2s * invT);
            const double Fc = (1.0 - al) * e3 + al * e1x + e2;
            const double dFc = -(1.0 - al) * i3 * e3 - al * i1 * e1x + T2s * invT * invT * e2;
            const double L = log(Pr) * kInvLn10, Lc = log(Fc) * kInvLn10;
            const double c = -0.4 - 0.67 * Lc, n = 0.75 - 1.27 * Lc;
            const double num = L + c, den = n - 0.14 * num;
            const double iden = 1.0 / den;
            const double f1 = num * iden;
            const double one_f = 1.0 + f1 * f1, ione_f = 1.0 / one_f;
            const double F = qss_exp(kLn10 * Lc * ione_f);
            const double i1pr = 1.0 / (1.0 + Pr);
            k = k * (Pr * i1pr) * F;
            const double df1_dL = n * iden * iden;
            const double dlF_dL = -2.0 * Lc * f1 * df1_dL * ione_f * ione_f;
            dlm = (i1pr + dlF_dL) / Mc;
            if (JAC) {
                const double df1_dLc = (-0.67 * den - num * (-1.27 + 0.14 * 0.67)) * iden * iden;
                const double dlF_dLc = ione_f - 2.0 * Lc * f1 * df1_dLc * ione_f * ione_f;
                const double delta = dlnk0 - dlnkinf;
                dlnk = dlnkinf + delta * i1pr + dlF_dL * delta + dlF_dLc * dFc / Fc;
            }
        }
        if (JAC) WS(t.w_DLM, tb) = dlm;
    }
    double kf = (mask & 1) ? k : 0.0, kb = 0.0, dlnKc = 0.0;
    if (mask & 2) {                                            // reverse rate from the equilibrium constant (G10)
        double dG = 0.0, dH = 0.0;
        const int n0 = t.I[t.i_net_ptr + j], n1 = t.I[t.i_net_ptr + j + 1];
        for (int p = n0; p < n1; ++p) {
            const int s = t.I[t.i_net_sp + p];
            const double nu = (double)t.I[t.i_net_nu + p];
            dG += nu * WS(t.w_G, s);
            if (JAC) dH += nu * WS(t.w_H, s);
        }
        kb = k * qss_exp(dG - rd[10] * cx.lnP0RT);                 // k / Kc, ln Kc = -dG + dnu ln(P0/RT)
        dlnKc = (dH - rd[10]) * invT;
    }
    WS(t.w_K, 2 * j) = kf;
    WS(t.w_K, 2 * j + 1) = kb;
    if (JAC) { WS(t.w_DF, j) = dlnk; WS(t.w_DC, j) = dlnKc; }
    // kappa_d = k_d * product of TRANSPORTED reactant concentrations (the coefficient of the QSS reactant,
    // PAPER.md Eq. 6; or the whole rate when the direction consumes no QSS species)
#pragma unroll
    for (int dir = 0; dir < 2; ++dir) {
        double kap = dir == 0 ? kf : kb;
        const int s0 = t.I[t.i_side_ptr + 2 * j + dir], s1 = t.I[t.i_side_ptr + 2 * j + dir + 1];
        for (int p = s0; p < s1; ++p) {
            const int s = t.I[t.i_side_sp + p];
            if (s < t.N) kap *= ipow_d(cx.Cg[(size_t)s * cx.ld], t.I[t.i_side_nu + p]);
        }
        WS(t.w_KAP, 2 * j + dir) = kap;
    }
}

// Solve (diag D - P) x = rhs for one group with the stored elimination factors; rhs is addressed through
// `RHS(m)` and overwritten by the solution.  Subtraction-free for rhs >= 0.
#define QSS_GROUP_SOLVE(RHS)                                                                   \
    for (int k = sz - 1; k >= 1; --k) {                                                        \
        const double tk = RHS(k) * WS(base + sz * sz + 2 * sz, k);                             \
        for (int m = 0; m < k; ++m) RHS(m) += WS(base, m * sz + k) * tk;                       \
    }                                                                                          \
    for (int k = 0; k < sz; ++k) {                                                             \
        double acc = RHS(k);                                                                   \
        for (int jj = 0; jj < k; ++jj) acc += WS(base, k * sz + jj) * RHS(jj);                 \
        RHS(k) = acc * WS(base + sz * sz + 2 * sz, k);                                         \
    }

// step 5: one QSS group -- add the couplings to earlier groups, eliminate (Grassmann-Taksar-Heyman order,
// no subtraction anywhere), solve for y.  PAPER.md Eq. 6 (L150-157), L159-171, L475; reading G2, G8.
__device__ __forceinline__ void closure_group(const QssTab &t, const CellCtx &cx, int g) {
    const int32_t *gi = t.I + t.i_group + g * QSS_GI_STRIDE;
    const int sz = gi[0], moff = gi[1], base = t.w_CL + gi[2], x0 = gi[4], x1 = gi[5];
    const int oL = base + sz * sz, oP0 = oL + sz, oID = oP0 + sz;
    for (int x = x0; x < x1; ++x)
        WS(oP0, t.I[t.i_xp_m + x]) += WS(t.w_XP, x) * WS(t.w_Y, t.I[t.i_xp_n + x]);
    for (int k = sz - 1; k >= 1; --k) {
        double Dk = WS(oL, k);
        for (int m = 0; m < k; ++m) Dk += WS(base, m * sz + k);
        const double iD = 1.0 / Dk;
        WS(oID, k) = iD;
        const double lk = WS(oL, k);
        for (int jj = 0; jj < k; ++jj) {
            const double f = WS(base, k * sz + jj) * iD;
            WS(oL, jj) += f * lk;
            for (int m = 0; m < k; ++m)
                if (m != jj) WS(base, m * sz + jj) += WS(base, m * sz + k) * f;
        }
    }
    WS(oID, 0) = 1.0 / WS(oL, 0);
#define RHS_P0(m) WS(oP0, m)
    QSS_GROUP_SOLVE(RHS_P0)
#undef RHS_P0
    for (int m = 0; m < sz; ++m) WS(t.w_Y, t.I[t.i_gmember + moff + m]) = WS(oP0, m);
}

template <bool JAC>
__global__ void __launch_bounds__(1024) qss_slab_kernel(const QssTab t, const int64_t ncells, const int64_t ld,
                                                       const double *__restrict__ C, const double *__restrict__ Tin,
                                                       double *__restrict__ wdot, double *__restrict__ cqss,
                                                       double *__restrict__ jac, double *__restrict__ wsbase,
                                                       const int64_t ws_stride) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
    const int N = t.N, Nq = t.Nq, M = t.M, nsp = t.nsp;
    const int64_t nslab = (ncells + 31) / 32;
    CellCtx cx;
    cx.ld = ld;
    cx.ws = wsbase + (size_t)blockIdx.x * ws_stride + lane;
    for (int64_t slab = blockIdx.x; slab < nslab; slab += gridDim.x) {
        const int64_t cell = slab * 32 + lane;
        const bool active = cell < ncells;
        const int64_t cc = active ? cell : ncells - 1;        // idle lanes of a ragged tail shadow the last cell
        cx.Cg = C + cc;
        cx.T = Tin[cc];
        cx.lnT = log(cx.T);
        cx.invT = 1.0 / cx.T;
        cx.lnP0RT = log(kPref / (kRgas * cx.T));
        double ct = 0.0;
        for (int k = 0; k < N; ++k) ct += cx.Cg[(size_t)k * ld];
        cx.Ctot = ct;
        // ---- thermo
        for (int s = warp; s < nsp; s += nwarp) thermo(t, cx, s);
        __syncthreads();
        // ---- rate constants and direction coefficients
        for (int r = warp; r < M; r += nwarp) rates<JAC>(t, cx, t.I[t.i_rorder + r]);
        __syncthreads();
        // ---- closure assembly: every P / leak / p0 slot gathers the kappas feeding it (no atomics)
        for (int e = warp; e < t.n_centry; e += nwarp) {
            double acc = 0.0;
            for (int p = t.I[t.i_ce_ptr + e]; p < t.I[t.i_ce_ptr + e + 1]; ++p) acc += WS(t.w_KAP, t.I[t.i_ce_dir + p]);
            WS(t.w_CL, t.I[t.i_ce_dst + e]) = acc;
        }
        for (int e = warp; e < t.n_xp; e += nwarp) {
            double acc = 0.0;
            for (int p = t.I[t.i_xp_ptr + e]; p < t.I[t.i_xp_ptr + e + 1]; ++p) acc += WS(t.w_KAP, t.I[t.i_xp_dir + p]);
            WS(t.w_XP, e) = acc;
        }
        __syncthreads();
        // ---- closure solve, level by level of the condensed DAG
        for (int l = 0; l < t.n_levels; ++l) {
            const int g0 = t.I[t.i_level_ptr + l], g1 = t.I[t.i_level_ptr + l + 1];
            for (int g = g0 + warp; g < g1; g += nwarp) closure_group(t, cx, g);
            __syncthreads();
        }
        // ---- net rates of progress
        for (int j = warp; j < M; j += nwarp) {
            const int32_t *ri = t.I + t.i_reac + j * QSS_RI_STRIDE;
            double rf = WS(t.w_KAP, 2 * j), rb = WS(t.w_KAP, 2 * j + 1);
            if (ri[3] >= 0) rf *= WS(t.w_Y, ri[3]);
            if (ri[4] >= 0) rb *= WS(t.w_Y, ri[4]);
            const double Q = rf - rb;
            WS(t.w_Q, j) = Q;
            if (JAC) {
                WS(t.w_QT, j) = Q * WS(t.w_DF, j) + rb * WS(t.w_DC, j);    // dQ/dT at fixed y and M
                if (ri[2] >= 0) WS(t.w_QM, ri[2]) = Q * WS(t.w_DLM, ri[2]); // dQ/dM
            }
        }
        __syncthreads();
        // ---- species sums: wdot (Eq. 3), and for the Jacobian the T column and the third-body vector
        for (int s = warp; s < nsp; s += nwarp) {
            double w = 0.0, et = 0.0, tv = 0.0;
            for (int p = t.I[t.i_sp_ptr + s]; p < t.I[t.i_sp_ptr + s + 1]; ++p) {
                const int j = t.I[t.i_sp_reac + p];
                const double nu = (double)t.I[t.i_sp_nu + p];
                w += nu * WS(t.w_Q, j);
                if (JAC) {
                    et += nu * WS(t.w_QT, j);
                    const int tb = t.I[t.i_reac + j * QSS_RI_STRIDE + 2];
                    if (tb >= 0) tv += nu * WS(t.w_QM, tb);
                }
            }
            if (s < N && wdot && active) wdot[(size_t)s * ld + cell] = w;
            if (JAC) { WS(t.w_ET, s) = et; WS(t.w_TV, s) = tv; }
        }
        if (cqss && active)
            for (int q = warp; q < Nq; q += nwarp) cqss[(size_t)q * ld + cell] = WS(t.w_Y, q);
        if (JAC) {
            // ---- W_y[i][q] = d wdot_i / d y_q at fixed x: sums of kappas (Eq. 9 second parenthesis, L224)
            for (int e = warp; e < t.n_wy; e += nwarp) {
                double acc = 0.0;
                for (int p = t.I[t.i_wy_ptr + e]; p < t.I[t.i_wy_ptr + e + 1]; ++p)
                    acc += (double)t.I[t.i_wy_coef + p] * WS(t.w_KAP, t.I[t.i_wy_dir + p]);
                WS(t.w_WY, e) = acc;
            }
            __syncthreads();
            // ---- column sweep: one column of [W_x; G_x] -> solve for dy/dx_k -> J[:,k] = W_x[:,k] + W_y dy/dx_k
            const int oCOL = t.w_COL + warp * nsp;
            for (int k = warp; k <= N; k += nwarp) {
                if (k < N) {
                    for (int s = 0; s < nsp; ++s) WS(oCOL, s) = WS(t.w_TV, s);       // rank-1 third-body term
                    for (int p = t.I[t.i_col_ptr + k]; p < t.I[t.i_col_ptr + k + 1]; ++p) {
                        const int d = t.I[t.i_col_dir + p], pos = t.I[t.i_col_pos + p], j = d >> 1;
                        double part = WS(t.w_K, d);                                   // d r_d / d C_k: product of the others
                        const int s0 = t.I[t.i_side_ptr + d], s1 = t.I[t.i_side_ptr + d + 1];
                        for (int x = s0; x < s1; ++x) {
                            const int s = t.I[t.i_side_sp + x], nu = t.I[t.i_side_nu + x];
                            const double c = conc(t, cx, s);
                            if (x - s0 == pos) { part *= (double)nu; if (nu > 1) part *= ipow_d(c, nu - 1); }
                            else part *= ipow_d(c, nu);
                        }
                        if (d & 1) part = -part;
                        for (int x = t.I[t.i_net_ptr + j]; x < t.I[t.i_net_ptr + j + 1]; ++x)
                            WS(oCOL, t.I[t.i_net_sp + x]) += (double)t.I[t.i_net_nu + x] * part;
                    }
                    for (int p = t.I[t.i_effc_ptr + k]; p < t.I[t.i_effc_ptr + k + 1]; ++p) {   // (alpha_k - 1) dQ/dM
                        const int j = t.I[t.i_effc_reac + p];
                        const double v = t.D[t.d_effc + p] * WS(t.w_QM, t.I[t.i_reac + j * QSS_RI_STRIDE + 2]);
                        for (int x = t.I[t.i_net_ptr + j]; x < t.I[t.i_net_ptr + j + 1]; ++x)
                            WS(oCOL, t.I[t.i_net_sp + x]) += (double)t.I[t.i_net_nu + x] * v;
                    }
                } else {
                    for (int s = 0; s < nsp; ++s) WS(oCOL, s) = WS(t.w_ET, s);
                }
                // dy/dx_k: (diag D - P) ycol = G_x[:,k], group by group with the closure's factors
                for (int g = 0; g < t.n_groups; ++g) {
                    const int32_t *gi = t.I + t.i_group + g * QSS_GI_STRIDE;
                    const int sz = gi[0], moff = gi[1], base = t.w_CL + gi[2];
                    for (int x = gi[4]; x < gi[5]; ++x)
                        WS(oCOL, N + t.I[t.i_gmember + moff + t.I[t.i_xp_m + x]]) += WS(t.w_XP, x) * WS(oCOL, N + t.I[t.i_xp_n + x]);
#define RHS_COL(m) WS(oCOL, N + t.I[t.i_gmember + moff + (m)])
                    QSS_GROUP_SOLVE(RHS_COL)
#undef RHS_COL
                }
                for (int i = 0; i < N; ++i) {
                    double acc = WS(oCOL, i);
                    for (int p = t.I[t.i_wyrow_ptr + i]; p < t.I[t.i_wyrow_ptr + i + 1]; ++p)
                        acc += WS(t.w_WY, t.I[t.i_wyrow_e + p]) * WS(oCOL, N + t.I[t.i_wyrow_q + p]);
                    if (active) jac[((size_t)i * (N + 1) + k) * ld + cell] = acc;
                }
            }
        }
        __syncthreads();      // the workspace slab is reused by the next cell slab
    }
}

// fp64 FMA-pipe micro-benchmark: 8 independent chains per thread (the roofline denominator)
__global__ void __launch_bounds__(256) qss_dfma_kernel(int iters, double *sink) {
    double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-9, a2 = a0 + 2e-9, a3 = a0 + 3e-9;
    double a4 = a0 + 4e-9, a5 = a0 + 5e-9, a6 = a0 + 6e-9, a7 = a0 + 7e-9;
    const double m = 0.999999999, c = 1e-12;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 16; ++u) {
            a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
            a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
        }
    }
    const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (s == 123.456) sink[0] = s;
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// launchers (called by qss_api.cu)
// ---------------------------------------------------------------------------------------------------
size_t qss_slab_ws_doubles(const QssTab &t, bool jac, int nwarp) {
    return (size_t)(jac ? t.ws_jac_base + nwarp * t.nsp : t.ws_wdot) * 32;
}

cudaError_t qss_launch_slab(const QssTab &t, bool jac, int64_t ncells, int64_t ld, const double *C, const double *T,
                            double *wdot, double *cqss, double *jacp, double *ws, int nblocks, int nwarp,
                            cudaStream_t stream) {
    const int64_t nslab = (ncells + 31) / 32;
    if (nslab == 0) return cudaSuccess;
    const int grid = (int)(nslab < nblocks ? nslab : nblocks);
    const int64_t stride = (int64_t)qss_slab_ws_doubles(t, jac, nwarp);
    if (jac) qss_slab_kernel<true><<<grid, nwarp * 32, 0, stream>>>(t, ncells, ld, C, T, wdot, cqss, jacp, ws, stride);
    else qss_slab_kernel<false><<<grid, nwarp * 32, 0, stream>>>(t, ncells, ld, C, T, wdot, cqss, jacp, ws, stride);
    return cudaGetLastError();
}

cudaError_t qss_launch_dfma(int blocks, int iters, double *sink, cudaStream_t stream) {
    qss_dfma_kernel<<<blocks, 256, 0, stream>>>(iters, sink);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------------------
// Allocation-free variant of the general slab kernel (qss_eval_wdot_static, include/qss.h): the per-cell workspace that
// qss_eval_wdot takes from the caller lives in a file-scope device array of QSS_STATIC_SCRATCH_BYTES bytes, which every GPU that
// loads this library holds until the process exits.  The array's name is a device symbol: host code may not pass it to a
// kernel; its device address comes from cudaGetSymbolAddress, taken once per device at handle creation (qss_static_scratch_setup,
// with that device current) and cached here.  The launch uses as many persistent blocks as fit the array.
// The kernel writes every workspace row of a slab before it reads it (the caller-supplied workspace of qss_eval_wdot is
// uninitialised memory too), so nothing has to be cleared between calls; calls that overlap on the GPU share the array and race.
// ---------------------------------------------------------------------------------------------------
#ifndef QSS_STATIC_MIB
#define QSS_STATIC_MIB 8
#endif
#define QSS_STATIC_SCRATCH_BYTES_ ((unsigned)QSS_STATIC_MIB << 20)
static __device__ __align__(256) unsigned char qss_static_scratch[QSS_STATIC_SCRATCH_BYTES_];

namespace {
constexpr int QSS_STATIC_MAX_DEVICES = 64;
double *g_static_ptr[QSS_STATIC_MAX_DEVICES] = {nullptr};      // device address of qss_static_scratch per device ordinal
}

// Set-up, once per device, with `device` current (called by qss_mech_create): no allocation, the array came with the module.
cudaError_t qss_static_scratch_setup(int device) {
    if (device < 0 || device >= QSS_STATIC_MAX_DEVICES) return cudaErrorInvalidDevice;
    if (g_static_ptr[device]) return cudaSuccess;
    void *p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, qss_static_scratch);
    if (e != cudaSuccess) return e;
    g_static_ptr[device] = (double *)p;
    return cudaSuccess;
}

size_t qss_static_scratch_capacity() { return (size_t)QSS_STATIC_SCRATCH_BYTES_; }

// wdot (and C_QSS) by the general slab kernel with the static workspace.  *blocks_out: persistent blocks used.  Returns
// cudaErrorMemoryAllocation when not even one block's workspace fits the array, cudaErrorNotReady when set-up has not run.
cudaError_t qss_launch_slab_static(const QssTab &t, int device, int64_t ncells, int64_t ld, const double *C, const double *T, double *wdot,
                                   double *cqss, int nblocks, int nwarp, cudaStream_t stream, int *blocks_out) {
    const int64_t nslab = (ncells + 31) / 32;
    if (nslab == 0) return cudaSuccess;
    if (device < 0 || device >= QSS_STATIC_MAX_DEVICES || !g_static_ptr[device]) return cudaErrorNotReady;
    const size_t per_block = qss_slab_ws_doubles(t, false, nwarp) * sizeof(double);
    const size_t fit = per_block ? (size_t)QSS_STATIC_SCRATCH_BYTES_ / per_block : (size_t)nblocks;
    if (fit == 0) return cudaErrorMemoryAllocation;
    int grid = (int)(nslab < nblocks ? nslab : nblocks);
    if ((size_t)grid > fit) grid = (int)fit;
    if (blocks_out) *blocks_out = grid;
    qss_slab_kernel<false><<<grid, nwarp * 32, 0, stream>>>(t, ncells, ld, C, T, wdot, cqss, nullptr, g_static_ptr[device],
                                                           (int64_t)qss_slab_ws_doubles(t, false, nwarp));
    return cudaGetLastError();
}
