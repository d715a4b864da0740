// Kernel variant 1 ("slab-smem") for sm_100a: per-cell QSS chemistry -- rate constants -> QSS closure -> wdot ->
// analytical Jacobian with the chain rule through the closure (Eq. 2-4, 6, 7, 9).
//
// Mapping: one thread block per SM works on a slab of 32 consecutive cells; lane l of EVERY
// warp is cell l of the slab, the warps split the items of each phase (species, reactions, closure slots, QSS
// groups, Jacobian columns) and meet at block barriers.  Consequences:
//   - every table read is warp-uniform (tables come from the kernel-parameter constant bank, `p.h`);
//   - every per-cell array access is one conflict-free 256-byte row, in shared memory for the hot state
//     (concentrations, closure factors, W_y, third-body vectors, dy/dx column) and in an L2-resident scratch slab
//     for the write-once / read-once per-direction arrays (k_d, kappa_d, dlnk/dT);
//   - the Jacobian is swept in rounds of 12 columns.  Pass A: each warp accumulates ONE column of [W_x; G_x] (the
//     temporaries that replace the paper's CSE scalars) in its own shared-memory column buffer: a
//     packed column stream is interpreted, the (distinct) rows of a record are loaded together, updated and stored
//     back, so no dependent chain builds up; then the dy/dx_k solve program runs in place on the QSS rows.  Pass B:
//     the warps switch to ROWS and add W_y * dy/dx for all 12 columns of the round from a register tile (one W_y
//     load and one table word per 12 FMAs); every entry leaves as one coalesced 256-byte streaming store.
#ifndef __CUDACC_RTC__
#include <cuda_runtime.h>
#endif

#include "qss_stdint.h"

#include "qss_tables.h"
#include "qss_math.h"
#include "qss_v1.h"

#ifndef QSS_GEN          // (the run-time specialised build exports its one kernel by name)
namespace {
#endif

constexpr double kLn10 = 2.302585092994045684017991454684;
constexpr double kInvLn10 = 0.434294481903251827651128918916605;
constexpr double kLnP0R = 9.4080919689433160;  // ln(101325 / 8.31446261815324)

extern __shared__ double qss_smem[];

#define HT(off, i) p.h[(off) + (i)]
#define SM(row, i) qss_smem[((row) + (i)) * 32 + lane]
#define SC(row, i) sc[(size_t)((row) + (i)) * 32]

// shared memory through 32-bit shared-window addresses (a generic pointer costs a window-base computation per access)
__device__ __forceinline__ double lds(unsigned a) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(a) : "memory");
    return v;
}
__device__ __forceinline__ void sts(unsigned a, double v) { asm volatile("st.shared.f64 [%0], %1;" ::"r"(a), "d"(v) : "memory"); }
// scratch-slab read pinned where it is written in the source (the prefetch distance is the point)
__device__ __forceinline__ double ldg_pin(const double *q) {
    double v;
    asm volatile("ld.global.f64 %0, [%1];" : "=d"(v) : "l"(q) : "memory");
    return v;
}
__device__ __forceinline__ int2 ldc2(const int32_t *q) { return *reinterpret_cast<const int2 *>(q); }
// mechanism tables in global memory: read-only loads with an L2 evict_last policy, so that the 10 GB of Jacobian
// entries streaming through the L2 do not push the (tiny, re-read by every block for every slab) tables out to DRAM
__device__ __forceinline__ unsigned long long l2_keep_policy() {
    unsigned long long pol;
    asm("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ int4 ldg_keep(const int4 *q, unsigned long long pol) {
    int4 v;
    asm volatile("ld.global.nc.L2::cache_hint.v4.s32 {%0, %1, %2, %3}, [%4], %5;" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(q), "l"(pol));
    return v;
}
__device__ __forceinline__ double ldg_keep(const double *q, unsigned long long pol) {
    double v;
    asm volatile("ld.global.nc.L2::cache_hint.f64 %0, [%1], %2;" : "=d"(v) : "l"(q), "l"(pol));
    return v;
}

// Third-body (type 1) and Troe fall-off (type 2) factor of a rate constant (Eq. 2; DESIGN.md readings
// G5-G7): k (in: k_inf, out: the effective rate constant), dlm = d ln k / dM, dlnk = d ln k / dT.  Mc = sum alpha_k C_k.
template <bool JACT>
__device__ __forceinline__ void qss_pressure_factor(const int type, const double Mc, const double lnkinf, const double dlnkinf,
                                                    const double t3, const double t4, const double t5, const double t6, const double t7,
                                                    const double t8, const double t9, const double T, const double lnT, const double invT,
                                                    double &k, double &dlm, double &dlnk) {
    if (type == 1) {
        k *= Mc;
        dlm = qss_rcp(Mc);
    } else {                                       // Troe fall-off
        const double lnk0 = t3 + t4 * lnT - t5 * invT;
        const double dlnk0 = (t4 + t5 * invT) * invT;
        const double Pr = qss_exp(lnk0 - lnkinf) * Mc;
        const double al = t6, i3 = t7, i1 = t8, T2s = t9;
        const double e3 = qss_exp_sat(-T * i3), e1x = qss_exp_sat(-T * i1), e2 = qss_exp_sat(-T2s * invT);
        const double Fc = (1.0 - al) * e3 + al * e1x + e2;
        const double L = log(Pr) * kInvLn10, Lc = log(Fc) * kInvLn10;
        const double c = -0.4 - 0.67 * Lc, n = 0.75 - 1.27 * Lc;
        const double num = L + c, den = n - 0.14 * num;
        const double iden = qss_rcp(den);
        const double f1 = num * iden;
        const double ione_f = qss_rcp(1.0 + f1 * f1);
        const double F = qss_exp(kLn10 * Lc * ione_f);
        const double i1pr = qss_rcp(1.0 + Pr);
        k = k * (Pr * i1pr) * F;
        const double df1_dL = n * iden * iden;
        const double dlF_dL = -2.0 * Lc * f1 * df1_dL * ione_f * ione_f;
        dlm = (i1pr + dlF_dL) * qss_rcp(Mc);
        if (JACT) {
            const double dFc = -(1.0 - al) * i3 * e3 - al * i1 * e1x + T2s * invT * invT * e2;
            const double df1_dLc = (-0.67 * den - num * (-1.27 + 0.14 * 0.67)) * iden * iden;
            const double dlF_dLc = ione_f - 2.0 * Lc * f1 * df1_dLc * ione_f * ione_f;
            const double delta = dlnk0 - dlnkinf;
            dlnk = dlnkinf + delta * i1pr + dlF_dL * delta + dlF_dLc * dFc * qss_rcp(Fc);
        }
    }
}

#ifdef QSS_GEN
// run-time specialised build (qss_jit.cpp): loads / stores with immediate offsets for the generated pass A
template <int O> __device__ __forceinline__ double lS(unsigned b) {
    double v;
    asm volatile("ld.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(b), "n"(O) : "memory");
    return v;
}
template <int O> __device__ __forceinline__ void sS(unsigned b, double v) { asm volatile("st.shared.f64 [%0+%1], %2;" ::"r"(b), "n"(O), "d"(v) : "memory"); }
template <int O> __device__ __forceinline__ void sG(double *b, double v) { asm volatile("st.global.f64 [%0+%1], %2;" ::"l"(b), "n"(O), "d"(v) : "memory"); }
template <int O> __device__ __forceinline__ double lG(const double *b) {
    double v;
    asm volatile("ld.global.f64 %0, [%1+%2];" : "=d"(v) : "l"(b), "n"(O) : "memory");
    return v;
}
#include "qss_gen.h"
#endif

// optional phase timing (development builds, QSS_TIMING=1): thread 0 of block 0 accumulates the cycles between block barriers
#ifndef QSS_DEVTOOLS
#define QSS_TICK(ph) do { } while (0)
#else
#define QSS_TICK(ph)                                                                   \
    do {                                                                               \
        if (p.timing && blockIdx.x == 0 && threadIdx.x == 0) {                         \
            const long long t_ = clock64();                                            \
            p.timing[ph] += t_ - tick_;                                                \
            tick_ = t_;                                                                \
        }                                                                              \
    } while (0)
#endif

#ifdef QSS_GEN
// run-time specialised build: one entry point, Jacobian on, column stream replaced by the generated pass A
constexpr bool JAC = true, CSG = false;
extern "C" __global__ void __launch_bounds__(QSS_V1_NW * 32, 1) qss_v1_jit(const __grid_constant__ QssV1 p) {
#else
template <bool JAC, bool CSG>
__global__ void __launch_bounds__(QSS_V1_NW * 32, 1) qss_v1_kernel(const __grid_constant__ QssV1 p) {
#endif
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
    const int N = p.N, Nq = p.Nq, M = p.M, nsp = p.nsp;
    const int64_t ld = p.ld;
    const int64_t nslab = (p.ncells + 31) / 32;
    double *sc = p.scratch + (size_t)blockIdx.x * p.scratch_stride + lane;
    const int32_t *gI = p.gI;
    const double *gD = p.gD;
    const unsigned sml = (unsigned)__cvta_generic_to_shared(qss_smem) + lane * 8;   // this lane's column of the rows
    const unsigned long long keep = l2_keep_policy();

    // stage the W_y assembly lists behind the per-cell rows (once per block; the block is persistent over slabs)
    const int *tab = reinterpret_cast<const int *>(qss_smem + (size_t)p.s_TAB * 32);
    for (int i = threadIdx.x; i < p.n_tab_words; i += blockDim.x) reinterpret_cast<int *>(qss_smem + (size_t)p.s_TAB * 32)[i] = __ldg(gI + p.i_wya_ptr + i);
    __syncthreads();

#ifdef QSS_DEVTOOLS
    long long tick_ = clock64();
#endif
    for (int64_t slab = blockIdx.x; slab < nslab; slab += gridDim.x) {
        const int64_t cell = slab * 32 + lane;
        const bool active = cell < p.ncells;
        const int64_t cc = active ? cell : p.ncells - 1;       // idle lanes of a ragged tail shadow the last cell
#ifdef QSS_GEN
        // ---- P0: the inputs of every slab but the block's first were fetched into spare shared-memory rows during the
        //      previous slab's sweep (cp.async below); every warp waits for and moves the rows it fetched itself
        double T;
        const int st_row = p.s_KAP + p.n_wy;                     // [N] C rows, then one T row per warp
        if (slab != blockIdx.x) {
            asm volatile("cp.async.wait_all;" ::: "memory");
            T = lds(sml + (st_row + N + warp) * 256);
            for (int s = warp; s < N; s += nw) sts(sml + (p.s_V + s) * 256, lds(sml + (st_row + s) * 256));
        } else {
            T = p.T[cc];
            for (int s = warp; s < N; s += nw) SM(p.s_V, s) = p.C[(size_t)s * ld + cc];
        }
        const double lnT = log(T), invT = 1.0 / T;
        const double lnP0RT = kLnP0R - lnT;                    // ln(P0 / (R T))
#else
        const double T = p.T[cc];
        const double lnT = log(T), invT = 1.0 / T;
        const double lnP0RT = kLnP0R - lnT;                    // ln(P0 / (R T))
        // ---- P0: stage the concentrations
        for (int s = warp; s < N; s += nw) SM(p.s_V, s) = p.C[(size_t)s * ld + cc];
#endif
        if (warp == 0) { SM(p.s_V, N) = 1.0; SM(p.s_Z0, 0) = 0.0; }
        __syncthreads();
        // (the zero rows behind g/RT and h/RT lie in the time-shared region and may coincide with staged input rows of other
        //  warps: they are written only now, after every warp has moved its staged rows; P2, behind the next barrier, reads them)
        if (warp == 0) { SM(p.s_G, nsp) = 0.0; SM(p.s_H, nsp) = 0.0; }
        QSS_TICK(0);
        // ---- P1: NASA-7 thermo (readings G4, G9); total concentration
        //      the coefficients are L2 reads behind a data-dependent range select: those of three of the warp's species
        //      are in flight together (two latencies per batch instead of two per species)
        for (int s0 = warp; s0 < nsp; s0 += 3 * nw) {
            const double *a[3];
            double tm[3], cf[3][11];
#pragma unroll
            for (int u = 0; u < 3; ++u) tm[u] = ldg_keep(gD + p.d_thermo + min(s0 + u * nw, nsp - 1) * QSS_TH_STRIDE, keep);
#pragma unroll
            for (int u = 0; u < 3; ++u) {
                a[u] = gD + p.d_thermo + min(s0 + u * nw, nsp - 1) * QSS_TH_STRIDE + 1 + (T < tm[u] ? 0 : 11);
#pragma unroll
                for (int i = 0; i < 11; ++i) cf[u][i] = ldg_keep(a[u] + i, keep);
            }
#pragma unroll
            for (int u = 0; u < 3; ++u) {
                const int s = s0 + u * nw;
                if (s < nsp) {
                    const double h = cf[u][0] + T * (cf[u][1] + T * (cf[u][2] + T * (cf[u][3] + T * cf[u][4]))) + cf[u][5] * invT;
                    const double sR = cf[u][0] * lnT + T * (cf[u][6] + T * (cf[u][7] + T * (cf[u][8] + T * cf[u][9]))) + cf[u][10];
                    SM(p.s_H, s) = h;
                    SM(p.s_G, s) = h - sR;
                }
            }
        }
        if (warp == nw - 1) {
            double ct_ = 0.0;
            for (int k = 0; k < N; ++k) ct_ += SM(p.s_V, k);
            SM(p.s_CT, 0) = ct_;
        }
        __syncthreads();
        QSS_TICK(1);
        // ---- P2: rate constants, direction coefficients kappa_d (Eq. 2, Eq. 6)
        {
            const double Ctot = SM(p.s_CT, 0);
            const unsigned gbase = sml + p.s_G * 256, hbase = sml + p.s_H * 256, kbase = sml + p.s_KAP * 256;
            // records and Arrhenius parameters are stored in processing order; those of the warp's NEXT reaction are
            // fetched (L2 reads, the L1 is a few KB next to the shared memory) before the current one is evaluated
            const int n_typed = p.n_tb;                            // third-body and fall-off reactions come first
            // The typed reactions are latency-bound (one long chain of exponentials, logarithms and reciprocals per warp),
            // the Arrhenius pairs issue-bound: half of the warps take the typed reactions first, the other half last, so
            // that every scheduler always has both kinds to pick from.
#pragma unroll 1
            for (int pass = 0; pass < 2; ++pass) {
            if ((pass == 0) == ((warp % 6) < 3)) {
            int4 nra = make_int4(0, 0, 0, 0), nrb = nra;
            double nq0 = 0.0, nq1 = 0.0, nq2 = 0.0, nq10 = 0.0;
            if (warp < n_typed) {
                nra = ldg_keep(reinterpret_cast<const int4 *>(gI + p.i_rrec + warp * QSS_V1_RREC), keep);
                nrb = ldg_keep(reinterpret_cast<const int4 *>(gI + p.i_rrec + warp * QSS_V1_RREC + 4), keep);
                const double *rn = gD + p.d_rate_r + warp * QSS_RD_STRIDE;
                nq0 = ldg_keep(rn, keep); nq1 = ldg_keep(rn + 1, keep); nq2 = ldg_keep(rn + 2, keep); nq10 = ldg_keep(rn + 10, keep);
            }
#pragma unroll 1
            for (int r = warp; r < n_typed; r += nw) {
                const int4 ra = nra, rb = nrb;
                const double q0 = nq0, q1 = nq1, q2 = nq2, q10 = nq10;
                const double *rd = gD + p.d_rate_r + r * QSS_RD_STRIDE;
                if (r + nw < n_typed) {
                    nra = ldg_keep(reinterpret_cast<const int4 *>(gI + p.i_rrec + (r + nw) * QSS_V1_RREC), keep);
                    nrb = ldg_keep(reinterpret_cast<const int4 *>(gI + p.i_rrec + (r + nw) * QSS_V1_RREC + 4), keep);
                    const double *rn = rd + nw * QSS_RD_STRIDE;
                    nq0 = ldg_keep(rn, keep); nq1 = ldg_keep(rn + 1, keep); nq2 = ldg_keep(rn + 2, keep); nq10 = ldg_keep(rn + 10, keep);
                }
                const int j = ra.x & 4095, type = (ra.x >> 12) & 3, mask = (ra.x >> 14) & 3, tb = (ra.x >> 16) - 1;
                double t3 = 0.0, t4 = 0.0, t5 = 0.0, t6 = 0.0, t7 = 0.0, t8 = 0.0, t9 = 0.0;   // fall-off parameters (L2 reads, issued early)
                if (type == 2) {
                    t3 = ldg_keep(rd + 3, keep); t4 = ldg_keep(rd + 4, keep); t5 = ldg_keep(rd + 5, keep); t6 = ldg_keep(rd + 6, keep);
                    t7 = ldg_keep(rd + 7, keep); t8 = ldg_keep(rd + 8, keep); t9 = ldg_keep(rd + 9, keep);
                }
                // all shared-memory reads of the reaction first, then the two exponentials side by side (two independent
                // Horner chains), then the type-specific factor
                const unsigned g0 = rb.x & 0xffff, g1 = (unsigned)rb.x >> 16, g2 = rb.y & 0xffff;      // reactant molecules
                const unsigned g3 = (unsigned)rb.y >> 16, g4 = rb.z & 0xffff, g5 = (unsigned)rb.z >> 16;  // product molecules
                const double dG = (lds(gbase + g3) + lds(gbase + g4) + lds(gbase + g5)) - (lds(gbase + g0) + lds(gbase + g1) + lds(gbase + g2));
                double dH = 0.0;
                if (JAC) dH = (lds(hbase + g3) + lds(hbase + g4) + lds(hbase + g5)) - (lds(hbase + g0) + lds(hbase + g1) + lds(hbase + g2));
                const double vf = lds(sml + (ra.y & 0xffff)) * lds(sml + ((unsigned)ra.y >> 16)) * lds(sml + (ra.z & 0xffff));
                const double vb = lds(sml + ((unsigned)ra.z >> 16)) * lds(sml + (ra.w & 0xffff)) * lds(sml + ((unsigned)ra.w >> 16));
                const double lnkinf = q0 + q1 * lnT - q2 * invT;
                const double dlnkinf = (q1 + q2 * invT) * invT;
                double k = qss_exp(lnkinf), dlnk = dlnkinf;
                const double iKc = qss_exp(dG - q10 * lnP0RT);      // 1 / Kc, ln Kc = -dG + dnu ln(P0/RT)
                if (type >= 1) {
                    double Mc = Ctot;                              // M = sum_k alpha_k C_k, transported only (G7)
                    for (int e = rb.w & 0xffff, ee = e + ((unsigned)rb.w >> 16); e < ee; ++e) {
                        const unsigned off = ((unsigned)HT(p.h_eff_off, e >> 1) >> ((e & 1) * 16)) & 0xffffu;
                        Mc = fma(*reinterpret_cast<const double *>(&p.h[p.h_eff_val + 2 * e]), lds(sml + off), Mc);
                    }
                    double dlm;
                    qss_pressure_factor<JAC>(type, Mc, lnkinf, dlnkinf, t3, t4, t5, t6, t7, t8, t9, T, lnT, invT, k, dlm, dlnk);
                    if (JAC) SC(p.g_QM, tb) = dlm;
                }
                // reverse rate from the equilibrium constant; a disabled direction contributes nothing (G10)
                const double kf = (mask & 1) ? k : 0.0, kb = (mask & 2) ? k * iKc : 0.0;
                const double dlnKc = (mask & 2) ? (dH - q10) * invT : 0.0;
                SC(p.g_K, 2 * j) = kf;
                SC(p.g_K, 2 * j + 1) = kb;
                // kappa_d = k_d * product of the TRANSPORTED reactant molecules (QSS and empty slots read the 1.0 row)
                sts(kbase + j * 512, kf * vf);
                sts(kbase + j * 512 + 256, kb * vb);
                if (JAC) { SC(p.g_DF, j) = dlnk; SC(p.g_DC, j) = dlnKc; }
            }
            } else {
            // Arrhenius reactions, two at a time (four independent exponential chains): reads of both, arithmetic, stores
#define QSS_RX_FETCH(R_, A_, B_, Q0_, Q1_, Q2_, Q10_)                                                            \
    if ((R_) < M) {                                                                                              \
        A_ = ldg_keep(reinterpret_cast<const int4 *>(gI + p.i_rrec + (R_) * QSS_V1_RREC), keep);                   \
        B_ = ldg_keep(reinterpret_cast<const int4 *>(gI + p.i_rrec + (R_) * QSS_V1_RREC + 4), keep);               \
        const double *rn_ = gD + p.d_rate_r + (size_t)(R_) * QSS_RD_STRIDE;                                       \
        Q0_ = ldg_keep(rn_, keep); Q1_ = ldg_keep(rn_ + 1, keep); Q2_ = ldg_keep(rn_ + 2, keep); Q10_ = ldg_keep(rn_ + 10, keep); \
    }
#define QSS_RX_READ(A_, B_, DG_, DH_, VF_, VB_)                                                                   \
    const double DG_ = (lds(gbase + ((unsigned)B_.y >> 16)) + lds(gbase + (B_.z & 0xffff)) + lds(gbase + ((unsigned)B_.z >> 16))) -  \
                       (lds(gbase + (B_.x & 0xffff)) + lds(gbase + ((unsigned)B_.x >> 16)) + lds(gbase + (B_.y & 0xffff)));        \
    double DH_ = 0.0;                                                                                             \
    if (JAC) DH_ = (lds(hbase + ((unsigned)B_.y >> 16)) + lds(hbase + (B_.z & 0xffff)) + lds(hbase + ((unsigned)B_.z >> 16))) -    \
                   (lds(hbase + (B_.x & 0xffff)) + lds(hbase + ((unsigned)B_.x >> 16)) + lds(hbase + (B_.y & 0xffff)));            \
    const double VF_ = lds(sml + (A_.y & 0xffff)) * lds(sml + ((unsigned)A_.y >> 16)) * lds(sml + (A_.z & 0xffff));                \
    const double VB_ = lds(sml + ((unsigned)A_.z >> 16)) * lds(sml + (A_.w & 0xffff)) * lds(sml + ((unsigned)A_.w >> 16))
#define QSS_RX_STORE(A_, Q1_, Q2_, Q10_, K_, IKC_, DH_, VF_, VB_)                                                 \
    {                                                                                                             \
        const int j_ = A_.x & 4095, mask_ = (A_.x >> 14) & 3;                                                     \
        const double kf_ = (mask_ & 1) ? K_ : 0.0, kb_ = (mask_ & 2) ? K_ * IKC_ : 0.0;                           \
        SC(p.g_K, 2 * j_) = kf_; SC(p.g_K, 2 * j_ + 1) = kb_;                                                     \
        sts(kbase + j_ * 512, kf_ * VF_); sts(kbase + j_ * 512 + 256, kb_ * VB_);                                 \
        if (JAC) { SC(p.g_DF, j_) = (Q1_ + Q2_ * invT) * invT; SC(p.g_DC, j_) = (mask_ & 2) ? (DH_ - Q10_) * invT : 0.0; } \
    }
            {
                int4 xa = make_int4(0, 0, 0, 0), xb = xa, ya = xa, yb = xa;
                double xq0 = 0.0, xq1 = 0.0, xq2 = 0.0, xq10 = 0.0, yq0 = 0.0, yq1 = 0.0, yq2 = 0.0, yq10 = 0.0;
                int r = n_typed + warp;
                QSS_RX_FETCH(r, xa, xb, xq0, xq1, xq2, xq10)
                QSS_RX_FETCH(r + nw, ya, yb, yq0, yq1, yq2, yq10)
#pragma unroll 1
                for (; r < M; r += 2 * nw) {
                    const int4 a0 = xa, b0 = xb, a1 = ya, b1 = yb;
                    const double p0 = xq0, p1 = xq1, p2 = xq2, p10 = xq10, s0 = yq0, s1 = yq1, s2 = yq2, s10 = yq10;
                    const bool two = r + nw < M;
                    QSS_RX_FETCH(r + 2 * nw, xa, xb, xq0, xq1, xq2, xq10)
                    QSS_RX_FETCH(r + 3 * nw, ya, yb, yq0, yq1, yq2, yq10)
                    QSS_RX_READ(a0, b0, dG0, dH0, vf0, vb0);
                    if (two) {
                        QSS_RX_READ(a1, b1, dG1, dH1, vf1, vb1);
                        const double k0 = qss_exp(p0 + p1 * lnT - p2 * invT), k1 = qss_exp(s0 + s1 * lnT - s2 * invT);
                        const double i0 = qss_exp(dG0 - p10 * lnP0RT), i1 = qss_exp(dG1 - s10 * lnP0RT);
                        QSS_RX_STORE(a0, p1, p2, p10, k0, i0, dH0, vf0, vb0)
                        QSS_RX_STORE(a1, s1, s2, s10, k1, i1, dH1, vf1, vb1)
                    } else {
                        const double k0 = qss_exp(p0 + p1 * lnT - p2 * invT), i0 = qss_exp(dG0 - p10 * lnP0RT);
                        QSS_RX_STORE(a0, p1, p2, p10, k0, i0, dH0, vf0, vb0)
                    }
                }
            }
#undef QSS_RX_FETCH
#undef QSS_RX_READ
#undef QSS_RX_STORE
            }
            }
        }
        __syncthreads();
        QSS_TICK(2);
#ifdef QSS_GEN
        // ---- P3 + P7, specialised: signed sums of kappas as straight-line code (closure slots, couplings, W_y entries)
        qss_gen_gather(warp, sml, sc);
#else
        // ---- P3: closure assembly: every P / leak / p0 slot gathers the kappas feeding it (no atomics)
        for (int e = warp; e < p.n_centry; e += nw) {
            double acc = 0.0;
            for (int x = tab[p.t_ce_ptr + e], xe = tab[p.t_ce_ptr + e + 1]; x < xe; ++x) acc += SM(p.s_KAP, tab[p.t_ce_dir + x]);
            SM(p.s_CL, tab[p.t_ce_dst + e]) = acc;
        }
        for (int e = warp; e < p.n_xp; e += nw) {
            double acc = 0.0;
            for (int x = HT(p.h_xp_ptr, e); x < HT(p.h_xp_ptr, e + 1); ++x) acc += SM(p.s_KAP, HT(p.h_xp_dir, x));
            SM(p.s_XP, e) = acc;
        }
        if (JAC) {
            // ---- P7 (same phase: reads kappa only): W_y[i][q] = d wdot_i / d y_q at fixed x, sums of kappas
            //      (Eq. 9 second parenthesis, L224); the entries go to the scratch slab, pass B reads each once per round
            const unsigned kb = sml + p.s_KAP * 256;
            for (int e = warp; e < p.n_wy; e += nw) {
                double acc = 0.0;
                const int xe = tab[e + 1];
                for (int x = tab[e]; x < xe; ++x) {
                    const int w = tab[p.n_wy + 1 + x], sg = w & 0x80000000;
                    const double kap = lds(kb + (w & 0x7fffffff));
                    acc += __hiloint2double(__double2hiint(kap) ^ sg, __double2loint(kap));
                }
                SC(p.g_WY, e) = acc;
            }
        }
#endif
        __syncthreads();
        QSS_TICK(3);
        // ---- P4: closure solve, level by level of the condensed DAG; subtraction-free elimination
        //          (Eq. 6; readings G2, G8)
#ifdef QSS_GEN
        qss_gen_closure(warp, sml);        // (block barrier after every level inside)
        QSS_TICK(4);
#else
        for (int l = 0; l < p.n_levels; ++l) {
            for (int g = HT(p.h_level_ptr, l) + warp; g < HT(p.h_level_ptr, l + 1); g += nw) {
                const int gi = p.h_group + g * QSS_GI_STRIDE;
                const int sz = HT(gi, 0), moff = HT(gi, 1), base = p.s_CL + HT(gi, 2), x0 = HT(gi, 4), x1 = HT(gi, 5);
                const int oL = base + sz * sz, oP0 = oL + sz, oID = oP0 + sz;
                for (int x = x0; x < x1; ++x) SM(oP0, HT(p.h_xp_m, x)) += SM(p.s_XP, x) * SM(p.s_V, N + 1 + HT(p.h_xp_n, x));
                for (int k = sz - 1; k >= 1; --k) {
                    const double lk = SM(oL, k);
                    double Dk = lk;
                    for (int m = 0; m < k; ++m) Dk += SM(base, m * sz + k);
                    const double iD = qss_rcp(Dk);
                    SM(oID, k) = iD;
                    for (int jj = 0; jj < k; ++jj) {
                        const double f = SM(base, k * sz + jj) * iD;
                        SM(oL, jj) += f * lk;
                        for (int m = 0; m < k; ++m)
                            if (m != jj) SM(base, m * sz + jj) += SM(base, m * sz + k) * f;
                    }
                }
                SM(oID, 0) = qss_rcp(SM(oL, 0));
                for (int k = sz - 1; k >= 1; --k) {          // U[m][k] = P[m][k] / D_k (reused by every dy/dx solve)
                    const double iD = SM(oID, k), tk = SM(oP0, k) * iD;
                    for (int m = 0; m < k; ++m) {
                        const double pmk = SM(base, m * sz + k);
                        SM(base, m * sz + k) = pmk * iD;
                        SM(oP0, m) += pmk * tk;
                    }
                }
                for (int k = 0; k < sz; ++k) {
                    double acc = SM(oP0, k);
                    for (int jj = 0; jj < k; ++jj) acc += SM(base, k * sz + jj) * SM(oP0, jj);
                    acc *= SM(oID, k);
                    SM(oP0, k) = acc;
                    SM(p.s_V, N + 1 + HT(p.h_gmember, moff + k)) = acc;
                }
            }
            __syncthreads();
            QSS_TICK(4);
        }
#endif
        // ---- P5: net rates of progress Q_j (Eq. 2), dQ/dT at fixed y and M, dQ/dM.  dlnk/dT, dlnKc/dT and dlnk/dM are L2
        //      reads (~700 cycles): those of 8 of the warp's reactions are in flight together.  dQ/dM goes to the scratch
        //      slab (the column streams read it) and to the dead g/RT rows of shared memory (the species sums read it).
        for (int j0 = warp; j0 < M; j0 += 8 * nw) {
            int wq[8];
            double df[8], dc[8], qm[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int j = j0 + u * nw;
                wq[u] = j < M ? tab[p.t_q + j] : 0;
                df[u] = dc[u] = qm[u] = 0.0;
                if (JAC && j < M) {
                    df[u] = ldg_pin(&SC(p.g_DF, j)); dc[u] = ldg_pin(&SC(p.g_DC, j));
                    if ((wq[u] >> 16) > 0) qm[u] = ldg_pin(&SC(p.g_QM, (wq[u] >> 16) - 1));
                }
            }
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const int j = j0 + u * nw;
                if (j < M) {
                    const int w = wq[u];
                    const double rf = SM(p.s_KAP, 2 * j) * SM(p.s_V, w & 255);
                    const double rb = SM(p.s_KAP, 2 * j + 1) * SM(p.s_V, (w >> 8) & 255);
                    const double Q = rf - rb;
                    SM(p.s_KAP, 2 * j) = Q;                         // Q_j and dQ_j/dT replace the two kappas in place
                    if (JAC) {
                        SM(p.s_KAP, 2 * j + 1) = Q * df[u] + rb * dc[u];
                        const int tb = (w >> 16) - 1;
                        if (tb >= 0) { SC(p.g_QM, tb) = qm[u] * Q; SM(p.s_G, tb) = qm[u] * Q; }
                    }
                }
            }
        }
        __syncthreads();
        QSS_TICK(5);
        // ---- P6: species sums: wdot (Eq. 3); for the Jacobian the T-column vector and the third-body vector.
        //      One table entry per unit of |nu|: the sign bit of the entry flips the sign bit of the value.
        {
            const unsigned kbase = sml + p.s_KAP * 256;
            for (int u = HT(p.h_ssw_ptr, warp); u < HT(p.h_ssw_ptr, warp + 1); ++u) {
                const int s = HT(p.h_ssw, u);
                double w = 0.0, et = 0.0, tv = 0.0;
                // software pipeline: the table word two entries ahead and the values one entry ahead are read while the current
                // entry is added (the words past the end of the list belong to the next list or table and address valid rows)
                const int xe = HT(p.h_ss_ptr, s + 1);
                int x = HT(p.h_ss_ptr, s);
                int e0 = HT(p.h_ss, x), e1 = HT(p.h_ss, x + 1);
                double q0 = lds(kbase + (e0 & 0x7fffffff)), t0 = JAC ? lds(kbase + (e0 & 0x7fffffff) + 256) : 0.0;
                for (; x < xe; ++x) {
                    const int e2 = HT(p.h_ss, x + 2);
                    const unsigned a1 = kbase + (e1 & 0x7fffffff);
                    const double q1 = lds(a1), t1 = JAC ? lds(a1 + 256) : 0.0;
                    const int sg = e0 & 0x80000000;
                    w += __hiloint2double(__double2hiint(q0) ^ sg, __double2loint(q0));
                    if (JAC) et += __hiloint2double(__double2hiint(t0) ^ sg, __double2loint(t0));
                    e0 = e1; e1 = e2; q0 = q1; t0 = t1;
                }
                if (JAC) {
                    const int te = HT(p.h_st_ptr, s + 1);
                    for (int x = HT(p.h_st_ptr, s); x < te; ++x) {
                        const int e = HT(p.h_st, x), sg = e & 0x80000000;
                        const double qm = SM(p.s_G, e & 0x7fffffff);
                        tv += __hiloint2double(__double2hiint(qm) ^ sg, __double2loint(qm));
                    }
                }
                if (s < N && p.wdot && active) p.wdot[(size_t)s * ld + cell] = w;
                if (JAC) { SM(p.s_TV, s) = tv; SC(p.g_ET, s) = et; }
            }
        }
        if (p.cqss && active)
            for (int q = warp; q < Nq; q += nw) p.cqss[(size_t)q * ld + cell] = SM(p.s_V, N + 1 + q);
        if (JAC) {
            __syncthreads();
            QSS_TICK(6);
#ifdef QSS_GEN
            // ---- P8, specialised: W_y moves from the scratch slab to shared memory (the kappa region is free now); then each
            //      warp takes its columns one after the other, everything in registers (qss_gen_column), no barrier between
            //      (QSS_GEN_NROWS rows: the W_y entries, or kappa_d of the QSS-consuming directions when those are fewer)
            for (int e0 = warp * 8; e0 < QSS_GEN_NROWS; e0 += nw * 8) {
                double t[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) t[u] = ldg_pin(&SC(p.g_WY, min(e0 + u, QSS_GEN_NROWS - 1)));
#pragma unroll
                for (int u = 0; u < 8; ++u) if (e0 + u < QSS_GEN_NROWS) sts(sml + (p.s_KAP + e0 + u) * 256, t[u]);
            }
            __syncthreads();
            QSS_TICK(11);
            if (slab + gridDim.x < nslab) {      // inputs of the block's next slab -> spare rows behind W_y, under the sweep
                const int64_t cell2 = (slab + gridDim.x) * 32 + lane;
                const int64_t cc2 = cell2 < p.ncells ? cell2 : p.ncells - 1;
                for (int s = warp; s < N; s += nw)
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sml + (st_row + s) * 256), "l"(p.C + (size_t)s * ld + cc2) : "memory");
                asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sml + (st_row + N + warp) * 256), "l"(p.T + cc2) : "memory");
            }
            for (int d = 0; d < QSS_GEN_DEPTH; ++d) {
                const int k = qss_gen_cols[warp * QSS_GEN_DEPTH + d];
                if (k >= 0) qss_gen_column(k, sml, sc, p.jac + (size_t)(unsigned)k * (size_t)ld + cell, (long long)(N + 1) * ld, active);
            }
            QSS_TICK(13);
#else
            // ---- P8: Jacobian sweep in rounds of nw columns (Eq. 7, Eq. 9)
            constexpr unsigned RS = QSS_V1_NW * 256;                 // byte stride between rows of a column buffer
            const unsigned colw = sml + (p.s_WX + warp) * 256;       // this warp's column of [W_x; G_x]: species row r at + r * RS
            const unsigned ycw = colw + N * RS;                      //   its QSS part, solved in place into dy/dx_k
            for (int r = 0; r < p.n_rounds; ++r) {
                // -- pass A: warp = column k.  [W_x; G_x][:,k] in shared memory, then (diag D - P) dy/dx_k = G_x[:,k]
                const int k = HT(p.h_cw, r * nw + warp);
                if (k >= 0) {
                    // initialise the column: rank-1 third-body vector (every species column) or the T-column vector;
                    // 8 rows are read before they are written so that the copies do not serialise on the load latency
                    if (k < N) {
                        for (int s0 = 0; s0 < nsp; s0 += 8) {
                            double t[8];
#pragma unroll
                            for (int u = 0; u < 8; ++u) t[u] = lds(sml + (p.s_TV + min(s0 + u, nsp - 1)) * 256);
#pragma unroll
                            for (int u = 0; u < 8; ++u) if (s0 + u < nsp) sts(colw + (s0 + u) * RS, t[u]);
                        }
                    } else {
                        for (int s0 = 0; s0 < nsp; s0 += 16) {          // L2 reads: 16 in flight together
                            double t[16];
#pragma unroll
                            for (int u = 0; u < 16; ++u) t[u] = ldg_pin(&SC(p.g_ET, min(s0 + u, nsp - 1)));
#pragma unroll
                            for (int u = 0; u < 16; ++u) if (s0 + u < nsp) sts(colw + (s0 + u) * RS, t[u]);
                        }
                    }
                    QSS_TICK(11);
                    // column stream: part = |nu| * A * V[o1] * V[o2] (* val), added to / subtracted from up to 8 rows of the
                    // column.  Records come in PAIRS with disjoint rows.  Software pipeline over pairs: while pair i is
                    // applied (the rows of both records are loaded together, updated, stored back), the factors of pair
                    // i+1 are read from shared memory and the table words and A (L2 reads) of pair i+2 are fetched.  Reads
                    // past the end of a column hit the next column's records or the sentinel pairs and are discarded.
                    {
                        const int x0 = p.h_cs + HT(p.h_cs_ptr, k);
                        const int npair = (HT(p.h_cs_ptr, k + 1) - HT(p.h_cs_ptr, k)) >> 3;
                        const unsigned one = sml + (p.s_V + N) * 256;
#define QSS_FETCH(XO, ra, rb, rA, rV)                                                    \
    if (CSG) {                                                                           \
        const int4 r4_ = ldg_keep(reinterpret_cast<const int4 *>(gI + (XO)), keep);      \
        ra = make_int2(r4_.x, r4_.y); rb = make_int2(r4_.z, r4_.w);                      \
    } else {                                                                             \
        ra = ldc2(&p.h[XO]); rb = ldc2(&p.h[(XO) + 2]);                                  \
    }                                                                                    \
    rA = sc[(size_t)(ra.x & 0xffff) * 32];                                               \
    rV = (ra.x & (1 << 20)) ? ldg_keep(gD + p.d_effv + ra.y, keep) : 1.0
#define QSS_FACTORS(ra, f1, f2)                                                          \
    const double f1 = lds((ra.x & (1 << 20)) ? one : sml + (ra.y & 0xffff)),             \
                 f2 = lds((ra.x & (1 << 20)) ? one : sml + ((unsigned)ra.y >> 16))
#define QSS_PART(ra, rA, rV, f1, f2, out)                                                \
    double out = rA * rV * f1 * f2;                                                      \
    if (((ra.x >> 21) & 7) > 1) out *= (double)((ra.x >> 21) & 7)
#define QSS_ROWS(w, q0, q1, q2, q3)                                                      \
    const unsigned q0 = colw + ((w) & 127) * RS, q1 = colw + (((w) >> 8) & 127) * RS,    \
                   q2 = colw + (((w) >> 16) & 127) * RS, q3 = colw + (((w) >> 24) & 127) * RS
#define QSS_SIGNED(pt, w, sh) __hiloint2double(__double2hiint(pt) ^ (int)(((w) << (sh)) & 0x80000000u), __double2loint(pt))
#define QSS_APPLY(w, q0, q1, q2, q3, v0, v1, v2, v3, pt)                                 \
    sts(q0, v0 + QSS_SIGNED(pt, w, 24)); sts(q1, v1 + QSS_SIGNED(pt, w, 16));            \
    sts(q2, v2 + QSS_SIGNED(pt, w, 8)); sts(q3, v3 + QSS_SIGNED(pt, w, 0))
                        double own = 0.0;                                 // contributions to the column's own row k
                        int2 sa0, sb0, sa1, sb1, ma0, mb0, ma1, mb1;
                        double tA, tV, mA0, mV0, mA1, mV1, part0, part1;
                        {
                            QSS_FETCH(x0, sa0, sb0, tA, tV);
                            QSS_FACTORS(sa0, f1, f2);
                            QSS_PART(sa0, tA, tV, f1, f2, pt);
                            part0 = pt;
                        }
                        {
                            QSS_FETCH(x0 + 4, sa1, sb1, tA, tV);
                            QSS_FACTORS(sa1, f1, f2);
                            QSS_PART(sa1, tA, tV, f1, f2, pt);
                            part1 = pt;
                        }
                        QSS_FETCH(x0 + 8, ma0, mb0, mA0, mV0);
                        QSS_FETCH(x0 + 12, ma1, mb1, mA1, mV1);
#pragma unroll 1
                        for (int i = 0; i < npair; ++i) {
                            // apply pair i, first half: load the rows of both records
                            const unsigned w0 = (unsigned)sb0.x, w1 = (unsigned)sb1.x;
                            QSS_ROWS(w0, a0, a1, a2, a3);
                            QSS_ROWS(w1, c0, c1, c2, c3);
                            const double v0 = lds(a0), v1 = lds(a1), v2 = lds(a2), v3 = lds(a3);
                            const double t0 = lds(c0), t1 = lds(c1), t2 = lds(c2), t3 = lds(c3);
                            // factors of pair i + 1
                            QSS_FACTORS(ma0, f1, f2);
                            QSS_FACTORS(ma1, g1, g2);
                            // table words and A of pair i + 2
                            const int xl = x0 + 8 * (i + 2);
                            int2 na0, nb0, na1, nb1;
                            double nA0, nV0, nA1, nV1;
                            QSS_FETCH(xl, na0, nb0, nA0, nV0);
                            QSS_FETCH(xl + 4, na1, nb1, nA1, nV1);
                            // apply pair i, second half
                            own += (sa0.x & (1 << 24)) ? part0 : ((sa0.x & (2 << 24)) ? -part0 : 0.0);
                            own += (sa1.x & (1 << 24)) ? part1 : ((sa1.x & (2 << 24)) ? -part1 : 0.0);
                            QSS_APPLY(w0, a0, a1, a2, a3, v0, v1, v2, v3, part0);
                            QSS_APPLY(w1, c0, c1, c2, c3, t0, t1, t2, t3, part1);
                            if (((sa0.x >> 16) & 15) > 4) {
                                const unsigned w2 = (unsigned)sb0.y;
                                QSS_ROWS(w2, d0, d1, d2, d3);
                                const double u0 = lds(d0), u1 = lds(d1), u2 = lds(d2), u3 = lds(d3);
                                QSS_APPLY(w2, d0, d1, d2, d3, u0, u1, u2, u3, part0);
                            }
                            if (((sa1.x >> 16) & 15) > 4) {
                                const unsigned w2 = (unsigned)sb1.y;
                                QSS_ROWS(w2, d0, d1, d2, d3);
                                const double u0 = lds(d0), u1 = lds(d1), u2 = lds(d2), u3 = lds(d3);
                                QSS_APPLY(w2, d0, d1, d2, d3, u0, u1, u2, u3, part1);
                            }
                            // parts of pair i + 1; rotate the pipeline
                            QSS_PART(ma0, mA0, mV0, f1, f2, np0);
                            QSS_PART(ma1, mA1, mV1, g1, g2, np1);
                            part0 = np0; part1 = np1;
                            sa0 = ma0; sb0 = mb0; sa1 = ma1; sb1 = mb1;
                            ma0 = na0; mb0 = nb0; mA0 = nA0; mV0 = nV0;
                            ma1 = na1; mb1 = nb1; mA1 = nA1; mV1 = nV1;
                        }
                        if (k < N) sts(colw + k * RS, lds(colw + k * RS) + own);
#undef QSS_FETCH
#undef QSS_FACTORS
#undef QSS_PART
#undef QSS_ROWS
#undef QSS_APPLY
#undef QSS_SIGNED
                    }
                    QSS_TICK(12);
                    // dy/dx solve program: pairs of independent fixed-format row operations
                    // y[a] = (y[a] + F0 y[b0] + F1 y[b1] + F2 y[b2]) * S; all 16 loads of a pair are issued together
                    // (a thread only touches its own lane)
#pragma unroll 1
                    for (int pc = p.h_sp, pe = p.h_sp + 8 * p.n_sp_ops; pc < pe; pc += 8) {
                        const int2 A0 = ldc2(&p.h[pc]), A1 = ldc2(&p.h[pc + 2]), B0 = ldc2(&p.h[pc + 4]), B1 = ldc2(&p.h[pc + 6]);
                        const unsigned ya = ycw + (A0.x & 0xfff) * 256, yb = ycw + (B0.x & 0xfff) * 256;
                        const int na_ = (A0.x >> 12) & 3, nb_ = (B0.x >> 12) & 3;        // terms actually present (the rest is padding)
                        double acc = lds(ya), bcc = lds(yb);
                        const double sa_ = lds(sml + ((unsigned)A1.y >> 16) * 256), sb_ = lds(sml + ((unsigned)B1.y >> 16) * 256);
                        double y0 = 0.0, y1 = 0.0, y2 = 0.0, f0 = 0.0, f1 = 0.0, f2 = 0.0, z0 = 0.0, z1 = 0.0, z2 = 0.0, g0 = 0.0, g1 = 0.0, g2 = 0.0;
                        if (na_ > 0) { y0 = lds(ycw + ((unsigned)A0.x >> 16) * 256); f0 = lds(sml + (A1.x & 0xffff) * 256); }
                        if (nb_ > 0) { z0 = lds(ycw + ((unsigned)B0.x >> 16) * 256); g0 = lds(sml + (B1.x & 0xffff) * 256); }
                        if (na_ > 1) { y1 = lds(ycw + (A0.y & 0xffff) * 256); f1 = lds(sml + ((unsigned)A1.x >> 16) * 256); }
                        if (nb_ > 1) { z1 = lds(ycw + (B0.y & 0xffff) * 256); g1 = lds(sml + ((unsigned)B1.x >> 16) * 256); }
                        if (na_ > 2) { y2 = lds(ycw + ((unsigned)A0.y >> 16) * 256); f2 = lds(sml + (A1.y & 0xffff) * 256); }
                        if (nb_ > 2) { z2 = lds(ycw + ((unsigned)B0.y >> 16) * 256); g2 = lds(sml + (B1.y & 0xffff) * 256); }
                        acc = fma(f0, y0, acc); bcc = fma(g0, z0, bcc);
                        acc = fma(f1, y1, acc); bcc = fma(g1, z1, bcc);
                        acc = fma(f2, y2, acc); bcc = fma(g2, z2, bcc);
                        sts(ya, acc * sa_);
                        sts(yb, bcc * sb_);
                    }
                }
                QSS_TICK(13);
                __syncthreads();
                QSS_TICK(7);
                // -- pass B: warp = a tile of up to 3 rows x the 12 columns of the round.
                //    J[i, round] = W_x[i, round] + sum_q W_y[i][q] * dy_q/dx[round]: dy_q/dx (12 LDS) is read once for the
                //    rows of the tile that have a W_y entry in column q; the W_y entries are L2 reads fetched two steps ahead
                {
                    const int i0 = HT(p.h_rw, warp * 3), i1 = HT(p.h_rw, warp * 3 + 1), i2 = HT(p.h_rw, warp * 3 + 2);
                    double acc0[QSS_V1_NW], acc1[QSS_V1_NW], acc2[QSS_V1_NW];
#pragma unroll
                    for (int w = 0; w < QSS_V1_NW; ++w) {
                        acc0[w] = i0 >= 0 ? lds(sml + (p.s_WX + i0 * nw + w) * 256) : 0.0;
                        acc1[w] = i1 >= 0 ? lds(sml + (p.s_WX + i1 * nw + w) * 256) : 0.0;
                        acc2[w] = i2 >= 0 ? lds(sml + (p.s_WX + i2 * nw + w) * 256) : 0.0;
                    }
                    int x0 = i0 >= 0 ? HT(p.h_wr_ptr, i0) : 0, x1 = i1 >= 0 ? HT(p.h_wr_ptr, i1) : 0, x2 = i2 >= 0 ? HT(p.h_wr_ptr, i2) : 0;
                    int e = HT(p.h_tile_ptr, warp);
                    const int ee = HT(p.h_tile_ptr, warp + 1);
                    int w0 = e < ee ? HT(p.h_tile, e) : 0, w1 = e + 1 < ee ? HT(p.h_tile, e + 1) : 0;
                    double a00 = 0.0, a01 = 0.0, a02 = 0.0, a10 = 0.0, a11 = 0.0, a12 = 0.0;
                    if (w0 & 0x100) a00 = SC(p.g_WY, x0++);
                    if (w0 & 0x200) a01 = SC(p.g_WY, x1++);
                    if (w0 & 0x400) a02 = SC(p.g_WY, x2++);
                    if (w1 & 0x100) a10 = SC(p.g_WY, x0++);
                    if (w1 & 0x200) a11 = SC(p.g_WY, x1++);
                    if (w1 & 0x400) a12 = SC(p.g_WY, x2++);
#pragma unroll 1
                    for (; e < ee; ++e) {
                        const int w2 = e + 2 < ee ? HT(p.h_tile, e + 2) : 0;
                        double a20 = 0.0, a21 = 0.0, a22 = 0.0;
                        if (w2 & 0x100) a20 = SC(p.g_WY, x0++);
                        if (w2 & 0x200) a21 = SC(p.g_WY, x1++);
                        if (w2 & 0x400) a22 = SC(p.g_WY, x2++);
                        const unsigned yr = sml + p.s_YC * 256 + (w0 & 255) * RS;
                        double y[QSS_V1_NW];
#pragma unroll
                        for (int w = 0; w < QSS_V1_NW; ++w) y[w] = lds(yr + w * 256);
                        if (w0 & 0x100) {
#pragma unroll
                            for (int w = 0; w < QSS_V1_NW; ++w) acc0[w] = fma(a00, y[w], acc0[w]);
                        }
                        if (w0 & 0x200) {
#pragma unroll
                            for (int w = 0; w < QSS_V1_NW; ++w) acc1[w] = fma(a01, y[w], acc1[w]);
                        }
                        if (w0 & 0x400) {
#pragma unroll
                            for (int w = 0; w < QSS_V1_NW; ++w) acc2[w] = fma(a02, y[w], acc2[w]);
                        }
                        w0 = w1; w1 = w2;
                        a00 = a10; a01 = a11; a02 = a12; a10 = a20; a11 = a21; a12 = a22;
                    }
                    QSS_TICK(9);
                    if (active) {
#pragma unroll
                        for (int w = 0; w < QSS_V1_NW; ++w) {
                            const int kk = HT(p.h_cw, r * nw + w);
                            if (kk >= 0) {
                                double *jc = p.jac + (size_t)(unsigned)kk * (size_t)ld + cell;
                                if (i0 >= 0) __stcs(jc + (size_t)i0 * (N + 1) * ld, acc0[w]);
                                if (i1 >= 0) __stcs(jc + (size_t)i1 * (N + 1) * ld, acc1[w]);
                                if (i2 >= 0) __stcs(jc + (size_t)i2 * (N + 1) * ld, acc2[w]);
                            }
                        }
                    }
                }
                QSS_TICK(10);
                __syncthreads();
                QSS_TICK(8);
            }
#endif
        }
        __syncthreads();      // shared memory and the scratch slab are reused by the next cell slab
    }
}

#ifndef QSS_GEN
}  // namespace

// ---------------------------------------------------------------------------------------------------
// launcher (called by qss_api.cu)
// ---------------------------------------------------------------------------------------------------
size_t qss_v1_smem_bytes(const QssV1 &v) { return (size_t)v.smem_rows * 256; }
size_t qss_v1_scratch_doubles(const QssV1 &v) { return (size_t)v.scratch_rows * 32; }

cudaError_t qss_v1_prepare() {
    cudaError_t e = cudaFuncSetAttribute(qss_v1_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    if ((e = cudaFuncSetAttribute(qss_v1_kernel<true, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024)) != cudaSuccess) return e;
    return cudaFuncSetAttribute(qss_v1_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

cudaError_t qss_launch_v1(const QssV1 &v, bool jac, int nblocks, cudaStream_t stream) {
    const int64_t nslab = (v.ncells + 31) / 32;
    if (nslab == 0) return cudaSuccess;
    const int grid = (int)(nslab < nblocks ? nslab : nblocks);
    const size_t smem = qss_v1_smem_bytes(v);
    if (jac && v.cs_global) qss_v1_kernel<true, true><<<grid, v.nw * 32, smem, stream>>>(v);
    else if (jac) qss_v1_kernel<true, false><<<grid, v.nw * 32, smem, stream>>>(v);
    else qss_v1_kernel<false, false><<<grid, v.nw * 32, smem, stream>>>(v);
    return cudaGetLastError();
}
#endif  // QSS_GEN
