// NEXT-1: temperature right-hand side and energy row of the (N+1) x (N+1) chemical Jacobian (Eq. 7
// L185; L278: "the contribution of the heat release rate can be simply obtained from the species production rates") for the
// adiabatic constant-volume reactor (L190; reading G17), from wdot and the species block J = d wdot / d[C, T]:
//     Tdot = -T E / Cv,        E = sum_i u_i wdot_i,  u_i = h_i/RT - 1,       Cv = sum_i C_i a_i,  a_i = cp_i/R - 1
//     d Tdot / d C_k = -(T / Cv) sum_i u_i J_ik - Tdot a_k / Cv
//     d Tdot / d T   = Tdot / T - (T / Cv) sum_i (u_i J_iT + wdot_i (cp_i/R - h_i/RT) / T) - Tdot sum_i C_i d(cp_i/R)/dT / Cv
// (sums over the transported species).  Mapping: block = 32 consecutive cells x 8 warps, lane = cell; the warps first split the
// species (NASA-7 polynomials into shared memory), then the columns of the row; every global access is a coalesced 256-byte
// row.  The kernel is bound by reading J once: 8 N (N+1) bytes per cell.
#include <cuda_runtime.h>
#include <stdint.h>

#include "qss_tables.h"

namespace {

constexpr int NWY = 8;

extern __shared__ double qss_en_smem[];

__global__ void __launch_bounds__(32 * NWY) qss_energy_kernel(const double *__restrict__ D, const int d_thermo, const int N, const int64_t ncells,
                                                               const int64_t ld, const double *__restrict__ C, const double *__restrict__ T,
                                                               const double *__restrict__ wdot, const double *__restrict__ jac,
                                                               double *__restrict__ tdot, double *__restrict__ erow) {
    const int x = threadIdx.x, y = threadIdx.y;
    const int64_t cell = (int64_t)blockIdx.x * 32 + x;
    const bool active = cell < ncells;
    const int64_t cc = active ? cell : ncells - 1;
    double *su = qss_en_smem, *sa = su + (size_t)N * 32, *spart = sa + (size_t)N * 32;       // u_i, a_i; partial sums [NWY][4][32]
    const double Tc = T[cc], invT = 1.0 / Tc;
    // species split over the warps: u_i, a_i to shared memory, partial sums of E, Cv, dCv/dT and sum_i wdot_i d(h_i/RT)/dT
    double pE = 0.0, pCv = 0.0, pdCv = 0.0, pdE = 0.0;
    for (int i = y; i < N; i += NWY) {
        const double *th = D + d_thermo + (size_t)i * QSS_TH_STRIDE;
        const double *a = th + 1 + (Tc < __ldg(th) ? 0 : 11);      // {a1, a2/2, a3/3, a4/4, a5/5, a6; a2, a3/2, a4/3, a5/4, a7}
        const double a1 = __ldg(a), a2 = __ldg(a + 6), a3 = 2.0 * __ldg(a + 7), a4 = 3.0 * __ldg(a + 8), a5 = 4.0 * __ldg(a + 9);
        const double hRT = a1 + Tc * (__ldg(a + 1) + Tc * (__ldg(a + 2) + Tc * (__ldg(a + 3) + Tc * __ldg(a + 4)))) + __ldg(a + 5) * invT;
        const double cpR = a1 + Tc * (a2 + Tc * (a3 + Tc * (a4 + Tc * a5)));
        const double dcp = a2 + Tc * (2.0 * a3 + Tc * (3.0 * a4 + Tc * 4.0 * a5));
        const double w = wdot[(size_t)i * ld + cc], c = C[(size_t)i * ld + cc];
        su[i * 32 + x] = hRT - 1.0;
        sa[i * 32 + x] = cpR - 1.0;
        pE = fma(hRT - 1.0, w, pE);
        pCv = fma(c, cpR - 1.0, pCv);
        pdCv = fma(c, dcp, pdCv);
        pdE = fma((cpR - hRT) * invT, w, pdE);
    }
    spart[(y * 4 + 0) * 32 + x] = pE; spart[(y * 4 + 1) * 32 + x] = pCv; spart[(y * 4 + 2) * 32 + x] = pdCv; spart[(y * 4 + 3) * 32 + x] = pdE;
    __syncthreads();
    double E = 0.0, Cv = 0.0, dCv = 0.0, dE = 0.0;
#pragma unroll
    for (int w = 0; w < NWY; ++w) {          // (the same order in every warp: the four sums are identical across the block)
        E += spart[(w * 4 + 0) * 32 + x]; Cv += spart[(w * 4 + 1) * 32 + x]; dCv += spart[(w * 4 + 2) * 32 + x]; dE += spart[(w * 4 + 3) * 32 + x];
    }
    const double iCv = 1.0 / Cv, Td = -Tc * E * iCv, g = Tc * iCv;
    if (y == 0 && active) tdot[cell] = Td;
    // columns split over the warps: e_k = sum_i u_i J_ik, eight rows of J in flight
    const int NC = N + 1;
    for (int k = y; k < NC; k += NWY) {
        const double *jk = jac + (size_t)k * ld + cc;
        double e0 = 0.0, e1 = 0.0;
        int i = 0;
        for (; i + 8 <= N; i += 8) {
            double v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = __ldcs(jk + (size_t)(i + u) * NC * ld);
#pragma unroll
            for (int u = 0; u < 8; u += 2) { e0 = fma(su[(i + u) * 32 + x], v[u], e0); e1 = fma(su[(i + u + 1) * 32 + x], v[u + 1], e1); }
        }
        for (; i < N; ++i) e0 = fma(su[i * 32 + x], __ldcs(jk + (size_t)i * NC * ld), e0);
        const double e = e0 + e1;
        const double row = k < N ? -g * e - Td * sa[k * 32 + x] * iCv : Td * invT - g * (e + dE) - Td * dCv * iCv;
        if (active) erow[(size_t)k * ld + cell] = row;
    }
}

}  // namespace

// Two cells per lane (ld even: every row is 16-byte aligned): the same arithmetic per cell, every global access a 512-byte run
// (16 bytes per lane), which is what the HBM wants (qss_jac_aos_kernel: 4.1 -> 5.4 TB/s from 256- to 512-byte runs).
namespace {
__device__ __forceinline__ double2 ld2(const double *p) { return __ldcs(reinterpret_cast<const double2 *>(p)); }

__global__ void __launch_bounds__(32 * NWY) qss_energy_kernel2(const double *__restrict__ D, const int d_thermo, const int N, const int64_t ncells,
                                                                const int64_t ld, const double *__restrict__ C, const double *__restrict__ T,
                                                                const double *__restrict__ wdot, const double *__restrict__ jac,
                                                                double *__restrict__ tdot, double *__restrict__ erow) {
    const int x = threadIdx.x, y = threadIdx.y;
    const int64_t cell = (int64_t)blockIdx.x * 64 + 2 * x;                   // this lane: cells cell, cell + 1
    const bool act0 = cell < ncells, act1 = cell + 1 < ncells;
    const int64_t cc = act0 ? cell : ((ncells - 1) & ~(int64_t)1);           // idle lanes shadow the last pair (in bounds: ld is even)
    double2 *su = reinterpret_cast<double2 *>(qss_en_smem), *sa = su + (size_t)N * 32, *spart = sa + (size_t)N * 32;
    const double2 Tc = *reinterpret_cast<const double2 *>(T + cc);
    const double Tv[2] = {Tc.x, Tc.y};
    const double invT[2] = {1.0 / Tc.x, 1.0 / Tc.y};
    double pE[2] = {0.0, 0.0}, pCv[2] = {0.0, 0.0}, pdCv[2] = {0.0, 0.0}, pdE[2] = {0.0, 0.0};
    for (int i = y; i < N; i += NWY) {
        const double *th = D + d_thermo + (size_t)i * QSS_TH_STRIDE;
        const double2 w2 = *reinterpret_cast<const double2 *>(wdot + (size_t)i * ld + cc), c2 = *reinterpret_cast<const double2 *>(C + (size_t)i * ld + cc);
        const double wv[2] = {w2.x, w2.y}, cv[2] = {c2.x, c2.y};
        double u[2], aa[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double t = Tv[h];
            const double *a = th + 1 + (t < __ldg(th) ? 0 : 11);
            const double a1 = __ldg(a), a2 = __ldg(a + 6), a3 = 2.0 * __ldg(a + 7), a4 = 3.0 * __ldg(a + 8), a5 = 4.0 * __ldg(a + 9);
            const double hRT = a1 + t * (__ldg(a + 1) + t * (__ldg(a + 2) + t * (__ldg(a + 3) + t * __ldg(a + 4)))) + __ldg(a + 5) * invT[h];
            const double cpR = a1 + t * (a2 + t * (a3 + t * (a4 + t * a5)));
            const double dcp = a2 + t * (2.0 * a3 + t * (3.0 * a4 + t * 4.0 * a5));
            u[h] = hRT - 1.0; aa[h] = cpR - 1.0;
            pE[h] = fma(hRT - 1.0, wv[h], pE[h]);
            pCv[h] = fma(cv[h], cpR - 1.0, pCv[h]);
            pdCv[h] = fma(cv[h], dcp, pdCv[h]);
            pdE[h] = fma((cpR - hRT) * invT[h], wv[h], pdE[h]);
        }
        su[i * 32 + x] = make_double2(u[0], u[1]);
        sa[i * 32 + x] = make_double2(aa[0], aa[1]);
    }
    spart[(y * 4 + 0) * 32 + x] = make_double2(pE[0], pE[1]); spart[(y * 4 + 1) * 32 + x] = make_double2(pCv[0], pCv[1]);
    spart[(y * 4 + 2) * 32 + x] = make_double2(pdCv[0], pdCv[1]); spart[(y * 4 + 3) * 32 + x] = make_double2(pdE[0], pdE[1]);
    __syncthreads();
    double E[2] = {0.0, 0.0}, Cv[2] = {0.0, 0.0}, dCv[2] = {0.0, 0.0}, dE[2] = {0.0, 0.0};
#pragma unroll
    for (int w = 0; w < NWY; ++w) {
        const double2 p0 = spart[(w * 4 + 0) * 32 + x], p1 = spart[(w * 4 + 1) * 32 + x], p2 = spart[(w * 4 + 2) * 32 + x], p3 = spart[(w * 4 + 3) * 32 + x];
        E[0] += p0.x; E[1] += p0.y; Cv[0] += p1.x; Cv[1] += p1.y; dCv[0] += p2.x; dCv[1] += p2.y; dE[0] += p3.x; dE[1] += p3.y;
    }
    double iCv[2], Td[2], g[2];
#pragma unroll
    for (int h = 0; h < 2; ++h) { iCv[h] = 1.0 / Cv[h]; Td[h] = -Tv[h] * E[h] * iCv[h]; g[h] = Tv[h] * iCv[h]; }
    if (y == 0) {
        if (act1) *reinterpret_cast<double2 *>(tdot + cell) = make_double2(Td[0], Td[1]);
        else if (act0) tdot[cell] = Td[0];
    }
    const int NC = N + 1;
    for (int k = y; k < NC; k += NWY) {
        const double *jk = jac + (size_t)k * ld + cc;
        double e0[2] = {0.0, 0.0}, e1[2] = {0.0, 0.0};
        int i = 0;
        for (; i + 8 <= N; i += 8) {
            double2 v[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) v[u] = ld2(jk + (size_t)(i + u) * NC * ld);
#pragma unroll
            for (int u = 0; u < 8; u += 2) {
                const double2 s0 = su[(i + u) * 32 + x], s1 = su[(i + u + 1) * 32 + x];
                e0[0] = fma(s0.x, v[u].x, e0[0]); e0[1] = fma(s0.y, v[u].y, e0[1]);
                e1[0] = fma(s1.x, v[u + 1].x, e1[0]); e1[1] = fma(s1.y, v[u + 1].y, e1[1]);
            }
        }
        for (; i < N; ++i) {
            const double2 s0 = su[i * 32 + x], v = ld2(jk + (size_t)i * NC * ld);
            e0[0] = fma(s0.x, v.x, e0[0]); e0[1] = fma(s0.y, v.y, e0[1]);
        }
        double row[2];
        const double2 ak = k < N ? sa[k * 32 + x] : make_double2(0.0, 0.0);
        const double akv[2] = {ak.x, ak.y};
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const double e = e0[h] + e1[h];
            row[h] = k < N ? -g[h] * e - Td[h] * akv[h] * iCv[h] : Td[h] * invT[h] - g[h] * (e + dE[h]) - Td[h] * dCv[h] * iCv[h];
        }
        if (act1) *reinterpret_cast<double2 *>(erow + (size_t)k * ld + cell) = make_double2(row[0], row[1]);
        else if (act0) erow[(size_t)k * ld + cell] = row[0];
    }
}
}  // namespace

// launcher (called by qss_api.cu); shared memory: (2 N + 4 NWY) rows of 32 doubles
cudaError_t qss_launch_energy(const double *D, int d_thermo, int N, int64_t ncells, int64_t ld, const double *C, const double *T, const double *wdot,
                              const double *jac, double *tdot, double *erow, cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    const size_t smem = (size_t)(2 * N + 4 * NWY) * 32 * sizeof(double);
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(qss_energy_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    const size_t smem2 = 2 * smem;
    if ((ld & 1) == 0 && smem2 <= 227 * 1024) {               // two cells per lane: 512-byte runs
        if (smem2 > 48 * 1024) {
            cudaError_t e = cudaFuncSetAttribute(qss_energy_kernel2, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem2);
            if (e != cudaSuccess) return e;
        }
        qss_energy_kernel2<<<(unsigned)((ncells + 63) / 64), dim3(32, NWY), smem2, stream>>>(D, d_thermo, N, ncells, ld, C, T, wdot, jac, tdot, erow);
        return cudaGetLastError();
    }
    const int64_t nblk = (ncells + 31) / 32;
    qss_energy_kernel<<<(unsigned)nblk, dim3(32, NWY), smem, stream>>>(D, d_thermo, N, ncells, ld, C, T, wdot, jac, tdot, erow);
    return cudaGetLastError();
}
