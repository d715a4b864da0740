// Mapping micro-benchmark (north_star subsystem 3: "a cell-to-thread vs cell-to-warp mapping, with warp shuffles for species-parallel
// reductions"): the species sums wdot_i = sum_j nu_ij Q_j (Eq. 3) of a slab of 32 cells, from given rates of progress Q
// [M][ld], in the two mappings, so that the choice made in the kernels (lane = cell for every row-wise phase) rests on a measurement
// and not on an instruction count alone.  Not on the product path: qss_eval_wdot / qss_eval_jac never call this.
//   mode 0  cell-to-thread: lane = cell; the 8 warps of a block split the species, each walks the species' reaction list (CSR by
//           species) over the slab staged in shared memory; no cross-lane traffic at all.
//   mode 1  cell-to-warp: a warp owns a cell, lane = reaction (j = lane + 32 t); every lane scatters its reactions' contributions
//           nu_ij Q_j into its own column of a [species][lane] array (CSR by reaction), then every species is reduced over the lanes
//           by a 5-step SHFL butterfly.
// Both stage the same slab of Q [M][33] through shared memory with coalesced loads and write wdot coalesced.
#include <cuda_runtime.h>
#include <stdint.h>

#include "qss_tables.h"

namespace {

constexpr int MB_WARPS = 8;

extern __shared__ double mb_smem[];

template <int MODE>
__global__ void __launch_bounds__(32 * MB_WARPS) qss_mapbench_kernel(const QssTab t, const int64_t ncells, const int64_t ld, const double *__restrict__ Q,
                                                                      double *__restrict__ wdot) {
    const int x = threadIdx.x, y = threadIdx.y, N = t.N, M = t.M;
    double *Qs = mb_smem;                                             // [M][33]
    double *cs = Qs + (size_t)M * 33;                                 // mode 1: [MB_WARPS][N][33] per-lane columns of contributions
    double *ws = cs + (MODE == 1 ? (size_t)MB_WARPS * N * 33 : 0);    // mode 1: [N][33] results of the slab
    const int32_t *I = t.I;
    for (int64_t slab = blockIdx.x; slab * 32 < ncells; slab += gridDim.x) {
        const int64_t cell = slab * 32 + x;
        const bool active = cell < ncells;
        const int64_t cc = active ? cell : ncells - 1;
        __syncthreads();
        for (int j = y; j < M; j += MB_WARPS) Qs[j * 33 + x] = Q[(size_t)j * ld + cc];
        __syncthreads();
        if (MODE == 0) {
            for (int i = y; i < N; i += MB_WARPS) {
                double s = 0.0;
                for (int e = __ldg(I + t.i_sp_ptr + i); e < __ldg(I + t.i_sp_ptr + i + 1); ++e)
                    s = fma((double)__ldg(I + t.i_sp_nu + e), Qs[__ldg(I + t.i_sp_reac + e) * 33 + x], s);
                if (active) wdot[(size_t)i * ld + cell] = s;
            }
        } else {
            double *col = cs + (size_t)y * N * 33 + x;                 // this lane's column
            for (int c = y; c < 32; c += MB_WARPS) {                   // this warp's cells of the slab
                for (int i = 0; i < N; ++i) col[i * 33] = 0.0;
                for (int j = x; j < M; j += 32) {                      // lane = reaction
                    const double qj = Qs[j * 33 + c];
                    for (int e = __ldg(I + t.i_net_ptr + j); e < __ldg(I + t.i_net_ptr + j + 1); ++e) {
                        const int sp = __ldg(I + t.i_net_sp + e);
                        if (sp < N) col[sp * 33] = fma((double)__ldg(I + t.i_net_nu + e), qj, col[sp * 33]);
                    }
                }
                __syncwarp();
                for (int i = 0; i < N; ++i) {                          // species-parallel reduction over the lanes: SHFL butterfly
                    double v = col[i * 33];
#pragma unroll
                    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                    if (x == 0) ws[i * 33 + c] = v;
                }
                __syncwarp();
            }
            __syncthreads();
            for (int i = y; i < N; i += MB_WARPS)
                if (active) wdot[(size_t)i * ld + cell] = ws[i * 33 + x];
        }
    }
}

}  // namespace

// returns cudaErrorInvalidValue when the slab does not fit the shared memory of one SM in the chosen mapping
cudaError_t qss_launch_mapbench(const QssTab &t, int mode, int64_t ncells, int64_t ld, const double *Q, double *wdot, int n_sm, cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    const size_t smem = ((size_t)t.M * 33 + (mode == 1 ? (size_t)MB_WARPS * t.N * 33 + (size_t)t.N * 33 : 0)) * sizeof(double);
    if (smem > 227 * 1024) return cudaErrorInvalidValue;
    const void *k = mode == 1 ? (const void *)qss_mapbench_kernel<1> : (const void *)qss_mapbench_kernel<0>;
    cudaError_t e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int per_sm = 1;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k, 32 * MB_WARPS, smem) != cudaSuccess || per_sm < 1) { cudaGetLastError(); per_sm = 1; }
    const int64_t nslab = (ncells + 31) / 32;
    const int64_t grid = nslab < (int64_t)n_sm * per_sm ? nslab : (int64_t)n_sm * per_sm;
    if (mode == 1) qss_mapbench_kernel<1><<<(unsigned)grid, dim3(32, MB_WARPS), smem, stream>>>(t, ncells, ld, Q, wdot);
    else qss_mapbench_kernel<0><<<(unsigned)grid, dim3(32, MB_WARPS), smem, stream>>>(t, ncells, ld, Q, wdot);
    return cudaGetLastError();
}
