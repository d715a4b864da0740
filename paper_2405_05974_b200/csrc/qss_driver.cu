// NEXT-4 (first half): the element-wise kernels of the 0-D constant-volume integrator qss_bdf1_advance
// (the interval "divided into substeps over which the chemical state is advanced"; L183-188: implicit scheme, Newton
// method with the chemical Jacobian; reading G21).  The heavy steps of a Newton iteration are the library's own calls
// (qss_eval_jac, qss_eval_energy, qss_newton_solve); what is left is the residual and the update of the state phi = (C, T):
//     b     = (phi^n - phi_m) + h f(phi_m)           f = (wdot, Tdot), rows 0..N-1 and N of `F`
//     phi_{m+1} = phi_m + delta,   C := max(C, 0)
// SoA, cell innermost: every access is a coalesced row; thread = (row, cell).
#include <cuda_runtime.h>
#include <stdint.h>

namespace {

__global__ void __launch_bounds__(256) qss_bdf1_residual_kernel(int N, int64_t ncells, int64_t ld, const double *__restrict__ C, const double *__restrict__ T,
                                                                 const double *__restrict__ phin, const double *__restrict__ F,
                                                                 const double *__restrict__ dt, double *__restrict__ b) {
    const int64_t c = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (c >= ncells) return;
    const double h = dt[c];
    for (int i = blockIdx.y; i <= N; i += gridDim.y) {
        const double phi = i < N ? C[(size_t)i * ld + c] : T[c];
        b[(size_t)i * ld + c] = (phin[(size_t)i * ld + c] - phi) + h * F[(size_t)i * ld + c];
    }
}

__global__ void __launch_bounds__(256) qss_bdf1_update_kernel(int N, int64_t ncells, int64_t ld, double *__restrict__ C, double *__restrict__ T,
                                                               const double *__restrict__ x) {
    const int64_t c = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (c >= ncells) return;
    for (int i = blockIdx.y; i <= N; i += gridDim.y) {
        const double d = x[(size_t)i * ld + c];
        if (i < N) C[(size_t)i * ld + c] = fmax(C[(size_t)i * ld + c] + d, 0.0);
        else T[c] = T[c] + d;
    }
}

}  // namespace

cudaError_t qss_launch_bdf1_residual(int N, int64_t ncells, int64_t ld, const double *C, const double *T, const double *phin, const double *F,
                                     const double *dt, double *b, cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    const dim3 grid((unsigned)((ncells + 255) / 256), (unsigned)(N + 1 < 8 ? N + 1 : 8));
    qss_bdf1_residual_kernel<<<grid, 256, 0, stream>>>(N, ncells, ld, C, T, phin, F, dt, b);
    return cudaGetLastError();
}

cudaError_t qss_launch_bdf1_update(int N, int64_t ncells, int64_t ld, double *C, double *T, const double *x, cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    const dim3 grid((unsigned)((ncells + 255) / 256), (unsigned)(N + 1 < 8 ? N + 1 : 8));
    qss_bdf1_update_kernel<<<grid, 256, 0, stream>>>(N, ncells, ld, C, T, x);
    return cudaGetLastError();
}

// ---- NEXT-3: the temperature column by finite differences ("computing the species' production rate twice at
// different temperatures"; L234: central differences, perturbation 1e-4; reading G22): the two element-wise steps around
// the two qss_eval_wdot calls.  dT = 1e-4 T, T+ = T + dT, T- = T - dT (each operation rounded on its own: no contraction, so
// that the oracle's numpy expression gives the same bits), column = (w+ - w-) / (T+ - T-).
namespace {

__global__ void __launch_bounds__(256) qss_fdT_perturb_kernel(int64_t ncells, const double *__restrict__ T, double *__restrict__ Tp, double *__restrict__ Tm) {
    const int64_t c = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (c >= ncells) return;
    const double t = T[c], d = __dmul_rn(1e-4, t);
    Tp[c] = __dadd_rn(t, d);
    Tm[c] = __dsub_rn(t, d);
}

__global__ void __launch_bounds__(256) qss_fdT_column_kernel(int N, int64_t ncells, int64_t ld, const double *__restrict__ wp, const double *__restrict__ wm,
                                                              const double *__restrict__ Tp, const double *__restrict__ Tm, double *__restrict__ jac) {
    const int64_t c = (int64_t)blockIdx.x * 256 + threadIdx.x;
    if (c >= ncells) return;
    const double h = __dsub_rn(Tp[c], Tm[c]);
    for (int i = blockIdx.y; i < N; i += gridDim.y)
        jac[((size_t)i * (N + 1) + N) * ld + c] = __ddiv_rn(__dsub_rn(wp[(size_t)i * ld + c], wm[(size_t)i * ld + c]), h);
}

}  // namespace

cudaError_t qss_launch_fdT_perturb(int64_t ncells, const double *T, double *Tp, double *Tm, cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    qss_fdT_perturb_kernel<<<(unsigned)((ncells + 255) / 256), 256, 0, stream>>>(ncells, T, Tp, Tm);
    return cudaGetLastError();
}

cudaError_t qss_launch_fdT_column(int N, int64_t ncells, int64_t ld, const double *wp, const double *wm, const double *Tp, const double *Tm, double *jac,
                                  cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    const dim3 grid((unsigned)((ncells + 255) / 256), (unsigned)(N < 8 ? N : 8));
    qss_fdT_column_kernel<<<grid, 256, 0, stream>>>(N, ncells, ld, wp, wm, Tp, Tm, jac);
    return cudaGetLastError();
}

// ---- NEXT-3: packed Jacobian (Table 4): row e of the output = row idx[e] of the dense SoA Jacobian (cells innermost, so a
// row is contiguous: the pack is a gather of whole rows, 16 bytes per thread)
namespace {
__global__ void __launch_bounds__(256) qss_jac_pack_kernel(int nnz, int64_t ncells, int64_t ld, const int32_t *__restrict__ idx, const double *__restrict__ jac,
                                                            double *__restrict__ out) {
    const int64_t c = ((int64_t)blockIdx.x * 256 + threadIdx.x) * 2;
    if (c >= ncells) return;
    for (int e = blockIdx.y; e < nnz; e += gridDim.y) {
        const double *src = jac + (size_t)idx[e] * ld + c;
        double *dst = out + (size_t)e * ld + c;
        if (c + 1 < ncells) *reinterpret_cast<double2 *>(dst) = *reinterpret_cast<const double2 *>(src);
        else dst[0] = src[0];
    }
}
}  // namespace

cudaError_t qss_launch_jac_pack(int nnz, int64_t ncells, int64_t ld, const int32_t *idx, const double *jac, double *out, cudaStream_t stream) {
    if (ncells == 0 || nnz == 0) return cudaSuccess;
    const dim3 grid((unsigned)((ncells + 511) / 512), (unsigned)(nnz < 64 ? nnz : 64));
    qss_jac_pack_kernel<<<grid, 256, 0, stream>>>(nnz, ncells, ld, idx, jac, out);
    return cudaGetLastError();
}

// ---- NEXT-2 ("optional AoS output layout for external batched solvers"; the Jacobian is handed
// to a batched dense solver that wants one contiguous matrix per cell): the SoA Jacobian [entry][cell] (and the energy row) as
// out[cell][rows][cols], row-major or column-major.  A tile of 64 output entries x 64 cells goes through shared memory: reads are
// coalesced over cells, writes over the entries of one cell.  Pure data movement: bit-exact.
namespace {
__global__ void __launch_bounds__(256) qss_jac_aos_kernel(int N, int rows, int64_t ncells, int64_t ld, const double *__restrict__ jac,
                                                           const double *__restrict__ erow, int col_major, double *__restrict__ out) {
    constexpr int TC = 64, TE = 64;                            // tile: 64 cells x 64 output entries (512-byte runs on both sides)
    __shared__ double tile[TE][TC + 1];
    const int cols = N + 1, E = rows * cols;
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    const int n_et = (E + TE - 1) / TE;                        // consecutive blocks: consecutive entry tiles of the same cells, so
    const int64_t c0 = (int64_t)(blockIdx.x / n_et) * TC;      // that their writes fill those cells' matrices front to back
    const int o0 = (int)(blockIdx.x % n_et) * TE;
    for (int u = w; u < TE; u += 8) {                          // output entry o0 + u of the cells c0 .. c0 + 63
        const int o = o0 + u;
        if (o >= E) break;
        const int i = col_major ? o % rows : o / cols, j = col_major ? o / rows : o % cols;
        const double *src = i < N ? jac + ((size_t)i * cols + j) * ld : erow + (size_t)j * ld;
#pragma unroll
        for (int h = 0; h < TC; h += 32) {
            const int64_t c = c0 + h + lane;
            if (c < ncells) tile[u][h + lane] = src[c];
        }
    }
    __syncthreads();
    for (int u = w; u < TC; u += 8) {                          // cell c0 + u, output entries o0 .. o0 + 63
        const int64_t c = c0 + u;
        if (c >= ncells) break;
#pragma unroll
        for (int h = 0; h < TE; h += 32) {
            const int o = o0 + h + lane;
            if (o < E) out[(size_t)c * E + o] = tile[h + lane][u];
        }
    }
}
}  // namespace

cudaError_t qss_launch_jac_aos(int N, int rows, int64_t ncells, int64_t ld, const double *jac, const double *erow, int col_major, double *out,
                               cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    const int E = rows * (N + 1);
    const int64_t nblocks = ((ncells + 63) / 64) * ((E + 63) / 64);
    if (nblocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    const dim3 grid((unsigned)nblocks);
    qss_jac_aos_kernel<<<grid, 256, 0, stream>>>(N, rows, ncells, ld, jac, erow, col_major, out);
    return cudaGetLastError();
}
