// Internal: run-time specialisation of kernel variant 1 (qss_jit.cpp -> qss_api.cu).
//
// The mechanism compiler (qss_compile.cpp) emits the Jacobian sweep's pass A for ONE mechanism as straight-line CUDA
// source (`QssCompiled::v1_gen`).  qss_jit_create compiles qss_kernel_v1.cu (its source is embedded in libqss.so by
// build.py) together with that source with NVRTC for the device's architecture and loads the result; the kernel it
// launches is the same slab-smem kernel with `qss_gen_pass_a` in place of the column-stream interpreter.
#ifndef QSS_JIT_H
#define QSS_JIT_H
#include <cuda_runtime.h>

#include <string>

#include "qss_v1.h"
#include "qss_v3.h"

struct QssJit;

// Returns NULL and sets `err` when NVRTC is not available or the compilation fails (the caller then keeps the
// interpreter kernel, which computes the same thing).  Compiled images are cached per process by source text.
QssJit *qss_jit_create(const std::string &gen_src, int cc_major, int cc_minor, std::string &err);
// Compilation only (no device needed): used by qss_mech_specialise_check.
bool qss_jit_compile_only(const std::string &gen_src, int cc_major, int cc_minor, size_t *image_bytes, std::string &err);
cudaError_t qss_jit_launch(const QssJit *j, const QssV1 &v, int nblocks, cudaStream_t stream);
void qss_jit_destroy(QssJit *j);

// Kernel variant 3 (qss_kernel_v3.cu + the generated qss_gen3.h): exists only as a run-time compiled program.  `jac`
// selects the Jacobian build (kernel qss_v3_jac) or the wdot-only build (qss_v3_wdot).  Compiled images are cached per
// process and on disk ($QSS_CACHE_DIR, default ~/.cache/libqss; QSS_CACHE=0 disables), keyed by a hash of every source.
QssJit *qss_jit3_create(const std::string &gen_src, bool jac, int cc_major, int cc_minor, std::string &err);
bool qss_jit3_compile_only(const std::string &gen_src, bool jac, int cc_major, int cc_minor, size_t *image_bytes, std::string &err);
cudaError_t qss_jit3_launch(const QssJit *j, const QssV3 &v, int nblocks, int nw, size_t smem_bytes, cudaStream_t stream);

// Newton solve (qss_newton_kernel.cu): compiled for one matrix order n (= N + 1 with the energy row, else N), nj = N + 1 columns
// of the Jacobian array, cpb cells (= warps) per block.  Same caches as above.
QssJit *qss_jit_newton_create(int n, int nj, bool has_e, int cpb, int cc_major, int cc_minor, std::string &err);
bool qss_jit_newton_compile_only(int n, int nj, bool has_e, int cpb, int cc_major, int cc_minor, size_t *image_bytes, std::string &err);
size_t qss_jit_newton_smem(int n, int cpb);
int qss_jit_newton_blocks_per_sm(const QssJit *j, int n, int cpb);
// One Newton iteration of qss_bdf1_advance behind the Jacobian kernel (qss_newton_step_kernel of the same image, n = N + 1 only): energy row,
// right-hand side, solve and update of (C, T) in place.  thermo: device NASA-7 table of the transported species ([N][24], qss_tables.h).
QssJit *qss_jit_newton_step_create(int n, int nj, int cpb, int cc_major, int cc_minor, std::string &err);
size_t qss_jit_newton_step_smem(int n, int cpb);
int qss_jit_newton_step_blocks_per_sm(const QssJit *j, int n, int cpb);
struct QssStepAdapt {           // adaptive form (qss_ignition_advance): per-cell time, step size, ignition time; tolerances (reading G23)
    int adapt;                  // 1: a Newton iteration of an attempt, 2: its last one (accept / reject)
    double *tcur, *dtio, *tign;
    const double *T0;
    double t_end, rtol, atolC, atolT, dT_ign, grow, shrink;
};
cudaError_t qss_jit_newton_step_launch(const QssJit *j, int n, int cpb, int max_blocks, const double *jac, const double *wdot, const double *phin,
                                       const double *dt, const double *thermo, double *C, double *T, int64_t ncells, int64_t ld, cudaStream_t stream,
                                       const QssStepAdapt *adapt = nullptr);
cudaError_t qss_jit_newton_launch(const QssJit *j, int n, int cpb, int max_blocks, const double *jac, const double *erow, const double *gamma,
                                  const double *b, double *x, int64_t ncells, int64_t ld, cudaStream_t stream);

#endif
