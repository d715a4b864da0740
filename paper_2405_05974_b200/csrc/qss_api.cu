// C-ABI of libqss (include/qss.h): handle management, argument checks, kernel selection and launch.
#include <cuda_runtime.h>

#include <cstdio>
#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>

#include "../../include/qss.h"
#include "qss_compile.h"
#include "qss_jit.h"
#include "qss_devtools.h"

size_t qss_slab_ws_doubles(const QssTab &t, bool jac, int nwarp);
cudaError_t qss_static_scratch_setup(int device);
size_t qss_static_scratch_capacity();
cudaError_t qss_launch_slab_static(const QssTab &t, int device, int64_t ncells, int64_t ld, const double *C, const double *T, double *wdot,
                                   double *cqss, int nblocks, int nwarp, cudaStream_t stream, int *blocks_out);
cudaError_t qss_launch_slab(const QssTab &t, bool jac, int64_t ncells, int64_t ld, const double *C, const double *T,
                            double *wdot, double *cqss, double *jacp, double *ws, int nblocks, int nwarp,
                            cudaStream_t stream);
cudaError_t qss_launch_dfma(int blocks, int iters, double *sink, cudaStream_t stream);
cudaError_t qss_launch_energy(const double *D, int d_thermo, int N, int64_t ncells, int64_t ld, const double *C, const double *T, const double *wdot,
                              const double *jac, double *tdot, double *erow, cudaStream_t stream);
size_t qss_v1_scratch_doubles(const QssV1 &v);
cudaError_t qss_v1_prepare();
cudaError_t qss_launch_v1(const QssV1 &v, bool jac, int nblocks, cudaStream_t stream);

struct qss_mech {
    QssCompiled c;
    int device = 0;
    int n_sm = 0;
    int32_t *dI = nullptr;
    double *dD = nullptr;
    int nwarp = 32;           // warps per block of the general slab kernel
    int blocks_per_sm = 1;    // general kernel: 1 x 32 warps per SM (64 registers): a quarter of the workspace slabs in flight; measured on cfg3 /
                              // cfg5: 108.8 / 306.9 ms against 122.6 / 324.7 ms with 4 blocks of 8 warps (193 ms with 2 x 8)
    int nblocks = 0;
    cudaStream_t copy_stream = nullptr;   // qss_eval_jac_host: device-to-host copies overlap the next chunk's kernel (created with the handle)
    mutable std::mutex host_mu;           // qss_eval_jac_host calls on one handle are serialised (they share copy_stream and the event)
    cudaEvent_t ev[2] = {nullptr, nullptr};
    long long *timing = nullptr;   // device counters when QSS_TIMING=1 (variant 1 only)
    int variant = 0;          // 0: general slab kernel (workspace in global memory); 1: slab-smem kernel (qss_kernel_v1.cu)
    QssJit *jit = nullptr;    // variant 1 with the Jacobian sweep's pass A specialised for this mechanism at run time (qss_jit.cpp)
    QssJit *jit3 = nullptr;   // variant 3 (qss_kernel_v3.cu, generated per mechanism): the Jacobian kernel
    QssJit *jit3w = nullptr;  //   and its wdot-only build
    double *dP3 = nullptr;    // variant 3: parameter blobs of the reaction-per-lane phases
    int32_t *iP3 = nullptr;
    int cc_major = 0, cc_minor = 0;
    bool static_scratch_ok = false;   // qss_static_scratch_setup succeeded on this device
    mutable int newton_blocks[2] = {0, 0};            //   persistent blocks of that kernel (SMs x resident blocks per SM)
    mutable QssJit *newton_step = nullptr;            // qss_bdf1_advance: the fused Newton step (energy row, right-hand side, solve, update), built on first use
    mutable int newton_step_blocks = 0;
    mutable bool newton_step_tried = false;
    mutable QssJit *newton[2] = {nullptr, nullptr};   // qss_newton_solve: [0] species block (n = N), [1] with the energy row (n = N + 1); built on first use
};

namespace {

thread_local std::string g_err;

int fail(int code, const std::string &msg) { g_err = msg; return code; }
int cuda_fail(cudaError_t e, const char *what) {
    g_err = std::string(what) + ": " + cudaGetErrorString(e);
    return QSS_E_CUDA;
}

struct DeviceGuard {
    int prev = -1; bool ok = false;
    explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && cudaSetDevice(dev) == cudaSuccess) ok = true; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int check_eval(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, const void *out,
               const void *ws, size_t ws_bytes, size_t need) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld");
    if (ncells == 0) return QSS_OK;
    if (!C || !T || !out) return fail(QSS_E_INVALID, "C, T or the output pointer is NULL");
    if (((uintptr_t)C | (uintptr_t)T | (uintptr_t)out) & 15) return fail(QSS_E_INVALID, "device pointers must be 16-byte aligned");
    if (!ws || ws_bytes < need) return fail(QSS_E_INVALID, "workspace is NULL or smaller than qss_mech_info reports");
    if ((uintptr_t)ws & 255) return fail(QSS_E_INVALID, "workspace must be 256-byte aligned");
    return QSS_OK;
}

}  // namespace

extern "C" const char *qss_last_error(void) { return g_err.c_str(); }

extern "C" int qss_mech_create(const qss_mech_desc_t *desc, int device, qss_mech_t **out) {
    if (!out) return fail(QSS_E_INVALID, "out is NULL");
    *out = nullptr;
    qss_mech *m = new (std::nothrow) qss_mech();
    if (!m) return fail(QSS_E_INVALID, "out of host memory");
    std::string err;
    int rc;
    try {
        rc = qss_compile(desc, m->c, err);
    } catch (const std::exception &e) {
        rc = QSS_E_INVALID; err = std::string("mechanism compiler: ") + e.what();
    }
    if (rc != QSS_OK) { delete m; return fail(rc, err); }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) { delete m; return e != cudaSuccess ? cuda_fail(e, "cudaGetDeviceCount") : fail(QSS_E_CUDA, "no CUDA device (libqss has no CPU fallback)"); }
    if (device < 0 || device >= ndev) { delete m; return fail(QSS_E_INVALID, "device index out of range"); }
    DeviceGuard guard(device);
    if (!guard.ok) { delete m; return fail(QSS_E_CUDA, "cudaSetDevice failed"); }
    m->device = device;
    cudaDeviceProp prop;
    if ((e = cudaGetDeviceProperties(&prop, device)) != cudaSuccess) { delete m; return cuda_fail(e, "cudaGetDeviceProperties"); }
    m->n_sm = prop.multiProcessorCount;
    m->cc_major = prop.major; m->cc_minor = prop.minor;
    m->static_scratch_ok = qss_static_scratch_setup(device) == cudaSuccess;      // address of the static workspace of qss_eval_wdot_static (no allocation)
    if (!m->static_scratch_ok) cudaGetLastError();
    if (const char *bps = qss_devenv("QSS_V0_BLOCKS_PER_SM")) m->blocks_per_sm = std::max(1, std::atoi(bps));   // tuning aid for the general kernel
    if (const char *nw = qss_devenv("QSS_V0_NWARP")) m->nwarp = std::max(1, std::min(32, std::atoi(nw)));
    m->nblocks = m->n_sm * m->blocks_per_sm;
    const size_t nI = m->c.I.size() ? m->c.I.size() : 1, nD = m->c.D.size() ? m->c.D.size() : 1;
    if ((e = cudaMalloc(&m->dI, nI * sizeof(int32_t))) != cudaSuccess) { delete m; return cuda_fail(e, "cudaMalloc(tables)"); }
    if ((e = cudaMalloc(&m->dD, nD * sizeof(double))) != cudaSuccess) { cudaFree(m->dI); delete m; return cuda_fail(e, "cudaMalloc(tables)"); }
    if (m->c.I.size()) e = cudaMemcpy(m->dI, m->c.I.data(), m->c.I.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
    if (e == cudaSuccess && m->c.D.size()) e = cudaMemcpy(m->dD, m->c.D.data(), m->c.D.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaFree(m->dI); cudaFree(m->dD); delete m; return cuda_fail(e, "cudaMemcpy(tables)"); }
    m->c.tab.I = m->dI; m->c.tab.D = m->dD;
    if ((e = cudaStreamCreateWithFlags(&m->copy_stream, cudaStreamNonBlocking)) == cudaSuccess) e = cudaEventCreateWithFlags(&m->ev[0], cudaEventDisableTiming);
    if (e != cudaSuccess) { qss_mech_destroy(m); return cuda_fail(e, "cudaStreamCreate / cudaEventCreate"); }
    const char *force = std::getenv("QSS_VARIANT");
    // kernel variant 3 (reaction-per-lane rate phases, everything generated per mechanism, NVRTC): the Jacobian kernel of
    // choice when the mechanism fits it.  QSS_VARIANT=3 makes its absence an error; QSS_VARIANT=0/1/2 keep the older kernels.
    const char *jit_env = std::getenv("QSS_JIT");            // QSS_JIT=0: no run-time compilation at all
    const bool want3 = (!force || force[0] == '3') && !(jit_env && jit_env[0] == '0');
    if (m->c.v3_ok && want3) {
        std::string jerr;
        m->jit3 = qss_jit3_create(m->c.v3.gen, true, prop.major, prop.minor, jerr);
        if (m->jit3) m->jit3w = qss_jit3_create(m->c.v3.gen, false, prop.major, prop.minor, jerr);
        if (m->jit3) {
            const QssV3Host &h = m->c.v3;
            if ((e = cudaMalloc(&m->dP3, h.dP.size() * sizeof(double))) == cudaSuccess) e = cudaMalloc(&m->iP3, h.iP.size() * sizeof(int32_t));
            if (e == cudaSuccess) e = cudaMemcpy(m->dP3, h.dP.data(), h.dP.size() * sizeof(double), cudaMemcpyHostToDevice);
            if (e == cudaSuccess) e = cudaMemcpy(m->iP3, h.iP.data(), h.iP.size() * sizeof(int32_t), cudaMemcpyHostToDevice);
            if (e != cudaSuccess) { qss_mech_destroy(m); return cuda_fail(e, "cudaMalloc/cudaMemcpy(variant 3 parameters)"); }
        } else if (qss_devenv("QSS_DEBUG") || (force && force[0] == '3')) {
            std::fprintf(stderr, "[qss] kernel variant 3 unavailable: %s\n", jerr.c_str());
        }
        if (!m->jit3 && force && force[0] == '3') { qss_mech_destroy(m); return fail(QSS_E_CUDA, "QSS_VARIANT=3: " + jerr); }
    } else if (force && force[0] == '3') {
        const std::string w = m->c.v3_why;
        qss_mech_destroy(m);
        return fail(QSS_E_UNSUPPORTED, "QSS_VARIANT=3: kernel variant 3 does not apply: " + w);
    }
    if (m->jit3 && qss_devenv("QSS_TIMING") && cudaMalloc(&m->timing, 32 * sizeof(long long)) == cudaSuccess) cudaMemset(m->timing, 0, 32 * sizeof(long long));
    // kernel selection: variant 1 when the mechanism fits it (QSS_VARIANT=0 in the environment forces the general kernel)
    if (m->c.v1_ok && !(force && force[0] == '0')) {   // (also the wdot-only kernel next to variant 3)
        if ((e = qss_v1_prepare()) != cudaSuccess) { cudaFree(m->dI); cudaFree(m->dD); delete m; return cuda_fail(e, "cudaFuncSetAttribute(variant 1)"); }
        m->variant = 1;
        m->nblocks = m->n_sm;
        m->c.v1.gI = m->dI; m->c.v1.gD = m->dD;
        if (!m->timing && qss_devenv("QSS_TIMING") && cudaMalloc(&m->timing, 16 * sizeof(long long)) == cudaSuccess) cudaMemset(m->timing, 0, 16 * sizeof(long long));
        // Jacobian kernel specialised for this mechanism (NVRTC); QSS_JIT=0 keeps the table interpreter, which is also what
        // runs when NVRTC is missing or the compilation fails (qss_mech_info.kernel_variant_jac tells which: 2 = specialised)
        if (!m->jit3 && !(jit_env && jit_env[0] == '0') && !m->c.v1_gen.empty()) {
            std::string jerr;
            m->jit = qss_jit_create(m->c.v1_gen, prop.major, prop.minor, jerr);
            if (!m->jit && (qss_devenv("QSS_DEBUG") || (jit_env && jit_env[0] == '2'))) std::fprintf(stderr, "[qss] run-time specialisation unavailable: %s\n", jerr.c_str());
            if (!m->jit && jit_env && jit_env[0] == '2') { cudaFree(m->dI); cudaFree(m->dD); cudaFree(m->timing); delete m; return fail(QSS_E_CUDA, "QSS_JIT=2: " + jerr); }
        }
    }
    *out = m;
    return QSS_OK;
}

extern "C" int qss_mech_validate(const qss_mech_desc_t *desc, int32_t *n_groups, int32_t *order, int32_t *group_of) {
    QssCompiled c;
    std::string err;
    int rc;
    try {
        rc = qss_compile(desc, c, err);
    } catch (const std::exception &e) {
        rc = QSS_E_INVALID; err = std::string("mechanism compiler: ") + e.what();
    }
    if (rc != QSS_OK) return fail(rc, err);
    if (n_groups) *n_groups = c.tab.n_groups;
    for (int i = 0; i < c.tab.Nq; ++i) { if (order) order[i] = c.order[i]; if (group_of) group_of[i] = c.group_of[i]; }
    return QSS_OK;
}

extern "C" int qss_mech_specialise_check(const qss_mech_desc_t *desc, int cc_major, int cc_minor, size_t *image_bytes) {
    QssCompiled c;
    std::string err;
    int rc;
    try {
        rc = qss_compile(desc, c, err);
    } catch (const std::exception &e) {
        rc = QSS_E_INVALID; err = std::string("mechanism compiler: ") + e.what();
    }
    if (rc != QSS_OK) return fail(rc, err);
    if (c.v3_ok) {
        if (!qss_jit3_compile_only(c.v3.gen, true, cc_major, cc_minor, image_bytes, err)) return fail(QSS_E_CUDA, err);
        return QSS_OK;
    }
    if (!c.v1_ok) return fail(QSS_E_UNSUPPORTED, "kernel variants 1-3 do not apply: " + c.v1_why + "; " + c.v3_why);
    if (!qss_jit_compile_only(c.v1_gen, cc_major, cc_minor, image_bytes, err)) return fail(QSS_E_CUDA, err);
    return QSS_OK;
}

extern "C" int qss_mech_destroy(qss_mech_t *m) {
    if (!m) return QSS_OK;
    DeviceGuard guard(m->device);
    if (m->timing) {
        long long t[32] = {0};
        static const char *name1[15] = {"P0 stage", "P1 thermo", "P2 Arrhenius+wait", "P3+P7 gather", "P4 closure", "P5 net rates", "P6 sums", "A: barrier wait", "B: barrier wait",
                                         "B: tile", "B: stores", "A: init", "A: stream", "A: solve", "P2 third-body/fall-off"};
        static const char *name3[15] = {"P0 inputs", "P2 rate tasks", "P2 barrier wait", "P3 gather", "P4 closure", "P5 net tasks", "P6 sums", "kappa_d reload", "P8 columns",
                                         "end barrier wait", "P2c kappa", "", "", "", ""};
        const char **name = m->jit3 ? name3 : name1;
        if (cudaMemcpy(t, m->timing, (m->jit3 ? 32 : 16) * sizeof(long long), cudaMemcpyDeviceToHost) == cudaSuccess) {
            if (m->jit3) { std::fprintf(stderr, "[qss timing] rate phase per warp (cycles/1e6):"); for (int i = 16; i < 32; ++i) std::fprintf(stderr, " %.2f", (double)t[i] * 1e-6); std::fprintf(stderr, "\n"); }
            long long tot = 0;
            for (int i = 0; i < 15; ++i) tot += t[i];
            for (int i = 0; i < 15 && tot > 0; ++i) std::fprintf(stderr, "[qss timing] %-14s %6.2f %%\n", name[i], 100.0 * (double)t[i] / (double)tot);
        }
        cudaFree(m->timing);
    }
    cudaDeviceSynchronize();          // no kernel of this handle may still run when its module is unloaded
    qss_jit_destroy(m->jit);
    qss_jit_destroy(m->jit3);
    qss_jit_destroy(m->jit3w);
    qss_jit_destroy(m->newton_step);
    qss_jit_destroy(m->newton[0]);
    qss_jit_destroy(m->newton[1]);
    cudaFree(m->dP3); cudaFree(m->iP3);
    if (m->copy_stream) cudaStreamDestroy(m->copy_stream);
    if (m->ev[0]) cudaEventDestroy(m->ev[0]);
    cudaFree(m->dI); cudaFree(m->dD);
    delete m;
    return QSS_OK;
}

static size_t ws_bytes(const qss_mech_t *m, bool jac) {
    if (jac && m->jit3) return (size_t)m->c.v3.scratch_rows * 32 * sizeof(double) * (size_t)m->n_sm;
    if (m->variant == 1) return qss_v1_scratch_doubles(m->c.v1) * sizeof(double) * (size_t)m->nblocks;
    return qss_slab_ws_doubles(m->c.tab, jac, m->nwarp) * sizeof(double) * (size_t)m->nblocks;
}

extern "C" int qss_mech_info(const qss_mech_t *m, qss_mech_info_t *o) {
    if (!m || !o) return fail(QSS_E_INVALID, "NULL argument");
    std::memset(o, 0, sizeof *o);
    const QssTab &t = m->c.tab;
    o->n_nqss = t.N; o->n_qss = t.Nq; o->n_reac = t.M;
    o->n_groups = t.n_groups; o->max_group = t.max_group; o->n_levels = t.n_levels;
    for (int g = 0; g < t.n_groups && g < 64; ++g) o->group_size[g] = m->c.group_size[g];
    o->slots_wdot = m->c.slots_wdot; o->slots_jac = m->c.slots_jac;
    o->bytes_wdot = m->c.bytes_wdot; o->bytes_jac = m->c.bytes_jac;
    o->workspace_bytes_wdot = ws_bytes(m, false);
    o->workspace_bytes_jac = ws_bytes(m, true);
    o->kernel_variant_wdot = m->jit3w ? 3 : m->variant; o->kernel_variant_jac = m->jit3 ? 3 : (m->jit ? 2 : m->variant);
    return QSS_OK;
}

extern "C" int qss_mech_qss_order(const qss_mech_t *m, int32_t *order, int32_t *group_of) {
    if (!m || !order || !group_of) return fail(QSS_E_INVALID, "NULL argument");
    for (int i = 0; i < m->c.tab.Nq; ++i) { order[i] = m->c.order[i]; group_of[i] = m->c.group_of[i]; }
    return QSS_OK;
}

extern "C" int qss_eval_wdot(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T,
                             double *wdot, double *cqss, void *workspace, size_t workspace_bytes, void *stream) {
    int rc = check_eval(m, ncells, ld, C, T, wdot, workspace, workspace_bytes, m ? ws_bytes(m, false) : 0);
    if (rc != QSS_OK || ncells == 0) return rc;
    DeviceGuard guard(m->device);          // the handle's tables and kernels live on its device; `stream` must belong to it
    cudaError_t e;
    if (m->jit3w) {
        QssV3 v;
        v.C = C; v.T = T; v.wdot = wdot; v.cqss = cqss; v.jac = nullptr; v.scratch = (double *)workspace;
        v.ncells = ncells; v.ld = ld; v.scratch_stride = 0; v.dP = m->dP3; v.iP = m->iP3; v.timing = nullptr; v.mode = 0;
        e = qss_jit3_launch(m->jit3w, v, m->n_sm, m->c.v3.nw, (size_t)m->c.v3.smem_bytes, (cudaStream_t)stream);
    } else if (m->variant == 1) {
        QssV1 v = m->c.v1;
        v.C = C; v.T = T; v.wdot = wdot; v.cqss = cqss; v.jac = nullptr; v.scratch = (double *)workspace; v.timing = nullptr;
        v.ncells = ncells; v.ld = ld; v.scratch_stride = (int64_t)qss_v1_scratch_doubles(v);
        e = qss_launch_v1(v, false, m->nblocks, (cudaStream_t)stream);
    } else {
        e = qss_launch_slab(m->c.tab, false, ncells, ld, C, T, wdot, cqss, nullptr, (double *)workspace, m->nblocks, m->nwarp,
                            (cudaStream_t)stream);
    }
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_eval_wdot launch");
}

// ---- NEXT-2: the Newton solve (qss_newton_kernel.cu, compiled for this mechanism's matrix order on first use) ------------------
static const int QSS_NEWTON_MAX_N = 40;     // two register rows of n + 1 doubles per lane: 164 registers at n = 40
static int newton_cpb() {                  // cells (= warps) per block
    if (const char *e = qss_devenv("QSS_NEWTON_CPB")) return std::atoi(e);      // (development builds)
    return 8;                                // 64-byte segments per matrix entry; one block of 8 warps per SM (234 registers)
}
#define QSS_NEWTON_CPB newton_cpb()

extern "C" int qss_newton_specialise_check(int n_species, int with_energy, int cc_major, int cc_minor, size_t *image_bytes) {
    const int n = n_species + (with_energy ? 1 : 0);
    if (n_species < 1 || n > QSS_NEWTON_MAX_N) return fail(QSS_E_UNSUPPORTED, "qss_newton_solve: matrix order outside 1..40");
    std::string err;
    if (!qss_jit_newton_compile_only(n, n_species + 1, with_energy != 0, QSS_NEWTON_CPB, cc_major, cc_minor, image_bytes, err)) return fail(QSS_E_CUDA, err);
    return QSS_OK;
}

extern "C" int qss_newton_solve(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *jac, const double *erow, const double *gamma,
                                const double *b, double *x, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld");
    const int N = m->c.tab.N, n = N + (erow ? 1 : 0);
    if (n > QSS_NEWTON_MAX_N) return fail(QSS_E_UNSUPPORTED, "qss_newton_solve: matrix order above 40 (the matrix does not fit a warp's registers)");
    if (ncells == 0) return QSS_OK;
    if (!jac || !gamma || !b || !x) return fail(QSS_E_INVALID, "NULL device pointer");
    if (((uintptr_t)jac | (uintptr_t)erow | (uintptr_t)gamma | (uintptr_t)b | (uintptr_t)x) & 7) return fail(QSS_E_INVALID, "device pointers must be 8-byte aligned");
    DeviceGuard guard(m->device);
    const int which = erow ? 1 : 0;
    {
        std::lock_guard<std::mutex> lock(m->host_mu);
        if (!m->newton[which]) {
            std::string err;
            m->newton[which] = qss_jit_newton_create(n, N + 1, erow != nullptr, QSS_NEWTON_CPB, m->cc_major, m->cc_minor, err);
            if (!m->newton[which]) return fail(QSS_E_CUDA, "qss_newton_solve: run-time compilation failed (there is no other path): " + err);
            m->newton_blocks[which] = m->n_sm * qss_jit_newton_blocks_per_sm(m->newton[which], n, QSS_NEWTON_CPB);
        }
    }
    cudaError_t e = qss_jit_newton_launch(m->newton[which], n, QSS_NEWTON_CPB, m->newton_blocks[which], jac, erow, gamma, b, x, ncells, ld, (cudaStream_t)stream);
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_newton_solve launch");
}

static int eval_jac_mode(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac, double *wdot, int mode,
                         void *workspace, size_t workspace_bytes, void *stream);

extern "C" int qss_eval_jac(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T,
                            double *jac, double *wdot, void *workspace, size_t workspace_bytes, void *stream) {
    return eval_jac_mode(m, ncells, ld, C, T, jac, wdot, 0, workspace, workspace_bytes, stream);
}

extern "C" int qss_eval_jac_approx(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac,
                                   int mode, void *workspace, size_t workspace_bytes, void *stream) {
    if (mode < 0 || mode > 2) return fail(QSS_E_INVALID, "mode must be QSS_JAC_EXACT, QSS_JAC_CONST_QSS or QSS_JAC_ZERO_QSS");
    if (m && mode != 0 && !m->jit3) return fail(QSS_E_UNSUPPORTED, "the simplified Jacobians need kernel variant 3 (qss_mech_info.kernel_variant_jac)");
    return eval_jac_mode(m, ncells, ld, C, T, jac, nullptr, mode, workspace, workspace_bytes, stream);
}

extern "C" int qss_eval_energy(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, const double *wdot,
                               const double *jac, double *tdot, double *erow, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld");
    if (ncells == 0) return QSS_OK;
    if (!C || !T || !wdot || !jac || !tdot || !erow) return fail(QSS_E_INVALID, "NULL device pointer");
    if (((uintptr_t)C | (uintptr_t)T | (uintptr_t)wdot | (uintptr_t)jac | (uintptr_t)tdot | (uintptr_t)erow) & 15) return fail(QSS_E_INVALID, "device pointers must be 16-byte aligned");
    if (m->c.tab.N > 430) return fail(QSS_E_UNSUPPORTED, "qss_eval_energy: more than 430 transported species");
    DeviceGuard guard(m->device);
    cudaError_t e = qss_launch_energy(m->dD, m->c.tab.d_thermo, m->c.tab.N, ncells, ld, C, T, wdot, jac, tdot, erow, (cudaStream_t)stream);
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_eval_energy launch");
}

static int eval_jac_mode(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac, double *wdot, int mode,
                         void *workspace, size_t workspace_bytes, void *stream) {
    int rc = check_eval(m, ncells, ld, C, T, jac, workspace, workspace_bytes, m ? ws_bytes(m, true) : 0);
    if (rc != QSS_OK || ncells == 0) return rc;
    DeviceGuard guard(m->device);
    cudaError_t e;
    if (m->jit3) {
        QssV3 v;
        v.C = C; v.T = T; v.wdot = wdot; v.cqss = nullptr; v.jac = jac; v.scratch = (double *)workspace;
        v.ncells = ncells; v.ld = ld; v.scratch_stride = (int64_t)m->c.v3.scratch_rows * 32;
        v.dP = m->dP3; v.iP = m->iP3; v.timing = m->timing; v.mode = mode;
        int nb3 = m->n_sm;
        if (const char *bx = qss_devenv("QSS3_BLOCKS")) nb3 = std::max(1, std::min(m->n_sm, std::atoi(bx)));      // (development builds: fewer SMs)
        e = qss_jit3_launch(m->jit3, v, nb3, m->c.v3.nw, (size_t)m->c.v3.smem_bytes, (cudaStream_t)stream);
    } else if (m->variant == 1) {
        QssV1 v = m->c.v1;
        v.C = C; v.T = T; v.wdot = wdot; v.cqss = nullptr; v.jac = jac; v.scratch = (double *)workspace; v.timing = m->timing;
        v.ncells = ncells; v.ld = ld; v.scratch_stride = (int64_t)qss_v1_scratch_doubles(v);
        e = m->jit ? qss_jit_launch(m->jit, v, m->nblocks, (cudaStream_t)stream) : qss_launch_v1(v, true, m->nblocks, (cudaStream_t)stream);
    } else {
        e = qss_launch_slab(m->c.tab, true, ncells, ld, C, T, wdot, nullptr, jac, (double *)workspace, m->nblocks, m->nwarp,
                            (cudaStream_t)stream);
    }
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_eval_jac launch");
}

static size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }


// ---- allocation-free entry point: wdot with the workspace in a static device array (qss_kernels.cu) ------------------------------
extern "C" int qss_eval_wdot_static(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, double *wdot,
                                    double *cqss, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld");
    if (ncells == 0) return QSS_OK;
    if (!C || !T || !wdot) return fail(QSS_E_INVALID, "C, T or the output pointer is NULL");
    if (((uintptr_t)C | (uintptr_t)T | (uintptr_t)wdot | (uintptr_t)cqss) & 15) return fail(QSS_E_INVALID, "device pointers must be 16-byte aligned");
    if (!m->static_scratch_ok) return fail(QSS_E_CUDA, "qss_eval_wdot_static: the address of the static workspace could not be taken at qss_mech_create");
    const size_t per_block = qss_slab_ws_doubles(m->c.tab, false, m->nwarp) * sizeof(double);
    if (per_block > qss_static_scratch_capacity()) {
        char msg[200];
        std::snprintf(msg, sizeof msg, "qss_eval_wdot_static: one block of this mechanism needs %zu bytes of workspace, the static array holds %zu (QSS_STATIC_SCRATCH_BYTES); use qss_eval_wdot",
                      per_block, qss_static_scratch_capacity());
        return fail(QSS_E_UNSUPPORTED, msg);
    }
    DeviceGuard guard(m->device);
    cudaError_t e = qss_launch_slab_static(m->c.tab, m->device, ncells, ld, C, T, wdot, cqss, m->nblocks, m->nwarp, (cudaStream_t)stream, nullptr);
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_eval_wdot_static launch");
}

// ---- mapping micro-benchmark (qss_mapbench.cu): species sums in the cell-to-thread and in the cell-to-warp mapping ------------------
cudaError_t qss_launch_mapbench(const QssTab &t, int mode, int64_t ncells, int64_t ld, const double *Q, double *wdot, int n_sm, cudaStream_t stream);

extern "C" int qss_bench_species_sums(const qss_mech_t *m, int mode, int64_t ncells, int64_t ld, const double *Q, double *wdot, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (mode < 0 || mode > 1 || ncells < 0 || ld < ncells) return fail(QSS_E_INVALID, "need mode 0 or 1 and 0 <= ncells <= ld");
    if (ncells == 0) return QSS_OK;
    if (!Q || !wdot) return fail(QSS_E_INVALID, "NULL device pointer");
    DeviceGuard guard(m->device);
    cudaError_t e = qss_launch_mapbench(m->c.tab, mode, ncells, ld, Q, wdot, m->n_sm, (cudaStream_t)stream);
    if (e == cudaErrorInvalidValue) { cudaGetLastError(); return fail(QSS_E_UNSUPPORTED, "qss_bench_species_sums: the slab of this mechanism does not fit the shared memory of one SM in this mapping"); }
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_bench_species_sums launch");
}

// ---- NEXT-1 in one call: the full (N+1) x (N+1) Jacobian and both right-hand sides (the two launches in sequence; a version with
// the energy row formed inside the sweep of kernel variant 3 was built and measured at 14.0 ms against 13.6 ms: DESIGN.md section 6)
extern "C" int qss_eval_jac_full(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac, double *wdot,
                                 double *tdot, double *erow, void *workspace, size_t workspace_bytes, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (!wdot || !tdot || !erow) return fail(QSS_E_INVALID, "qss_eval_jac_full: wdot, tdot and erow are required");
    int rc = eval_jac_mode(m, ncells, ld, C, T, jac, wdot, 0, workspace, workspace_bytes, stream);
    if (rc != QSS_OK || ncells == 0) return rc;
    return qss_eval_energy(m, ncells, ld, C, T, wdot, jac, tdot, erow, stream);
}

// ---- NEXT-3: structural sparsity pattern (qss_pattern.cpp) and packed output (qss_driver.cu) -----------------------------------
int qss_pattern_build(const qss_mech_desc_t *d, int mode, uint8_t *pat);
cudaError_t qss_launch_jac_pack(int nnz, int64_t ncells, int64_t ld, const int32_t *idx, const double *jac, double *out, cudaStream_t stream);

extern "C" int qss_mech_jac_pattern(const qss_mech_desc_t *desc, int mode, uint8_t *pattern) {
    if (!desc || !pattern) return fail(QSS_E_INVALID, "NULL argument");
    if (mode < 0 || mode > 2) return fail(QSS_E_INVALID, "mode must be QSS_JAC_EXACT, QSS_JAC_CONST_QSS or QSS_JAC_ZERO_QSS");
    QssCompiled c;
    std::string err;
    int rc;
    try {
        rc = qss_compile(desc, c, err);                                 // (validation: the pattern is defined for mechanisms the library accepts)
    } catch (const std::exception &e) {
        rc = QSS_E_INVALID; err = std::string("mechanism compiler: ") + e.what();
    }
    if (rc != QSS_OK) return fail(rc, err);
    return qss_pattern_build(desc, mode, pattern);
}

extern "C" int qss_jac_pack(const qss_mech_t *m, int64_t ncells, int64_t ld, int32_t nnz, const int32_t *idx, const double *jac, double *packed, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells || nnz < 0 || (ld & 1)) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld, ld even, nnz >= 0");
    if (ncells == 0 || nnz == 0) return QSS_OK;
    if (!idx || !jac || !packed) return fail(QSS_E_INVALID, "NULL device pointer");
    if (((uintptr_t)jac | (uintptr_t)packed) & 15) return fail(QSS_E_INVALID, "device pointers must be 16-byte aligned");
    DeviceGuard guard(m->device);
    cudaError_t e = qss_launch_jac_pack(nnz, ncells, ld, idx, jac, packed, (cudaStream_t)stream);
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_jac_pack launch");
}

// ---- NEXT-2: AoS export for external batched solvers (kernel in qss_driver.cu) --------------------------------------------------------
cudaError_t qss_launch_jac_aos(int N, int rows, int64_t ncells, int64_t ld, const double *jac, const double *erow, int col_major, double *out,
                               cudaStream_t stream);

extern "C" int qss_jac_to_aos(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *jac, const double *erow, int col_major, double *out,
                              void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld");
    if (ncells == 0) return QSS_OK;
    if (!jac || !out) return fail(QSS_E_INVALID, "NULL device pointer");
    DeviceGuard guard(m->device);
    const int N = m->c.tab.N;
    cudaError_t e = qss_launch_jac_aos(N, erow ? N + 1 : N, ncells, ld, jac, erow, col_major != 0, out, (cudaStream_t)stream);
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_jac_to_aos launch");
}

// ---- NEXT-3: temperature column by finite differences (reading G22; kernels in qss_driver.cu) ---------------
cudaError_t qss_launch_fdT_perturb(int64_t ncells, const double *T, double *Tp, double *Tm, cudaStream_t stream);
cudaError_t qss_launch_fdT_column(int N, int64_t ncells, int64_t ld, const double *wp, const double *wm, const double *Tp, const double *Tm, double *jac,
                                  cudaStream_t stream);

extern "C" size_t qss_jac_fdt_workspace_bytes(const qss_mech_t *m, int64_t ld) {
    if (!m || ld < 0) return 0;
    const size_t row = align256((size_t)ld * sizeof(double));
    return std::max(align256(ws_bytes(m, true)), align256(ws_bytes(m, false))) + row * (2 + 2 * (size_t)m->c.tab.N) + 256;
}

extern "C" int qss_eval_jac_fdt(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *C, const double *T, double *jac, double *wdot,
                                void *workspace, size_t workspace_bytes, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ld & 1) return fail(QSS_E_INVALID, "qss_eval_jac_fdt: ld must be even (16-byte aligned rows)");
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < qss_jac_fdt_workspace_bytes(m, ld)) return fail(QSS_E_INVALID, "workspace is NULL, misaligned or smaller than qss_jac_fdt_workspace_bytes");
    const size_t wsk = std::max(align256(ws_bytes(m, true)), align256(ws_bytes(m, false)));
    int rc = eval_jac_mode(m, ncells, ld, C, T, jac, wdot, 0, workspace, wsk, stream);          // species columns (and the analytic T column, overwritten below)
    if (rc != QSS_OK || ncells == 0) return rc;
    DeviceGuard guard(m->device);
    const int N = m->c.tab.N;
    char *p = (char *)workspace + wsk;
    auto take = [&](size_t rows) { double *q = (double *)p; p += align256(rows * (size_t)ld * sizeof(double)); return q; };
    double *Tp = take(1), *Tm = take(1), *wp = take(N), *wm = take(N);
    cudaError_t e = qss_launch_fdT_perturb(ncells, T, Tp, Tm, (cudaStream_t)stream);
    if (e != cudaSuccess) return cuda_fail(e, "qss_eval_jac_fdt: perturbation kernel");
    rc = qss_eval_wdot(m, ncells, ld, C, Tp, wp, nullptr, workspace, wsk, stream);
    if (rc == QSS_OK) rc = qss_eval_wdot(m, ncells, ld, C, Tm, wm, nullptr, workspace, wsk, stream);
    if (rc != QSS_OK) return rc;
    e = qss_launch_fdT_column(N, ncells, ld, wp, wm, Tp, Tm, jac, (cudaStream_t)stream);
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_eval_jac_fdt: column kernel");
}

// ---- NEXT-4: 0-D constant-volume integrator (backward-Euler substeps, full Newton iterations; qss_driver.cu) --------------------
cudaError_t qss_launch_bdf1_residual(int N, int64_t ncells, int64_t ld, const double *C, const double *T, const double *phin, const double *F,
                                     const double *dt, double *b, cudaStream_t stream);
cudaError_t qss_launch_bdf1_update(int N, int64_t ncells, int64_t ld, double *C, double *T, const double *x, cudaStream_t stream);

extern "C" size_t qss_bdf1_workspace_bytes(const qss_mech_t *m, int64_t ld) {
    if (!m || ld < 0) return 0;
    const size_t N = (size_t)m->c.tab.N, row = align256((size_t)ld * sizeof(double));
    // jac N (N+1) rows | F N+1 | erow N+1 | phi^n N+1 | b (and x in place) N+1 | workspace of qss_eval_jac
    return row * (N * (N + 1) + 4 * (N + 1)) + align256(ws_bytes(m, true)) + 256;
}

extern "C" int qss_bdf1_advance(const qss_mech_t *m, int64_t ncells, int64_t ld, double *C, double *T, const double *dt, int nsub, int newton_iters,
                                void *workspace, size_t workspace_bytes, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells || nsub < 0 || newton_iters < 1) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld, nsub >= 0, newton_iters >= 1");
    const int N = m->c.tab.N;
    if (N + 1 > QSS_NEWTON_MAX_N) return fail(QSS_E_UNSUPPORTED, "qss_bdf1_advance: more than 39 transported species (limit of qss_newton_solve)");
    if (ncells == 0 || nsub == 0) return QSS_OK;
    if (!C || !T || !dt) return fail(QSS_E_INVALID, "NULL device pointer");
    if (ld & 1) return fail(QSS_E_INVALID, "qss_bdf1_advance: ld must be even (16-byte aligned rows)");
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < qss_bdf1_workspace_bytes(m, ld)) return fail(QSS_E_INVALID, "workspace is NULL, misaligned or smaller than qss_bdf1_workspace_bytes");
    DeviceGuard guard(m->device);
    cudaStream_t st = (cudaStream_t)stream;
    // the rows of one array are contiguous with stride ld (the layout every call of the library uses)
    const size_t nrow = (size_t)ld;
    char *p = (char *)workspace;
    auto take = [&](size_t rows) { double *q = (double *)p; p += align256(rows * nrow * sizeof(double)); return q; };
    double *jac = take((size_t)N * (N + 1)), *F = take(N + 1), *erow = take(N + 1), *phin = take(N + 1), *b = take(N + 1);
    void *ws = (void *)(((uintptr_t)p + 255) & ~(uintptr_t)255);
    const size_t wsb = ws_bytes(m, true);
    QssJit *step = nullptr;
    {
        std::lock_guard<std::mutex> lock(m->host_mu);
        if (!m->newton_step_tried) {
            m->newton_step_tried = true;
            std::string jerr;
            if (!qss_devenv("QSS_BDF1_UNFUSED")) m->newton_step = qss_jit_newton_step_create(N + 1, N + 1, QSS_NEWTON_CPB, m->cc_major, m->cc_minor, jerr);
            if (m->newton_step) m->newton_step_blocks = m->n_sm * qss_jit_newton_step_blocks_per_sm(m->newton_step, N + 1, QSS_NEWTON_CPB);
            else if (qss_devenv("QSS_DEBUG")) std::fprintf(stderr, "[qss] fused Newton step unavailable: %s\n", jerr.c_str());
        }
        step = m->newton_step;      // NULL: the five-launch sequence below (same arithmetic up to the summation order of the energy row)
    }
    for (int s = 0; s < nsub; ++s) {
        cudaError_t e = cudaMemcpyAsync(phin, C, (size_t)N * nrow * sizeof(double), cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(phin + (size_t)N * nrow, T, nrow * sizeof(double), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return cuda_fail(e, "qss_bdf1_advance: saving the state");
        for (int it = 0; it < newton_iters; ++it) {
            if (step) {      // two launches per iteration: the Jacobian kernel (J, wdot), then energy row + right-hand side + solve + update in one kernel
                int rc = eval_jac_mode(m, ncells, ld, C, T, jac, F, 0, ws, wsb, stream);
                if (rc != QSS_OK) return rc;
                e = qss_jit_newton_step_launch(step, N + 1, QSS_NEWTON_CPB, m->newton_step_blocks, jac, F, phin, dt, m->dD + m->c.tab.d_thermo, C, T, ncells, ld, st);
                if (e != cudaSuccess) return cuda_fail(e, "qss_bdf1_advance: fused Newton step");
                continue;
            }
            int rc = qss_eval_jac_full(m, ncells, ld, C, T, jac, F, F + (size_t)N * nrow, erow, ws, wsb, stream);      // J, wdot -> F[0..N-1], Tdot -> F[N], energy row
            if (rc != QSS_OK) return rc;
            e = qss_launch_bdf1_residual(N, ncells, ld, C, T, phin, F, dt, b, st);
            if (e != cudaSuccess) return cuda_fail(e, "qss_bdf1_advance: residual kernel");
            rc = qss_newton_solve(m, ncells, ld, jac, erow, dt, b, b, stream);                             // gamma = h: (I - h J) delta = b, in place
            if (rc != QSS_OK) return rc;
            e = qss_launch_bdf1_update(N, ncells, ld, C, T, b, st);
            if (e != cudaSuccess) return cuda_fail(e, "qss_bdf1_advance: update kernel");
        }
    }
    return QSS_OK;
}


// ---- NEXT-4: adaptive form with ignition time (reading G23) ---------------------------------------------------------------
extern "C" int qss_ignition_advance(const qss_mech_t *m, int64_t ncells, int64_t ld, double *C, double *T, double *dt, double *t, double t_end,
                                    double *t_ign, const double *T0, double dT_ign, int n_attempts, int newton_iters, double rtol, double atol_C,
                                    double atol_T, void *workspace, size_t workspace_bytes, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells || n_attempts < 0 || newton_iters < 1) return fail(QSS_E_INVALID, "need 0 <= ncells <= ld, n_attempts >= 0, newton_iters >= 1");
    if (!(rtol >= 0.0) || !(atol_C >= 0.0) || !(atol_T >= 0.0) || !(rtol + atol_C > 0.0) || !(rtol + atol_T > 0.0)) return fail(QSS_E_INVALID, "tolerances must be non-negative and not both zero");
    const int N = m->c.tab.N;
    if (N + 1 > QSS_NEWTON_MAX_N) return fail(QSS_E_UNSUPPORTED, "qss_ignition_advance: more than 39 transported species (limit of qss_newton_solve)");
    if (ncells == 0 || n_attempts == 0) return QSS_OK;
    if (!C || !T || !dt || !t || (t_ign && !T0)) return fail(QSS_E_INVALID, "NULL device pointer (T0 is required with t_ign)");
    if (ld & 1) return fail(QSS_E_INVALID, "qss_ignition_advance: ld must be even (16-byte aligned rows)");
    if (!workspace || ((uintptr_t)workspace & 255) || workspace_bytes < qss_bdf1_workspace_bytes(m, ld)) return fail(QSS_E_INVALID, "workspace is NULL, misaligned or smaller than qss_bdf1_workspace_bytes");
    DeviceGuard guard(m->device);
    cudaStream_t st = (cudaStream_t)stream;
    QssJit *step = nullptr;
    {
        std::lock_guard<std::mutex> lock(m->host_mu);
        if (!m->newton_step_tried) {
            m->newton_step_tried = true;
            std::string jerr;
            m->newton_step = qss_jit_newton_step_create(N + 1, N + 1, QSS_NEWTON_CPB, m->cc_major, m->cc_minor, jerr);
            if (m->newton_step) m->newton_step_blocks = m->n_sm * qss_jit_newton_step_blocks_per_sm(m->newton_step, N + 1, QSS_NEWTON_CPB);
        }
        step = m->newton_step;
    }
    if (!step) return fail(QSS_E_CUDA, "qss_ignition_advance needs the run-time compiled Newton step kernel (NVRTC unavailable)");
    const size_t nrow = (size_t)ld;
    char *p = (char *)workspace;
    auto take = [&](size_t rows) { double *q = (double *)p; p += align256(rows * nrow * sizeof(double)); return q; };
    double *jac = take((size_t)N * (N + 1)), *F = take(N + 1);
    (void)take(N + 1);                                          // (the energy row of the unfused sequence: not used here)
    double *phin = take(N + 1);
    (void)take(N + 1);
    void *ws = (void *)(((uintptr_t)p + 255) & ~(uintptr_t)255);
    const size_t wsb = ws_bytes(m, true);
    QssStepAdapt ad = {1, t, dt, t_ign, T0, t_end, rtol, atol_C, atol_T, dT_ign, 1.5, 0.25};
    for (int a = 0; a < n_attempts; ++a) {
        cudaError_t e = cudaMemcpyAsync(phin, C, (size_t)N * nrow * sizeof(double), cudaMemcpyDeviceToDevice, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(phin + (size_t)N * nrow, T, nrow * sizeof(double), cudaMemcpyDeviceToDevice, st);
        if (e != cudaSuccess) return cuda_fail(e, "qss_ignition_advance: saving the state");
        for (int it = 0; it < newton_iters; ++it) {
            int rc = eval_jac_mode(m, ncells, ld, C, T, jac, F, 0, ws, wsb, stream);
            if (rc != QSS_OK) return rc;
            ad.adapt = it == newton_iters - 1 ? 2 : 1;
            e = qss_jit_newton_step_launch(step, N + 1, QSS_NEWTON_CPB, m->newton_step_blocks, jac, F, phin, dt, m->dD + m->c.tab.d_thermo, C, T, ncells, ld, st, &ad);
            if (e != cudaSuccess) return cuda_fail(e, "qss_ignition_advance: Newton step");
        }
    }
    return QSS_OK;
}

extern "C" size_t qss_host_scratch_bytes(const qss_mech_t *m, int64_t ncells, int64_t ld) {
    if (!m || ncells < 0 || ld < ncells) return 0;
    const size_t N = m->c.tab.N, L = (size_t)ld * sizeof(double);
    return align256(N * L) + align256(L) + align256(N * L) + align256(N * (N + 1) * L) + align256(ws_bytes(m, true));
}

extern "C" int qss_eval_jac_host(const qss_mech_t *m, int64_t ncells, int64_t ld, const double *Ch, const double *Th,
                                 double *jach, double *wdoth, void *scratch, size_t scratch_bytes, void *stream) {
    if (!m) return fail(QSS_E_INVALID, "mech is NULL");
    if (ncells < 0 || ld < ncells || !Ch || !Th || !jach) return fail(QSS_E_INVALID, "bad host arguments");
    if (ncells == 0) return QSS_OK;
    if (!scratch || scratch_bytes < qss_host_scratch_bytes(m, ncells, ld) || ((uintptr_t)scratch & 255))
        return fail(QSS_E_INVALID, "dev_scratch is NULL, misaligned or smaller than qss_host_scratch_bytes()");
    const size_t N = m->c.tab.N, L = (size_t)ld * sizeof(double);
    char *p = (char *)scratch;
    double *dC = (double *)p; p += align256(N * L);
    double *dT = (double *)p; p += align256(L);
    double *dW = (double *)p; p += align256(N * L);
    double *dJ = (double *)p; p += align256(N * (N + 1) * L);
    void *ws = p;
    cudaStream_t s = (cudaStream_t)stream;
    cudaError_t e;
    // Pipelined over chunks of cells: the kernel of chunk c runs on `stream` while the Jacobian of chunk c-1 streams back
    // to the host on an internal copy stream (the device-to-host copy of N(N+1) doubles per cell dominates the call).
    // The SoA arrays are copied as 2D blocks: `rows` rows of `chunk` cells with row pitch ld.
    std::lock_guard<std::mutex> lock(m->host_mu);
    DeviceGuard guard(m->device);
    // on any failure: no copy into the caller's host buffers may still be pending when the call returns
    auto bail = [&](int rc) { cudaStreamSynchronize(m->copy_stream); cudaStreamSynchronize(s); return rc; };
    const int64_t nchunk = ncells >= (1 << 16) ? 8 : 1;
    const int64_t chunk = ((ncells + nchunk - 1) / nchunk + 31) / 32 * 32;
    if ((e = cudaMemcpyAsync(dT, Th, L, cudaMemcpyHostToDevice, s)) != cudaSuccess) return bail(cuda_fail(e, "H2D T"));
    for (int64_t c0 = 0; c0 < ncells; c0 += chunk) {
        const int64_t nc = std::min(chunk, ncells - c0);
        const size_t wbytes = (size_t)nc * sizeof(double);
        if ((e = cudaMemcpy2DAsync(dC + c0, L, Ch + c0, L, wbytes, N, cudaMemcpyHostToDevice, s)) != cudaSuccess) return bail(cuda_fail(e, "H2D C"));
        int rc = qss_eval_jac(m, nc, ld, dC + c0, dT + c0, dJ + c0, wdoth ? dW + c0 : nullptr, ws, ws_bytes(m, true), stream);
        if (rc != QSS_OK) return bail(rc);
        if ((e = cudaEventRecord(m->ev[0], s)) != cudaSuccess) return bail(cuda_fail(e, "cudaEventRecord"));
        if ((e = cudaStreamWaitEvent(m->copy_stream, m->ev[0], 0)) != cudaSuccess) return bail(cuda_fail(e, "cudaStreamWaitEvent"));
        if ((e = cudaMemcpy2DAsync(jach + c0, L, dJ + c0, L, wbytes, N * (N + 1), cudaMemcpyDeviceToHost, m->copy_stream)) != cudaSuccess) return bail(cuda_fail(e, "D2H jac"));
        if (wdoth && (e = cudaMemcpy2DAsync(wdoth + c0, L, dW + c0, L, wbytes, N, cudaMemcpyDeviceToHost, m->copy_stream)) != cudaSuccess) return bail(cuda_fail(e, "D2H wdot"));
    }
    if ((e = cudaStreamSynchronize(m->copy_stream)) != cudaSuccess) return bail(cuda_fail(e, "cudaStreamSynchronize(copy)"));
    if ((e = cudaStreamSynchronize(s)) != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize");
    return QSS_OK;
}

extern "C" int qss_bench_dfma(int blocks, int iters, double *sink, double *n_fma, void *stream) {
    if (blocks < 1 || iters < 1 || !sink) return fail(QSS_E_INVALID, "bad arguments");
    cudaError_t e = qss_launch_dfma(blocks, iters, sink, (cudaStream_t)stream);
    if (n_fma) *n_fma = (double)blocks * 256.0 * (double)iters * 16.0 * 8.0;
    return e == cudaSuccess ? QSS_OK : cuda_fail(e, "qss_bench_dfma launch");
}
