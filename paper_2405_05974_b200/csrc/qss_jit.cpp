// Run-time specialisation of kernel variant 1: NVRTC compile of qss_kernel_v1.cu + the generated pass A, load, launch.
// NVRTC is opened with dlopen so that libqss.so loads (and the interpreter kernels work) on a box without it.
#include "qss_jit.h"
#include "qss_devtools.h"

#include <dlfcn.h>
#include <nvrtc.h>
#include <sys/stat.h>
#include <sys/types.h>
#include <unistd.h>

#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <memory>
#include <mutex>
#include <vector>

// written by build.py (build/qss_embed.cpp): the sources the run-time compilation needs
extern const int qss_embed_count;
extern const char *const qss_embed_name[];
extern const char *const qss_embed_text[];

struct QssJit {
    cudaLibrary_t lib = nullptr;
    cudaKernel_t kernel = nullptr;
};

namespace {

struct Nvrtc {
    void *so = nullptr;
    decltype(&nvrtcCreateProgram) createProgram = nullptr;
    decltype(&nvrtcCompileProgram) compileProgram = nullptr;
    decltype(&nvrtcGetCUBINSize) getCUBINSize = nullptr;
    decltype(&nvrtcGetCUBIN) getCUBIN = nullptr;
    decltype(&nvrtcGetProgramLogSize) getProgramLogSize = nullptr;
    decltype(&nvrtcGetProgramLog) getProgramLog = nullptr;
    decltype(&nvrtcDestroyProgram) destroyProgram = nullptr;
    decltype(&nvrtcGetErrorString) getErrorString = nullptr;
    bool ok = false;
};

const Nvrtc &nvrtc() {
    static Nvrtc n = [] {
        Nvrtc r;
        const char *cand[] = {"libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so"};
        for (const char *c : cand) if ((r.so = dlopen(c, RTLD_NOW | RTLD_LOCAL))) break;
        if (!r.so) return r;
#define QSS_SYM(field, name) r.field = reinterpret_cast<decltype(r.field)>(dlsym(r.so, name))
        QSS_SYM(createProgram, "nvrtcCreateProgram"); QSS_SYM(compileProgram, "nvrtcCompileProgram");
        QSS_SYM(getCUBINSize, "nvrtcGetCUBINSize"); QSS_SYM(getCUBIN, "nvrtcGetCUBIN");
        QSS_SYM(getProgramLogSize, "nvrtcGetProgramLogSize"); QSS_SYM(getProgramLog, "nvrtcGetProgramLog");
        QSS_SYM(destroyProgram, "nvrtcDestroyProgram"); QSS_SYM(getErrorString, "nvrtcGetErrorString");
#undef QSS_SYM
        r.ok = r.createProgram && r.compileProgram && r.getCUBINSize && r.getCUBIN && r.getProgramLogSize && r.getProgramLog &&
               r.destroyProgram && r.getErrorString;
        return r;
    }();
    return n;
}

std::mutex g_mu;
std::map<std::string, std::shared_ptr<std::vector<char>>> g_cubin;      // key: architecture + generated source

// ---- on-disk cache of compiled images: $QSS_CACHE_DIR, else $XDG_CACHE_HOME/libqss, else ~/.cache/libqss; QSS_CACHE=0
//      turns it off.  The key hashes everything the image depends on (architecture, options, every embedded source, the
//      generated header), so a new library build or another mechanism never finds a stale image.
uint64_t fnv1a(const std::string &s, uint64_t h) {
    for (unsigned char ch : s) { h ^= ch; h *= 1099511628211ull; }
    return h;
}

std::string cache_path(const std::string &key) {
    const char *off = std::getenv("QSS_CACHE");
    if (off && off[0] == '0') return "";
    std::string dir;
    if (const char *d = std::getenv("QSS_CACHE_DIR")) dir = d;
    else if (const char *x = std::getenv("XDG_CACHE_HOME")) dir = std::string(x) + "/libqss";
    else if (const char *h = std::getenv("HOME")) dir = std::string(h) + "/.cache/libqss";
    if (dir.empty()) return "";
    std::string full = key;
    for (int i = 0; i < qss_embed_count; ++i) { full += qss_embed_name[i]; full += qss_embed_text[i]; }
    char name[64];
    std::snprintf(name, sizeof name, "/%016llx%016llx.cubin", (unsigned long long)fnv1a(full, 14695981039346656037ull),
                  (unsigned long long)fnv1a(full, 0x9e3779b97f4a7c15ull));
    // mkdir -p (two levels are enough for the defaults)
    const size_t cut = dir.find_last_of('/');
    if (cut != std::string::npos && cut > 0) mkdir(dir.substr(0, cut).c_str(), 0700);
    mkdir(dir.c_str(), 0700);
    return dir + name;
}

std::shared_ptr<std::vector<char>> cache_load(const std::string &path) {
    if (path.empty()) return nullptr;
    FILE *f = std::fopen(path.c_str(), "rb");
    if (!f) return nullptr;
    std::fseek(f, 0, SEEK_END);
    const long sz = std::ftell(f);
    std::fseek(f, 0, SEEK_SET);
    auto bin = std::make_shared<std::vector<char>>(sz > 0 ? (size_t)sz : 0);
    const bool ok = sz > 64 && std::fread(bin->data(), 1, (size_t)sz, f) == (size_t)sz && std::memcmp(bin->data(), "\x7f" "ELF", 4) == 0;
    std::fclose(f);
    return ok ? bin : nullptr;
}

void cache_store(const std::string &path, const std::vector<char> &bin) {
    if (path.empty()) return;
    const std::string tmp = path + ".tmp" + std::to_string((long long)getpid());
    FILE *f = std::fopen(tmp.c_str(), "wb");
    if (!f) return;
    const bool ok = std::fwrite(bin.data(), 1, bin.size(), f) == bin.size();
    std::fclose(f);
    if (!ok || std::rename(tmp.c_str(), path.c_str()) != 0) std::remove(tmp.c_str());
}

// main_name: embedded source that holds the kernel; gen_name / gen_src: the generated header it includes; defs: -D options
std::shared_ptr<std::vector<char>> compile(const std::string &main_name, const std::string &gen_name, const std::string &gen_src,
                                           const std::vector<std::string> &defs, const std::string &arch, std::string &err) {
    std::string key = arch + "\n" + main_name + "\n";
    for (const std::string &dd : defs) key += dd + "\n";
    key += gen_src;
    std::lock_guard<std::mutex> lock(g_mu);
    auto it = g_cubin.find(key);
    if (it != g_cubin.end()) return it->second;
    const std::string cpath = cache_path(key);
    if (auto hit = cache_load(cpath)) { g_cubin[key] = hit; return hit; }
    const Nvrtc &n = nvrtc();
    if (!n.ok) { err = "NVRTC (libnvrtc.so.12) not found"; return nullptr; }
    std::vector<const char *> names, texts;
    const char *main_src = nullptr;
    for (int i = 0; i < qss_embed_count; ++i) {
        if (main_name == qss_embed_name[i]) main_src = qss_embed_text[i];
        else { names.push_back(qss_embed_name[i]); texts.push_back(qss_embed_text[i]); }
    }
    if (!main_src) { err = "kernel source not embedded"; return nullptr; }
    names.push_back(gen_name.c_str()); texts.push_back(gen_src.c_str());
    nvrtcProgram prog = nullptr;
    nvrtcResult r = n.createProgram(&prog, main_src, main_name.c_str(), (int)names.size(), texts.data(), names.data());
    if (r != NVRTC_SUCCESS) { err = std::string("nvrtcCreateProgram: ") + n.getErrorString(r); return nullptr; }
    const std::string archopt = "--gpu-architecture=" + arch;
    std::vector<const char *> opts = {archopt.c_str(), "-std=c++17", "-lineinfo", "--fmad=true"};
    for (const std::string &dd : defs) opts.push_back(dd.c_str());
    r = n.compileProgram(prog, (int)opts.size(), opts.data());
    if (r != NVRTC_SUCCESS) {
        size_t ls = 0;
        n.getProgramLogSize(prog, &ls);
        std::string log(ls, '\0');
        if (ls) n.getProgramLog(prog, &log[0]);
        if (log.size() > 2000) log.resize(2000);
        err = std::string("nvrtcCompileProgram: ") + n.getErrorString(r) + "\n" + log;
        n.destroyProgram(&prog);
        return nullptr;
    }
    size_t sz = 0;
    r = n.getCUBINSize(prog, &sz);
    auto bin = std::make_shared<std::vector<char>>(sz);
    if (r == NVRTC_SUCCESS && sz) r = n.getCUBIN(prog, bin->data());
    n.destroyProgram(&prog);
    if (r != NVRTC_SUCCESS || !sz) { err = std::string("nvrtcGetCUBIN: ") + n.getErrorString(r); return nullptr; }
    if (const char *dump = qss_devenv("QSS_JIT_DUMP")) {       // debugging aid: the device image, for cuobjdump -sass
        if (FILE *f = std::fopen(dump, "wb")) { std::fwrite(bin->data(), 1, bin->size(), f); std::fclose(f); }
    }
    cache_store(cpath, *bin);
    g_cubin[key] = bin;
    return bin;
}

std::string arch_of(int cc_major, int cc_minor) {
    char arch[32];
    std::snprintf(arch, sizeof arch, "sm_%d%d%s", cc_major, cc_minor, cc_major >= 9 ? "a" : "");
    return arch;
}

QssJit *load_image(const std::vector<char> &bin, const char *kernel, std::string &err) {
    QssJit *j = new QssJit();
    cudaError_t e = cudaLibraryLoadData(&j->lib, bin.data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->kernel, j->lib, kernel);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(reinterpret_cast<const void *>(j->kernel), cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) {
        err = std::string("loading the specialised kernel: ") + cudaGetErrorString(e);
        if (j->lib) cudaLibraryUnload(j->lib);
        delete j;
        cudaGetLastError();
        return nullptr;
    }
    return j;
}

}  // namespace

std::vector<std::string> defs3(bool jac);

std::vector<std::string> defs1() {
    std::vector<std::string> d = {"-DQSS_GEN"};
    if (qss_devenv("QSS_TIMING")) d.push_back("-DQSS_DEVTOOLS");
    return d;
}

bool qss_jit_compile_only(const std::string &gen_src, int cc_major, int cc_minor, size_t *image_bytes, std::string &err) {
    std::shared_ptr<std::vector<char>> bin = compile("qss_kernel_v1.cu", "qss_gen.h", gen_src, defs1(), arch_of(cc_major, cc_minor), err);
    if (bin && image_bytes) *image_bytes = bin->size();
    return (bool)bin;
}

QssJit *qss_jit_create(const std::string &gen_src, int cc_major, int cc_minor, std::string &err) {
    std::shared_ptr<std::vector<char>> bin = compile("qss_kernel_v1.cu", "qss_gen.h", gen_src, defs1(), arch_of(cc_major, cc_minor), err);
    return bin ? load_image(*bin, "qss_v1_jit", err) : nullptr;
}

std::vector<std::string> defs3(bool jac) {
    std::vector<std::string> d = {jac ? "-DQSS3_JAC=1" : "-DQSS3_JAC=0"};
    if (qss_devenv("QSS_TIMING")) d.push_back("-DQSS3_TIMING=1");
    if (const char *x = qss_devenv("QSS3_EXP")) d.push_back(std::string("-DQSS3_X=") + x);      // (development builds: experiment switches)
    return d;
}

bool qss_jit3_compile_only(const std::string &gen_src, bool jac, int cc_major, int cc_minor, size_t *image_bytes, std::string &err) {
    std::shared_ptr<std::vector<char>> bin = compile("qss_kernel_v3.cu", "qss_gen3.h", gen_src, defs3(jac), arch_of(cc_major, cc_minor), err);
    if (bin && image_bytes) *image_bytes = bin->size();
    return (bool)bin;
}

QssJit *qss_jit3_create(const std::string &gen_src, bool jac, int cc_major, int cc_minor, std::string &err) {
    std::shared_ptr<std::vector<char>> bin = compile("qss_kernel_v3.cu", "qss_gen3.h", gen_src, defs3(jac), arch_of(cc_major, cc_minor), err);
    return bin ? load_image(*bin, jac ? "qss_v3_jac" : "qss_v3_wdot", err) : nullptr;
}

cudaError_t qss_jit3_launch(const QssJit *j, const QssV3 &v, int nblocks, int nw, size_t smem_bytes, cudaStream_t stream) {
    const int64_t nslab = (v.ncells + 31) / 32;
    if (nslab == 0) return cudaSuccess;
    const int grid = (int)(nslab < nblocks ? nslab : nblocks);
    void *args[] = {const_cast<QssV3 *>(&v)};
    return cudaLaunchKernel(reinterpret_cast<const void *>(j->kernel), dim3(grid), dim3(nw * 32), args, smem_bytes, stream);
}

cudaError_t qss_jit_launch(const QssJit *j, const QssV1 &v, int nblocks, cudaStream_t stream) {
    const int64_t nslab = (v.ncells + 31) / 32;
    if (nslab == 0) return cudaSuccess;
    const int grid = (int)(nslab < nblocks ? nslab : nblocks);
    void *args[] = {const_cast<QssV1 *>(&v)};
    return cudaLaunchKernel(reinterpret_cast<const void *>(j->kernel), dim3(grid), dim3(v.nw * 32), args, (size_t)v.smem_rows * 256, stream);
}

// ---- Newton solve ------------------------------------------------------------------------------------------------------
namespace {
bool newton_packed() {          // the mapping of qss_newton_kernel.cu: rows of 8 cells packed over a block (1) or one warp per cell (0)
    if (const char *e = qss_devenv("QSS_NEWTON_PACKED")) return std::atoi(e) != 0;      // (development builds: measured 14.7 against 14.1 ms)
    return false;
}
std::string newton_gen(int n, int nj, bool has_e, int cpb) {
    char buf[320];
    int minb = newton_packed() ? 2 : 1;
    if (const char *e = qss_devenv("QSS_NEWTON_MINB")) minb = std::atoi(e);      // (development builds: register limit experiments)
    std::snprintf(buf, sizeof buf, "#define LU_N %d\n#define LU_NJ %d\n#define LU_HAS_E %d\n#define LU_CPB %d\n#define LU_MINB %d\n#define LU_PACKED %d\n",
                  n, nj, has_e ? 1 : 0, cpb, minb, newton_packed() ? 1 : 0);
    return buf;
}
int newton_threads(int n, int cpb) { return newton_packed() ? (cpb * n + 31) / 32 * 32 : 32 * cpb; }
struct QssNewtonArgs {          // = struct QssNewton of qss_newton_kernel.cu
    const double *jac, *erow, *gamma, *b;
    double *x;
    int64_t ncells, ld;
};
}  // namespace

bool qss_jit_newton_compile_only(int n, int nj, bool has_e, int cpb, int cc_major, int cc_minor, size_t *image_bytes, std::string &err) {
    std::shared_ptr<std::vector<char>> bin = compile("qss_newton_kernel.cu", "qss_newton_gen.h", newton_gen(n, nj, has_e, cpb), {}, arch_of(cc_major, cc_minor), err);
    if (bin && image_bytes) *image_bytes = bin->size();
    return (bool)bin;
}

QssJit *qss_jit_newton_create(int n, int nj, bool has_e, int cpb, int cc_major, int cc_minor, std::string &err) {
    std::shared_ptr<std::vector<char>> bin = compile("qss_newton_kernel.cu", "qss_newton_gen.h", newton_gen(n, nj, has_e, cpb), {}, arch_of(cc_major, cc_minor), err);
    return bin ? load_image(*bin, "qss_newton_kernel", err) : nullptr;
}

size_t qss_jit_newton_smem(int n, int cpb) {
    const size_t nc = (size_t)n + 1, pitch = nc | 1, ub = (nc + 4) & ~(size_t)1;
    if (newton_packed()) return ((size_t)cpb * n * pitch + (size_t)cpb * ((nc + 5) & ~(size_t)1) + (size_t)cpb * n) * sizeof(double) + (size_t)2 * cpb * sizeof(unsigned);
    return ((size_t)2 * cpb * n * pitch + (size_t)cpb * 2 * ub + (size_t)cpb * n) * sizeof(double) + (size_t)cpb * n * sizeof(int);
}

int qss_jit_newton_blocks_per_sm(const QssJit *j, int n, int cpb) {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, reinterpret_cast<const void *>(j->kernel), newton_threads(n, cpb), qss_jit_newton_smem(n, cpb)) != cudaSuccess) { cudaGetLastError(); nb = 1; }
    return nb < 1 ? 1 : nb;
}

cudaError_t qss_jit_newton_launch(const QssJit *j, int n, int cpb, int max_blocks, const double *jac, const double *erow, const double *gamma,
                                  const double *b, double *x, int64_t ncells, int64_t ld, cudaStream_t stream) {
    if (ncells == 0) return cudaSuccess;
    QssNewtonArgs a = {jac, erow, gamma, b, x, ncells, ld};
    void *args[] = {&a};
    const int64_t ntiles = (ncells + cpb - 1) / cpb;
    const int64_t grid = ntiles < max_blocks ? ntiles : max_blocks;          // persistent blocks: tile t, t + grid, ...
    return cudaLaunchKernel(reinterpret_cast<const void *>(j->kernel), dim3((unsigned)grid), dim3(newton_threads(n, cpb)), args, qss_jit_newton_smem(n, cpb), stream);
}

// ---- fused Newton step (qss_newton_step_kernel) ----------------------------------------------------------------------------
namespace {
struct QssStepArgs {            // = struct QssStep of qss_newton_kernel.cu
    const double *jac, *wdot, *phin, *dt, *thermo;
    double *C, *T;
    int64_t ncells, ld;
    int adapt;
    double *tcur, *dtio, *tign;
    const double *T0;
    double t_end, rtol, atolC, atolT, dT_ign, grow, shrink;
};
}  // namespace

QssJit *qss_jit_newton_step_create(int n, int nj, int cpb, int cc_major, int cc_minor, std::string &err) {
    if (newton_packed()) { err = "the fused step exists for the warp-per-cell mapping only"; return nullptr; }
    std::shared_ptr<std::vector<char>> bin = compile("qss_newton_kernel.cu", "qss_newton_gen.h", newton_gen(n, nj, true, cpb), {}, arch_of(cc_major, cc_minor), err);
    return bin ? load_image(*bin, "qss_newton_step_kernel", err) : nullptr;
}

size_t qss_jit_newton_step_smem(int n, int cpb) {
    const size_t nc = (size_t)n + 1, pitch = nc | 1, ub = (nc + 4) & ~(size_t)1, N = (size_t)n - 1, aux = 3 * N + 2;
    return ((size_t)2 * cpb * n * pitch + (size_t)2 * cpb * aux + (size_t)cpb * 2 * ub + (size_t)cpb * n + (size_t)cpb * 2 * N) * sizeof(double) + (size_t)cpb * n * sizeof(int);
}

int qss_jit_newton_step_blocks_per_sm(const QssJit *j, int n, int cpb) {
    int nb = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, reinterpret_cast<const void *>(j->kernel), 32 * cpb, qss_jit_newton_step_smem(n, cpb)) != cudaSuccess) { cudaGetLastError(); nb = 1; }
    return nb < 1 ? 1 : nb;
}

cudaError_t qss_jit_newton_step_launch(const QssJit *j, int n, int cpb, int max_blocks, const double *jac, const double *wdot, const double *phin,
                                       const double *dt, const double *thermo, double *C, double *T, int64_t ncells, int64_t ld, cudaStream_t stream,
                                       const QssStepAdapt *ad) {
    if (ncells == 0) return cudaSuccess;
    QssStepArgs a = {jac, wdot, phin, dt, thermo, C, T, ncells, ld, 0, nullptr, nullptr, nullptr, nullptr, 0, 0, 0, 0, 0, 0, 0};
    if (ad) {
        a.adapt = ad->adapt; a.tcur = ad->tcur; a.dtio = ad->dtio; a.tign = ad->tign; a.T0 = ad->T0;
        a.t_end = ad->t_end; a.rtol = ad->rtol; a.atolC = ad->atolC; a.atolT = ad->atolT; a.dT_ign = ad->dT_ign; a.grow = ad->grow; a.shrink = ad->shrink;
    }
    void *args[] = {&a};
    const int64_t ntiles = (ncells + cpb - 1) / cpb;
    const int64_t grid = ntiles < max_blocks ? ntiles : max_blocks;
    return cudaLaunchKernel(reinterpret_cast<const void *>(j->kernel), dim3((unsigned)grid), dim3(32 * cpb), args, qss_jit_newton_step_smem(n, cpb), stream);
}

void qss_jit_destroy(QssJit *j) {
    if (!j) return;
    if (j->lib) cudaLibraryUnload(j->lib);
    delete j;
}
