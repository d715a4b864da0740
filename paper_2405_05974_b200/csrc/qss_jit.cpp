// Run-time specialisation of kernel variant 1: NVRTC compile of qss_kernel_v1.cu + the generated pass A, load, launch.
// NVRTC is opened with dlopen so that libqss.so loads (and the interpreter kernels work) on a box without it.
#include "qss_jit.h"

#include <dlfcn.h>
#include <nvrtc.h>

#include <cstdio>
#include <cstdlib>
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

std::shared_ptr<std::vector<char>> compile(const std::string &gen_src, const std::string &arch, std::string &err) {
    const std::string key = arch + "\n" + gen_src;
    std::lock_guard<std::mutex> lock(g_mu);
    auto it = g_cubin.find(key);
    if (it != g_cubin.end()) return it->second;
    const Nvrtc &n = nvrtc();
    if (!n.ok) { err = "NVRTC (libnvrtc.so.12) not found"; return nullptr; }
    std::vector<const char *> names, texts;
    const char *main_src = nullptr;
    for (int i = 0; i < qss_embed_count; ++i) {
        if (std::string(qss_embed_name[i]) == "qss_kernel_v1.cu") main_src = qss_embed_text[i];
        else { names.push_back(qss_embed_name[i]); texts.push_back(qss_embed_text[i]); }
    }
    if (!main_src) { err = "kernel source not embedded"; return nullptr; }
    names.push_back("qss_gen.h"); texts.push_back(gen_src.c_str());
    nvrtcProgram prog = nullptr;
    nvrtcResult r = n.createProgram(&prog, main_src, "qss_kernel_v1.cu", (int)names.size(), texts.data(), names.data());
    if (r != NVRTC_SUCCESS) { err = std::string("nvrtcCreateProgram: ") + n.getErrorString(r); return nullptr; }
    const std::string archopt = "--gpu-architecture=" + arch;
    const char *opts[] = {archopt.c_str(), "-std=c++17", "-DQSS_GEN", "-lineinfo", "--fmad=true"};
    r = n.compileProgram(prog, (int)(sizeof opts / sizeof opts[0]), opts);
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
    if (const char *dump = std::getenv("QSS_JIT_DUMP")) {       // debugging aid: the device image, for cuobjdump -sass
        if (FILE *f = std::fopen(dump, "wb")) { std::fwrite(bin->data(), 1, bin->size(), f); std::fclose(f); }
    }
    g_cubin[key] = bin;
    return bin;
}

}  // namespace

bool qss_jit_compile_only(const std::string &gen_src, int cc_major, int cc_minor, size_t *image_bytes, std::string &err) {
    char arch[32];
    std::snprintf(arch, sizeof arch, "sm_%d%d%s", cc_major, cc_minor, cc_major >= 9 ? "a" : "");
    std::shared_ptr<std::vector<char>> bin = compile(gen_src, arch, err);
    if (bin && image_bytes) *image_bytes = bin->size();
    return (bool)bin;
}

QssJit *qss_jit_create(const std::string &gen_src, int cc_major, int cc_minor, std::string &err) {
    char arch[32];
    std::snprintf(arch, sizeof arch, "sm_%d%d%s", cc_major, cc_minor, cc_major >= 9 ? "a" : "");
    std::shared_ptr<std::vector<char>> bin = compile(gen_src, arch, err);
    if (!bin) return nullptr;
    QssJit *j = new QssJit();
    cudaError_t e = cudaLibraryLoadData(&j->lib, bin->data(), nullptr, nullptr, 0, nullptr, nullptr, 0);
    if (e == cudaSuccess) e = cudaLibraryGetKernel(&j->kernel, j->lib, "qss_v1_jit");
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

cudaError_t qss_jit_launch(const QssJit *j, const QssV1 &v, int nblocks, cudaStream_t stream) {
    const int64_t nslab = (v.ncells + 31) / 32;
    if (nslab == 0) return cudaSuccess;
    const int grid = (int)(nslab < nblocks ? nslab : nblocks);
    void *args[] = {const_cast<QssV1 *>(&v)};
    return cudaLaunchKernel(reinterpret_cast<const void *>(j->kernel), dim3(grid), dim3(v.nw * 32), args, (size_t)v.smem_rows * 256, stream);
}

void qss_jit_destroy(QssJit *j) {
    if (!j) return;
    if (j->lib) cudaLibraryUnload(j->lib);
    delete j;
}
