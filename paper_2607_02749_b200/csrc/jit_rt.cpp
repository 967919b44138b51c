// jit_rt.cpp -- run-time side of the specialised gate-block kernels (jit.h): NVRTC (found with dlopen, no link-time
// dependency) turns the generated source into an sm_100a cubin, the CUDA driver entry points (obtained from the runtime,
// no libcuda link) load and launch it.  Compiled images are cached per process by source text.
#include <cuda.h>
#include <cuda_runtime.h>
#include <dlfcn.h>

#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "jit.h"

namespace gv {
namespace {

typedef struct _nvrtcProgram *nvrtcProgram_t;
struct Nvrtc {
    void *h = nullptr;
    int (*CreateProgram)(nvrtcProgram_t *, const char *, const char *, int, const char *const *, const char *const *) = nullptr;
    int (*CompileProgram)(nvrtcProgram_t, int, const char *const *) = nullptr;
    int (*GetCUBINSize)(nvrtcProgram_t, size_t *) = nullptr;
    int (*GetCUBIN)(nvrtcProgram_t, char *) = nullptr;
    int (*GetProgramLogSize)(nvrtcProgram_t, size_t *) = nullptr;
    int (*GetProgramLog)(nvrtcProgram_t, char *) = nullptr;
    int (*DestroyProgram)(nvrtcProgram_t *) = nullptr;
    std::string why;
};

Nvrtc &nvrtc()
{
    static Nvrtc N;
    static std::once_flag once;
    std::call_once(once, [] {
        const char *names[] = {"libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so"};
        for (const char *nm : names) {
            N.h = dlopen(nm, RTLD_NOW | RTLD_LOCAL);
            if (N.h) break;
        }
        if (!N.h) { N.why = "libnvrtc not found"; return; }
#define GV_SYM(field, sym) *(void **)(&N.field) = dlsym(N.h, sym); if (!N.field) { N.why = std::string("missing ") + sym; N.h = nullptr; return; }
        GV_SYM(CreateProgram, "nvrtcCreateProgram") GV_SYM(CompileProgram, "nvrtcCompileProgram") GV_SYM(GetCUBINSize, "nvrtcGetCUBINSize")
        GV_SYM(GetCUBIN, "nvrtcGetCUBIN") GV_SYM(GetProgramLogSize, "nvrtcGetProgramLogSize") GV_SYM(GetProgramLog, "nvrtcGetProgramLog")
        GV_SYM(DestroyProgram, "nvrtcDestroyProgram")
#undef GV_SYM
    });
    return N;
}

struct Driver {
    CUresult (*ModuleLoadData)(CUmodule *, const void *) = nullptr;
    CUresult (*ModuleGetFunction)(CUfunction *, CUmodule, const char *) = nullptr;
    CUresult (*ModuleUnload)(CUmodule) = nullptr;
    CUresult (*FuncSetAttribute)(CUfunction, CUfunction_attribute, int) = nullptr;
    CUresult (*LaunchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream, void **, void **) = nullptr;
    bool ok = false;
    std::string why;
};

Driver &driver()
{
    static Driver D;
    static std::once_flag once;
    std::call_once(once, [] {
        auto get = [](const char *sym, void **fn) {
            cudaDriverEntryPointQueryResult qr;
            return cudaGetDriverEntryPoint(sym, fn, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess && *fn;
        };
        if (!get("cuModuleLoadData", (void **)&D.ModuleLoadData) || !get("cuModuleGetFunction", (void **)&D.ModuleGetFunction) ||
            !get("cuModuleUnload", (void **)&D.ModuleUnload) || !get("cuFuncSetAttribute", (void **)&D.FuncSetAttribute) ||
            !get("cuLaunchKernel", (void **)&D.LaunchKernel)) {
            D.why = "CUDA driver entry points unavailable";
            (void)cudaGetLastError();
            return;
        }
        D.ok = true;
    });
    return D;
}

std::mutex g_cache_mu;
std::map<std::string, std::vector<char>> g_cubins;   // source text -> cubin

bool compile(const JitBlock &blk, std::vector<char> &cubin, std::string &err)
{
    {
        std::lock_guard<std::mutex> lk(g_cache_mu);
        auto it = g_cubins.find(blk.source);
        if (it != g_cubins.end()) { cubin = it->second; return true; }
    }
    Nvrtc &N = nvrtc();
    if (!N.h) { err = "jit: " + N.why; return false; }
    nvrtcProgram_t prog = nullptr;
    if (N.CreateProgram(&prog, blk.source.c_str(), (blk.name + ".cu").c_str(), 0, nullptr, nullptr) != 0) { err = "jit: nvrtcCreateProgram failed"; return false; }
    const char *opts[] = {"--gpu-architecture=sm_100a", "-lineinfo", "--std=c++17", "-default-device"};
    const int rc = N.CompileProgram(prog, 4, opts);
    if (rc != 0) {
        size_t ls = 0;
        N.GetProgramLogSize(prog, &ls);
        std::string log(ls, ' ');
        if (ls) N.GetProgramLog(prog, &log[0]);
        err = "jit: compilation of " + blk.name + " failed: " + log.substr(0, 1500);
        N.DestroyProgram(&prog);
        return false;
    }
    size_t cs = 0;
    if (N.GetCUBINSize(prog, &cs) != 0 || cs == 0) { err = "jit: no cubin"; N.DestroyProgram(&prog); return false; }
    cubin.resize(cs);
    N.GetCUBIN(prog, cubin.data());
    N.DestroyProgram(&prog);
    std::lock_guard<std::mutex> lk(g_cache_mu);
    g_cubins[blk.source] = cubin;
    return true;
}

}  // namespace

struct JitModule {
    CUmodule mod = nullptr;
    CUfunction fn = nullptr;
};

bool jit_runtime_available(std::string &why)
{
    if (!nvrtc().h) { why = nvrtc().why; return false; }
    return true;
}

bool jit_compile_only(const JitBlock &blk, std::vector<char> &cubin, std::string &err) { return compile(blk, cubin, err); }

JitModule *jit_load(const JitBlock &blk, std::string &err)
{
    std::vector<char> cubin;
    if (!compile(blk, cubin, err)) return nullptr;
    Driver &D = driver();
    if (!D.ok) { err = "jit: " + D.why; return nullptr; }
    (void)cudaFree(nullptr);   // make sure the primary context is current
    JitModule *m = new JitModule();
    CUresult r = D.ModuleLoadData(&m->mod, cubin.data());
    if (r == CUDA_SUCCESS) r = D.ModuleGetFunction(&m->fn, m->mod, blk.name.c_str());
    if (r == CUDA_SUCCESS) r = D.FuncSetAttribute(m->fn, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)blk.smem_bytes);
    if (r != CUDA_SUCCESS) {
        char b[96];
        snprintf(b, sizeof b, "jit: loading %s failed (CUresult %d)", blk.name.c_str(), (int)r);
        err = b;
        if (m->mod) D.ModuleUnload(m->mod);
        delete m;
        return nullptr;
    }
    return m;
}

void jit_unload(JitModule *m)
{
    if (!m) return;
    if (m->mod && driver().ok) driver().ModuleUnload(m->mod);
    delete m;
}

int jit_launch(JitModule *m, const JitBlock &blk, void *states, uint64_t stride, const void *ry, const void *cs, int nb, int P,
               int per_cta, void *stream, const void *src, uint64_t src_stride)
{
    if (!src) { src = states; src_stride = stride; }
    if (!m || !m->fn || nb <= 0 || per_cta < 1) return (int)cudaErrorInvalidValue;
    const uint64_t total = (uint64_t)nb << blk.tiles_log2;
    const uint64_t grid64 = (total + (uint64_t)per_cta - 1) / (uint64_t)per_cta;
    if (grid64 > 0x7fffffffull) return (int)cudaErrorInvalidValue;
    const unsigned grid = (unsigned)grid64;
    void *args[] = {&states, &stride, &ry, &cs, &nb, &P, &per_cta, &src, &src_stride};
    const CUresult r = driver().LaunchKernel(m->fn, grid, 1, 1, blk.threads, 1, 1, blk.smem_bytes, (CUstream)stream, args, nullptr);
    return r == CUDA_SUCCESS ? 0 : (int)cudaErrorLaunchFailure;
}

int jit_launch_expect(JitModule *m, const JitBlock &blk, const void *states, uint64_t stride, const void *table, const void *wst,
                      const void *pats, const void *terms, double *partial, uint32_t slots_per_b, uint32_t slot_off, int nb,
                      int per_cta, void *stream)
{
    if (!m || !m->fn || nb <= 0 || per_cta < 1) return (int)cudaErrorInvalidValue;
    const uint64_t total = (uint64_t)nb << blk.tiles_log2;
    const uint64_t grid64 = (total + (uint64_t)per_cta - 1) / (uint64_t)per_cta;
    if (grid64 > 0x7fffffffull) return (int)cudaErrorInvalidValue;
    const unsigned grid = (unsigned)grid64;
    void *args[] = {&states, &stride, &table, &wst, &pats, &terms, &partial, &slots_per_b, &slot_off, &nb, &per_cta};
    const CUresult r = driver().LaunchKernel(m->fn, grid, 1, 1, blk.threads, 1, 1, blk.smem_bytes, (CUstream)stream, args, nullptr);
    return r == CUDA_SUCCESS ? 0 : (int)cudaErrorLaunchFailure;
}

}  // namespace gv
