// pm_jit.cpp — NVRTC compilation and driver-API launch of run-time specialised fill kernels (see pm_jit.hpp).
#include "pm_jit.hpp"

#include <cstdio>
#include <cstdlib>
#include <map>
#include <mutex>
#include <sstream>
#include <vector>

#include <cuda.h>
#include <dlfcn.h>
#include <nvrtc.h>

#include "pm_emit.hpp"

namespace pm {

namespace {

// the kernel's headers as text (written by csrc/build.py): kJitDeviceCuh, kJitYlmH, kJitFillCuh
#include "gen/pm_jit_src.inc"

struct Api {
    bool tried = false, ok = false;          // NVRTC
    bool tried_cu = false, ok_cu = false;    // driver API
    std::string why;
    // NVRTC
    decltype(&nvrtcCreateProgram) createProgram = nullptr;
    decltype(&nvrtcCompileProgram) compileProgram = nullptr;
    decltype(&nvrtcDestroyProgram) destroyProgram = nullptr;
    decltype(&nvrtcGetProgramLogSize) getLogSize = nullptr;
    decltype(&nvrtcGetProgramLog) getLog = nullptr;
    decltype(&nvrtcAddNameExpression) addName = nullptr;
    decltype(&nvrtcGetLoweredName) getLowered = nullptr;
    decltype(&nvrtcGetCUBINSize) getCubinSize = nullptr;
    decltype(&nvrtcGetCUBIN) getCubin = nullptr;
    decltype(&nvrtcGetErrorString) errString = nullptr;
    // driver
    CUresult (*moduleLoadData)(CUmodule*, const void*) = nullptr;
    CUresult (*moduleGetFunction)(CUfunction*, CUmodule, const char*) = nullptr;
    CUresult (*funcSetAttribute)(CUfunction, CUfunction_attribute, int) = nullptr;
    CUresult (*launchKernel)(CUfunction, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, CUstream, void**, void**) = nullptr;
    CUresult (*occupancy)(int*, CUfunction, int, size_t) = nullptr;
    CUresult (*ctxGetDevice)(int*) = nullptr;
};

Api g_api;
std::mutex g_mu;
std::map<std::string, JitFill> g_cache;          // key: device / hash / nw / rb (a CUfunction belongs to the context it was loaded in)
std::map<void*, int> g_fn_smem;                  // per function: the dynamic shared-memory limit set so far
bool g_enabled = std::getenv("PM_NO_JIT") == nullptr;

template <class F>
bool sym(void* h, const char* name, F& f, std::string& why)
{
    f = reinterpret_cast<F>(dlsym(h, name));
    if (!f) { why = std::string("symbol ") + name + " not found"; return false; }
    return true;
}

bool load_nvrtc()
{
    Api& a = g_api;
    if (a.tried) return a.ok;
    a.tried = true;
    void* hn = nullptr;
    for (const char* n : {"libnvrtc.so.12", "libnvrtc.so", "/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/lib64/libnvrtc.so"})
        if ((hn = dlopen(n, RTLD_NOW | RTLD_LOCAL))) break;
    if (!hn) { a.why = "libnvrtc not found"; return false; }
    a.ok = sym(hn, "nvrtcCreateProgram", a.createProgram, a.why) && sym(hn, "nvrtcCompileProgram", a.compileProgram, a.why)
        && sym(hn, "nvrtcDestroyProgram", a.destroyProgram, a.why) && sym(hn, "nvrtcGetProgramLogSize", a.getLogSize, a.why)
        && sym(hn, "nvrtcGetProgramLog", a.getLog, a.why) && sym(hn, "nvrtcAddNameExpression", a.addName, a.why)
        && sym(hn, "nvrtcGetLoweredName", a.getLowered, a.why) && sym(hn, "nvrtcGetCUBINSize", a.getCubinSize, a.why)
        && sym(hn, "nvrtcGetCUBIN", a.getCubin, a.why) && sym(hn, "nvrtcGetErrorString", a.errString, a.why);
    return a.ok;
}

bool load_driver()
{
    Api& a = g_api;
    if (a.tried_cu) return a.ok_cu;
    a.tried_cu = true;
    void* hc = dlopen("libcuda.so.1", RTLD_NOW | RTLD_LOCAL);
    if (!hc) { a.why = "libcuda.so.1 not found"; return false; }
    a.ok_cu = sym(hc, "cuModuleLoadData", a.moduleLoadData, a.why) && sym(hc, "cuModuleGetFunction", a.moduleGetFunction, a.why)
        && sym(hc, "cuFuncSetAttribute", a.funcSetAttribute, a.why) && sym(hc, "cuLaunchKernel", a.launchKernel, a.why)
        && sym(hc, "cuOccupancyMaxActiveBlocksPerMultiprocessor", a.occupancy, a.why) && sym(hc, "cuCtxGetDevice", a.ctxGetDevice, a.why);
    return a.ok_cu;
}

// NVRTC only (no device needed): cubin and the lowered names of the two kernel variants
bool compile_cubin(const Tables& T, int nw, int rb, std::vector<char>& cubin, std::string low[2], std::string& err)
{
    if (!load_nvrtc()) { err = g_api.why; return false; }
    const Api& a = g_api;
    EmitStats st;
    std::ostringstream src;
    src << "#include \"pm_fill.cuh\"\nnamespace pm {\nnamespace gen {\n" << emit_spec("jit", T, st) << "}\n}\n";
    const std::string text = src.str();
    const char* hdr_src[] = {kJitDeviceCuh, kJitYlmH, kJitFillCuh};
    const char* hdr_name[] = {"pm_device.cuh", "pm_ylm.h", "pm_fill.cuh"};
    nvrtcProgram prog = nullptr;
    nvrtcResult r = a.createProgram(&prog, text.c_str(), "pm_fill_jit.cu", 3, hdr_src, hdr_name);
    if (r != NVRTC_SUCCESS) { err = std::string("nvrtcCreateProgram: ") + a.errString(r); return false; }
    std::string names[2];
    for (int c = 0; c < 2; ++c) {
        std::ostringstream n;
        n << "pm::k_fill_warp<pm::gen::Spec_jit, " << nw << ", " << rb << ", " << (c ? "true" : "false") << ">";
        names[c] = n.str();
        a.addName(prog, names[c].c_str());
    }
    const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-lineinfo", "-default-device"};
    r = a.compileProgram(prog, 4, opts);
    if (r != NVRTC_SUCCESS) {
        size_t n = 0;
        a.getLogSize(prog, &n);
        std::string log(n, '\0');
        if (n) a.getLog(prog, &log[0]);
        err = std::string("nvrtcCompileProgram: ") + a.errString(r) + "\n" + log.substr(0, 4000);
        a.destroyProgram(&prog);
        return false;
    }
    size_t nbin = 0;
    a.getCubinSize(prog, &nbin);
    cubin.resize(nbin);
    a.getCubin(prog, cubin.data());
    for (int c = 0; c < 2; ++c) { const char* l = nullptr; a.getLowered(prog, names[c].c_str(), &l); low[c] = l ? l : ""; }
    a.destroyProgram(&prog);
    return true;
}

}  // namespace

void jit_set_enabled(bool on) { std::lock_guard<std::mutex> g(g_mu); g_enabled = on; }
bool jit_enabled() { std::lock_guard<std::mutex> g(g_mu); return g_enabled; }

bool jit_compile_check(const Tables& T, int nw, int rb, size_t* cubin_bytes, std::string& err)
{
    std::lock_guard<std::mutex> g(g_mu);
    std::vector<char> cubin;
    std::string low[2];
    if (!compile_cubin(T, nw, rb, cubin, low, err)) return false;
    if (cubin_bytes) *cubin_bytes = cubin.size();
    return !low[0].empty() && !low[1].empty();
}

bool jit_fill(const Tables& T, unsigned long long hash, int nw, int rb, JitFill* out, std::string& err)
{
    std::lock_guard<std::mutex> g(g_mu);
    if (!g_enabled) { err = "run-time compilation is disabled"; return false; }
    char key[80];
    int dev = -1;
    if (load_driver() && g_api.ctxGetDevice) g_api.ctxGetDevice(&dev);
    std::snprintf(key, sizeof key, "%d/%016llx/%d/%d", dev, hash, nw, rb);
    auto it = g_cache.find(key);
    if (it != g_cache.end()) { *out = it->second; return true; }
    std::vector<char> cubin;
    std::string low[2];
    if (!compile_cubin(T, nw, rb, cubin, low, err)) return false;
    if (!load_driver()) { err = g_api.why; return false; }
    const Api& a = g_api;
    CUmodule mod = nullptr;
    CUresult cr = a.moduleLoadData(&mod, cubin.data());
    JitFill k;
    k.nw = nw; k.rb = rb;
    if (cr == CUDA_SUCCESS) {
        CUfunction f0 = nullptr, f1 = nullptr;
        cr = a.moduleGetFunction(&f0, mod, low[0].c_str());
        if (cr == CUDA_SUCCESS) cr = a.moduleGetFunction(&f1, mod, low[1].c_str());
        k.fn = f0; k.fn_cols = f1;
    }
    if (cr != CUDA_SUCCESS) { err = "loading the compiled kernel failed (CUresult " + std::to_string((int)cr) + ")"; return false; }
    g_cache[key] = k;                                // the module stays loaded for the life of the process
    *out = k;
    return true;
}

int jit_prepare_fn(void* fn, int smem_bytes)
{
    std::lock_guard<std::mutex> g(g_mu);
    if (!g_api.ok_cu) return -1;
    auto it = g_fn_smem.find(fn);
    if (it != g_fn_smem.end() && it->second >= smem_bytes) return 0;
    if (g_api.funcSetAttribute((CUfunction)fn, CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, smem_bytes) != CUDA_SUCCESS) return -1;
    g_fn_smem[fn] = smem_bytes;
    return 0;
}

int jit_prepare(const JitFill& k, bool cols, int smem_bytes)
{
    if (!g_api.ok_cu) return 0;
    CUfunction f = (CUfunction)(cols ? k.fn_cols : k.fn);
    if (jit_prepare_fn((void*)f, smem_bytes) != 0) return 0;
    int per_sm = 0;
    if (g_api.occupancy(&per_sm, f, k.nw * 32, (size_t)smem_bytes) != CUDA_SUCCESS) return 0;
    return per_sm;
}

int jit_launch(void* fn, int grid, int block, int smem_bytes, void* stream, void** args)
{
    if (!g_api.ok_cu) return (int)CUDA_ERROR_NOT_INITIALIZED;
    return (int)g_api.launchKernel((CUfunction)fn, (unsigned)grid, 1, 1, (unsigned)block, 1, 1, (unsigned)smem_bytes, (CUstream)stream, args, nullptr);
}

}  // namespace pm
