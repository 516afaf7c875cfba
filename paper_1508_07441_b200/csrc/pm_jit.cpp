// pm_jit.cpp — NVRTC compilation and driver-API launch of run-time specialised fill kernels (see pm_jit.hpp).
#include "pm_jit.hpp"

#include <cstdio>
#include <cstdlib>
#include <algorithm>
#include <atomic>
#include <map>
#include <mutex>
#include <thread>
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
bool compile_cubin(const KetView& T, int nw, int rb, int variants, std::vector<char>& cubin, std::string low[3], std::string& err)
{
    if (!g_api.ok) { err = g_api.why.empty() ? "NVRTC is not loaded" : g_api.why; return false; }      // (load_nvrtc() ran under the lock)
    const Api& a = g_api;
    EmitStats st;
    std::ostringstream src;
    src << "#include \"pm_fill.cuh\"\nnamespace pm {\nnamespace gen {\n" << emit_spec("jit", T, st) << "}\n}\n";
    const std::string text = src.str();
    if (const char* dump = std::getenv("PM_JIT_DUMP")) {        // debugging aid: the generated translation unit
        if (FILE* f = std::fopen(dump, "w")) { std::fputs(text.c_str(), f); std::fclose(f); }
    }
    const char* hdr_src[] = {kJitDeviceCuh, kJitYlmH, kJitFillCuh};
    const char* hdr_name[] = {"pm_device.cuh", "pm_ylm.h", "pm_fill.cuh"};
    nvrtcProgram prog = nullptr;
    nvrtcResult r = a.createProgram(&prog, text.c_str(), "pm_fill_jit.cu", 3, hdr_src, hdr_name);
    if (r != NVRTC_SUCCESS) { err = std::string("nvrtcCreateProgram: ") + a.errString(r); return false; }
    std::string names[3];
    for (int c = 0; c < 3; ++c) {
        if (!(variants & (1 << c))) continue;
        std::ostringstream n;
        n << "pm::k_fill_warp<pm::gen::Spec_jit, " << nw << ", " << rb << ", " << c << ">";
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
    for (int c = 0; c < 3; ++c) {
        low[c].clear();
        if (!(variants & (1 << c))) continue;
        const char* l = nullptr;
        a.getLowered(prog, names[c].c_str(), &l);
        low[c] = l ? l : "";
    }
    a.destroyProgram(&prog);
    return true;
}

}  // namespace

void jit_set_enabled(bool on) { std::lock_guard<std::mutex> g(g_mu); g_enabled = on; }
bool jit_enabled() { std::lock_guard<std::mutex> g(g_mu); return g_enabled; }

bool jit_compile_check(const KetView& V, int nw, int rb, size_t* cubin_bytes, std::string& err)
{
    {
        std::lock_guard<std::mutex> g(g_mu);
        if (!load_nvrtc()) { err = g_api.why; return false; }
    }
    std::vector<char> cubin;
    std::string low[3];
    if (!compile_cubin(V, nw, rb, 2, cubin, low, err)) return false;      // the variant pm_build launches
    if (cubin_bytes) *cubin_bytes = cubin.size();
    return !low[1].empty();
}

bool jit_fill_many(const std::vector<KetView>& views, int nw, int rb, int mode, std::vector<JitFill>& out, std::string& err)
{
    const size_t n = views.size();
    out.assign(n, JitFill{});
    std::vector<std::string> keys(n);
    std::vector<size_t> todo;
    {
        std::lock_guard<std::mutex> g(g_mu);
        if (!g_enabled) { err = "run-time compilation is disabled"; return false; }
        int dev = -1;
        if (load_driver() && g_api.ctxGetDevice) g_api.ctxGetDevice(&dev);
        for (size_t i = 0; i < n; ++i) {
            char key[96];
            std::snprintf(key, sizeof key, "%d/%016llx/%d/%d/%d/%d/%d", dev, (unsigned long long)views[i].hash, nw, rb, views[i].bra_smem ? 1 : 0, views[i].n_bra > 254 ? 1 : 0, mode);
            keys[i] = key;
            auto it = g_cache.find(keys[i]);
            if (it != g_cache.end()) out[i] = it->second; else todo.push_back(i);
        }
        if (todo.empty()) return true;
        if (!load_nvrtc()) { err = g_api.why; return false; }
        if (!load_driver()) { err = g_api.why; return false; }
    }
    // NVRTC runs outside the lock, one host thread per kernel (the programs are independent)
    std::vector<std::vector<char>> cubin(todo.size());
    std::vector<std::string> lowm(todo.size()), errs(todo.size());
    std::vector<char> ok(todo.size(), 0);
    {
        const size_t nt = std::min<size_t>(todo.size(), std::max(1u, std::thread::hardware_concurrency()));
        std::atomic<size_t> next{0};
        auto work = [&] {
            for (size_t j = next++; j < todo.size(); j = next++) {
                std::string low[3];
                ok[j] = compile_cubin(views[todo[j]], nw, rb, 1 << mode, cubin[j], low, errs[j]) ? 1 : 0;
                lowm[j] = low[mode];
            }
        };
        std::vector<std::thread> th;
        for (size_t t = 1; t < nt; ++t) th.emplace_back(work);
        work();
        for (std::thread& t : th) t.join();
    }
    // modules are loaded by the calling thread (it holds the CUDA context)
    std::lock_guard<std::mutex> g(g_mu);
    const Api& a = g_api;
    for (size_t j = 0; j < todo.size(); ++j) {
        if (!ok[j]) { err = errs[j]; return false; }
        CUmodule mod = nullptr;
        CUresult cr = a.moduleLoadData(&mod, cubin[j].data());
        JitFill k;
        k.nw = nw; k.rb = rb;
        if (cr == CUDA_SUCCESS) {
            CUfunction f = nullptr;
            cr = a.moduleGetFunction(&f, mod, lowm[j].c_str());
            (mode == 2 ? k.fn_op : mode == 1 ? k.fn_cols : k.fn) = f;
        }
        if (cr != CUDA_SUCCESS) { err = "loading the compiled kernel failed (CUresult " + std::to_string((int)cr) + ")"; return false; }
        g_cache[keys[todo[j]]] = k;                  // the module stays loaded for the life of the process
        out[todo[j]] = k;
    }
    return true;
}

bool jit_fill(const KetView& V, int nw, int rb, int mode, JitFill* out, std::string& err)
{
    std::vector<JitFill> r;
    if (!jit_fill_many(std::vector<KetView>{V}, nw, rb, mode, r, err)) return false;
    *out = r[0];
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

int jit_prepare(const JitFill& k, int mode, int smem_bytes)
{
    if (!g_api.ok_cu) return 0;
    CUfunction f = (CUfunction)(mode == 2 ? k.fn_op : mode == 1 ? k.fn_cols : k.fn);
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
