// pm_fill.cu — instantiations and launcher of the fill kernel (pm_fill.cuh): one instantiation per generated
// channel-set specialisation (gen/pm_spec_gen.cuh, written by pm_codegen at build time) plus the table-driven one.
#include "pm_fill.cuh"

#include <cstdlib>
#include <map>
#include <mutex>

#include "gen/pm_spec_gen.cuh"
#include "pm_jit.hpp"
#include "pm_kernels.cuh"

namespace pm {

namespace {

constexpr int kSmemLimit = 227 * 1024;

using FillKernel = void (*)(DevLattice, FillSmem, NodeLists, int, int, const int64_t*, double*, int32_t*, int*, const int64_t*);

struct FillVariant { unsigned long long hash; int nw, rb, n_oterm; FillKernel fn, fn_cols; const char* name; };

#define PM_VAR(S, NW, RB) {gen::S::kHash, NW, RB, gen::S::NOT, k_fill_warp<gen::S, NW, RB, false>, k_fill_warp<gen::S, NW, RB, true>, #S}
#define PM_SPEC(S) PM_VAR(S, 4, 4), PM_VAR(S, 8, 4), PM_VAR(S, 12, 4),
const FillVariant kVariants[] = {
    PM_SPEC_LIST
    {0ull, 2, 4, SpecGeneric::NOT, k_fill_warp<SpecGeneric, 2, 4, false>, k_fill_warp<SpecGeneric, 2, 4, true>, "generic"},
    {0ull, 4, 4, SpecGeneric::NOT, k_fill_warp<SpecGeneric, 4, 4, false>, k_fill_warp<SpecGeneric, 4, 4, true>, "generic"},
    {0ull, 8, 4, SpecGeneric::NOT, k_fill_warp<SpecGeneric, 8, 4, false>, k_fill_warp<SpecGeneric, 8, 4, true>, "generic"},
};
#undef PM_VAR
#undef PM_SPEC

// The dynamic shared-memory limit is an attribute of the kernel FUNCTION, shared by every lattice that selects it, while
// the bytes a launch needs depend on the lattice (grids, orders): keep a per-function monotone maximum and raise it
// before any launch that needs more (never lowered, so interleaved lattices of different shape cannot starve each other).
std::mutex g_attr_mu;
std::map<const void*, int> g_attr_max;

cudaError_t ensure_smem_limit(const void* fn, int bytes)
{
    std::lock_guard<std::mutex> g(g_attr_mu);
    int dev = 0;
    cudaGetDevice(&dev);
    const void* key = (const char*)fn + dev;              // per (function, device)
    auto it = g_attr_max.find(key);
    if (it != g_attr_max.end() && it->second >= bytes) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
    if (e == cudaSuccess) g_attr_max[key] = bytes;
    return e;
}

int preferred_warps()
{
    static const int v = [] { const char* e = std::getenv("PM_FILL_WARPS"); return e ? std::atoi(e) : 12; }();
    return v;
}

}  // namespace

bool fill_has_spec(unsigned long long hash)
{
    for (const FillVariant& v : kVariants) if (v.hash == hash && hash != 0ull) return true;
    return false;
}

const char* fill_variant_name(unsigned long long hash)
{
    for (const FillVariant& v : kVariants) if (v.hash == hash && hash != 0ull) return v.name;
    return "generic";
}

// Picks the variant (specialised when `hash` matches a generated kernel, else table-driven; the preferred warp count
// if its shared memory fits, else a smaller one) and the persistent grid.  Returns cudaErrorInvalidConfiguration
// when no variant fits in shared memory.
cudaError_t fill_plan(const DevLattice& L, unsigned long long hash, int n_sm, FillLaunch* out)
{
    const unsigned long long key = fill_has_spec(hash) ? hash : 0ull;
    const int want = preferred_warps();
    const FillVariant* best = nullptr;          // largest warp count <= want whose shared memory fits, else the smallest that fits
    auto plan_of = [&](const FillVariant& v) {         // the bra table moves to global memory when it does not fit beside the tiles
        FillSmem s = fill_smem_plan(L, v.nw, v.rb, v.n_oterm, true, v.hash == 0ull);
        if (s.total > kSmemLimit && v.hash == 0ull) s = fill_smem_plan(L, v.nw, v.rb, v.n_oterm, false, true);
        return s;
    };
    for (const FillVariant& v : kVariants) {
        if (v.hash != key || plan_of(v).total > kSmemLimit) continue;
        if (!best) { best = &v; continue; }
        const bool v_ok = v.nw <= want, b_ok = best->nw <= want;
        if ((v_ok && (!b_ok || v.nw > best->nw)) || (!v_ok && !b_ok && v.nw < best->nw)) best = &v;
    }
    if (!best) return cudaErrorInvalidConfiguration;
    out->fn = (const void*)best->fn;
    out->fn_cols = (const void*)best->fn_cols;
    out->fn_op = nullptr;
    out->nw = best->nw;
    out->name = best->name;
    out->jit = false;
    out->smem = plan_of(*best);
    cudaError_t e = ensure_smem_limit(out->fn, out->smem.total);
    if (e != cudaSuccess) return e;
    if ((e = ensure_smem_limit(out->fn_cols, out->smem.total)) != cudaSuccess) return e;
    int per_sm = 1;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, out->fn, best->nw * 32, (size_t)out->smem.total);
    if (e != cudaSuccess) return e;
    out->grid = n_sm * (per_sm > 0 ? per_sm : 1);
    return cudaSuccess;
}

// Run-time compiled kernels for the column-channel groups `views` of one lattice (devs[g]: the group's device view).
// One warp count and one bra placement for all groups: the most warps whose shared memory fits with the bra harmonics
// beside them, else the most warps with the bra harmonics read from global memory.
bool fill_plan_jit(const std::vector<DevLattice>& devs, std::vector<KetView> views, int n_sm, int mode, std::vector<FillLaunch>& out, std::string& err)
{
    const int rb = 4;
    const size_t n = devs.size();
    auto fits = [&](int w, bool bra_smem) {
        for (size_t g = 0; g < n; ++g) if (fill_smem_plan(devs[g], w, rb, views[g].n_oterm, bra_smem).total > kSmemLimit) return false;
        return true;
    };
    int nw = 0;
    bool bra_smem = true;
    const int want = preferred_warps();
    for (int w : {want, 12, 8, 4}) {
        if (w < 1 || w > 32) continue;
        if (fits(w, true)) { nw = w; bra_smem = true; break; }
        if (w >= 8 && fits(w, false)) { nw = w; bra_smem = false; break; }
    }
    if (!nw) for (int w : {4, 2}) if (fits(w, false)) { nw = w; bra_smem = false; break; }
    if (!nw) { err = "no warp count fits in shared memory"; return false; }
    for (KetView& v : views) v.bra_smem = bra_smem;
    std::vector<JitFill> k;
    if (!jit_fill_many(views, nw, rb, mode, k, err)) return false;
    if (out.size() != n) out.assign(n, FillLaunch{});       // (a second call adds the other variant to the plans of the first)
    for (size_t g = 0; g < n; ++g) {
        FillLaunch& F = out[g];
        (mode == 2 ? F.fn_op : mode == 1 ? F.fn_cols : F.fn) = mode == 2 ? k[g].fn_op : mode == 1 ? k[g].fn_cols : k[g].fn;
        F.nw = nw; F.name = n > 1 ? "jit-grouped" : "jit"; F.jit = true;
        F.smem = fill_smem_plan(devs[g], nw, rb, views[g].n_oterm, bra_smem);
        const int per_sm = jit_prepare(k[g], mode, F.smem.total);
        if (per_sm < 1) { err = "the compiled kernel does not fit on an SM"; return false; }
        F.grid = n_sm * per_sm;
    }
    return true;
}

cudaError_t launch_fill(const DevLattice& L, const FillLaunch& F, int cell_begin, int n_blk, const NodeLists& nl,
                        const int64_t* rowptr, double* vals, int32_t* colidx, int* counter, const int64_t* guard, cudaStream_t st, bool op_mode)
{
    const int need = (n_blk + F.nw - 1) / F.nw;                        // one cell per warp at a time
    const int grid = need < F.grid ? need : F.grid;
    DevLattice Lc = L;
    FillSmem S = F.smem;
    NodeLists N = nl;
    cudaError_t e = cudaMemsetAsync(counter, 0, sizeof(int), st);      // the work counter the warps draw cells from
    if (e != cudaSuccess) return e;
    void* args[] = {&Lc, &S, &N, &cell_begin, &n_blk, (void*)&rowptr, &vals, &colidx, &counter, (void*)&guard};
    if (F.jit) {
        void* fn = const_cast<void*>(op_mode ? F.fn_op : colidx ? F.fn_cols : F.fn);
        if (!fn || jit_prepare_fn(fn, S.total) != 0) return cudaErrorInvalidValue;
        const int cr = jit_launch(fn, grid, F.nw * 32, S.total, (void*)st, args);
        count_launch();
        return cr == 0 ? cudaGetLastError() : cudaErrorLaunchFailure;
    }
    if ((e = ensure_smem_limit(colidx ? F.fn_cols : F.fn, S.total)) != cudaSuccess) return e;
    e = cudaLaunchKernel(colidx ? F.fn_cols : F.fn, dim3((unsigned)grid), dim3((unsigned)(F.nw * 32)), args, (size_t)S.total, st);
    count_launch();
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace pm
