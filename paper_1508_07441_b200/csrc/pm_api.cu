// pm_api.cu — the C ABI of libpm (include/pm.h): handle management, validation, table upload and the
// entry points pm_pattern / pm_fill / pm_spmv / pm_build_host.  No torch types, no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/pm.h"
#include "pm_jit.hpp"
#include "pm_kernels.cuh"
#include "pm_tables.hpp"

namespace {

thread_local std::string g_err = "";

int32_t fail(int32_t code, const std::string& msg) { g_err = msg; return code; }
int32_t cuda_fail(cudaError_t e, const char* where)
{
    g_err = std::string(where) + ": " + cudaGetErrorString(e);
    return e == cudaErrorMemoryAllocation ? PM_ERR_NOMEM : PM_ERR_CUDA;
}

int next_pow2(int n) { int p = 1; while (p < n) p <<= 1; return p; }

}  // namespace

namespace pm {
// used by the other translation units of the library (pm_stream.cu): every failing path leaves a message for pm_last_error()
int32_t set_error(int32_t code, const std::string& msg) { return fail(code, msg); }
int32_t set_cuda_error(cudaError_t e, const char* where) { cudaGetLastError(); return cuda_fail(e, where); }
}  // namespace pm

struct pm_lattice {
    int Np = 0, Nq = 0, n_ch = 0, J2 = 0, parity = 1, T2 = 0, stat = 0, n_p = 0, n_q = 0, n_x = 0;
    std::vector<double> pe, qe;
    std::vector<double> rule_t[3], rule_w[3];
    std::vector<pm_channel> ch;
    pm::Tables T;
    // device side
    bool dirty = true;                 // tables need (re)upload
    int device = -1;
    char* d_blob = nullptr;            // all small tables
    pm::NodeLists nl{};                // sorted node lists of the last pattern call (cells [pat_begin, pat_end))
    int64_t* d_cellbase = nullptr;
    int64_t* d_summary = nullptr;      // {nnz, hmax}
    int64_t* h_summary = nullptr;      // pinned
    int hits_cap = 0;
    int hmax = -1, pat_begin = -1, pat_end = -1;     // max hit cells, and the cell range, of the last pattern call
    bool pat_count_only = false;       // the last pattern call only counted: an emit call for the same range reuses its lists
    int64_t counts[3] = {0, 0, 0};     // nodes on the grid, (target, x-node) segments, hit cells of the last pattern call
    bool have_plan = false;
    bool jit_failed = false;           // run-time compilation was tried for this lattice and failed (jit_error says why)
    std::string jit_error;
    pm::FillLaunch plan{};
    int* d_counter = nullptr;          // work counter of the fill kernel
    int* d_hitlist = nullptr;          // hit cells of every source cell of the last pattern call (pm_spmv_implicit), lazily built
    int64_t hitlist_cap = 0;
    bool hitlist_valid = false;
    cudaEvent_t ev_fill0 = nullptr, ev_fill1 = nullptr;   // around the last fill kernel, on its stream (pm_last_fill_ms)
    bool fill_timed = false;
    unsigned long long hash = 0;       // pm::tables_hash of T (selects a generated fill kernel)
    int n_sm = 0;
    pm::DevLattice dev{};
};

namespace {

void free_device(pm_lattice* L)
{
    if (L->d_blob) cudaFree(L->d_blob);
    if (L->nl.key) cudaFree(L->nl.key);
    if (L->nl.rkpos) cudaFree(L->nl.rkpos);
    if (L->nl.ntot) cudaFree(L->nl.ntot);
    if (L->nl.hits) cudaFree(L->nl.hits);
    if (L->nl.nseg) cudaFree(L->nl.nseg);
    if (L->d_cellbase) cudaFree(L->d_cellbase);
    if (L->d_summary) cudaFree(L->d_summary);
    if (L->h_summary) cudaFreeHost(L->h_summary);
    if (L->d_counter) cudaFree(L->d_counter);
    L->d_counter = nullptr;
    if (L->d_hitlist) cudaFree(L->d_hitlist);
    L->d_hitlist = nullptr; L->hitlist_cap = 0; L->hitlist_valid = false;
    if (L->ev_fill0) cudaEventDestroy(L->ev_fill0);
    if (L->ev_fill1) cudaEventDestroy(L->ev_fill1);
    L->ev_fill0 = L->ev_fill1 = nullptr; L->fill_timed = false;
    L->d_blob = nullptr; L->nl = pm::NodeLists{}; L->d_cellbase = nullptr; L->d_summary = nullptr; L->h_summary = nullptr;
    L->hits_cap = 0;
}

// device check + upload of every small table as one blob
int32_t ensure_device(pm_lattice* L)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(PM_ERR_DEVICE, std::string("no CUDA device: ") + cudaGetErrorString(e)); }
    if (!L->dirty && L->device == dev) return PM_OK;     // (cudaGetDeviceProperties costs milliseconds: first use only)
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return fail(PM_ERR_DEVICE, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e));
    if (prop.major < 10) return fail(PM_ERR_DEVICE, "libpm is built for sm_100a (B200); this device is older");
    free_device(L);
    L->device = dev;
    L->n_sm = prop.multiProcessorCount;

    const pm::Tables& T = L->T;
    pm::DevLattice D{};
    D.Np = L->Np; D.Nq = L->Nq; D.n_ch = L->n_ch; D.n_p = L->n_p; D.n_q = L->n_q; D.n_x = L->n_x;
    D.nnode = L->n_p * L->n_q * L->n_x; D.n_cells = L->Np * L->Nq; D.n_words = (D.n_cells + 31) / 32;
    D.pe_pad = next_pow2(L->Np + 2); D.qe_pad = next_pow2(L->Nq + 2);     // at least one +inf sentinel after the last edge
    D.totcoup = T.totcoup; D.n_slot = T.n_slot; D.n_fun = (int)T.fun.size(); D.lmax = T.lmax;
    D.ny = pm::ylm_index(T.lmax, T.lmax) + 1;
    auto magic = [](int d) { return d <= 1 ? 0u : (unsigned)(((1ull << 32) + (unsigned)d - 1) / (unsigned)d); };
    D.mg_npq = magic(L->n_p * L->n_q); D.mg_nq = magic(L->n_q); D.mg_Nq = magic(L->Nq);

    std::vector<char> blob;
    auto put = [&](const void* src, size_t bytes) {
        size_t off = (blob.size() + 15) & ~size_t(15);
        blob.resize(off + bytes);
        if (bytes) std::memcpy(blob.data() + off, src, bytes);
        return off;
    };
    const double inf = std::numeric_limits<double>::infinity();
    std::vector<double> pe(D.pe_pad, inf), qe(D.qe_pad, inf);
    std::copy(L->pe.begin(), L->pe.end(), pe.begin());
    std::copy(L->qe.begin(), L->qe.end(), qe.begin());
    std::vector<double> thp(D.pe_pad, inf), thq(D.qe_pad, inf);          // +inf has the largest bit pattern of all
    for (int k = 0; k <= L->Np; ++k) thp[(size_t)k] = pm::sqrt_threshold(L->pe[(size_t)k]);
    for (int k = 0; k <= L->Nq; ++k) thq[(size_t)k] = pm::sqrt_threshold(L->qe[(size_t)k]);
    std::vector<double> sx(L->n_x), bra;
    for (int c = 0; c < L->n_x; ++c) { const double x = L->rule_t[2][c]; sx[c] = std::sqrt((1.0 - x) * (1.0 + x)); }
    pm::build_bra(T, L->rule_t[2], bra);
    std::vector<int32_t> o_alpha(T.totcoup);
    for (int a = 0; a < L->n_ch; ++a) for (int o = T.cl_off[a]; o < T.cl_off[a + 1]; ++o) o_alpha[o] = a;
    std::vector<int4> fun(T.fun.size());
    for (size_t f = 0; f < T.fun.size(); ++f) fun[f] = make_int4(T.fun[f].sa0, T.fun[f].sb0, T.fun[f].nM, T.fun[f].L);

    const size_t o_pe = put(pe.data(), 8 * pe.size()), o_qe = put(qe.data(), 8 * qe.size());
    const size_t o_thp = put(thp.data(), 8 * thp.size()), o_thq = put(thq.data(), 8 * thq.size());
    std::vector<uint16_t> bkp, bkq;
    pm::bucket_table(thp, L->Np + 1, pm::kBuckets, D.bk_hmin_p, D.bk_sh_p, bkp);
    pm::bucket_table(thq, L->Nq + 1, pm::kBuckets, D.bk_hmin_q, D.bk_sh_q, bkq);
    const size_t o_bkp = put(bkp.data(), 2 * bkp.size()), o_bkq = put(bkq.data(), 2 * bkq.size());
    size_t o_t[3], o_w[3];
    for (int k = 0; k < 3; ++k) { o_t[k] = put(L->rule_t[k].data(), 8 * L->rule_t[k].size()); o_w[k] = put(L->rule_w[k].data(), 8 * L->rule_w[k].size()); }
    const size_t o_sx = put(sx.data(), 8 * sx.size());
    const size_t o_cloff = put(T.cl_off.data(), 4 * T.cl_off.size()), o_cl = put(T.cl.data(), 4 * T.cl.size());
    const size_t o_oa = put(o_alpha.data(), 4 * o_alpha.size());
    const size_t o_bra = put(bra.data(), 8 * bra.size());
    const size_t o_ktoff = put(T.kt_off.data(), 4 * T.kt_off.size()), o_ktip = put(T.kt_ip.data(), 4 * T.kt_ip.size());
    const size_t o_ktiq = put(T.kt_iq.data(), 4 * T.kt_iq.size()), o_ktc = put(T.kt_c.data(), 8 * T.kt_c.size());
    const size_t o_fun = put(fun.data(), sizeof(int4) * fun.size());
    const size_t o_otoff = put(T.ot_off.data(), 4 * T.ot_off.size()), o_otf = put(T.ot_f.data(), 4 * T.ot_f.size());
    const size_t o_otc = put(T.ot_c.data(), 8 * T.ot_c.size());
    const size_t o_ya = put(T.ya.data(), 8 * T.ya.size()), o_yb = put(T.yb.data(), 8 * T.yb.size());
    const size_t o_yd = put(T.ydiag.data(), 8 * T.ydiag.size());

    if ((e = cudaMalloc(&L->d_blob, blob.size())) != cudaSuccess) return cuda_fail(e, "cudaMalloc(tables)");
    if ((e = cudaMemcpy(L->d_blob, blob.data(), blob.size(), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e, "cudaMemcpy(tables)");
    if ((e = cudaMalloc(&L->d_summary, 4 * sizeof(int64_t))) != cudaSuccess) return cuda_fail(e, "cudaMalloc(summary)");
    if ((e = cudaMalloc(&L->d_counter, sizeof(int))) != cudaSuccess) return cuda_fail(e, "cudaMalloc(counter)");
    if ((e = cudaEventCreate(&L->ev_fill0)) != cudaSuccess || (e = cudaEventCreate(&L->ev_fill1)) != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
    if ((e = cudaMallocHost(&L->h_summary, 4 * sizeof(int64_t))) != cudaSuccess) return cuda_fail(e, "cudaMallocHost(summary)");
    char* b = L->d_blob;
    D.pe = (const double*)(b + o_pe); D.qe = (const double*)(b + o_qe);
    D.thr_p = (const double*)(b + o_thp); D.thr_q = (const double*)(b + o_thq);
    D.bk_p = (const unsigned short*)(b + o_bkp); D.bk_q = (const unsigned short*)(b + o_bkq);
    D.tp = (const double*)(b + o_t[0]); D.wp = (const double*)(b + o_w[0]);
    D.tq = (const double*)(b + o_t[1]); D.wq = (const double*)(b + o_w[1]);
    D.tx = (const double*)(b + o_t[2]); D.wx = (const double*)(b + o_w[2]);
    D.sx = (const double*)(b + o_sx);
    D.cl_off = (const int*)(b + o_cloff); D.cl = (const int*)(b + o_cl); D.o_alpha = (const int*)(b + o_oa);
    D.bra = (const double*)(b + o_bra);
    D.kt_off = (const int*)(b + o_ktoff); D.kt_ip = (const int*)(b + o_ktip); D.kt_iq = (const int*)(b + o_ktiq);
    D.kt_c = (const double*)(b + o_ktc);
    D.fun = (const int4*)(b + o_fun);
    D.ot_off = (const int*)(b + o_otoff); D.ot_f = (const int*)(b + o_otf); D.ot_c = (const double*)(b + o_otc);
    D.ya = (const double*)(b + o_ya); D.yb = (const double*)(b + o_yb); D.ydiag = (const double*)(b + o_yd);
    L->dev = D;
    L->dirty = false;
    L->hmax = -1;
    L->have_plan = false;
    return PM_OK;
}

int32_t ensure_cell_scratch(pm_lattice* L, int n_blk)
{
    if (n_blk <= L->hits_cap) return PM_OK;
    if (L->nl.key) cudaFree(L->nl.key);
    if (L->nl.rkpos) cudaFree(L->nl.rkpos);
    if (L->nl.ntot) cudaFree(L->nl.ntot);
    if (L->nl.hits) cudaFree(L->nl.hits);
    if (L->nl.nseg) cudaFree(L->nl.nseg);
    if (L->d_cellbase) cudaFree(L->d_cellbase);
    L->nl = pm::NodeLists{}; L->d_cellbase = nullptr; L->hits_cap = 0;
    const size_t nn = (size_t)n_blk * (size_t)L->dev.nnode;
    cudaError_t e;
    if ((e = cudaMalloc(&L->nl.key, sizeof(unsigned) * nn)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(node lists)");
    if ((e = cudaMalloc(&L->nl.rkpos, sizeof(unsigned short) * nn)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(node lists)");
    if ((e = cudaMalloc(&L->nl.ntot, sizeof(int) * (size_t)n_blk)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(ntot)");
    if ((e = cudaMalloc(&L->nl.hits, sizeof(int) * (size_t)n_blk)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(hits)");
    if ((e = cudaMalloc(&L->nl.nseg, sizeof(int) * (size_t)n_blk)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(nseg)");
    if ((e = cudaMalloc(&L->d_cellbase, sizeof(int64_t) * ((size_t)n_blk + 1))) != cudaSuccess) return cuda_fail(e, "cudaMalloc(cellbase)");
    L->hits_cap = n_blk;
    return PM_OK;
}

bool bad_edges(const double* e, int N)
{
    if (!(e[0] >= 0.0)) return true;
    for (int k = 0; k <= N; ++k) if (!std::isfinite(e[k]) || e[k] > 1e150) return true;      // e*e must stay finite
    for (int k = 0; k < N; ++k) if (!(e[k + 1] > e[k])) return true;
    return false;
}

}  // namespace

extern "C" {

const char* pm_last_error(void) { return g_err.c_str(); }
int64_t pm_launch_count(void) { return pm::launch_count(); }

int32_t pm_lattice_create(const double* p_edges, int32_t Np, const double* q_edges, int32_t Nq,
                          const pm_channel* ch, int32_t n_ch, int32_t J2, int32_t parity, int32_t T2, int32_t statistics,
                          int32_t n_p, int32_t n_q, int32_t n_x, pm_lattice** out)
{
    if (!out) return fail(PM_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (!p_edges || !q_edges || !ch) return fail(PM_ERR_ARG, "NULL input pointer");
    if (Np < 1 || Nq < 1) return fail(PM_ERR_GRID, "need at least one cell per axis");
    if ((int64_t)Np * Nq > 262144) return fail(PM_ERR_GRID, "Np*Nq exceeds 262144");
    if ((int64_t)Np * Nq * Nq >= (int64_t(1) << 32)) return fail(PM_ERR_GRID, "Np*Nq*Nq must be below 2^32 (exact division of cell ids by Nq)");
    if (bad_edges(p_edges, Np)) return fail(PM_ERR_GRID, "p_edges must be finite (at most 1e150), strictly increasing, p_edges[0] >= 0");
    if (bad_edges(q_edges, Nq)) return fail(PM_ERR_GRID, "q_edges must be finite (at most 1e150), strictly increasing, q_edges[0] >= 0");
    if (n_ch < 1 || n_ch > PM_MAX_CHANNELS) return fail(PM_ERR_CHANNEL, "n_ch out of range");
    if (n_p < 1 || n_q < 1 || n_x < 1 || n_p > PM_MAX_ORDER || n_q > PM_MAX_ORDER || n_x > PM_MAX_ORDER)
        return fail(PM_ERR_ORDER, "quadrature order out of range 1..64");
    if ((int64_t)n_p * n_q * n_x > 16384) return fail(PM_ERR_ORDER, "n_p*n_q*n_x exceeds 16384");
    if ((int64_t)Np * Nq * n_ch >= (int64_t(1) << 31)) return fail(PM_ERR_OVERFLOW, "M = n_ch*Np*Nq must be below 2^31");
    std::string msg = pm::validate_channels(ch, n_ch, J2, parity, T2, statistics);
    if (!msg.empty()) return fail(PM_ERR_CHANNEL, msg);
    pm_lattice* L = new (std::nothrow) pm_lattice();
    if (!L) return fail(PM_ERR_NOMEM, "out of host memory");
    L->Np = Np; L->Nq = Nq; L->n_ch = n_ch; L->J2 = J2; L->parity = parity; L->T2 = T2; L->stat = statistics;
    L->n_p = n_p; L->n_q = n_q; L->n_x = n_x;
    L->pe.assign(p_edges, p_edges + Np + 1); L->qe.assign(q_edges, q_edges + Nq + 1);
    L->ch.assign(ch, ch + n_ch);
    msg = pm::build_tables(ch, n_ch, J2, T2, statistics, L->T);
    if (!msg.empty()) { delete L; return fail(PM_ERR_CHANNEL, msg); }
    L->hash = pm::tables_hash(L->T);
    if ((int)L->T.fun.size() > pm::kFillMaxFun || L->T.n_slot > pm::kFillMaxSlot) {
        delete L; return fail(PM_ERR_CHANNEL, "channel set needs more orbital functions than this build supports");
    }
    const int orders[3] = {n_p, n_q, n_x};
    for (int k = 0; k < 3; ++k) pm::gauss_legendre(orders[k], L->rule_t[k], L->rule_w[k]);
    *out = L;
    return PM_OK;
}

int32_t pm_lattice_destroy(pm_lattice* lat)
{
    if (!lat) return PM_OK;
    free_device(lat);
    delete lat;
    return PM_OK;
}

int32_t pm_lattice_dims(const pm_lattice* lat, int64_t* M, int32_t* n_cells)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    if (M) *M = (int64_t)lat->Np * lat->Nq * lat->n_ch;
    if (n_cells) *n_cells = lat->Np * lat->Nq;
    return PM_OK;
}

int32_t pm_lattice_rule(const pm_lattice* lat, int32_t axis, double* nodes, double* weights)
{
    if (!lat || axis < 0 || axis > 2) return fail(PM_ERR_ARG, "bad lattice or axis");
    if (nodes) std::copy(lat->rule_t[axis].begin(), lat->rule_t[axis].end(), nodes);
    if (weights) std::copy(lat->rule_w[axis].begin(), lat->rule_w[axis].end(), weights);
    return PM_OK;
}

int32_t pm_lattice_set_rule(pm_lattice* lat, int32_t axis, const double* nodes, const double* weights)
{
    if (!lat || axis < 0 || axis > 2 || !nodes || !weights) return fail(PM_ERR_ARG, "bad lattice, axis or NULL rule");
    const int n = (int)lat->rule_t[axis].size();
    for (int k = 0; k < n; ++k) {
        if (!std::isfinite(nodes[k]) || !std::isfinite(weights[k]) || !(nodes[k] > -1.0 && nodes[k] < 1.0))
            return fail(PM_ERR_ORDER, "rule nodes must lie inside (-1,1) and be finite");
        if (k && !(nodes[k] > nodes[k - 1])) return fail(PM_ERR_ORDER, "rule nodes must be strictly increasing");
    }
    if (axis == 2)
        for (int k = 0; k < n; ++k)
            if (nodes[k] != -nodes[n - 1 - k] || weights[k] != weights[n - 1 - k])
                return fail(PM_ERR_ORDER, "the x-rule must be symmetric under x -> -x (both cyclic terms are folded into one)");
    lat->rule_t[axis].assign(nodes, nodes + n);
    lat->rule_w[axis].assign(weights, weights + n);
    lat->dirty = true;
    return PM_OK;
}

int32_t pm_lattice_coupling(const pm_lattice* lat, uint8_t* coupled, int32_t* n_functions)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    if (coupled) std::copy(lat->T.coupled.begin(), lat->T.coupled.end(), coupled);
    if (n_functions) *n_functions = (int32_t)lat->T.fun.size();
    return PM_OK;
}

int32_t pm_lattice_work(const pm_lattice* lat, double* flop_per_node, double* flop_per_segment, double* flop_per_hit_cell,
                        int32_t* n_coupled_pairs)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    const pm::Tables& T = lat->T;
    // per node on the grid (pm_fill.cuh, phase C): node map 16, weight and omega 7 (one rsqrt), rotated directions 20
    // (two rsqrt), the generated ket code, and one add per slot in the segment sum (phase D)
    if (flop_per_node) *flop_per_node = 16.0 + 7.0 + 20.0 + pm::ket_flops(T) + (double)T.n_slot;
    // per (target, x-node) segment: sum_M bra*S per orbital function (nM multiply-adds) and one add into the target sum
    double seg = 0.0;
    for (const pm::OrbFun& f : T.fun) seg += 2.0 * f.nM;
    if (flop_per_segment) *flop_per_segment = seg;
    // per hit cell: normalisation 5, per output one multiply-add per (channel pair, L) term and the scaling by the norm
    if (flop_per_hit_cell) *flop_per_hit_cell = 5.0 + 2.0 * (double)T.ot_c.size();
    if (n_coupled_pairs) *n_coupled_pairs = T.totcoup;
    return PM_OK;
}

int32_t pm_pattern_counts(const pm_lattice* lat, int64_t* nodes_on_grid, int64_t* segments, int64_t* hit_cells)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    if (lat->hmax < 0) return fail(PM_ERR_STATE, "pm_pattern_counts needs a preceding pm_pattern");
    if (nodes_on_grid) *nodes_on_grid = lat->counts[0];
    if (segments) *segments = lat->counts[1];
    if (hit_cells) *hit_cells = lat->counts[2];
    return PM_OK;
}

const char* pm_lattice_fill_kernel(const pm_lattice* lat)
{
    if (!lat) return "";
    if (pm::fill_has_spec(lat->hash)) return pm::fill_variant_name(lat->hash);
    if (lat->have_plan) return lat->plan.name;                              // what the last fill ran: "jit" or "generic"
    return (pm::jit_enabled() && !lat->jit_failed) ? "jit" : "generic";
}

int32_t pm_set_jit(int32_t enabled)
{
    pm::jit_set_enabled(enabled != 0);
    return PM_OK;
}

int32_t pm_diag_jit_compile(const pm_lattice* lat, int64_t* cubin_bytes)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    std::string err;
    size_t n = 0;
    if (!pm::jit_compile_check(lat->T, 12, 4, &n, err)) return fail(PM_ERR_STATE, err);
    if (cubin_bytes) *cubin_bytes = (int64_t)n;
    return PM_OK;
}

double pm_diag_sqrt_threshold(double edge) { return pm::sqrt_threshold(edge); }

int32_t pm_diag_dfma_tflops(double* tflops, void* cuda_stream)
{
    if (!tflops) return fail(PM_ERR_ARG, "NULL argument");
    int dev = -1;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) {
        cudaGetLastError();
        return fail(PM_ERR_DEVICE, "no CUDA device");
    }
    if (prop.major < 10) return fail(PM_ERR_DEVICE, "libpm is built for sm_100a (B200); this device is older");
    cudaError_t e = pm::measure_dfma(prop.multiProcessorCount, tflops, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "k_dfma_peak");
    return PM_OK;
}

int32_t pm_pattern(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx,
                   int64_t colidx_capacity, int64_t* nnz_host, void* cuda_stream)
{
    if (!lat || !d_rowptr || !nnz_host) return fail(PM_ERR_ARG, "NULL argument");
    const int n_cells = lat->Np * lat->Nq;
    if (cell_begin < 0 || cell_end > n_cells || cell_begin > cell_end) return fail(PM_ERR_ARG, "bad cell range");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int n_blk = cell_end - cell_begin;
    cudaError_t e;
    if (n_blk == 0) {
        if ((e = cudaMemsetAsync(d_rowptr, 0, sizeof(int64_t), st)) != cudaSuccess) return cuda_fail(e, "memset");
        if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e, "sync");
        *nnz_host = 0; lat->hmax = 0; lat->pat_begin = cell_begin; lat->pat_end = cell_end;
        lat->counts[0] = lat->counts[1] = lat->counts[2] = 0;
        return PM_OK;
    }
    // Two-phase use (count, allocate, emit): the emit call reuses the node lists of the count call of the same range,
    // so the nodes are mapped once.  Any other call maps afresh.
    const bool reuse = lat->hmax >= 0 && lat->pat_count_only && d_colidx && lat->pat_begin == cell_begin && lat->pat_end == cell_end
                    && lat->hits_cap >= n_blk;
    lat->pat_count_only = (d_colidx == nullptr);
    if (!reuse) lat->hitlist_valid = false;
    if (!reuse) {
        lat->hmax = -1;
        if ((rc = ensure_cell_scratch(lat, n_blk))) return rc;
        if ((e = pm::launch_map_sort(lat->dev, cell_begin, n_blk, lat->nl, st)) != cudaSuccess) return cuda_fail(e, "k_map_sort");
    }
    if ((e = pm::launch_scan_rows(lat->dev, n_blk, lat->nl, lat->d_cellbase, d_rowptr, lat->d_summary, st)) != cudaSuccess)
        return cuda_fail(e, "k_scan_rows");
    if ((e = cudaMemcpyAsync(lat->h_summary, lat->d_summary, 4 * sizeof(int64_t), cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(e, "cudaMemcpyAsync(summary)");
    if ((e = cudaStreamSynchronize(st)) != cudaSuccess) return cuda_fail(e, "pattern: map/scan");
    *nnz_host = lat->h_summary[0];
    lat->hmax = (int)lat->h_summary[1]; lat->pat_begin = cell_begin; lat->pat_end = cell_end;
    lat->counts[0] = lat->h_summary[2]; lat->counts[1] = lat->h_summary[3]; lat->counts[2] = *nnz_host / lat->T.totcoup;
    if (!d_colidx) return PM_OK;
    if (*nnz_host > colidx_capacity) return fail(PM_ERR_OVERFLOW, "d_colidx too small for this block's nnz");
    if ((e = pm::launch_emit_cols(lat->dev, n_blk, lat->nl, lat->hmax, d_rowptr, d_colidx, st)) != cudaSuccess)
        return cuda_fail(e, "k_emit_cols");
    return PM_OK;
}

}  // extern "C"

namespace {

// values (and, when d_colidx is given, column indices) of the block of the last pattern call
int32_t fill_block(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, const int64_t* d_rowptr, double* d_vals,
                   int32_t* d_colidx, cudaStream_t st)
{
    if (lat->hmax < 0 || cell_begin != lat->pat_begin || cell_end != lat->pat_end)
        return fail(PM_ERR_STATE, "pm_fill needs a preceding pm_pattern of the same cell range on this lattice");
    if (cell_begin == cell_end) return PM_OK;
    const int n_blk = cell_end - cell_begin;
    cudaError_t e;
    if (!lat->have_plan && !pm::fill_has_spec(lat->hash) && pm::jit_enabled() && !lat->jit_failed) {
        // no build-time kernel for this channel set: specialise at run time (pm_jit.hpp), else fall back below
        if (pm::fill_plan_jit(lat->dev, lat->T, lat->hash, lat->n_sm, &lat->plan, lat->jit_error)) lat->have_plan = true;
        else lat->jit_failed = true;
    }
    if (!lat->have_plan) {
        e = pm::fill_plan(lat->dev, lat->hash, lat->n_sm, &lat->plan);
        if (e == cudaErrorInvalidConfiguration) { cudaGetLastError(); return fail(PM_ERR_NOMEM, "channel set needs more shared memory than one SM has"); }
        if (e != cudaSuccess) return cuda_fail(e, "fill_plan");
        lat->have_plan = true;
    }
    if ((e = cudaEventRecord(lat->ev_fill0, st)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    e = pm::launch_fill(lat->dev, lat->plan, cell_begin, n_blk, lat->nl, d_rowptr, d_vals, d_colidx, lat->d_counter, st);
    if (e != cudaSuccess) return cuda_fail(e, "k_fill");
    if ((e = cudaEventRecord(lat->ev_fill1, st)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    lat->fill_timed = true;
    return PM_OK;
}

}  // namespace

extern "C" {

int32_t pm_fill(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, const int64_t* d_rowptr, double* d_vals, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_vals) return fail(PM_ERR_ARG, "NULL argument");
    const int n_cells = lat->Np * lat->Nq;
    if (cell_begin < 0 || cell_end > n_cells || cell_begin > cell_end) return fail(PM_ERR_ARG, "bad cell range");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    return fill_block(lat, cell_begin, cell_end, d_rowptr, d_vals, nullptr, (cudaStream_t)cuda_stream);
}

int32_t pm_spmv_implicit(pm_lattice* lat, const int64_t* d_rowptr, const double* d_vals, const double* d_x, double* d_y, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_vals || !d_x || !d_y) return fail(PM_ERR_ARG, "NULL argument");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    const int n_cells = lat->Np * lat->Nq;
    if (lat->hmax < 0 || lat->pat_begin != 0 || lat->pat_end != n_cells)
        return fail(PM_ERR_STATE, "pm_spmv_implicit needs the node lists of a pm_pattern / pm_build call over the whole lattice");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e;
    if (!lat->hitlist_valid) {
        const int64_t need = std::max<int64_t>(lat->counts[2], 1);
        if (need > lat->hitlist_cap) {
            if (lat->d_hitlist) cudaFree(lat->d_hitlist);
            lat->d_hitlist = nullptr; lat->hitlist_cap = 0;
            if ((e = cudaMalloc(&lat->d_hitlist, sizeof(int) * (size_t)need)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(hit list)");
            lat->hitlist_cap = need;
        }
        if ((e = pm::launch_hit_list(lat->dev, n_cells, lat->nl, lat->d_cellbase, lat->d_hitlist, st)) != cudaSuccess) return cuda_fail(e, "k_hit_list");
        lat->hitlist_valid = true;
    }
    e = pm::launch_spmv_implicit(lat->dev, (int64_t)n_cells * lat->n_ch, d_rowptr, lat->nl.hits, lat->d_cellbase, lat->d_hitlist, d_vals, d_x, d_y, st);
    if (e != cudaSuccess) return cuda_fail(e, "k_spmv_implicit");
    return PM_OK;
}

int32_t pm_block_apply(pm_lattice* lat, const double* d_blocks, const double* d_diag, const double* d_in, double* d_out, void* cuda_stream)
{
    if (!lat || !d_blocks || !d_in || !d_out) return fail(PM_ERR_ARG, "NULL argument");
    if (d_in == d_out) return fail(PM_ERR_ARG, "pm_block_apply cannot work in place");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    cudaError_t e = pm::launch_block_apply(lat->Np, lat->Nq, lat->n_ch, d_blocks, d_diag, d_in, d_out, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "k_block_apply");
    return PM_OK;
}

int32_t pm_kernel_apply(pm_lattice* lat, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                        const double* d_O, const double* d_Vt, const double* d_g1, const double* d_u, double* d_out,
                        double* d_work, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_vals || !d_O || !d_Vt || !d_g1 || !d_u || !d_out || !d_work)
        return fail(PM_ERR_ARG, "NULL argument");
    const int64_t M = (int64_t)lat->Np * lat->Nq * lat->n_ch;
    double* t1 = d_work;                                   // V~1 G1 u
    double* t2 = d_work + M;                               // P0 V~1 G1 u
    int32_t rc = pm_block_apply(lat, d_Vt, d_g1, d_u, t1, cuda_stream);
    if (rc) return rc;
    rc = d_colidx ? pm_spmv(lat, M, d_rowptr, d_colidx, d_vals, t1, t2, cuda_stream)
                  : pm_spmv_implicit(lat, d_rowptr, d_vals, t1, t2, cuda_stream);      // columns implied by the hit lists
    if (rc) return rc;
    return pm_block_apply(lat, d_O, nullptr, t2, d_out, cuda_stream);
}

int32_t pm_last_fill_ms(pm_lattice* lat, float* ms)
{
    if (!lat || !ms) return fail(PM_ERR_ARG, "NULL argument");
    if (!lat->fill_timed) return fail(PM_ERR_STATE, "no fill kernel has been launched on this lattice");
    cudaError_t e = cudaEventSynchronize(lat->ev_fill1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(ms, lat->ev_fill0, lat->ev_fill1);
    if (e != cudaSuccess) return cuda_fail(e, "pm_last_fill_ms");
    return PM_OK;
}

int32_t pm_build(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                 int64_t capacity, int64_t* nnz_host, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_colidx || !d_vals || !nnz_host) return fail(PM_ERR_ARG, "NULL argument");
    // pattern pass without the column kernel: node lists, rowptr, nnz ...
    int32_t rc = pm_pattern(lat, cell_begin, cell_end, d_rowptr, nullptr, 0, nnz_host, cuda_stream);
    if (rc) return rc;
    if (*nnz_host > capacity) return fail(PM_ERR_OVERFLOW, "d_colidx / d_vals too small for this block's nnz");
    // ... then one kernel writes the column index and the value of every nonzero
    return fill_block(lat, cell_begin, cell_end, d_rowptr, d_vals, d_colidx, (cudaStream_t)cuda_stream);
}

int32_t pm_spmv(pm_lattice* lat, int64_t n_rows, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                const double* d_x, double* d_y, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_x || !d_y || n_rows < 0) return fail(PM_ERR_ARG, "NULL argument");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    if (n_rows == 0) return PM_OK;
    if (!d_colidx || !d_vals) return fail(PM_ERR_ARG, "NULL colidx/vals");
    cudaError_t e = pm::launch_spmv(n_rows, d_rowptr, d_colidx, d_vals, d_x, d_y, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "k_spmv");
    return PM_OK;
}

}  // extern "C"
