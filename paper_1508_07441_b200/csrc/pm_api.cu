// pm_api.cu — the C ABI of libpm (include/pm.h): handle management, validation, table upload and the entry points
// pm_pattern / pm_fill / pm_build / pm_spmv / iteration step / sharding helpers.  No torch types, no CPU fallback.
//
// Two host objects: a GEOMETRY (grids, quadrature rules, their device tables, and the node lists the pattern pass
// leaves: everything that does not depend on the channel set) shared by reference count between the lattices created
// by pm_lattice_attach, and the LATTICE proper (channel set, recoupling tables, fill kernel).  The geometric pattern of
// a cell range is therefore computed once for every J^pi on the same grids (PAPER.md:L374,
// L394: "62 spin-orbital channels and all states ... up to J_max = 17/2").
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <new>
#include <mutex>
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
    cudaGetLastError();
    return e == cudaErrorMemoryAllocation ? PM_ERR_NOMEM : PM_ERR_CUDA;
}

int next_pow2(int n) { int p = 1; while (p < n) p <<= 1; return p; }

}  // namespace

namespace pm {
// used by the other translation units of the library (pm_stream.cu): every failing path leaves a message for pm_last_error()
int32_t set_error(int32_t code, const std::string& msg) { return fail(code, msg); }
int32_t set_cuda_error(cudaError_t e, const char* where) { return cuda_fail(e, where); }
}  // namespace pm

// Everything that depends on the grids and the quadrature orders only.
struct pm_geometry {
    int refs = 1;
    int Np = 0, Nq = 0, n_p = 0, n_q = 0, n_x = 0;
    std::vector<double> pe, qe;
    std::vector<double> rule_t[3], rule_w[3];
    uint64_t version = 1;              // bumped by pm_lattice_set_rule: device tables and node lists are stale
    // device side
    uint64_t dev_version = 0;          // version the device tables were built from (0: none)
    int device = -1, n_sm = 0;
    char* d_blob = nullptr;            // edges, sqrt-thresholds, bucket tables, rules
    pm::DevLattice geo{};              // the geometric fields of DevLattice
    pm::NodeLists nl{};                // sorted node lists of the last pattern call (cells [pat_begin, pat_end))
    int64_t* d_cellbase = nullptr;     // exclusive scan of the hit counts of that call
    int cells_cap = 0;
    int64_t* d_summary = nullptr;      // {nnz, max hits, nodes on the grid, segments, overflow flag}
    int64_t* h_summary = nullptr;      // pinned copy
    cudaEvent_t ev_summary = nullptr;  // recorded after the copy
    bool summary_pending = false;      // the host has not looked at h_summary yet
    int* d_counter = nullptr;          // [0] work counter of the fill kernel, [1] of k_map_sort
    void* d_sort_scratch = nullptr;    // k_map_sort: targets of the cells in flight (a few MB)
    size_t sort_scratch_bytes = 0;
    int* d_hitlist = nullptr;          // hit cells of every source cell of the last pattern call, lazily built
    int64_t hitlist_cap = 0;
    bool hitlist_valid = false;
    bool lists_valid = false;          // nl holds the lists of [pat_begin, pat_end)
    bool pat_count_only = false;       // the last pattern call only counted: an emit call of the same range reuses its lists
    int pat_begin = -1, pat_end = -1;
    uint64_t pattern_serial = 0;       // counts the pattern passes (pm_operator_apply checks its sums against it)
    int totcoup_of_scan = 0;           // the channel-pair count the last scan multiplied the hit counts with
    int hmax = -1;
    int64_t nnz = 0, nodes_on_grid = 0, hit_cells = 0, segments = -1, overflow = 0, chunks = 0;
    cudaStream_t last_stream = nullptr;
};

struct pm_lattice {
    uint64_t id = 0;                   // unique per created lattice (pm_stream.cu keys its cached block plan with it)
    pm_geometry* G = nullptr;
    int n_ch = 0, J2 = 0, parity = 1, T2 = 0, stat = 0;
    int norm = 0;                      // cell normalisation (pm_lattice_set_normalisation)
    std::vector<pm_channel> ch;
    pm::Tables T;
    // device side
    uint64_t geo_version = 0;          // geometry version the channel tables were uploaded for
    int device = -1;
    char* d_blob = nullptr;            // channel tables (coupled lists, bra harmonics, term lists)
    bool have_plan = false;            // every group has its launch plan
    bool jit_failed = false;           // run-time compilation was tried for this lattice and failed (jit_error says why)
    std::string jit_error;
    std::vector<pm::GroupTables> groups;   // column-channel groups the table-driven kernel can hold (one for small sets)
    std::vector<pm::GroupTables> jgroups;  // the groups a specialised kernel can hold (ket slots in registers): one for the sets of
                                           // BASELINE.json's configs, up to 13 for the 62-channel sets
    struct GroupDev { pm::DevLattice dev; pm::FillLaunch plan; };
    std::vector<GroupDev> gdev, gdev_j;
    bool use_j = false;                // the last plan runs the specialised kernels of jgroups
    // several groups: the fill goes through the per-pair sums (pm_fill.cuh mode 2 + k_op_expand)
    int op_stride = 0;                 // doubles per hit cell pair: the groups' functions, each group's range padded to 4
    std::vector<int> op_off;           // first position of each group of jgroups
    const unsigned short* d_xpos = nullptr;    // [totcoup][4] position of each term's function in a pair's sums (in d_blob)
    const double* d_xc = nullptr;              // [totcoup][4] coefficients
    double* d_opA = nullptr;           // the sums of the last fill, library-owned scratch
    int64_t opA_cap = 0;
    uint64_t op_serial = 0;            // pattern pass the sums of pm_operator_build belong to (0: none)
    int op_norm = 0;
    cudaEvent_t ev_fill0 = nullptr, ev_fill1 = nullptr;   // around the last fill kernel, on its stream (pm_last_fill_ms)
    bool fill_timed = false;
    unsigned long long hash = 0;       // pm::tables_hash of T (selects a generated fill kernel)
    pm::DevLattice dev{};
};

namespace {

void free_lists(pm_geometry* G)
{
    if (G->nl.key) cudaFree(G->nl.key);
    if (G->nl.ntot) cudaFree(G->nl.ntot);
    if (G->nl.hits) cudaFree(G->nl.hits);
    if (G->nl.chunk) cudaFree(G->nl.chunk);
    if (G->nl.nchunk) cudaFree(G->nl.nchunk);
    if (G->d_cellbase) cudaFree(G->d_cellbase);
    G->nl = pm::NodeLists{}; G->d_cellbase = nullptr; G->cells_cap = 0;
    G->lists_valid = false; G->hitlist_valid = false; G->hmax = -1;
}

void free_geometry_device(pm_geometry* G)
{
    free_lists(G);
    if (G->d_blob) cudaFree(G->d_blob);
    if (G->d_summary) cudaFree(G->d_summary);
    if (G->h_summary) cudaFreeHost(G->h_summary);
    if (G->ev_summary) cudaEventDestroy(G->ev_summary);
    if (G->d_counter) cudaFree(G->d_counter);
    if (G->d_hitlist) cudaFree(G->d_hitlist);
    if (G->d_sort_scratch) cudaFree(G->d_sort_scratch);
    G->d_sort_scratch = nullptr; G->sort_scratch_bytes = 0;
    G->d_blob = nullptr; G->d_summary = nullptr; G->h_summary = nullptr; G->ev_summary = nullptr; G->d_counter = nullptr;
    G->d_hitlist = nullptr; G->hitlist_cap = 0; G->summary_pending = false; G->dev_version = 0;
}

void free_lattice_device(pm_lattice* L)
{
    if (L->d_blob) cudaFree(L->d_blob);
    if (L->ev_fill0) cudaEventDestroy(L->ev_fill0);
    if (L->ev_fill1) cudaEventDestroy(L->ev_fill1);
    if (L->d_opA) cudaFree(L->d_opA);
    L->d_opA = nullptr; L->opA_cap = 0;
    L->d_blob = nullptr; L->ev_fill0 = L->ev_fill1 = nullptr; L->fill_timed = false; L->geo_version = 0; L->have_plan = false; L->use_j = false;
}

struct Blob {
    std::vector<char> b;
    size_t put(const void* src, size_t bytes)
    {
        const size_t off = (b.size() + 15) & ~size_t(15);
        b.resize(off + bytes);
        if (bytes) std::memcpy(b.data() + off, src, bytes);
        return off;
    }
};

// device check + upload of the geometric tables
int32_t ensure_geometry(pm_geometry* G)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(PM_ERR_DEVICE, std::string("no CUDA device: ") + cudaGetErrorString(e)); }
    if (G->dev_version == G->version && G->device == dev) return PM_OK;     // (cudaGetDeviceProperties costs milliseconds: first use only)
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(PM_ERR_DEVICE, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e)); }
    if (prop.major < 10) return fail(PM_ERR_DEVICE, "libpm is built for sm_100a (B200); this device is older");
    free_geometry_device(G);
    G->device = dev;
    G->n_sm = prop.multiProcessorCount;

    pm::DevLattice D{};
    D.Np = G->Np; D.Nq = G->Nq; D.n_p = G->n_p; D.n_q = G->n_q; D.n_x = G->n_x;
    D.nnode = G->n_p * G->n_q * G->n_x; D.n_cells = G->Np * G->Nq; D.n_words = (D.n_cells + 31) / 32;
    D.pe_pad = next_pow2(G->Np + 2); D.qe_pad = next_pow2(G->Nq + 2);     // at least one +inf sentinel after the last edge
    auto magic = [](int d) { return d <= 1 ? 0u : (unsigned)(((1ull << 32) + (unsigned)d - 1) / (unsigned)d); };
    D.mg_npq = magic(G->n_p * G->n_q); D.mg_nq = magic(G->n_q); D.mg_Nq = magic(G->Nq);

    Blob B;
    const double inf = std::numeric_limits<double>::infinity();
    std::vector<double> pe(D.pe_pad, inf), qe(D.qe_pad, inf);
    std::copy(G->pe.begin(), G->pe.end(), pe.begin());
    std::copy(G->qe.begin(), G->qe.end(), qe.begin());
    std::vector<double> thp(D.pe_pad, inf), thq(D.qe_pad, inf);          // +inf has the largest bit pattern of all
    for (int k = 0; k <= G->Np; ++k) thp[(size_t)k] = pm::sqrt_threshold(G->pe[(size_t)k]);
    for (int k = 0; k <= G->Nq; ++k) thq[(size_t)k] = pm::sqrt_threshold(G->qe[(size_t)k]);
    std::vector<double> sx(G->n_x);
    for (int c = 0; c < G->n_x; ++c) { const double x = G->rule_t[2][c]; sx[c] = std::sqrt((1.0 - x) * (1.0 + x)); }
    const size_t o_pe = B.put(pe.data(), 8 * pe.size()), o_qe = B.put(qe.data(), 8 * qe.size());
    const size_t o_thp = B.put(thp.data(), 8 * thp.size()), o_thq = B.put(thq.data(), 8 * thq.size());
    std::vector<uint16_t> bkp, bkq;
    pm::bucket_table(thp, G->Np + 1, pm::kBuckets, D.bk_hmin_p, D.bk_sh_p, bkp);
    pm::bucket_table(thq, G->Nq + 1, pm::kBuckets, D.bk_hmin_q, D.bk_sh_q, bkq);
    const size_t o_bkp = B.put(bkp.data(), 2 * bkp.size()), o_bkq = B.put(bkq.data(), 2 * bkq.size());
    D.bk_kmax = 0;                                      // most thresholds in one bucket (the fast location compares kLocK of them at once)
    for (int k = 0; k < pm::kBuckets; ++k) {
        D.bk_kmax = std::max(D.bk_kmax, (k + 1 < pm::kBuckets ? (int)bkp[(size_t)k + 1] : G->Np + 1) - (int)bkp[(size_t)k]);
        D.bk_kmax = std::max(D.bk_kmax, (k + 1 < pm::kBuckets ? (int)bkq[(size_t)k + 1] : G->Nq + 1) - (int)bkq[(size_t)k]);
    }
    size_t o_t[3], o_w[3];
    for (int k = 0; k < 3; ++k) { o_t[k] = B.put(G->rule_t[k].data(), 8 * G->rule_t[k].size()); o_w[k] = B.put(G->rule_w[k].data(), 8 * G->rule_w[k].size()); }
    const size_t o_sx = B.put(sx.data(), 8 * sx.size());

    if ((e = cudaMalloc(&G->d_blob, B.b.size())) != cudaSuccess) return cuda_fail(e, "cudaMalloc(geometry tables)");
    if ((e = cudaMemcpy(G->d_blob, B.b.data(), B.b.size(), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e, "cudaMemcpy(geometry tables)");
    if ((e = cudaMalloc(&G->d_summary, 8 * sizeof(int64_t))) != cudaSuccess) return cuda_fail(e, "cudaMalloc(summary)");
    if ((e = cudaMemset(G->d_summary, 0, 8 * sizeof(int64_t))) != cudaSuccess) return cuda_fail(e, "cudaMemset(summary)");
    if ((e = cudaMalloc(&G->d_counter, 2 * sizeof(int))) != cudaSuccess) return cuda_fail(e, "cudaMalloc(counter)");
    if ((e = cudaEventCreateWithFlags(&G->ev_summary, cudaEventDisableTiming)) != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
    if ((e = cudaMallocHost(&G->h_summary, 8 * sizeof(int64_t))) != cudaSuccess) return cuda_fail(e, "cudaMallocHost(summary)");
    char* b = G->d_blob;
    D.pe = (const double*)(b + o_pe); D.qe = (const double*)(b + o_qe);
    D.thr_p = (const double*)(b + o_thp); D.thr_q = (const double*)(b + o_thq);
    D.bk_p = (const unsigned short*)(b + o_bkp); D.bk_q = (const unsigned short*)(b + o_bkq);
    D.tp = (const double*)(b + o_t[0]); D.wp = (const double*)(b + o_w[0]);
    D.tq = (const double*)(b + o_t[1]); D.wq = (const double*)(b + o_w[1]);
    D.tx = (const double*)(b + o_t[2]); D.wx = (const double*)(b + o_w[2]);
    D.sx = (const double*)(b + o_sx);
    G->geo = D;
    G->dev_version = G->version;
    return PM_OK;
}

// geometry + the lattice's channel tables as one blob
int32_t ensure_device(pm_lattice* L)
{
    pm_geometry* G = L->G;
    int32_t rc = ensure_geometry(G);
    if (rc) return rc;
    if (L->d_blob && L->geo_version == G->version && L->device == G->device) return PM_OK;
    free_lattice_device(L);
    L->device = G->device;
    const pm::Tables& T = L->T;
    pm::DevLattice D = G->geo;
    D.n_ch = L->n_ch; D.norm = L->norm;
    D.totcoup = T.totcoup; D.n_bra = T.n_slot; D.lmax = T.lmax;
    D.ny = pm::ylm_index(T.lmax, T.lmax) + 1;
    std::vector<double> bra;
    {   // rows of n_slot + 1 entries: one trailing zero slot for the unused terms of a function
        std::vector<double> b0;
        pm::build_bra(T, G->rule_t[2], b0);
        const size_t ns = (size_t)T.n_slot, nx = G->rule_t[2].size();
        bra.assign(nx * (ns + 1), 0.0);
        for (size_t c = 0; c < nx; ++c) std::copy(b0.begin() + (ptrdiff_t)(c * ns), b0.begin() + (ptrdiff_t)((c + 1) * ns), bra.begin() + (ptrdiff_t)(c * (ns + 1)));
    }
    std::vector<int32_t> o_alpha(T.totcoup);
    for (int a = 0; a < L->n_ch; ++a) for (int o = T.cl_off[a]; o < T.cl_off[a + 1]; ++o) o_alpha[o] = a;
    Blob B;
    const size_t o_cloff = B.put(T.cl_off.data(), 4 * T.cl_off.size()), o_cl = B.put(T.cl.data(), 4 * T.cl.size());
    const size_t o_oa = B.put(o_alpha.data(), 4 * o_alpha.size());
    const size_t o_bra = B.put(bra.data(), 8 * bra.size());
    const size_t o_ya = B.put(T.ya.data(), 8 * T.ya.size()), o_yb = B.put(T.yb.data(), 8 * T.yb.size());
    const size_t o_yd = B.put(T.ydiag.data(), 8 * T.ydiag.size());
    struct GOff { size_t ktoff, ktip, ktiq, ktc, fun, otoff, otf, otc, ga, gm, gap; };
    std::vector<const pm::GroupTables*> all;           // the groups of the table-driven kernel, then those of the specialised kernels
    for (const pm::GroupTables& Gt : L->groups) all.push_back(&Gt);
    for (const pm::GroupTables& Gt : L->jgroups) all.push_back(&Gt);
    std::vector<GOff> go(all.size());
    for (size_t g = 0; g < all.size(); ++g) {
        const pm::GroupTables& Gt = *all[g];
        std::vector<int4> fun(Gt.fun.size());
        for (size_t f = 0; f < Gt.fun.size(); ++f) fun[f] = make_int4(Gt.fun[f].sa0, Gt.fun[f].sb0, Gt.fun[f].nM, Gt.fun[f].L);
        go[g].ktoff = B.put(Gt.kt_off.data(), 4 * Gt.kt_off.size()); go[g].ktip = B.put(Gt.kt_ip.data(), 4 * Gt.kt_ip.size());
        go[g].ktiq = B.put(Gt.kt_iq.data(), 4 * Gt.kt_iq.size()); go[g].ktc = B.put(Gt.kt_c.data(), 8 * Gt.kt_c.size());
        go[g].fun = B.put(fun.data(), sizeof(int4) * fun.size());
        go[g].otoff = B.put(Gt.ot_off.data(), 4 * Gt.ot_off.size()); go[g].otf = B.put(Gt.ot_f.data(), 4 * Gt.ot_f.size());
        go[g].otc = B.put(Gt.ot_c.data(), 8 * Gt.ot_c.size());
        go[g].ga = B.put(Gt.o_alpha.data(), 4 * Gt.o_alpha.size()); go[g].gm = B.put(Gt.o_m.data(), 4 * Gt.o_m.size());
        go[g].gap = B.put(Gt.o_ap.data(), 4 * Gt.o_ap.size());
    }
    // per-pair sums layout of jgroups and the whole set's outputs in terms of it (k_op_expand)
    size_t o_xpos = 0, o_xc = 0;
    L->op_off.clear(); L->op_stride = 0;
    if (!L->jgroups.empty()) {
        std::vector<int> pos(T.fun.size(), 0);
        for (const pm::GroupTables& Gt : L->jgroups) {
            L->op_off.push_back(L->op_stride);
            for (size_t f = 0; f < Gt.f_global.size(); ++f) pos[(size_t)Gt.f_global[f]] = L->op_stride + (int)f;
            L->op_stride += ((int)Gt.fun.size() + 3) & ~3;
        }
        std::vector<uint16_t> xpos(4 * (size_t)T.totcoup, 0);
        std::vector<double> xc(4 * (size_t)T.totcoup, 0.0);
        bool ok = L->op_stride <= 2048;                // (k_op_apply packs byte offsets into 16 bits; k_op_expand keeps 8 pairs' sums in shared memory)
        // Term slot i of every output of a row belongs to the row's i-th L value (coefficient 0 where the output has no term
        // with that L): neighbouring outputs of a row then read, slot by slot, sums of one bra triple and neighbouring ket
        // triples — neighbouring or equal positions, few shared-memory bank conflicts in k_op_expand / k_op_apply.
        for (int a = 0; a < L->n_ch && ok; ++a) {
            std::vector<int> Ls;                        // distinct L of the row's terms, ascending
            for (int o = T.cl_off[(size_t)a]; o < T.cl_off[(size_t)a + 1]; ++o)
                for (int t = T.ot_off[(size_t)o]; t < T.ot_off[(size_t)o + 1]; ++t) {
                    const int Lt = T.fun[(size_t)T.ot_f[(size_t)t]].L;
                    if (std::find(Ls.begin(), Ls.end(), Lt) == Ls.end()) Ls.push_back(Lt);
                }
            std::sort(Ls.begin(), Ls.end());
            if (Ls.size() > 4) { ok = false; break; }
            int last_pos[4] = {0, 0, 0, 0};             // an output without the slot's L repeats its neighbour's position
            for (size_t i = 0; i < Ls.size(); ++i)
                for (int o = T.cl_off[(size_t)a]; o < T.cl_off[(size_t)a + 1] && last_pos[i] == 0; ++o)
                    for (int t = T.ot_off[(size_t)o]; t < T.ot_off[(size_t)o + 1]; ++t)
                        if (T.fun[(size_t)T.ot_f[(size_t)t]].L == Ls[i]) { last_pos[i] = pos[(size_t)T.ot_f[(size_t)t]]; break; }
            for (int o = T.cl_off[(size_t)a]; o < T.cl_off[(size_t)a + 1]; ++o) {
                for (size_t i = 0; i < Ls.size(); ++i) {
                    for (int t = T.ot_off[(size_t)o]; t < T.ot_off[(size_t)o + 1]; ++t)
                        if (T.fun[(size_t)T.ot_f[(size_t)t]].L == Ls[i]) { last_pos[i] = pos[(size_t)T.ot_f[(size_t)t]]; xc[4 * (size_t)o + i] = T.ot_c[(size_t)t]; }
                    xpos[4 * (size_t)o + i] = (uint16_t)last_pos[i];
                }
            }
        }
        if (ok) { o_xpos = B.put(xpos.data(), 2 * xpos.size()); o_xc = B.put(xc.data(), 8 * xc.size()); }
        else { L->op_stride = 0; L->op_off.clear(); }          // (more than four terms per output: group by group into the CSR)
    }
    cudaError_t e;
    if ((e = cudaMalloc(&L->d_blob, B.b.size())) != cudaSuccess) return cuda_fail(e, "cudaMalloc(channel tables)");
    if ((e = cudaMemcpy(L->d_blob, B.b.data(), B.b.size(), cudaMemcpyHostToDevice)) != cudaSuccess) return cuda_fail(e, "cudaMemcpy(channel tables)");
    if ((e = cudaEventCreate(&L->ev_fill0)) != cudaSuccess || (e = cudaEventCreate(&L->ev_fill1)) != cudaSuccess) return cuda_fail(e, "cudaEventCreate");
    char* b = L->d_blob;
    D.cl_off = (const int*)(b + o_cloff); D.cl = (const int*)(b + o_cl); D.o_alpha = (const int*)(b + o_oa);
    D.bra = (const double*)(b + o_bra);
    L->d_xpos = L->op_stride ? (const unsigned short*)(b + o_xpos) : nullptr; L->d_xc = L->op_stride ? (const double*)(b + o_xc) : nullptr;
    D.ya = (const double*)(b + o_ya); D.yb = (const double*)(b + o_yb); D.ydiag = (const double*)(b + o_yd);
    L->gdev.assign(L->groups.size(), pm_lattice::GroupDev{});
    L->gdev_j.assign(L->jgroups.size(), pm_lattice::GroupDev{});
    for (size_t g = 0; g < all.size(); ++g) {
        const pm::GroupTables& Gt = *all[g];
        pm::DevLattice Dg = D;
        Dg.n_slot = Gt.n_slot; Dg.n_fun = (int)Gt.fun.size(); Dg.n_out = (int)Gt.o_alpha.size(); Dg.n_out1 = Gt.n_out1; Dg.n_out2 = Gt.n_out2; Dg.n_out3 = Gt.n_out3;
        Dg.kt_off = (const int*)(b + go[g].ktoff); Dg.kt_ip = (const int*)(b + go[g].ktip); Dg.kt_iq = (const int*)(b + go[g].ktiq);
        Dg.kt_c = (const double*)(b + go[g].ktc);
        Dg.fun = (const int4*)(b + go[g].fun);
        Dg.ot_off = (const int*)(b + go[g].otoff); Dg.ot_f = (const int*)(b + go[g].otf); Dg.ot_c = (const double*)(b + go[g].otc);
        Dg.op_stride = L->op_stride; Dg.op_off = (g >= L->groups.size() && L->op_stride) ? L->op_off[g - L->groups.size()] : 0;
        Dg.g_alpha = (const int*)(b + go[g].ga); Dg.g_m = (const int*)(b + go[g].gm); Dg.g_ap = (const int*)(b + go[g].gap);
        (g < L->groups.size() ? L->gdev[g] : L->gdev_j[g - L->groups.size()]).dev = Dg;
    }
    D = L->gdev[0].dev;                                 // (the pattern kernels read the geometric and coupled-list fields only)
    L->dev = D;
    L->geo_version = G->version;
    L->have_plan = false;
    return PM_OK;
}

// nodes one lane of the fill kernel sums before the cross-lane segment sums (PM_CHUNK_LEN: tuning / test hook)
int chunk_len()
{
    static const int v = [] { const char* e = std::getenv("PM_CHUNK_LEN"); const int x = e ? std::atoi(e) : 4; return x < 1 ? 1 : (x > pm::kMaxChunkLen ? pm::kMaxChunkLen : x); }();
    return v;
}

int32_t ensure_cell_scratch(pm_geometry* G, int n_blk)
{
    if (n_blk <= G->cells_cap) return PM_OK;
    free_lists(G);
    const size_t nn = (size_t)n_blk * (size_t)G->geo.nnode;
    cudaError_t e;
    if ((e = cudaMalloc(&G->nl.key, sizeof(unsigned) * nn)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(node lists)");
    if ((e = cudaMalloc(&G->nl.ntot, sizeof(int) * (size_t)n_blk)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(ntot)");
    if ((e = cudaMalloc(&G->nl.hits, sizeof(int) * (size_t)n_blk)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(hits)");
    if ((e = cudaMalloc(&G->nl.chunk, sizeof(uint2) * nn)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(chunk lists)");
    if ((e = cudaMalloc(&G->nl.nchunk, sizeof(int) * (size_t)n_blk)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(nchunk)");
    {   // (a, b) indices are packed into 32 bits per chunk
        int bits = 1;
        while ((1 << bits) < G->geo.n_p * G->geo.n_q) ++bits;
        G->nl.ab_bits = bits;
        int r = 1;                                      // a power of two, r * bits <= 32
        while (2 * r <= chunk_len() && 2 * r * bits <= 32) r *= 2;
        G->nl.chunk_len = r;
    }
    if ((e = cudaMalloc(&G->d_cellbase, sizeof(int64_t) * ((size_t)n_blk + 1))) != cudaSuccess) return cuda_fail(e, "cudaMalloc(cellbase)");
    G->cells_cap = n_blk;
    return PM_OK;
}

// waits for the summary of the last pattern pass and takes it over into the host state
int32_t sync_summary(pm_geometry* G)
{
    if (!G->summary_pending) return PM_OK;
    cudaError_t e = cudaEventSynchronize(G->ev_summary);
    if (e != cudaSuccess) return cuda_fail(e, "pattern pass (map / sort / scan)");
    G->summary_pending = false;
    G->nnz = G->h_summary[0]; G->hmax = (int)G->h_summary[1]; G->nodes_on_grid = G->h_summary[2];
    G->overflow = G->h_summary[4];
    G->chunks = G->h_summary[5];
    G->hit_cells = G->totcoup_of_scan ? G->nnz / G->totcoup_of_scan : 0;
    return PM_OK;
}

bool bad_edges(const double* e, int N)
{
    if (!(e[0] >= 0.0)) return true;
    for (int k = 0; k <= N; ++k) if (!std::isfinite(e[k]) || e[k] > 1e150) return true;      // e*e must stay finite
    for (int k = 0; k < N; ++k) if (!(e[k + 1] > e[k])) return true;
    return false;
}

int32_t make_lattice(pm_geometry* G, const pm_channel* ch, int32_t n_ch, int32_t J2, int32_t parity, int32_t T2, int32_t statistics,
                     pm_lattice** out)
{
    if (n_ch < 1 || n_ch > PM_MAX_CHANNELS) return fail(PM_ERR_CHANNEL, "n_ch out of range");
    if ((int64_t)G->Np * G->Nq * n_ch >= (int64_t(1) << 31)) return fail(PM_ERR_OVERFLOW, "M = n_ch*Np*Nq must be below 2^31");
    std::string msg = pm::validate_channels(ch, n_ch, J2, parity, T2, statistics);
    if (!msg.empty()) return fail(PM_ERR_CHANNEL, msg);
    pm_lattice* L = new (std::nothrow) pm_lattice();
    if (!L) return fail(PM_ERR_NOMEM, "out of host memory");
    L->n_ch = n_ch; L->J2 = J2; L->parity = parity; L->T2 = T2; L->stat = statistics;
    L->ch.assign(ch, ch + n_ch);
    msg = pm::build_tables(ch, n_ch, J2, T2, statistics, L->T);
    if (!msg.empty()) { delete L; return fail(PM_ERR_CHANNEL, msg); }
    L->hash = pm::tables_hash(L->T);
    pm::build_groups(L->T, ch, pm::kFillMaxSlot, pm::kFillMaxFun, pm::kFillMaxOut, L->groups);
    pm::build_groups(L->T, ch, pm::kFillJitSlot, pm::kFillJitFun, pm::kFillJitOut, L->jgroups);
    for (const pm::GroupTables& Gt : L->jgroups)
        if (Gt.n_slot > pm::kFillJitSlot || (int)Gt.fun.size() > pm::kFillJitFun) { L->jgroups.clear(); break; }   // (one class too big: table-driven only)
    for (const pm::GroupTables& Gt : L->groups)
        if (Gt.n_slot > pm::kFillMaxSlot || (int)Gt.fun.size() > pm::kFillMaxFun) {
            delete L; return fail(PM_ERR_CHANNEL, "one orbital pair (l', lambda') of this channel set needs more ket slots than a kernel holds");
        }
    static std::atomic<uint64_t> next_id{1};
    L->id = next_id++;
    L->G = G;
    *out = L;
    return PM_OK;
}

}  // namespace

namespace pm {
void lattice_stamp(const pm_lattice* lat, uint64_t* id, uint64_t* version, int* nnode)
{
    *id = lat->id; *version = lat->G->version; *nnode = lat->G->n_p * lat->G->n_q * lat->G->n_x;
}
}  // namespace pm

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
    if (n_p < 1 || n_q < 1 || n_x < 1 || n_p > PM_MAX_ORDER || n_q > PM_MAX_ORDER || n_x > PM_MAX_ORDER)
        return fail(PM_ERR_ORDER, "quadrature order out of range 1..64");
    if ((int64_t)n_p * n_q * n_x > 16384) return fail(PM_ERR_ORDER, "n_p*n_q*n_x exceeds 16384");
    pm_geometry* G = new (std::nothrow) pm_geometry();
    if (!G) return fail(PM_ERR_NOMEM, "out of host memory");
    G->Np = Np; G->Nq = Nq; G->n_p = n_p; G->n_q = n_q; G->n_x = n_x;
    G->pe.assign(p_edges, p_edges + Np + 1); G->qe.assign(q_edges, q_edges + Nq + 1);
    const int orders[3] = {n_p, n_q, n_x};
    for (int k = 0; k < 3; ++k) pm::gauss_legendre(orders[k], G->rule_t[k], G->rule_w[k]);
    const int32_t rc = make_lattice(G, ch, n_ch, J2, parity, T2, statistics, out);
    if (rc) delete G;
    return rc;
}

int32_t pm_lattice_attach(pm_lattice* base, const pm_channel* ch, int32_t n_ch, int32_t J2, int32_t parity, int32_t T2,
                          int32_t statistics, pm_lattice** out)
{
    if (!out) return fail(PM_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (!base || !ch) return fail(PM_ERR_ARG, "NULL input pointer");
    const int32_t rc = make_lattice(base->G, ch, n_ch, J2, parity, T2, statistics, out);
    if (rc == PM_OK) ++base->G->refs;
    return rc;
}

int32_t pm_lattice_destroy(pm_lattice* lat)
{
    if (!lat) return PM_OK;
    free_lattice_device(lat);
    if (--lat->G->refs == 0) { free_geometry_device(lat->G); delete lat->G; }
    delete lat;
    return PM_OK;
}

int32_t pm_lattice_dims(const pm_lattice* lat, int64_t* M, int32_t* n_cells)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    if (M) *M = (int64_t)lat->G->Np * lat->G->Nq * lat->n_ch;
    if (n_cells) *n_cells = lat->G->Np * lat->G->Nq;
    return PM_OK;
}

int32_t pm_lattice_rule(const pm_lattice* lat, int32_t axis, double* nodes, double* weights)
{
    if (!lat || axis < 0 || axis > 2) return fail(PM_ERR_ARG, "bad lattice or axis");
    if (nodes) std::copy(lat->G->rule_t[axis].begin(), lat->G->rule_t[axis].end(), nodes);
    if (weights) std::copy(lat->G->rule_w[axis].begin(), lat->G->rule_w[axis].end(), weights);
    return PM_OK;
}

int32_t pm_lattice_set_rule(pm_lattice* lat, int32_t axis, const double* nodes, const double* weights)
{
    if (!lat || axis < 0 || axis > 2 || !nodes || !weights) return fail(PM_ERR_ARG, "bad lattice, axis or NULL rule");
    pm_geometry* G = lat->G;
    const int n = (int)G->rule_t[axis].size();
    for (int k = 0; k < n; ++k) {
        if (!std::isfinite(nodes[k]) || !std::isfinite(weights[k]) || !(nodes[k] > -1.0 && nodes[k] < 1.0))
            return fail(PM_ERR_ORDER, "rule nodes must lie inside (-1,1) and be finite");
        if (k && !(nodes[k] > nodes[k - 1])) return fail(PM_ERR_ORDER, "rule nodes must be strictly increasing");
    }
    if (axis == 2)
        for (int k = 0; k < n; ++k)
            if (nodes[k] != -nodes[n - 1 - k] || weights[k] != weights[n - 1 - k])
                return fail(PM_ERR_ORDER, "the x-rule must be symmetric under x -> -x (both cyclic terms are folded into one)");
    if (std::equal(nodes, nodes + n, G->rule_t[axis].begin()) && std::equal(weights, weights + n, G->rule_w[axis].begin())) return PM_OK;
    G->rule_t[axis].assign(nodes, nodes + n);
    G->rule_w[axis].assign(weights, weights + n);
    ++G->version;                      // every lattice of the group re-uploads its tables; the node lists are stale
    return PM_OK;
}

int32_t pm_lattice_set_normalisation(pm_lattice* lat, int32_t normalisation)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    if (normalisation != PM_NORM_WIDTH && normalisation != PM_NORM_P2) return fail(PM_ERR_ARG, "unknown normalisation");
    if (lat->norm != normalisation) { lat->norm = normalisation; lat->geo_version = 0; }      // the device tables are rebuilt at the next call
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
    // per node on the grid (pm_fill.cuh, phase C): weight and omega 5 (w = two products, p q, ra rb, two more products),
    // rotated directions 20 (two rsqrt), the generated ket code, and one add per slot into the chunk sum.  (The node map is
    // the pattern pass's work: the fill reads the nodes' (a, b, c) from the chunk words.)
    if (flop_per_node) *flop_per_node = 5.0 + 20.0 + pm::ket_flops(T) + (double)T.n_slot;
    // per (target, x-node) segment: sum_M bra*S per orbital function (nM multiply-adds) and one add into the target sum
    double seg = 0.0;
    for (const pm::OrbFun& f : T.fun) seg += 2.0 * f.nM;
    if (flop_per_segment) *flop_per_segment = seg;
    // per hit cell: normalisation 5, per output one multiply-add per (channel pair, L) term and the scaling by the norm
    if (flop_per_hit_cell) *flop_per_hit_cell = 5.0 + 2.0 * (double)T.ot_c.size();
    if (n_coupled_pairs) *n_coupled_pairs = T.totcoup;
    return PM_OK;
}

int32_t pm_pattern_counts(const pm_lattice* lat_c, int64_t* nodes_on_grid, int64_t* segments, int64_t* hit_cells)
{
    if (!lat_c) return fail(PM_ERR_ARG, "lat is NULL");
    pm_lattice* lat = const_cast<pm_lattice*>(lat_c);
    pm_geometry* G = lat->G;
    if (!G->lists_valid) return fail(PM_ERR_STATE, "pm_pattern_counts needs a preceding pm_pattern");
    int32_t rc = sync_summary(G);
    if (rc) return rc;
    if (G->segments < 0 && segments) {                 // counted on demand: statistics of the work model, not part of the build
        const int n_blk = G->pat_end - G->pat_begin;
        G->segments = 0;
        if (n_blk > 0) {
            cudaError_t e = pm::launch_count_segments(lat->dev, n_blk, G->nl, (unsigned long long*)(G->d_summary + 3), G->last_stream);
            if (e != cudaSuccess) return cuda_fail(e, "k_count_segments");
            int64_t v = 0;
            if ((e = cudaMemcpyAsync(&v, G->d_summary + 3, sizeof v, cudaMemcpyDeviceToHost, G->last_stream)) != cudaSuccess) return cuda_fail(e, "cudaMemcpy(segments)");
            if ((e = cudaStreamSynchronize(G->last_stream)) != cudaSuccess) return cuda_fail(e, "k_count_segments");
            G->segments = v;
        }
    }
    if (nodes_on_grid) *nodes_on_grid = G->nodes_on_grid;
    if (segments) *segments = G->segments;
    if (hit_cells) *hit_cells = G->hit_cells;
    return PM_OK;
}

int32_t pm_pattern_chunks(const pm_lattice* lat_c, int64_t* chunks)
{
    if (!lat_c || !chunks) return fail(PM_ERR_ARG, "NULL argument");
    pm_geometry* G = const_cast<pm_lattice*>(lat_c)->G;
    if (!G->lists_valid) return fail(PM_ERR_STATE, "pm_pattern_chunks needs a preceding pm_pattern");
    int32_t rc = sync_summary(G);
    if (rc) return rc;
    *chunks = G->chunks;
    return PM_OK;
}

const char* pm_lattice_fill_kernel(const pm_lattice* lat)
{
    if (!lat) return "";
    if (pm::fill_has_spec(lat->hash)) return pm::fill_variant_name(lat->hash);
    const bool may_jit = !lat->jgroups.empty() && pm::jit_enabled() && !lat->jit_failed;
    const char* jname = lat->jgroups.size() > 1 ? "jit-grouped" : "jit";
    if (lat->have_plan) return lat->use_j ? jname : (lat->groups.size() > 1 ? "generic-grouped" : lat->gdev[0].plan.name);
    return may_jit ? jname : (lat->groups.size() > 1 ? "generic-grouped" : "generic");
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
    if (lat->jgroups.empty()) return fail(PM_ERR_STATE, "one orbital pair of this channel set needs more ket slots than a specialised kernel holds: table-driven kernel only");
    for (const pm::GroupTables& Gt : lat->jgroups) {           // every column-channel group is one kernel
        size_t k = 0;
        if (!pm::jit_compile_check(pm::ket_view(Gt, lat->T.n_slot, lat->jgroups.size() == 1), 12, 4, &k, err)) return fail(PM_ERR_STATE, err);
        n += k;
    }
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

}  // extern "C"

namespace {

// The pattern pass up to rowptr, all asynchronous on `st`: node lists (unless `reuse_lists` and the group's lists cover
// the same range), scan, rowptr, and the copy of the summary to pinned host memory.  capacity < 0: no overflow flag.
int32_t pattern_async(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int64_t capacity, bool reuse_lists,
                      bool count_only, cudaStream_t st)
{
    pm_geometry* G = lat->G;
    const int n_cells = G->Np * G->Nq;
    if (cell_begin < 0 || cell_end > n_cells || cell_begin > cell_end) return fail(PM_ERR_ARG, "bad cell range");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    if ((rc = sync_summary(G))) return rc;             // at most one pattern pass in flight per geometry
    const int n_blk = cell_end - cell_begin;
    cudaError_t e;
    G->last_stream = st;
    G->totcoup_of_scan = lat->T.totcoup;
    if (n_blk == 0) {
        if ((e = cudaMemsetAsync(d_rowptr, 0, sizeof(int64_t), st)) != cudaSuccess) return cuda_fail(e, "memset");
        G->lists_valid = true; G->hitlist_valid = false; G->pat_begin = cell_begin; G->pat_end = cell_end; G->pat_count_only = count_only;
        G->hmax = 0; G->nnz = G->nodes_on_grid = G->hit_cells = G->segments = G->overflow = 0;
        return PM_OK;
    }
    const bool reuse = reuse_lists && G->lists_valid && G->pat_begin == cell_begin && G->pat_end == cell_end && G->cells_cap >= n_blk;
    if (!reuse) {
        G->lists_valid = false; G->hitlist_valid = false; G->segments = -1;
        if ((rc = ensure_cell_scratch(G, n_blk))) return rc;
        if ((e = cudaMemsetAsync(G->d_counter, 0, 2 * sizeof(int), st)) != cudaSuccess) return cuda_fail(e, "memset(counters)");
        const size_t need = pm::map_sort_scratch_bytes(lat->dev, G->n_sm);
        if (need > G->sort_scratch_bytes) {
            if (G->d_sort_scratch) cudaFree(G->d_sort_scratch);
            G->d_sort_scratch = nullptr; G->sort_scratch_bytes = 0;
            if ((e = cudaMalloc(&G->d_sort_scratch, need)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(sort scratch)");
            G->sort_scratch_bytes = need;
        }
        e = pm::launch_map_sort(lat->dev, cell_begin, n_blk, G->nl, G->n_sm, G->d_counter + 1, G->d_sort_scratch, st);
        if (e == cudaErrorInvalidConfiguration) { cudaGetLastError(); return fail(PM_ERR_NOMEM, "lattice needs more shared memory per source cell than one SM has"); }
        if (e != cudaSuccess) return cuda_fail(e, "k_map_sort");
    }
    if ((e = pm::launch_scan_rows(lat->dev, n_blk, G->nl, G->d_cellbase, d_rowptr, G->d_summary, capacity, st)) != cudaSuccess)
        return cuda_fail(e, "k_scan_rows");
    if ((e = cudaMemcpyAsync(G->h_summary, G->d_summary, 6 * sizeof(int64_t), cudaMemcpyDeviceToHost, st)) != cudaSuccess)
        return cuda_fail(e, "cudaMemcpyAsync(summary)");
    if ((e = cudaEventRecord(G->ev_summary, st)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    G->summary_pending = true;
    G->lists_valid = true; G->pat_begin = cell_begin; G->pat_end = cell_end; G->pat_count_only = count_only;
    ++G->pattern_serial;
    return PM_OK;
}

int32_t ensure_hitlist(pm_lattice* lat, cudaStream_t st)
{
    pm_geometry* G = lat->G;
    if (G->hitlist_valid) return PM_OK;
    int32_t rc = sync_summary(G);
    if (rc) return rc;
    const int n_blk = G->pat_end - G->pat_begin;
    const int64_t need = std::max<int64_t>(G->hit_cells, 1);
    cudaError_t e;
    if (need > G->hitlist_cap) {
        if (G->d_hitlist) cudaFree(G->d_hitlist);
        G->d_hitlist = nullptr; G->hitlist_cap = 0;
        if ((e = cudaMalloc(&G->d_hitlist, sizeof(int) * (size_t)need)) != cudaSuccess) return cuda_fail(e, "cudaMalloc(hit list)");
        G->hitlist_cap = need;
    }
    if (n_blk > 0 && (e = pm::launch_hit_list(lat->dev, n_blk, G->nl, G->d_cellbase, G->d_hitlist, st)) != cudaSuccess) return cuda_fail(e, "k_hit_list");
    G->hitlist_valid = true;
    return PM_OK;
}

// run-time specialised kernels (mode 2: per-pair sums) for every group of jgroups; false when NVRTC is off, missing or fails
bool ensure_sums_plans(pm_lattice* lat)
{
    if (lat->gdev_j.empty() || lat->op_stride <= 0) return false;
    bool ready = true;
    for (auto& gd : lat->gdev_j) ready = ready && gd.plan.fn_op != nullptr;
    if (ready) return true;
    if (!pm::jit_enabled() || lat->jit_failed) { if (lat->jit_error.empty()) lat->jit_error = "run-time compilation is switched off"; return false; }
    std::vector<pm::DevLattice> devs;
    std::vector<pm::KetView> views;
    for (size_t g = 0; g < lat->gdev_j.size(); ++g) { devs.push_back(lat->gdev_j[g].dev); views.push_back(pm::ket_view(lat->jgroups[g], lat->T.n_slot, true)); }
    std::vector<pm::FillLaunch> plans;
    for (auto& gd : lat->gdev_j) plans.push_back(gd.plan);
    if (!pm::fill_plan_jit(devs, views, lat->G->n_sm, 2, plans, lat->jit_error)) { lat->jit_failed = true; return false; }
    for (size_t g = 0; g < plans.size(); ++g) lat->gdev_j[g].plan = plans[g];
    return true;
}

// The per-pair sums of the cells [cell_begin, cell_begin + n_blk) of the last pattern call into lat->d_opA: every group of
// jgroups through its run-time specialised kernel in mode 2 (compiled on first use).
int32_t fill_sums(pm_lattice* lat, int32_t cell_begin, int n_blk, const int64_t* guard, cudaStream_t st)
{
    pm_geometry* G = lat->G;
    if (lat->gdev_j.empty() || lat->op_stride <= 0) return fail(PM_ERR_STATE, "this channel set has no per-pair sums form");
    if (!ensure_sums_plans(lat)) return fail(PM_ERR_STATE, "the per-pair sums need run-time compilation (NVRTC): " + lat->jit_error);
    int32_t rc = ensure_hitlist(lat, st);               // (waits for the pattern pass: the number of hit cell pairs sizes the sums)
    if (rc) return rc;
    if (G->overflow) return PM_OK;                      // (the caller reports it)
    cudaError_t e;
    const int64_t need = std::max<int64_t>(G->hit_cells, 1) * lat->op_stride;
    if (need > lat->opA_cap) {
        if (lat->d_opA) cudaFree(lat->d_opA);
        lat->d_opA = nullptr; lat->opA_cap = 0;
        if ((e = cudaMalloc(&lat->d_opA, sizeof(double) * (size_t)need)) != cudaSuccess) { cudaGetLastError(); return fail(PM_ERR_NOMEM, "out of device memory for the per-pair sums of this channel set"); }
        lat->opA_cap = need;
    }
    for (auto& gd : lat->gdev_j) {
        e = pm::launch_fill(gd.dev, gd.plan, cell_begin, n_blk, G->nl, G->d_cellbase, lat->d_opA, nullptr, G->d_counter, guard, st, true);
        if (e != cudaSuccess) return cuda_fail(e, "k_fill (per-pair sums)");
    }
    lat->op_serial = 0;                                 // (pm_operator_build stamps it)
    return PM_OK;
}

// values (and, when d_colidx is given, column indices) of the block of the last pattern call; `guard` (device) stops the
// kernel when the scan found nnz above the caller's capacity
int32_t fill_block(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, const int64_t* d_rowptr, double* d_vals,
                   int32_t* d_colidx, const int64_t* guard, cudaStream_t st)
{
    pm_geometry* G = lat->G;
    if (!G->lists_valid || cell_begin != G->pat_begin || cell_end != G->pat_end)
        return fail(PM_ERR_STATE, "pm_fill needs a preceding pm_pattern of the same cell range on this lattice");
    if (cell_begin == cell_end) return PM_OK;
    const int n_blk = cell_end - cell_begin;
    cudaError_t e;
    const bool grouped = lat->gdev.size() > 1;         // big channel sets: one launch per column-channel group
    const bool has_spec = !grouped && pm::fill_has_spec(lat->hash);
    // several specialised groups: each writes the per-pair sums of its functions, one kernel then writes whole CSR rows
    const bool via_sums = lat->gdev_j.size() > 1 && lat->op_stride > 0 && ensure_sums_plans(lat);       // (else the table-driven groups below)
    const int mode = d_colidx != nullptr ? 1 : 0;
    auto have_fn = [&](const pm::FillLaunch& F) { return mode == 1 ? F.fn_cols != nullptr : F.fn != nullptr; };
    const bool need_variant = !via_sums && lat->have_plan && lat->use_j && !have_fn(lat->gdev_j[0].plan);
    if (via_sums) { lat->have_plan = true; lat->use_j = true; }
    else if (lat->use_j && lat->gdev_j.size() > 1) { lat->have_plan = false; lat->use_j = false; }              // (run-time compilation went away)
    if (!via_sums && (!lat->have_plan || need_variant) && !has_spec && !lat->gdev_j.empty() && pm::jit_enabled() && !lat->jit_failed) {
        // no build-time kernel for this channel set: specialise at run time (pm_jit.hpp), one kernel per group of jgroups
        // and only the variant this call launches; else fall back to the table-driven kernel below
        std::vector<pm::DevLattice> devs;
        std::vector<pm::KetView> views;
        for (size_t g = 0; g < lat->gdev_j.size(); ++g) { devs.push_back(lat->gdev_j[g].dev); views.push_back(pm::ket_view(lat->jgroups[g], lat->T.n_slot, true)); }
        std::vector<pm::FillLaunch> plans;
        if (need_variant) for (auto& gd : lat->gdev_j) plans.push_back(gd.plan);
        if (pm::fill_plan_jit(devs, views, G->n_sm, mode, plans, lat->jit_error)) {
            for (size_t g = 0; g < plans.size(); ++g) lat->gdev_j[g].plan = plans[g];
            lat->have_plan = true; lat->use_j = true;
        } else { lat->jit_failed = true; lat->have_plan = false; }
    }
    if (!lat->have_plan) {
        lat->use_j = false;
        for (auto& gd : lat->gdev) {
            e = pm::fill_plan(gd.dev, grouped ? 0ull : lat->hash, G->n_sm, &gd.plan);
            if (e == cudaErrorInvalidConfiguration) { cudaGetLastError(); return fail(PM_ERR_NOMEM, "channel set needs more shared memory than one SM has"); }
            if (e != cudaSuccess) return cuda_fail(e, "fill_plan");
        }
        lat->have_plan = true;
    }
    if ((e = cudaEventRecord(lat->ev_fill0, st)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    if (lat->use_j && via_sums) {
        int32_t rc = fill_sums(lat, cell_begin, n_blk, guard, st);
        if (rc) return rc;
        if (G->overflow) return PM_OK;
        pm::DevLattice De = lat->dev;
        De.op_stride = lat->op_stride;
        e = pm::launch_op_expand(De, cell_begin, n_blk, G->nl, G->d_cellbase, G->d_hitlist, lat->d_opA, lat->d_xpos, lat->d_xc, d_rowptr, d_vals,
                                 d_colidx, G->d_counter, guard, G->n_sm, st);
        if (e != cudaSuccess) return cuda_fail(e, "k_op_expand");
    } else
    for (auto& gd : (lat->use_j ? lat->gdev_j : lat->gdev)) {
        e = pm::launch_fill(gd.dev, gd.plan, cell_begin, n_blk, G->nl, d_rowptr, d_vals, d_colidx, G->d_counter, guard, st);
        if (e != cudaSuccess) return cuda_fail(e, "k_fill");
    }
    if ((e = cudaEventRecord(lat->ev_fill1, st)) != cudaSuccess) return cuda_fail(e, "cudaEventRecord");
    lat->fill_timed = true;
    return PM_OK;
}

int32_t build_common(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                     int64_t capacity, bool reuse_lists, cudaStream_t st)
{
    if (capacity < 0) return fail(PM_ERR_ARG, "negative capacity");
    // pattern pass without the column kernel: node lists, rowptr, nnz and the overflow flag stay on the device ...
    int32_t rc = pattern_async(lat, cell_begin, cell_end, d_rowptr, capacity, reuse_lists, true, st);
    if (rc) return rc;
    // ... and the one kernel that writes the column index and the value of every nonzero follows on the stream at once
    return fill_block(lat, cell_begin, cell_end, d_rowptr, d_vals, d_colidx, lat->G->d_summary, st);
}

}  // namespace

extern "C" {

int32_t pm_pattern(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx,
                   int64_t colidx_capacity, int64_t* nnz_host, void* cuda_stream)
{
    if (!lat || !d_rowptr || !nnz_host) return fail(PM_ERR_ARG, "NULL argument");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    pm_geometry* G = lat->G;
    // Two-phase use (count, allocate, emit): the emit call reuses the node lists of the count call of the same range,
    // so the nodes are mapped once.  Any other call maps afresh.
    const bool reuse = d_colidx && G->pat_count_only;
    int32_t rc = pattern_async(lat, cell_begin, cell_end, d_rowptr, -1, reuse, d_colidx == nullptr, st);
    if (rc) return rc;
    if ((rc = sync_summary(G))) return rc;
    *nnz_host = G->nnz;
    if (!d_colidx || cell_begin == cell_end) return PM_OK;
    if (*nnz_host > colidx_capacity) return fail(PM_ERR_OVERFLOW, "d_colidx too small for this block's nnz");
    if ((rc = ensure_hitlist(lat, st))) return rc;
    cudaError_t e = pm::launch_emit_cols(lat->dev, cell_end - cell_begin, G->nl, G->d_cellbase, G->d_hitlist, d_rowptr, d_colidx, st);
    if (e != cudaSuccess) return cuda_fail(e, "k_emit_cols");
    return PM_OK;
}

int32_t pm_fill(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, const int64_t* d_rowptr, double* d_vals, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_vals) return fail(PM_ERR_ARG, "NULL argument");
    const int n_cells = lat->G->Np * lat->G->Nq;
    if (cell_begin < 0 || cell_end > n_cells || cell_begin > cell_end) return fail(PM_ERR_ARG, "bad cell range");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    return fill_block(lat, cell_begin, cell_end, d_rowptr, d_vals, nullptr, nullptr, (cudaStream_t)cuda_stream);
}

int32_t pm_build_async(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                       int64_t capacity, int32_t reuse_lists, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_colidx || !d_vals) return fail(PM_ERR_ARG, "NULL argument");
    return build_common(lat, cell_begin, cell_end, d_rowptr, d_colidx, d_vals, capacity, reuse_lists != 0, (cudaStream_t)cuda_stream);
}

int32_t pm_build_wait(pm_lattice* lat, int64_t* nnz_host)
{
    if (!lat) return fail(PM_ERR_ARG, "NULL argument");
    pm_geometry* G = lat->G;
    if (!G->lists_valid) return fail(PM_ERR_STATE, "no build has been started on this lattice");
    int32_t rc = sync_summary(G);
    if (rc) return rc;
    if (nnz_host) *nnz_host = G->nnz;
    if (G->overflow) return fail(PM_ERR_OVERFLOW, "d_colidx / d_vals too small for this block's nnz (nothing was written to them)");
    return PM_OK;
}

int32_t pm_build(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                 int64_t capacity, int64_t* nnz_host, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_colidx || !d_vals || !nnz_host) return fail(PM_ERR_ARG, "NULL argument");
    int32_t rc = build_common(lat, cell_begin, cell_end, d_rowptr, d_colidx, d_vals, capacity, false, (cudaStream_t)cuda_stream);
    if (rc) return rc;
    return pm_build_wait(lat, nnz_host);               // one host read-back, after the fill kernel has been queued
}

int32_t pm_build_reuse(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                       int64_t capacity, int64_t* nnz_host, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_colidx || !d_vals || !nnz_host) return fail(PM_ERR_ARG, "NULL argument");
    int32_t rc = build_common(lat, cell_begin, cell_end, d_rowptr, d_colidx, d_vals, capacity, true, (cudaStream_t)cuda_stream);
    if (rc) return rc;
    return pm_build_wait(lat, nnz_host);
}

int32_t pm_pattern_cell_hits(pm_lattice* lat, int32_t* h_hits, void* cuda_stream)
{
    if (!lat || !h_hits) return fail(PM_ERR_ARG, "NULL argument");
    pm_geometry* G = lat->G;
    if (!G->lists_valid) return fail(PM_ERR_STATE, "pm_pattern_cell_hits needs a preceding pm_pattern / pm_build");
    const int n_blk = G->pat_end - G->pat_begin;
    if (n_blk == 0) return PM_OK;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    cudaError_t e = cudaMemcpyAsync(h_hits, G->nl.hits, sizeof(int) * (size_t)n_blk, cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return cuda_fail(e, "pm_pattern_cell_hits");
    return PM_OK;
}

int32_t pm_partition_cells(const int32_t* hits, int32_t n_cells, double cell_cost, int32_t n_parts, int32_t* cuts)
{
    if (!hits || !cuts || n_cells < 0 || n_parts < 1 || !(cell_cost >= 0.0)) return fail(PM_ERR_ARG, "bad argument");
    // contiguous ranges of (almost) equal weight, weight of a cell = hit cells + cell_cost: cut r sits where the running
    // weight first reaches r/n_parts of the total (every cut is a function of the prefix sums only: deterministic)
    double total = 0.0;
    for (int k = 0; k < n_cells; ++k) total += (double)hits[k] + cell_cost;
    cuts[0] = 0;
    int k = 0;
    double run = 0.0;
    for (int r = 1; r < n_parts; ++r) {
        const double want = total * (double)r / (double)n_parts;
        while (k < n_cells && run + 0.5 * ((double)hits[k] + cell_cost) < want) { run += (double)hits[k] + cell_cost; ++k; }
        cuts[r] = k;
    }
    cuts[n_parts] = n_cells;
    return PM_OK;
}

int32_t pm_rowptr_offset(int64_t* d_rowptr, int64_t n, int64_t offset, void* cuda_stream)
{
    if (!d_rowptr || n < 0) return fail(PM_ERR_ARG, "bad argument");
    if (n == 0 || offset == 0) return PM_OK;
    cudaError_t e = pm::launch_add_offset(d_rowptr, n, offset, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "k_add_offset");
    return PM_OK;
}

int32_t pm_spmv_implicit(pm_lattice* lat, const int64_t* d_rowptr, const double* d_vals, const double* d_x, double* d_y, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_vals || !d_x || !d_y) return fail(PM_ERR_ARG, "NULL argument");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    pm_geometry* G = lat->G;
    const int n_cells = G->Np * G->Nq;
    if (!G->lists_valid || G->pat_begin != 0 || G->pat_end != n_cells)
        return fail(PM_ERR_STATE, "pm_spmv_implicit needs the node lists of a pm_pattern / pm_build call over the whole lattice");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = ensure_hitlist(lat, st))) return rc;
    cudaError_t e = pm::launch_spmv_implicit(lat->dev, (int64_t)n_cells * lat->n_ch, d_rowptr, G->nl.hits, G->d_cellbase, G->d_hitlist, d_vals, d_x, d_y, st);
    if (e != cudaSuccess) return cuda_fail(e, "k_spmv_implicit");
    return PM_OK;
}

int32_t pm_operator_build(pm_lattice* lat, int64_t* n_pairs, int64_t* bytes, void* cuda_stream)
{
    if (!lat) return fail(PM_ERR_ARG, "lat is NULL");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    pm_geometry* G = lat->G;
    const int n_cells = G->Np * G->Nq;
    if (!G->lists_valid || G->pat_begin != 0 || G->pat_end != n_cells)
        return fail(PM_ERR_STATE, "pm_operator_build needs the node lists of a pm_pattern / pm_build call over the whole lattice");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if ((rc = fill_sums(lat, 0, n_cells, nullptr, st))) return rc;
    lat->op_serial = G->pattern_serial; lat->op_norm = lat->norm;
    if (n_pairs) *n_pairs = G->hit_cells;
    if (bytes) *bytes = 8 * G->hit_cells * (int64_t)lat->op_stride;
    return PM_OK;
}

int32_t pm_operator_apply(pm_lattice* lat, const double* d_x, double* d_y, void* cuda_stream)
{
    if (!lat || !d_x || !d_y) return fail(PM_ERR_ARG, "NULL argument");
    if (d_x == d_y) return fail(PM_ERR_ARG, "pm_operator_apply cannot work in place");
    pm_geometry* G = lat->G;
    if (!lat->d_opA || lat->op_serial == 0 || lat->op_serial != G->pattern_serial || lat->op_norm != lat->norm)
        return fail(PM_ERR_STATE, "pm_operator_apply needs a pm_operator_build after the last pattern pass / change of normalisation");
    cudaStream_t st = (cudaStream_t)cuda_stream;
    pm::DevLattice De = lat->dev;
    De.op_stride = lat->op_stride;
    cudaError_t e = pm::launch_op_apply(De, G->Np * G->Nq, G->hmax, G->nl, G->d_cellbase, G->d_hitlist, lat->d_opA, lat->d_xpos, lat->d_xc, d_x, d_y,
                                        G->d_counter, G->n_sm, st);
    if (e != cudaSuccess) return cuda_fail(e, "k_op_apply");
    return PM_OK;
}

int32_t pm_block_apply(pm_lattice* lat, const double* d_blocks, const double* d_diag, const double* d_in, double* d_out, void* cuda_stream)
{
    if (!lat || !d_blocks || !d_in || !d_out) return fail(PM_ERR_ARG, "NULL argument");
    if (d_in == d_out) return fail(PM_ERR_ARG, "pm_block_apply cannot work in place");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    cudaError_t e = pm::launch_block_apply(lat->G->Np, lat->G->Nq, lat->n_ch, d_blocks, d_diag, d_in, d_out, 0, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "k_block_apply");
    return PM_OK;
}

int32_t pm_block_apply_t(pm_lattice* lat, const double* d_blocks, const double* d_in, double* d_out, void* cuda_stream)
{
    if (!lat || !d_blocks || !d_in || !d_out) return fail(PM_ERR_ARG, "NULL argument");
    if (d_in == d_out) return fail(PM_ERR_ARG, "pm_block_apply_t cannot work in place");
    int32_t rc = ensure_device(lat);
    if (rc) return rc;
    cudaError_t e = pm::launch_block_apply(lat->G->Np, lat->G->Nq, lat->n_ch, d_blocks, nullptr, d_in, d_out, 1, (cudaStream_t)cuda_stream);
    if (e != cudaSuccess) return cuda_fail(e, "k_block_apply (transposed)");
    return PM_OK;
}

int32_t pm_kernel_apply(pm_lattice* lat, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                        const double* d_O, const double* d_Vt, const double* d_g1, const double* d_u, double* d_out,
                        double* d_work, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_vals || !d_O || !d_Vt || !d_g1 || !d_u || !d_out || !d_work)
        return fail(PM_ERR_ARG, "NULL argument");
    const int64_t M = (int64_t)lat->G->Np * lat->G->Nq * lat->n_ch;
    double* t1 = d_work;                                   // V~1 G1 u
    double* t2 = d_work + M;                               // P0 V~1 G1 u
    int32_t rc = pm_block_apply(lat, d_Vt, d_g1, d_u, t1, cuda_stream);
    if (rc) return rc;
    rc = d_colidx ? pm_spmv(lat, M, d_rowptr, d_colidx, d_vals, t1, t2, cuda_stream)
                  : pm_spmv_implicit(lat, d_rowptr, d_vals, t1, t2, cuda_stream);      // columns implied by the hit lists
    if (rc) return rc;
    return pm_block_apply(lat, d_O, nullptr, t2, d_out, cuda_stream);
}

int32_t pm_rotate_apply(pm_lattice* lat, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                        const double* d_O, const double* d_x, double* d_out, double* d_work, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_vals || !d_O || !d_x || !d_out || !d_work) return fail(PM_ERR_ARG, "NULL argument");
    const int64_t M = (int64_t)lat->G->Np * lat->G->Nq * lat->n_ch;
    double* t1 = d_work;                                   // O^T x
    double* t2 = d_work + M;                               // P0 O^T x
    int32_t rc = pm_block_apply_t(lat, d_O, d_x, t1, cuda_stream);
    if (rc) return rc;
    rc = d_colidx ? pm_spmv(lat, M, d_rowptr, d_colidx, d_vals, t1, t2, cuda_stream)
                  : pm_spmv_implicit(lat, d_rowptr, d_vals, t1, t2, cuda_stream);
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

// ------------------------------------------------------------------------------------------------
// pm_rotate_apply_static — the rotation P x = O P0 O^T x (eq. 20) for callers that cannot allocate
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): the two intermediate vectors
// O^T x and P0 O^T x, which pm_rotate_apply takes from the caller's d_work, live in a file-scope device array of
// 2 * PM_STATIC_MAX_M doubles (1 MiB) that every GPU loading the library holds until exit.  The name of the array is a
// HOST-side stand-in in host code: its device address comes from cudaGetSymbolAddress, once per device, with that device
// current.  The call allocates nothing (no cudaMalloc / cudaFree, no lazily built library scratch): the lattice's device
// tables must already exist (any pm_pattern / pm_build / pm_block_apply call creates them), and d_colidx is required (the
// column-free SpMV builds its hit lists lazily).  All calls share the array, which keeps the last call's contents: both
// vectors are fully overwritten before they are read, so nothing has to be cleared; calls that overlap on the GPU (other
// streams, other host threads) race on it.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) double g_static_work[2 * PM_STATIC_MAX_M];

namespace {

constexpr int kStaticMaxDev = 64;
std::mutex g_static_mu;
double* g_static_ptr[kStaticMaxDev] = {};          // device address of g_static_work per device (nullptr: not asked yet)

// device address of the scratch array on the CURRENT device (asked once per device), or nullptr + error message
double* static_work_ptr()
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cuda_fail(e, "cudaGetDevice"); return nullptr; }
    if (dev < 0 || dev >= kStaticMaxDev) { fail(PM_ERR_DEVICE, "device index beyond the table of static scratch addresses"); return nullptr; }
    std::lock_guard<std::mutex> g(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        e = cudaGetSymbolAddress(&p, g_static_work);
        if (e != cudaSuccess || !p) { cuda_fail(e, "cudaGetSymbolAddress(static scratch)"); return nullptr; }
        g_static_ptr[dev] = (double*)p;
    }
    return g_static_ptr[dev];
}

}  // namespace

extern "C" {

int32_t pm_rotate_apply_static(pm_lattice* lat, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                               const double* d_O, const double* d_x, double* d_out, void* cuda_stream)
{
    if (!lat || !d_rowptr || !d_colidx || !d_vals || !d_O || !d_x || !d_out) return fail(PM_ERR_ARG, "NULL argument (pm_rotate_apply_static needs the column array)");
    if (d_x == d_out) return fail(PM_ERR_ARG, "pm_rotate_apply_static cannot work in place");
    pm_geometry* G = lat->G;
    const int64_t M = (int64_t)G->Np * G->Nq * lat->n_ch;
    if (M > PM_STATIC_MAX_M)
        return fail(PM_ERR_OVERFLOW, "M = " + std::to_string(M) + " exceeds PM_STATIC_MAX_M = " + std::to_string((int64_t)PM_STATIC_MAX_M) +
                                     ": the static scratch holds two vectors of at most that many doubles; use pm_rotate_apply with your own d_work");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (!lat->d_blob || lat->geo_version != G->version || lat->device != dev || G->device != dev)
        return fail(PM_ERR_STATE, "pm_rotate_apply_static allocates nothing: the lattice's device tables must exist on the current device "
                                  "(call pm_pattern / pm_build / pm_block_apply on it first)");
    double* work = static_work_ptr();
    if (!work) return PM_ERR_CUDA;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* t1 = work;                                      // O^T x
    double* t2 = work + M;                                  // P0 O^T x
    if ((e = pm::launch_block_apply(G->Np, G->Nq, lat->n_ch, d_O, nullptr, d_x, t1, 1, st)) != cudaSuccess) return cuda_fail(e, "k_block_apply");
    if ((e = pm::launch_spmv(M, d_rowptr, d_colidx, d_vals, t1, t2, st)) != cudaSuccess) return cuda_fail(e, "k_spmv");
    if ((e = pm::launch_block_apply(G->Np, G->Nq, lat->n_ch, d_O, nullptr, t2, d_out, 0, st)) != cudaSuccess) return cuda_fail(e, "k_block_apply");
    return PM_OK;
}

}  // extern "C"
