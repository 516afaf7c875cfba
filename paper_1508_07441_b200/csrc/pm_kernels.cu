// pm_kernels.cu — CUDA kernels of libpm for sm_100a: pattern pass (a6), SpMV (a9) with and without the column array, the block factors of the iteration step, FP64 peak diagnostic.
// One CTA per source cell D_ij; the node map and location live in pm_device.cuh.
// Paper's prior art: pre-selection of the nonzero elements by a separate GPU pass,
// one thread per element, constants in global memory (L341), CPU repack into CSR for coupled channels (L376).
// Here the pattern pass bins every quadrature node ONCE: k_map_sort leaves, per source cell, the node ids sorted
// by target cell (NodeLists); the column indices and the whole fill pass are driven by those lists, and the
// cell-major row order makes every row segment contiguous, so no repack exists.
#include "pm_kernels.cuh"

#include <cstdlib>

namespace pm {

__device__ __forceinline__ char* carve(char*& p, size_t bytes)
{
    char* r = p;
    p += (bytes + 15) & ~size_t(15);
    return r;
}

static size_t al16(size_t b) { return (b + 15) & ~size_t(15); }

// ------------------------------------------------------------------------------------------------
// Pattern pass, kernel A: ONE WARP per source cell (cells drawn from a work counter, tables staged once per CTA, no
// block barrier after start-up).  Pass 1 maps every node (exact ops, bucketed location), marks the hit cells in a bitset
// and keeps each node's target in shared memory; word-prefix popcounts turn a target into its rank; pass 2 counts the
// nodes per rank, pass 3 places the node ids in node order (a stable counting sort).  Node id m = c*(n_p*n_q) + a*n_q + b,
// so the sorted list is ordered by (target, x-node, a, b).  Lanes that meet the same rank in a step are grouped with
// match_any (32 consecutive nodes fall into one to three targets), so no shared-memory atomics are needed for the counts.
// Ranks are processed in windows of kHistCap counters: one window for every realistic lattice, any number otherwise.
// The targets of pass 1 wait for passes 2 and 3 in a per-warp global scratch (L2-resident, 2-4 bytes per node), which
// keeps the shared memory per warp small enough for 32 warps per SM.
// ------------------------------------------------------------------------------------------------
MapSortSmem map_sort_plan(const DevLattice& L, int max_warps)
{
    // rank counters per window (PM_HIST_CAP: test hook that forces several windows on small lattices)
    static const int hist_cap = [] { const char* e = std::getenv("PM_HIST_CAP"); return e ? std::max(1, std::min(kHistCap, std::atoi(e))) : kHistCap; }();
    MapSortSmem S{};
    S.hist_cap = hist_cap;
    int o = 0;
    auto take = [&](size_t bytes) { int r = o; o += (int)al16(bytes); return r; };
    S.thr_p = take(8 * (size_t)(L.pe_pad + kLocK)); S.thr_q = take(8 * (size_t)(L.qe_pad + kLocK));      // + sentinels of locate_k
    S.bk_p = take(2 * (size_t)kBuckets); S.bk_q = take(2 * (size_t)kBuckets);
    S.tp = take(8 * (size_t)L.n_p); S.tq = take(8 * (size_t)L.n_q); S.tx = take(8 * (size_t)L.n_x);
    S.wide = L.n_cells > 65535 ? 1 : 0;                 // targets kept as 16-bit ids when they fit
    // pass 1 items = (a, b) pairs x runs of n_x / nchunk consecutive x-nodes: the fewest runs that keep >= 90 % of the lanes busy
    S.nchunk = 1;
    {
        const int npq = L.n_p * L.n_q;
        double best = 0.0;
        for (int nc = 1; nc <= L.n_x; ++nc) {
            if (L.n_x % nc) continue;
            const int items = npq * nc;
            const double util = (double)items / (32.0 * ((items + 31) / 32));
            if (util > best + 1e-9) { best = util; S.nchunk = nc; }
            if (util >= 0.9) break;
        }
    }
    int w = 0;
    auto wtake = [&](size_t bytes) { int r = w; w += (int)al16(bytes); return r; };
    S.w_bits = wtake(4 * (size_t)L.n_words);
    S.w_wpre = wtake(2 * (size_t)L.n_words);
    S.w_hist = wtake(4 * (size_t)S.hist_cap);
    S.warp_bytes = w;
    // two CTAs per SM when 2 x (tables + max_warps warps) fit, else one CTA with as many warps as fit
    const int limit = 227 * 1024;
    if (2 * (o + w * max_warps + 1024) <= limit) { S.nw = max_warps; S.ctas = 2; }
    else { S.nw = std::max(0, std::min(max_warps, (limit - o) / w)); S.ctas = 1; }
    S.warp0 = take((size_t)w * std::max(S.nw, 1));
    S.total = o;
    return S;
}

template <class TT, bool kFast>
__global__ void __launch_bounds__(kMapSortMaxWarps * 32, 2)
k_map_sort(DevLattice L, MapSortSmem S, int cell_begin, int n_blk, NodeLists nl, int* __restrict__ counter, void* __restrict__ scratch)
{
    extern __shared__ __align__(16) char smem[];
    constexpr unsigned kOff = (unsigned)(TT)~(TT)0;             // marker of a node that left the grid
    const int T = blockDim.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    double* s_thr_p = (double*)(smem + S.thr_p); double* s_thr_q = (double*)(smem + S.thr_q);
    unsigned short* s_bk_p = (unsigned short*)(smem + S.bk_p); unsigned short* s_bk_q = (unsigned short*)(smem + S.bk_q);
    double* s_tp = (double*)(smem + S.tp); double* s_tq = (double*)(smem + S.tq); double* s_tx = (double*)(smem + S.tx);
    char* wsm = smem + S.warp0 + warp * S.warp_bytes;
    unsigned* bits = (unsigned*)(wsm + S.w_bits);
    unsigned short* wpre = (unsigned short*)(wsm + S.w_wpre);
    TT* s_t = (TT*)scratch + (size_t)(blockIdx.x * (T >> 5) + warp) * (size_t)((L.nnode + 31) & ~31);   // this warp's targets
    int* hist = (int*)(wsm + S.w_hist);

    for (int k = tid; k < L.pe_pad + kLocK; k += T) s_thr_p[k] = k < L.pe_pad ? L.thr_p[k] : __longlong_as_double(0x7ff0000000000000ll);
    for (int k = tid; k < L.qe_pad + kLocK; k += T) s_thr_q[k] = k < L.qe_pad ? L.thr_q[k] : __longlong_as_double(0x7ff0000000000000ll);
    for (int k = tid; k < kBuckets; k += T) { s_bk_p[k] = L.bk_p[k]; s_bk_q[k] = L.bk_q[k]; }
    for (int k = tid; k < L.n_p; k += T) s_tp[k] = L.tp[k];
    for (int k = tid; k < L.n_q; k += T) s_tq[k] = L.tq[k];
    for (int k = tid; k < L.n_x; k += T) s_tx[k] = L.tx[k];
    const Locator lc{s_thr_p, s_thr_q, s_bk_p, s_bk_q, L.bk_hmin_p, L.bk_sh_p, L.bk_hmin_q, L.bk_sh_q, L.Np, L.Nq};
    __syncthreads();                                            // the only block-level barrier

    const unsigned lt = (1u << lane) - 1u;
    const int wchunk = (L.n_words + 31) >> 5;                   // bitset words per lane in the rank prefix
    const int nsteps = (L.nnode + 31) >> 5;
    for (;;) {
        int cb = 0;
        if (lane == 0) cb = atomicAdd(counter, 1);
        cb = __shfl_sync(0xffffffffu, cb, 0);
        if (cb >= n_blk) break;
        const int cell = cell_begin + cb;
        const int ci = cell / L.Nq, cj = cell - ci * L.Nq;
        const CellGeom g = cell_geom(L.pe, L.qe, ci, cj);
        for (int k = lane; k < L.n_words; k += 32) bits[k] = 0u;
        __syncwarp();
        // ---- pass 1: map, locate, mark.  Lane = one (a, b) pair and one run of consecutive x-nodes: p, q and the
        // x-independent sums of the map are formed once per run (the very operations of map_node_sq, in its order), and
        // since p'^2 grows and q'^2 falls with x, the cell indices of a node follow from the previous node's by a few
        // comparisons (the first node of a run is located through the bucket tables).
        {
            const int npq = L.n_p * L.n_q, cpc = L.n_x / S.nchunk, items = npq * S.nchunk;
            for (int item = lane; item < items; item += 32) {
                const int ck = item / npq, ab = item - ck * npq;
                const int a = L.mg_nq ? (int)__umulhi((unsigned)ab, L.mg_nq) : ab, b = ab - a * L.n_q;
                const double p = __dadd_rn(g.cp, __dmul_rn(g.hp, s_tp[a])), q = __dadd_rn(g.cq, __dmul_rn(g.hq, s_tq[b]));
                const double pq = __dmul_rn(p, q), p2 = __dmul_rn(p, p), q2 = __dmul_rn(q, q);
                const double PA = __dadd_rn(__dmul_rn(0.25, p2), __dmul_rn(0.5625, q2)), QA = __dadd_rn(p2, __dmul_rn(0.25, q2));
                int ip = 0, iq = 0;
                for (int c = ck * cpc; c < (ck + 1) * cpc; ++c) {
                    const double pqx = __dmul_rn(pq, s_tx[c]);
                    double P2 = __dadd_rn(PA, __dmul_rn(0.75, pqx)), Q2 = __dsub_rn(QA, pqx);
                    P2 = P2 < 0.0 ? 0.0 : P2;
                    Q2 = Q2 < 0.0 ? 0.0 : Q2;
                    if (c == ck * cpc) {
                        ip = kFast ? locate_k<kLocK>(s_thr_p, s_bk_p, L.bk_hmin_p, L.bk_sh_p, P2) : locate(s_thr_p, s_bk_p, L.bk_hmin_p, L.bk_sh_p, P2);
                        iq = kFast ? locate_k<kLocK>(s_thr_q, s_bk_q, L.bk_hmin_q, L.bk_sh_q, Q2) : locate(s_thr_q, s_bk_q, L.bk_hmin_q, L.bk_sh_q, Q2);
                    } else {
                        while (s_thr_p[ip + 1] <= P2) ++ip;              // (+inf sentinel behind the last threshold)
                        while (iq >= 0 && s_thr_q[iq] > Q2) --iq;
                    }
                    const bool ok = (ip >= 0) & (ip < L.Np) & (iq >= 0) & (iq < L.Nq) & (P2 != 0.0) & (Q2 != 0.0);
                    const int t = ok ? ip * L.Nq + iq : -1;
                    if (t >= 0) atomicOr(&bits[t >> 5], 1u << (t & 31));
                    s_t[c * npq + ab] = t >= 0 ? (TT)t : (TT)~(TT)0;
                }
            }
        }
        __syncwarp();
        // ---- ranks: exclusive prefix of the word popcounts (lane = a contiguous run of words)
        int H;
        {
            const int k0 = min(lane * wchunk, L.n_words), k1 = min(k0 + wchunk, L.n_words);
            int mine = 0;
            for (int k = k0; k < k1; ++k) mine += __popc(bits[k]);
            int x = mine;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
            H = __shfl_sync(0xffffffffu, x, 31);
            int run = x - mine;
            for (int k = k0; k < k1; ++k) { wpre[k] = (unsigned short)run; run += __popc(bits[k]); }
        }
        __syncwarp();
        unsigned* g_key = nl.key + (size_t)cb * L.nnode;
        int placed = 0;
        for (int r0 = 0; r0 < H; r0 += S.hist_cap) {
            const int nr = min(S.hist_cap, H - r0);
            for (int k = lane; k < nr; k += 32) hist[k] = 0;
            __syncwarp();
            // ---- pass 2: nodes per rank (the targets of the next four steps are fetched while four are processed)
            {
                unsigned tn[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) { const int m = u * 32 + lane; tn[u] = m < L.nnode ? (unsigned)s_t[m] : kOff; }
                for (int st0 = 0; st0 < nsteps; st0 += 4) {
                    unsigned tt[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) { tt[u] = tn[u]; const int m = (st0 + 4 + u) * 32 + lane; tn[u] = m < L.nnode ? (unsigned)s_t[m] : kOff; }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (st0 + u >= nsteps) break;
                        const unsigned t = tt[u];
                        int r = -1;
                        if (t != kOff) r = (int)wpre[t >> 5] + __popc(bits[t >> 5] & ((1u << (t & 31)) - 1u)) - r0;
                        const bool in = r >= 0 && r < nr;
                        const unsigned same = __match_any_sync(0xffffffffu, in ? r : -1 - lane);
                        if (in && (same & lt) == 0u) hist[r] += __popc(same);
                        __syncwarp();
                    }
                }
            }
            // ---- exclusive scan of the counts, offset by what earlier windows placed
            for (int k0 = 0; k0 < nr; k0 += 32) {
                const int k = k0 + lane, v = k < nr ? hist[k] : 0;
                int x = v;
#pragma unroll
                for (int d = 1; d < 32; d <<= 1) { const int y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
                if (k < nr) hist[k] = placed + x - v;
                placed += __shfl_sync(0xffffffffu, x, 31);
            }
            __syncwarp();
            // ---- pass 3: placement in node order (stable)
            {
                unsigned tn[4];
#pragma unroll
                for (int u = 0; u < 4; ++u) { const int m = u * 32 + lane; tn[u] = m < L.nnode ? (unsigned)s_t[m] : kOff; }
                for (int st0 = 0; st0 < nsteps; st0 += 4) {
                    unsigned tt[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) { tt[u] = tn[u]; const int m = (st0 + 4 + u) * 32 + lane; tn[u] = m < L.nnode ? (unsigned)s_t[m] : kOff; }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        if (st0 + u >= nsteps) break;
                        const int m = (st0 + u) * 32 + lane;
                        const unsigned t = tt[u];
                        int r = -1;
                        if (t != kOff) r = (int)wpre[t >> 5] + __popc(bits[t >> 5] & ((1u << (t & 31)) - 1u)) - r0;
                        const bool in = r >= 0 && r < nr;
                        const unsigned same = __match_any_sync(0xffffffffu, in ? r : -1 - lane);
                        int base = 0;
                        if (in) { base = hist[r]; g_key[base + __popc(same & lt)] = (t << 14) | (unsigned)m; }
                        __syncwarp();
                        if (in && (same & lt) == 0u) hist[r] = base + __popc(same);
                        __syncwarp();
                    }
                }
            }
        }
        // ---- chunks of the sorted list (NodeLists): a chunk ends with its segment or after chunk_len nodes of it.
        // Lane = sorted position; a position's offset in its segment follows from the last segment start at or before it;
        // the lane that ends a chunk collects the (a, b) indices of the chunk's nodes from the lanes below it (those of
        // the previous step when the chunk began there).
        __syncwarp();
        int nck = 0;
        auto emit_chunks = [&](auto r_tag) {                    // r_tag: the chunk length at compile time (4: every config of BASELINE.json), 0: run time
            constexpr unsigned kR = decltype(r_tag)::value;
            uint2* g_chunk = nl.chunk + (size_t)cb * L.nnode;
            const unsigned R = kR ? kR : (unsigned)nl.chunk_len, bits = (unsigned)nl.ab_bits;      // R: a power of two, R * bits <= 32
            const unsigned npq = (unsigned)(L.n_p * L.n_q);
            int seg_start = 0;                                  // first position of the segment that is open at the start of a step
            unsigned carry = 1u;                                // the step's first position starts a segment
            unsigned prev[4] = {0u, 0u, 0u, 0u};                // the previous step's packed indices, level by level
            // keys of this step and of the next two (the last position's successor is the next step's first key, so the
            // loads run two steps ahead of their use)
            unsigned k = lane < placed ? g_key[lane] : 0u, kn = 32 + lane < placed ? g_key[32 + lane] : 0u;
            for (int base = 0; base < placed; base += 32) {
                const int pos = base + lane;
                const bool act = pos < placed;
                const unsigned knn = pos + 64 < placed ? g_key[pos + 64] : 0u;
                unsigned k1 = __shfl_down_sync(0xffffffffu, k, 1);
                const unsigned k1n = __shfl_sync(0xffffffffu, kn, 0);
                if (lane == 31) k1 = k1n;
                // (target, x-node) of a position = key with the (a, b) part removed: tc = t << 14 | c * npq
                const unsigned mk = k & 16383u;
                const unsigned ck = L.mg_npq ? __umulhi(mk, L.mg_npq) : mk;
                const unsigned ab = mk - ck * npq, tc = k - ab;
                unsigned tc1 = __shfl_down_sync(0xffffffffu, tc, 1);
                {   // lane 31's successor: the next step's first position
                    const unsigned mn = k1n & 16383u, cn = L.mg_npq ? __umulhi(mn, L.mg_npq) : mn;
                    if (lane == 31) tc1 = k1n - (mn - cn * npq);
                }
                const bool tend = act && (pos + 1 >= placed || (k1 >> 14) != (k >> 14));
                const bool send = act && (tend || tc1 != tc);
                const unsigned smask = __ballot_sync(0xffffffffu, send);
                const unsigned starts = (smask << 1) | carry;               // positions of this step that start a segment
                const unsigned below = starts & (0xffffffffu >> (31 - lane));
                const int start = below ? base + 31 - __clz(below) : seg_start;
                const unsigned off = (unsigned)(pos - start) & (R - 1u);    // position in its chunk
                const bool cend = act && (send || off == R - 1u);
                const unsigned cmask = __ballot_sync(0xffffffffu, cend);
                // v = the (a, b) indices of the R positions that end here, oldest in the low bits (doubling: 1, 2, 4, ... positions)
                unsigned v = ab;
#pragma unroll
                for (int lv = 0; lv < 4; ++lv) {
                    const unsigned d = 1u << lv;
                    if (kR ? d < kR : d < R) {
                        const unsigned src = (unsigned)(lane - (int)d) & 31u;
                        const unsigned va = __shfl_sync(0xffffffffu, v, src), vb = __shfl_sync(0xffffffffu, prev[lv], src);
                        prev[lv] = v;
                        v = ((unsigned)lane >= d ? va : vb) | (v << (d * bits));
                    }
                }
                if (cend) g_chunk[nck + __popc(cmask & lt)] =
                    make_uint2((k >> 14) | (off << 18) | ((unsigned)send << 22) | ((unsigned)tend << 23) | (ck << 24),
                               v >> ((R - 1u - off) * bits));
                nck += __popc(cmask);
                if (starts) seg_start = base + 31 - __clz(starts);
                carry = smask >> 31;
                k = kn; kn = knn;
            }
        };
        if (nl.chunk_len == 4) emit_chunks(std::integral_constant<unsigned, 4>{}); else emit_chunks(std::integral_constant<unsigned, 0>{});
        if (lane == 0) { nl.hits[cb] = H; nl.ntot[cb] = placed; nl.nchunk[cb] = nck; }
    }
}

// Pattern pass, kernel S: exclusive scan of the hit counts -> cellbase, nnz, max hits, nodes on the grid.  One CTA;
// thread = a contiguous run of cells (one load phase, one block scan, one store phase).
__global__ void __launch_bounds__(1024) k_scan_cells(DevLattice L, int n_blk, const int* __restrict__ hits,
                                                    const int* __restrict__ ntot, const int* __restrict__ nchunk,
                                                    int64_t* __restrict__ cellbase, int64_t* __restrict__ summary, int64_t capacity)
{
    __shared__ long long wsum[32], wnod[32], wchk[32];
    __shared__ int wmax[32];
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int chunk = (n_blk + 1023) >> 10;
    const int k0 = min(t * chunk, n_blk), k1 = min(k0 + chunk, n_blk);
    long long mine = 0, nodes = 0, chunks = 0;
    int mx = 0;
    for (int k = k0; k < k1; ++k) { const int h = hits[k]; mine += h; mx = max(mx, h); nodes += ntot[k]; chunks += nchunk[k]; }
    long long x = mine;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        nodes += __shfl_xor_sync(0xffffffffu, nodes, d); chunks += __shfl_xor_sync(0xffffffffu, chunks, d);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    }
    if (lane == 31) wsum[warp] = x;
    if (lane == 0) { wnod[warp] = nodes; wchk[warp] = chunks; wmax[warp] = mx; }
    __syncthreads();
    long long carry = 0;
    for (int w = 0; w < warp; ++w) carry += wsum[w];
    long long run = carry + x - mine;
    for (int k = k0; k < k1; ++k) { cellbase[k] = run; run += hits[k]; }
    if (t == 1023) {
        long long nn = 0, nc = 0; int m = 0;
        for (int w = 0; w < 32; ++w) { nn += wnod[w]; nc += wchk[w]; m = max(m, wmax[w]); }
        const long long total = carry + x;
        cellbase[n_blk] = total;
        summary[0] = total * L.totcoup;                 // nnz of the block
        summary[1] = m;                                 // max hit cells of any source cell
        summary[2] = nn;                                // nodes on the grid
        summary[5] = nc;                                // chunks of the sorted node lists (8 B each, read once by the fill)
        summary[4] = (capacity >= 0 && total * L.totcoup > capacity) ? 1 : 0;      // the fill of pm_build must not run
    }
}

// Pattern pass, kernel R: rowptr (block-local) from cellbase: row (cell k, alpha) starts at
// cellbase[k]*totcoup + H_k*cl_off[alpha] (PAPER.md:L339 keeps the row END addresses W; same information).
__global__ void __launch_bounds__(256) k_write_rowptr(DevLattice L, int n_blk, const int* __restrict__ hits,
                                                     const int64_t* __restrict__ cellbase, int64_t* __restrict__ rowptr)
{
    const int64_t n = (int64_t)n_blk * L.n_ch;
    for (int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; r <= n; r += (int64_t)gridDim.x * blockDim.x) {
        if (r == n) { rowptr[r] = cellbase[n_blk] * L.totcoup; continue; }
        const int k = (int)(r / L.n_ch), a = (int)(r - (int64_t)k * L.n_ch);
        rowptr[r] = cellbase[k] * L.totcoup + (int64_t)hits[k] * L.cl_off[a];
    }
}

// Hit cells of every source cell, ascending, at hitlist[cellbase[k] ..): the target at every change of target in the
// sorted node list.  One warp per source cell.  (Not on pm_build's path: pm_pattern with d_colidx and the SpMV without
// the column array use it.)
__global__ void __launch_bounds__(kThreads) k_hit_list(DevLattice L, int n_blk, NodeLists nl, const int64_t* __restrict__ cellbase,
                                                      int* __restrict__ hitlist)
{
    const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    for (int cb = blockIdx.x * wpb + (threadIdx.x >> 5); cb < n_blk; cb += gridDim.x * wpb) {
        const int ntot = nl.ntot[cb];
        const unsigned* g_key = nl.key + (size_t)cb * L.nnode;
        int* out = hitlist + cellbase[cb];
        int rank = 0;
        for (int p0 = 0; p0 < ntot; p0 += 32) {
            const int pos = p0 + lane;
            unsigned t = 0, tp = 0xffffffffu;
            if (pos < ntot) { t = g_key[pos] >> 14; if (pos) tp = g_key[pos - 1] >> 14; }
            const bool first = pos < ntot && t != tp;
            const unsigned b = __ballot_sync(0xffffffffu, first);
            if (first) out[rank + __popc(b & ((1u << lane) - 1u))] = (int)t;
            rank += __popc(b);
        }
    }
}

// (target, x-node) segments of the sorted lists (statistics for the work model only; run on demand)
__global__ void __launch_bounds__(kThreads) k_count_segments(DevLattice L, int n_blk, NodeLists nl, unsigned long long* __restrict__ total)
{
    const int lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    unsigned long long seg = 0;
    for (int cb = blockIdx.x * wpb + (threadIdx.x >> 5); cb < n_blk; cb += gridDim.x * wpb) {
        const int ntot = nl.ntot[cb];
        const unsigned* g_key = nl.key + (size_t)cb * L.nnode;
        for (int k = lane; k < ntot; k += 32) {
            const unsigned kk = g_key[k], kp = k ? g_key[k - 1] : 0u;
            const int mk = (int)(kk & 16383u), mp = (int)(kp & 16383u);
            const int ck = L.mg_npq ? (int)__umulhi((unsigned)mk, L.mg_npq) : mk, cp = L.mg_npq ? (int)__umulhi((unsigned)mp, L.mg_npq) : mp;
            seg += (k == 0 || (kk >> 14) != (kp >> 14) || ck != cp) ? 1 : 0;
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) seg += __shfl_xor_sync(0xffffffffu, seg, d);
    if (lane == 0 && seg) atomicAdd(total, seg);
}

// CSR rows from the per-pair sums (pm_fill.cuh, mode 2), for channel sets whose fill runs group by group: every nonzero
// of (source cell, k-th hit cell) is a combination of at most four of the pair's sums,
//   P[(cell, alpha), (cell_k, alpha')] = sum_i xc[4 o + i] * A[(cellbase + k) * stride + xpos[4 o + i]],   o = cl_off[alpha] + m.
// One CTA of 16 warps per source cell (cells from a work counter).  Every thread keeps the terms of its kOPL outputs in
// REGISTERS for the life of the kernel (output o = (warp * kOPL + j) * 32 + lane: a warp store covers consecutive alpha'
// of a row); the sums of kExpandTB hit cell pairs at a time arrive in shared memory by cp.async, double buffered.  Every
// 32-byte sector of vals / colidx is written once, in full (group-by-group fills of the CSR would write a few entries of
// every sector per group, which DRAM pays with a read-modify-write each time).
constexpr int kExpandWarps = 16, kExpandTB = 4;

template <int kOPL>
__global__ void __launch_bounds__(kExpandWarps * 32, 1)
k_op_expand(DevLattice L, int cell_begin, int n_blk, const int* __restrict__ hits, const int64_t* __restrict__ cellbase,
            const int* __restrict__ hitlist, const double* __restrict__ A, const unsigned short* __restrict__ g_xpos,
            const double* __restrict__ g_xc, const int64_t* __restrict__ rowptr, double* __restrict__ vals,
            int32_t* __restrict__ colidx, int* __restrict__ counter, const int64_t* __restrict__ guard)
{
    if (guard != nullptr && guard[4] != 0) return;
    extern __shared__ __align__(16) char smem[];
    constexpr int T = kExpandWarps * 32;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int nout = L.totcoup, stride = L.op_stride;           // stride: a multiple of 4 doubles
    double* s_A = (double*)smem;                                // [2][kExpandTB][stride]
    int* s_col = (int*)(smem + 2 * kExpandTB * stride * 8);     // [2][kExpandTB] first column of the batch's hit cells
    __shared__ int s_cb;
    // this thread's outputs: row offsets, column channel, positions and coefficients of up to four terms
    int od[kOPL];                                               // cl_off[alpha] | nc << 12 | m << 19 | alpha' << 25; -1: no output
    unsigned px[kOPL], py[kOPL];
    double c0[kOPL], c1[kOPL], c2[kOPL], c3[kOPL];
#pragma unroll
    for (int j = 0; j < kOPL; ++j) {
        const int o = (warp * kOPL + j) * 32 + lane;
        od[j] = -1; px[j] = py[j] = 0u; c0[j] = c1[j] = c2[j] = c3[j] = 0.0;
        if (o < nout) {
            const int al = L.o_alpha[o], off = L.cl_off[al], nc = L.cl_off[al + 1] - off;
            od[j] = off | (nc << 12) | ((o - off) << 19) | (L.cl[o] << 25);
            px[j] = (unsigned)g_xpos[4 * o] | ((unsigned)g_xpos[4 * o + 1] << 16);
            py[j] = (unsigned)g_xpos[4 * o + 2] | ((unsigned)g_xpos[4 * o + 3] << 16);
            c0[j] = g_xc[4 * o]; c1[j] = g_xc[4 * o + 1]; c2[j] = g_xc[4 * o + 2]; c3[j] = g_xc[4 * o + 3];
        }
    }
    const unsigned sA0 = (unsigned)__cvta_generic_to_shared(s_A);
    for (;;) {
        __syncthreads();
        if (tid == 0) s_cb = atomicAdd(counter, 1);
        __syncthreads();
        const int cb = s_cb;
        if (cb >= n_blk) break;
        const int H = hits[cb];
        const int64_t hbase = cellbase[cb], rbase = rowptr[(int64_t)cb * L.n_ch];
        double* __restrict__ row0 = vals + rbase;
        int32_t* __restrict__ col0 = colidx ? colidx + rbase : nullptr;
        // batch b of the cell's hit cell pairs -> buffer b & 1 (16-byte cp.async pieces; the pairs' sums are contiguous)
        auto fetch = [&](int b) {
            const int k0 = b * kExpandTB, nb = min(kExpandTB, H - k0);
            if (nb > 0) {
                const double* src = A + (hbase + k0) * (int64_t)stride;
                const unsigned dst = sA0 + (unsigned)((b & 1) * kExpandTB * stride * 8);
                for (int i = tid; i < nb * stride / 2; i += T)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * i), "l"(src + 2 * i) : "memory");
                if (tid < nb) s_col[(b & 1) * kExpandTB + tid] = hitlist[hbase + k0 + tid] * L.n_ch;
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        const int nbatch = (H + kExpandTB - 1) / kExpandTB;
        fetch(0);
        for (int b = 0; b < nbatch; ++b) {
            fetch(b + 1);
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            __syncthreads();
            const int k0 = b * kExpandTB, nb = min(kExpandTB, H - k0);
            const double* Ab = s_A + (b & 1) * kExpandTB * stride;
            const int* colb = s_col + (b & 1) * kExpandTB;
#pragma unroll
            for (int j = 0; j < kOPL; ++j) {
                if (od[j] < 0) continue;
                const int clo = od[j] & 4095, nc = (od[j] >> 12) & 127, mm = (od[j] >> 19) & 63, ap = (unsigned)od[j] >> 25;
                const unsigned p0 = px[j] & 65535u, p1 = px[j] >> 16, p2 = py[j] & 65535u, p3 = py[j] >> 16;
                unsigned e = (unsigned)(H * clo + k0 * nc + mm);
#pragma unroll
                for (int t = 0; t < kExpandTB; ++t) {
                    if (t < nb) {
                        const double* At = Ab + t * stride;
                        row0[e] = fma(c3[j], At[p3], fma(c2[j], At[p2], fma(c1[j], At[p1], c0[j] * At[p0])));
                        if (col0) col0[e] = colb[t] + ap;
                        e += (unsigned)nc;
                    }
                }
            }
            __syncthreads();                                    // the buffer is free for batch b + 2
        }
    }
}

cudaError_t launch_op_expand(const DevLattice& L, int cell_begin, int n_blk, const NodeLists& nl, const int64_t* cellbase, const int* hitlist,
                             const double* A, const unsigned short* xpos, const double* xc, const int64_t* rowptr, double* vals,
                             int32_t* colidx, int* counter, const int64_t* guard, int n_sm, cudaStream_t st)
{
    using Fn = void (*)(DevLattice, int, int, const int*, const int64_t*, const int*, const double*, const unsigned short*, const double*,
                        const int64_t*, double*, int32_t*, int*, const int64_t*);
    const int need = (L.totcoup + kExpandWarps * 32 - 1) / (kExpandWarps * 32);       // outputs per thread
    Fn fn = need <= 2 ? k_op_expand<2> : need <= 4 ? k_op_expand<4> : need <= 6 ? k_op_expand<6> : need <= 8 ? k_op_expand<8> : nullptr;
    if (!fn) return cudaErrorInvalidConfiguration;
    const size_t smem = 2 * (size_t)kExpandTB * (size_t)L.op_stride * 8 + 2 * kExpandTB * sizeof(int);
    if (smem > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(counter, 0, sizeof(int), st)) != cudaSuccess) return e;
    int per_sm = 1;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, kExpandWarps * 32, smem)) != cudaSuccess) return e;
    const int grid = std::max(1, std::min(n_sm * std::max(per_sm, 1), n_blk));
    fn<<<grid, kExpandWarps * 32, smem, st>>>(L, cell_begin, n_blk, nl.hits, cellbase, hitlist, A, xpos, xc, rowptr, vals, colidx, counter, guard);
    count_launch();
    return cudaGetLastError();
}

// y = P0 x straight from the per-pair sums (the operator form of P0: 8 * n_functions bytes per hit cell pair instead of
// 8 bytes per nonzero; PAPER.md:L408-410 — the iterations are what remains the bottleneck once P0 is on the GPU).
//   y[(cell, alpha)] = sum_k sum_{alpha'} ( sum_i xc[4 o + i] * A[(cellbase + k) * stride + xpos[4 o + i]] ) * x[(cell_k, alpha')]
// One CTA per source cell; a thread keeps the terms of its kOPL outputs AND their running products with x in registers over
// all hit cells of the cell, so nothing but the sums (cp.async, double buffered) and the x slices is read and nothing is
// written until the cell's rows are summed — in a fixed order: bitwise reproducible, no floating-point atomics.
constexpr int kApplyTB = 8, kApplyStages = 4;       // hit cell pairs per batch; batches in flight

template <int kOPL, int kWarps>
__global__ void __launch_bounds__(kWarps * 32, (kWarps <= 8 ? 2 : 1))
k_op_apply(DevLattice L, int n_blk, int hmax, const int* __restrict__ hits, const int64_t* __restrict__ cellbase, const int* __restrict__ hitlist,
           const double* __restrict__ A, const unsigned short* __restrict__ g_xpos, const double* __restrict__ g_xc,
           const double* __restrict__ x, double* __restrict__ y, int* __restrict__ counter)
{
    extern __shared__ __align__(16) char smem[];
    constexpr int T = kWarps * 32;
    const int tid = threadIdx.x;
    const int nout = L.totcoup, stride = L.op_stride, nch = L.n_ch;
    const int nchp = (nch + 1) & ~1;                                     // x slices padded to 16 bytes
    double* s_A = (double*)smem;                                        // [kApplyStages][kApplyTB][stride]
    double* s_x = s_A + kApplyStages * kApplyTB * stride;               // [kApplyStages][kApplyTB][nchp]
    double* s_y = s_x + kApplyStages * kApplyTB * nchp;                 // [totcoup] per-output sums of the cell
    int* s_hit = (int*)(s_y + nout);                                    // [hmax] the cell's hit cells
    __shared__ int s_cb;
    int ap[kOPL];                                                       // column channel of the output
    unsigned px[kOPL], py[kOPL];
    double c0[kOPL], c1[kOPL], c2[kOPL], c3[kOPL];
#pragma unroll
    for (int j = 0; j < kOPL; ++j) {
        const int o = j * T + tid;
        ap[j] = 0; px[j] = py[j] = 0u; c0[j] = c1[j] = c2[j] = c3[j] = 0.0;      // (no output: zero coefficients)
        if (o < nout) {
            ap[j] = L.cl[o];
            px[j] = 8u * g_xpos[4 * o] | (8u * g_xpos[4 * o + 1] << 16);         // byte offsets (8 * stride < 65536)
            py[j] = 8u * g_xpos[4 * o + 2] | (8u * g_xpos[4 * o + 3] << 16);
            c0[j] = g_xc[4 * o]; c1[j] = g_xc[4 * o + 1]; c2[j] = g_xc[4 * o + 2]; c3[j] = g_xc[4 * o + 3];
        }
    }
    const unsigned sA0 = (unsigned)__cvta_generic_to_shared(s_A), sX0 = (unsigned)__cvta_generic_to_shared(s_x);
    for (;;) {
        __syncthreads();
        if (tid == 0) s_cb = atomicAdd(counter, 1);
        __syncthreads();
        const int cb = s_cb;
        if (cb >= n_blk) break;
        const int H = min(hits[cb], hmax);
        const int64_t hbase = cellbase[cb];
        for (int k = tid; k < H; k += T) s_hit[k] = hitlist[hbase + k];
        __syncthreads();
        double acc[kOPL];
#pragma unroll
        for (int j = 0; j < kOPL; ++j) acc[j] = 0.0;
        // batch b of the cell's pairs -> ring slot b % kApplyStages: the pairs' sums (contiguous, 16-byte pieces) and the x
        // slices of their hit cells (8-byte pieces), all by cp.async
        auto fetch = [&](int b) {
            const int k0 = b * kApplyTB, nb = min(kApplyTB, H - k0), slot = b % kApplyStages;
            if (nb > 0) {
                const double* src = A + (hbase + k0) * (int64_t)stride;
                const unsigned dst = sA0 + (unsigned)(slot * kApplyTB * stride * 8);
                for (int i = tid; i < nb * stride / 2; i += T)
                    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst + 16u * i), "l"(src + 2 * i) : "memory");
                const unsigned dx = sX0 + (unsigned)(slot * kApplyTB * nchp * 8);
                for (int i = tid; i < nb * nch; i += T) {
                    const int t = i / nch, a = i - t * nch;
                    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dx + 8u * (t * nchp + a)), "l"(x + (int64_t)s_hit[k0 + t] * nch + a) : "memory");
                }
            }
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        const int nbatch = (H + kApplyTB - 1) / kApplyTB;
#pragma unroll
        for (int b = 0; b < kApplyStages - 1; ++b) fetch(b);
        for (int b = 0; b < nbatch; ++b) {
            fetch(b + kApplyStages - 1);
            asm volatile("cp.async.wait_group %0;" ::"n"(kApplyStages - 1) : "memory");
            __syncthreads();
            const int nb = min(kApplyTB, H - b * kApplyTB), slot = b % kApplyStages;
            const double* Ab = s_A + slot * kApplyTB * stride;
            const double* xb = s_x + slot * kApplyTB * nchp;
            // pair by pair (the pair's base address is the same for all threads), output by output: byte offsets of the four sums
            // come unpacked from registers, so a term is one add, one shared-memory load and one FMA
#pragma unroll
            for (int t = 0; t < kApplyTB; ++t) {
                if (t < nb) {
                    const char* At = (const char*)(Ab + t * stride);
                    const double* xt = xb + t * nchp;
#pragma unroll
                    for (int j = 0; j < kOPL; ++j) {
                        const double v = fma(c3[j], *(const double*)(At + (py[j] >> 16)),
                                         fma(c2[j], *(const double*)(At + (py[j] & 65535u)),
                                         fma(c1[j], *(const double*)(At + (px[j] >> 16)), c0[j] * *(const double*)(At + (px[j] & 65535u)))));
                        acc[j] = fma(v, xt[ap[j]], acc[j]);
                    }
                }
            }
            __syncthreads();                                            // the slot is free for batch b + kApplyStages
        }
#pragma unroll
        for (int j = 0; j < kOPL; ++j) { const int o = j * T + tid; if (o < nout) s_y[o] = acc[j]; }
        __syncthreads();
        if (tid < nch) {                                                // row alpha = the outputs cl_off[alpha] .. cl_off[alpha + 1], in order
            double r = 0.0;
            for (int o = L.cl_off[tid]; o < L.cl_off[tid + 1]; ++o) r += s_y[o];
            y[(int64_t)cb * nch + tid] = r;
        }
    }
}

cudaError_t launch_op_apply(const DevLattice& L, int n_blk, int hmax, const NodeLists& nl, const int64_t* cellbase, const int* hitlist, const double* A,
                            const unsigned short* xpos, const double* xc, const double* x, double* y, int* counter, int n_sm, cudaStream_t st)
{
    using Fn = void (*)(DevLattice, int, int, const int*, const int64_t*, const int*, const double*, const unsigned short*, const double*,
                        const double*, double*, int*);
    Fn fn = nullptr;
    int warps = 8;
    const int n = L.totcoup;
    if (n <= 256) fn = k_op_apply<1, 8>;
    else if (n <= 512) fn = k_op_apply<2, 8>;
    else if (n <= 768) fn = k_op_apply<3, 8>;
    else if (n <= 1024) fn = k_op_apply<4, 8>;
    else { warps = 16; fn = n <= 2048 ? k_op_apply<4, 16> : n <= 3072 ? k_op_apply<6, 16> : n <= 4096 ? k_op_apply<8, 16> : nullptr; }
    if (!fn) return cudaErrorInvalidConfiguration;
    const size_t nchp = ((size_t)L.n_ch + 1) & ~(size_t)1;
    const size_t smem = 8 * ((size_t)kApplyStages * kApplyTB * ((size_t)L.op_stride + nchp) + (size_t)L.totcoup) + 4 * (size_t)std::max(hmax, 1);
    if (smem > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(counter, 0, sizeof(int), st)) != cudaSuccess) return e;
    int per_sm = 1;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, (const void*)fn, warps * 32, smem)) != cudaSuccess) return e;
    const int grid = std::max(1, std::min(n_sm * std::max(per_sm, 1), n_blk));
    fn<<<grid, warps * 32, smem, st>>>(L, n_blk, hmax, nl.hits, cellbase, hitlist, A, xpos, xc, x, y, counter);
    count_launch();
    return cudaGetLastError();
}

// Pattern pass, kernel B: column indices, ascending within each row, from the hit lists.  Thread = output (alpha, m-th
// coupled alpha'), looping over the hit cells k: entry k of row alpha sits at row_start + k*nc + m, so the threads
// of a warp write runs of consecutive m and consecutive k fill the gaps (the same store pattern as the fill's rows).
__global__ void __launch_bounds__(1024) k_emit_cols(DevLattice L, NodeLists nl, const int64_t* __restrict__ cellbase,
                                                   const int* __restrict__ hitlist, const int64_t* __restrict__ rowptr,
                                                   int32_t* __restrict__ colidx)
{
    const int T = blockDim.x, tid = threadIdx.x;
    const int H = nl.hits[blockIdx.x];
    const int* __restrict__ hit = hitlist + cellbase[blockIdx.x];
    int32_t* __restrict__ row0 = colidx + rowptr[(int64_t)blockIdx.x * L.n_ch];
    // the block is G groups of `ow` threads: a group covers all outputs (in passes if totcoup > ow) for k = g, g+G, ...
    const int ow = min(T, (L.totcoup + 31) & ~31), G = T / ow, g = tid / ow;
    if (g < G)
        for (int o = tid - g * ow; o < L.totcoup; o += ow) {
            const int al = L.o_alpha[o], off = L.cl_off[al], nc = L.cl_off[al + 1] - off, ap = L.cl[o];
            int32_t* out = row0 + ((size_t)H * off + (o - off));
#pragma unroll 4
            for (int k = g; k < H; k += G) out[(size_t)k * nc] = hit[k] * L.n_ch + ap;
        }
}

// ------------------------------------------------------------------------------------------------
// SpMV check: one warp per row, y = A x.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_spmv(int64_t n_rows, const int64_t* __restrict__ rowptr,
                                             const int32_t* __restrict__ colidx, const double* __restrict__ vals,
                                             const double* __restrict__ x, double* __restrict__ y)
{
    const int lane = threadIdx.x & 31;
    const int64_t wpb = blockDim.x >> 5;
    for (int64_t r = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5); r < n_rows; r += (int64_t)gridDim.x * wpb) {
        double s = 0.0;
        int64_t k = rowptr[r] + lane;
        const int64_t ke = rowptr[r + 1];
        for (; k + 96 < ke; k += 128) {                    // four independent element chains in flight per lane
            double vv[4], xx[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) { vv[u] = vals[k + 32 * u]; xx[u] = x[colidx[k + 32 * u]]; }
#pragma unroll
            for (int u = 0; u < 4; ++u) s += vv[u] * xx[u];
        }
        for (; k < ke; k += 32) s += vals[k] * x[colidx[k]];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0) y[r] = s;
    }
}

// ------------------------------------------------------------------------------------------------
// SpMV without the column array.  A row (cell, alpha) holds, for each hit cell k of its source cell in ascending
// order, each alpha' coupled to alpha: column = hit[k]*n_ch + cl[alpha][m].  With the hit lists (4 B per hit cell pair,
// 6 MB on configs[4]) the 4 B per nonzero of colidx need not be read: 8 instead of 12 B per nonzero from HBM.
// Same lane striding and reduction as k_spmv, hence the same bits.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_spmv_implicit(DevLattice L, int64_t n_rows, const int64_t* __restrict__ rowptr,
                                                      const int* __restrict__ hits, const int64_t* __restrict__ cellbase,
                                                      const int* __restrict__ hitlist, const double* __restrict__ vals,
                                                      const double* __restrict__ x, double* __restrict__ y)
{
    const int lane = threadIdx.x & 31;
    const int64_t wpb = blockDim.x >> 5;
    for (int64_t r = (int64_t)blockIdx.x * wpb + (threadIdx.x >> 5); r < n_rows; r += (int64_t)gridDim.x * wpb) {
        const int cell = (int)(r / L.n_ch), al = (int)(r - (int64_t)cell * L.n_ch);
        const int off = L.cl_off[al], nc = L.cl_off[al + 1] - off, len = hits[cell] * nc;
        const unsigned mg = nc > 1 ? (unsigned)(((1ull << 32) + (unsigned)nc - 1) / (unsigned)nc) : 0u;
        const int* hl = hitlist + cellbase[cell];
        const int* cl = L.cl + off;
        const double* v = vals + rowptr[r];
        double s = 0.0;
        for (int idx = lane; idx < len; idx += 32) {
            const int k = mg ? (int)__umulhi((unsigned)idx, mg) : idx, m = idx - k * nc;
            s += v[idx] * x[hl[k] * L.n_ch + cl[m]];
        }
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
        if (lane == 0) y[r] = s;
    }
}

// ------------------------------------------------------------------------------------------------
// Host launchers
// ------------------------------------------------------------------------------------------------
static std::atomic<int64_t> g_launches{0};
int64_t launch_count() { return g_launches.load(); }
void count_launch() { ++g_launches; }

static int map_sort_warps()
{
    static const int want = [] { const char* e = std::getenv("PM_MAPSORT_WARPS"); return e ? std::max(1, std::min(kMapSortMaxWarps, std::atoi(e))) : kMapSortMaxWarps; }();
    return want;
}

size_t map_sort_scratch_bytes(const DevLattice& L, int n_sm)
{
    const MapSortSmem S = map_sort_plan(L, map_sort_warps());
    return (size_t)n_sm * S.ctas * std::max(S.nw, 1) * (size_t)((L.nnode + 31) & ~31) * (S.wide ? 4 : 2);
}

cudaError_t launch_map_sort(const DevLattice& L, int cell_begin, int n_blk, const NodeLists& nl, int n_sm, int* counter, void* scratch, cudaStream_t st)
{
    // warps per CTA: as many as shared memory holds, at most kMapSortMaxWarps (PM_MAPSORT_WARPS: test hook)
    const MapSortSmem S = map_sort_plan(L, map_sort_warps());
    if (S.nw < 1) return cudaErrorInvalidConfiguration;
    using Fn = void (*)(DevLattice, MapSortSmem, int, int, NodeLists, int*, void*);
    const bool fast = L.bk_kmax <= kLocK;
    const Fn fn = S.wide ? (fast ? k_map_sort<unsigned, true> : k_map_sort<unsigned, false>)
                         : (fast ? k_map_sort<unsigned short, true> : k_map_sort<unsigned short, false>);
    cudaError_t e = cudaFuncSetAttribute((const void*)fn, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e != cudaSuccess) return e;
    const int grid = std::max(1, std::min(n_sm * S.ctas, (n_blk + S.nw - 1) / S.nw));
    fn<<<grid, S.nw * 32, S.total, st>>>(L, S, cell_begin, n_blk, nl, counter, scratch);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_scan_rows(const DevLattice& L, int n_blk, const NodeLists& nl, int64_t* cellbase, int64_t* rowptr,
                             int64_t* summary, int64_t capacity, cudaStream_t st)
{
    k_scan_cells<<<1, 1024, 0, st>>>(L, n_blk, nl.hits, nl.ntot, nl.nchunk, cellbase, summary, capacity);
    ++g_launches;
    const int64_t n = (int64_t)n_blk * L.n_ch + 1;
    k_write_rowptr<<<(unsigned)std::min<int64_t>((n + 255) / 256, 148 * 8), 256, 0, st>>>(L, n_blk, nl.hits, cellbase, rowptr);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_emit_cols(const DevLattice& L, int n_blk, const NodeLists& nl, const int64_t* cellbase, const int* hitlist,
                             const int64_t* rowptr, int32_t* colidx, cudaStream_t st)
{
    const int threads = std::min(1024, std::max(128, (L.totcoup + 31) & ~31));
    k_emit_cols<<<n_blk, threads, 0, st>>>(L, nl, cellbase, hitlist, rowptr, colidx);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_hit_list(const DevLattice& L, int n_blk, const NodeLists& nl, const int64_t* cellbase, int* hitlist, cudaStream_t st)
{
    k_hit_list<<<std::max(1, std::min((n_blk + 7) / 8, 148 * 8)), kThreads, 0, st>>>(L, n_blk, nl, cellbase, hitlist);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_count_segments(const DevLattice& L, int n_blk, const NodeLists& nl, unsigned long long* total, cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(total, 0, sizeof(unsigned long long), st);
    if (e != cudaSuccess) return e;
    k_count_segments<<<std::max(1, std::min((n_blk + 7) / 8, 148 * 8)), kThreads, 0, st>>>(L, n_blk, nl, total);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_spmv_implicit(const DevLattice& L, int64_t n_rows, const int64_t* rowptr, const int* hits, const int64_t* cellbase,
                                 const int* hitlist, const double* vals, const double* x, double* y, cudaStream_t st)
{
    const int64_t blocks = std::min<int64_t>((n_rows + 7) / 8, 148 * 32);
    k_spmv_implicit<<<(unsigned)std::max<int64_t>(blocks, 1), 256, 0, st>>>(L, n_rows, rowptr, hits, cellbase, hitlist, vals, x, y);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_spmv(int64_t n_rows, const int64_t* rowptr, const int32_t* colidx, const double* vals,
                        const double* x, double* y, cudaStream_t st)
{
    const int64_t blocks = std::min<int64_t>((n_rows + 7) / 8, 148 * 32);
    k_spmv<<<(unsigned)std::max<int64_t>(blocks, 1), 256, 0, st>>>(n_rows, rowptr, colidx, vals, x, y);
    ++g_launches;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// FP64 peak diagnostic: 16 independent FMA chains per thread, 1024 threads per CTA, 2 CTAs per SM.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_dfma_peak(int iters, double seed, double* __restrict__ sink)
{
    double a[16];
#pragma unroll
    for (int k = 0; k < 16; ++k) a[k] = seed + k + threadIdx.x;
    const double m = 1.0000001, c = 1e-9;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int k = 0; k < 16; ++k) a[k] = fma(a[k], m, c);
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < 16; ++k) s += a[k];
    if (s == 12345.678) sink[0] = s;           // never true; keeps the chains alive
}

cudaError_t measure_dfma(int n_sm, double* tflops, cudaStream_t st)
{
    double* sink = nullptr;
    cudaError_t e = cudaMalloc(&sink, 8);
    if (e != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    const int iters = 4096, blocks = 2 * n_sm;
    float best = 1e30f;
    for (int rep = 0; rep < 6; ++rep) {
        cudaEventRecord(t0, st);
        k_dfma_peak<<<blocks, 1024, 0, st>>>(iters, 1.0, sink);
        ++g_launches;
        cudaEventRecord(t1, st);
        if ((e = cudaEventSynchronize(t1)) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, t0, t1);
        if (rep > 0 && ms < best) best = ms;
    }
    cudaEventDestroy(t0); cudaEventDestroy(t1); cudaFree(sink);
    if (e != cudaSuccess) return e;
    *tflops = 2.0 * 16.0 * iters * 1024.0 * blocks / (best * 1e-3) * 1e-12;
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// Iteration step (eq. 24):  K u = O P0 V~1 G1 u  with G1 diagonal,
// P0 the CSR matrix of this library and O, V~1 block matrices with (Np x Np) blocks acting on the pair index i for fixed
// (j, alpha).  k_block_apply is one block-matrix factor with an optional diagonal factor folded in:
//   out[(i,j,a)] = sum_i' B_a[i][i'] * (diag ? diag[(i',j,a)] : 1) * in[(i',j,a)] ,  index (i*Nq + j)*n_ch + a.
// The vectors (8 M bytes) and the blocks stay in L2; the step is bound by the P0 SpMV (12 B per nonzero from HBM).
// ------------------------------------------------------------------------------------------------
// Per channel a this is the product Out_a (Np x Nq) = B_a (Np x Np) * In_a (Np x Nq) on strided data.  CTA = (a, 32 x 32
// tile of (i, j)): the 32 rows of B_a and the Np x 32 slab of (diag*)in are staged in shared memory (each reused 32
// times), thread = 2 x 2 outputs.
constexpr int kBlkT = 32;

__global__ void __launch_bounds__(256) k_block_apply(int Np, int Nq, int n_ch, const double* __restrict__ B,
                                                    const double* __restrict__ diag, const double* __restrict__ in,
                                                    double* __restrict__ out, int transpose)
{
    extern __shared__ __align__(16) char smem[];
    const int ld = Np + 1;                                     // padded row length of the B tile
    double* sB = (double*)smem;                                 // [kBlkT][Np + 1]
    double* sX = sB + kBlkT * ld;                               // [Np][kBlkT]
    const int ti = (Np + kBlkT - 1) / kBlkT, tj = (Nq + kBlkT - 1) / kBlkT;
    const int a = blockIdx.x / (ti * tj), rem = blockIdx.x - a * ti * tj, i0 = (rem / tj) * kBlkT, j0 = (rem % tj) * kBlkT;
    const int64_t stride = (int64_t)Nq * n_ch;
    const double* Ba = B + (size_t)a * Np * Np;
    // staging by cp.async: all of a thread's loads are in flight at once (the strided 8-byte reads of the vector are what the
    // kernel waits for); out-of-range entries are zeroed with plain stores
    const unsigned sB0 = (unsigned)__cvta_generic_to_shared(sB), sX0 = (unsigned)__cvta_generic_to_shared(sX);
    for (int k = threadIdx.x; k < kBlkT * Np; k += blockDim.x) {
        const int r = k / Np, c = k - r * Np;
        if (i0 + r < Np) {
            const double* src = transpose ? Ba + (size_t)c * Np + (i0 + r) : Ba + (size_t)(i0 + r) * Np + c;     // B_a or its transpose
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sB0 + 8u * (unsigned)(r * ld + c)), "l"(src) : "memory");
        } else sB[r * ld + c] = 0.0;
    }
    for (int k = threadIdx.x; k < Np * kBlkT; k += blockDim.x) {
        const int ip = k / kBlkT, jj = k - ip * kBlkT;
        if (j0 + jj < Nq) {
            const int64_t c = (int64_t)ip * stride + (int64_t)(j0 + jj) * n_ch + a;
            asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(sX0 + 8u * (unsigned)k), "l"(in + c) : "memory");
        } else sX[k] = 0.0;
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
    if (diag) {                                                 // the diagonal factor: every thread scales the entries it copied
        for (int k = threadIdx.x; k < Np * kBlkT; k += blockDim.x) {
            const int ip = k / kBlkT, jj = k - ip * kBlkT;
            if (j0 + jj < Nq) sX[k] *= diag[(int64_t)ip * stride + (int64_t)(j0 + jj) * n_ch + a];
        }
    }
    __syncthreads();
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;     // outputs (i0 + ty, +16) x (j0 + tx, +16)
    double s00 = 0.0, s01 = 0.0, s10 = 0.0, s11 = 0.0;
    const double* b0 = sB + ty * ld;
    const double* b1 = sB + (ty + 16) * ld;
    for (int ip = 0; ip < Np; ++ip) {
        const double x0 = sX[ip * kBlkT + tx], x1 = sX[ip * kBlkT + tx + 16], v0 = b0[ip], v1 = b1[ip];
        s00 = fma(v0, x0, s00); s01 = fma(v0, x1, s01);
        s10 = fma(v1, x0, s10); s11 = fma(v1, x1, s11);
    }
    const int i = i0 + ty, j = j0 + tx;
    if (i < Np && j < Nq) out[(int64_t)i * stride + (int64_t)j * n_ch + a] = s00;
    if (i < Np && j + 16 < Nq) out[(int64_t)i * stride + (int64_t)(j + 16) * n_ch + a] = s01;
    if (i + 16 < Np && j < Nq) out[(int64_t)(i + 16) * stride + (int64_t)j * n_ch + a] = s10;
    if (i + 16 < Np && j + 16 < Nq) out[(int64_t)(i + 16) * stride + (int64_t)(j + 16) * n_ch + a] = s11;
}

cudaError_t launch_block_apply(int Np, int Nq, int n_ch, const double* B, const double* diag, const double* in, double* out,
                               int transpose, cudaStream_t st)
{
    const int ti = (Np + kBlkT - 1) / kBlkT, tj = (Nq + kBlkT - 1) / kBlkT;
    const size_t sm = sizeof(double) * ((size_t)kBlkT * (Np + 1) + (size_t)Np * kBlkT);
    if (sm > 227 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(k_block_apply, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    k_block_apply<<<(unsigned)(n_ch * ti * tj), 256, sm, st>>>(Np, Nq, n_ch, B, diag, in, out, transpose);
    count_launch();
    return cudaGetLastError();
}

// rowptr of a shard -> global offsets (sharded multi-GPU build: add the nonzeros of the shards before it)
__global__ void __launch_bounds__(256) k_add_offset(int64_t* __restrict__ a, int64_t n, int64_t off)
{
    for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) a[k] += off;
}

cudaError_t launch_add_offset(int64_t* a, int64_t n, int64_t off, cudaStream_t st)
{
    k_add_offset<<<(unsigned)std::max<int64_t>(1, std::min<int64_t>((n + 255) / 256, 148 * 8)), 256, 0, st>>>(a, n, off);
    count_launch();
    return cudaGetLastError();
}

}  // namespace pm
