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
// Pattern pass, kernel A: map every node of a source cell, rank the hit cells, stable counting sort of the
// node ids by rank.  Node id m = c*(n_p*n_q) + a*n_q + b, so the sorted list is ordered by (target, x-node, a, b).
// ------------------------------------------------------------------------------------------------
size_t map_sort_smem(const DevLattice& L, int hits_fast)
{
    const int nw = kThreads / 32;
    const int hcap = std::min(L.nnode, L.n_cells);
    return al16(8 * (size_t)L.pe_pad) + al16(8 * (size_t)L.qe_pad) + 2 * al16(2 * (size_t)kBuckets) + al16(8 * (size_t)L.n_p) + al16(8 * (size_t)L.n_q)
         + al16(8 * (size_t)L.n_x) + 2 * al16(4 * (size_t)L.n_words) + al16(4 * (size_t)(kThreads + 1))
         + al16(4 * (size_t)L.nnode) + al16(2 * (size_t)L.nnode) + al16(4 * (size_t)(hcap + 1))
         + al16(4 * (size_t)std::max(nw * std::min(hcap, hits_fast), hcap));
}

__global__ void __launch_bounds__(kThreads) k_map_sort(DevLattice L, int cell_begin, NodeLists nl, int hits_fast)
{
    extern __shared__ __align__(16) char smem[];
    constexpr int T = kThreads, NW = kThreads / 32;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int hcap = min(L.nnode, L.n_cells);
    char* sp = smem;
    double* s_thr_p = (double*)carve(sp, 8 * (size_t)L.pe_pad);
    double* s_thr_q = (double*)carve(sp, 8 * (size_t)L.qe_pad);
    unsigned short* s_bk_p = (unsigned short*)carve(sp, 2 * (size_t)kBuckets);
    unsigned short* s_bk_q = (unsigned short*)carve(sp, 2 * (size_t)kBuckets);
    double* s_tp = (double*)carve(sp, 8 * (size_t)L.n_p);
    double* s_tq = (double*)carve(sp, 8 * (size_t)L.n_q);
    double* s_tx = (double*)carve(sp, 8 * (size_t)L.n_x);
    HitSet hs;
    hs.bits = (unsigned*)carve(sp, 4 * (size_t)L.n_words);
    hs.wpre = (int*)carve(sp, 4 * (size_t)L.n_words);
    hs.scratch = (int*)carve(sp, 4 * (size_t)(T + 1));
    int* s_tgt = (int*)carve(sp, 4 * (size_t)L.nnode);
    unsigned short* s_rk = (unsigned short*)carve(sp, 2 * (size_t)L.nnode);     // rank of each node's target (0xffff: off the grid)
    int* s_start = (int*)carve(sp, 4 * (size_t)(hcap + 1));
    int* s_hist = (int*)carve(sp, 4 * (size_t)max(NW * min(hcap, hits_fast), hcap));

    for (int k = tid; k < L.pe_pad; k += T) s_thr_p[k] = L.thr_p[k];
    for (int k = tid; k < L.qe_pad; k += T) s_thr_q[k] = L.thr_q[k];
    for (int k = tid; k < kBuckets; k += T) { s_bk_p[k] = L.bk_p[k]; s_bk_q[k] = L.bk_q[k]; }
    const Locator lc{s_thr_p, s_thr_q, s_bk_p, s_bk_q, L.bk_hmin_p, L.bk_sh_p, L.bk_hmin_q, L.bk_sh_q, L.Np, L.Nq};
    for (int k = tid; k < L.n_p; k += T) s_tp[k] = L.tp[k];
    for (int k = tid; k < L.n_q; k += T) s_tq[k] = L.tq[k];
    for (int k = tid; k < L.n_x; k += T) s_tx[k] = L.tx[k];
    for (int k = tid; k < L.n_words; k += T) hs.bits[k] = 0u;
    const int cell = cell_begin + blockIdx.x;
    const int ci = cell / L.Nq, cj = cell - ci * L.Nq;
    const CellGeom g = cell_geom(L.pe, L.qe, ci, cj);
    __syncthreads();

    for (int m = tid; m < L.nnode; m += T) {
        int c, a, b;
        split_node(L, m, c, a, b);
        double p, q, P2, Q2;
        map_node_sq(g, s_tp[a], s_tq[b], s_tx[c], p, q, P2, Q2);
        const int t = target_cell_sq(lc, P2, Q2);
        if (t >= 0) atomicOr(&hs.bits[t >> 5], 1u << (t & 31));
        s_tgt[m] = t;
    }
    __syncthreads();
    const int H = rank_bits_n(L.n_words, hs);
    // stable counting sort: each of `nwe` warps owns a contiguous slice of node ids and a histogram of H counters
    // (all warps when H <= hits_fast, else warp 0 alone: rare, slow, same result)
    const int nwe = (H <= hits_fast) ? NW : 1;
    for (int k = tid; k < nwe * H; k += T) s_hist[k] = 0;
    __syncthreads();
    const int slice = (((L.nnode + nwe - 1) / nwe) + 31) & ~31;
    const int nb = min(warp * slice, L.nnode), ne = (warp < nwe) ? min(nb + slice, L.nnode) : nb;
    for (int m = nb + lane; m < ne; m += 32) {
        const int t = s_tgt[m];
        const int r = (t >= 0) ? rank_of(hs, t) : 0xffff;
        s_rk[m] = (unsigned short)r;
        if (t >= 0) atomicAdd(&s_hist[warp * H + r], 1);
    }
    __syncthreads();
    for (int k = tid; k < H; k += T) {
        int tot = 0;
        for (int w = 0; w < nwe; ++w) tot += s_hist[w * H + k];
        s_start[k] = tot;
    }
    if (tid == 0) s_start[H] = 0;
    __syncthreads();
    const int ntot = block_exclusive_scan(s_start, H + 1, hs.scratch);
    for (int k = tid; k < H; k += T) {
        int run = s_start[k];
        for (int w = 0; w < nwe; ++w) { const int v = s_hist[w * H + k]; s_hist[w * H + k] = run; run += v; }
    }
    __syncthreads();
    // placement straight into the node lists (scattered 4- and 2-byte stores inside the cell's 19 KB; L2 merges them)
    unsigned* g_key = nl.key + (size_t)blockIdx.x * L.nnode;
    unsigned short* g_rkpos = nl.rkpos + (size_t)blockIdx.x * L.nnode;
    for (int m0 = nb; m0 < ne; m0 += 32) {
        const int m = m0 + lane;
        const int key = (m < ne) ? (int)s_rk[m] : 0xffff;
        const unsigned same = __match_any_sync(0xffffffffu, key);
        if (key != 0xffff) {
            const int pos = s_hist[warp * H + key] + __popc(same & ((1u << lane) - 1u));
            g_key[pos] = ((unsigned)s_tgt[m] << 14) | (unsigned)m;
            g_rkpos[pos] = (unsigned short)key;
        }
        __syncwarp();
        if (key != 0xffff && lane == (__ffs(same) - 1)) s_hist[warp * H + key] += __popc(same);
        __syncwarp();
    }
    __syncthreads();
    // (target, x-node) segments of the sorted list (statistics for the work model): read back what this CTA just wrote
    int seg = 0;
    for (int k = tid; k < ntot; k += T) {
        const unsigned kk = g_key[k], kp = k ? g_key[k - 1] : 0u;
        const int mk = (int)(kk & 16383u), mp = (int)(kp & 16383u);
        const int ck = L.mg_npq ? (int)__umulhi((unsigned)mk, L.mg_npq) : mk, cp = L.mg_npq ? (int)__umulhi((unsigned)mp, L.mg_npq) : mp;
        seg += (k == 0 || (kk >> 14) != (kp >> 14) || ck != cp) ? 1 : 0;
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) seg += __shfl_xor_sync(0xffffffffu, seg, d);
    if (lane == 0) hs.scratch[warp] = seg;
    __syncthreads();
    if (tid == 0) {
        int tot = 0;
        for (int w = 0; w < NW; ++w) tot += hs.scratch[w];
        nl.hits[blockIdx.x] = H; nl.ntot[blockIdx.x] = ntot; nl.nseg[blockIdx.x] = tot;
    }
}

// Pattern pass, kernel S: exclusive scan of the hit counts -> cellbase, nnz and max hits.  One CTA.
__global__ void __launch_bounds__(1024) k_scan_cells(DevLattice L, int n_blk, const int* __restrict__ hits,
                                                    const int* __restrict__ ntot, const int* __restrict__ nseg,
                                                    int64_t* __restrict__ cellbase, int64_t* __restrict__ summary)
{
    // tiles of 1024 consecutive cells (coalesced reads and writes): warp scans, then the 32 warp totals, then the carry
    __shared__ long long wsum[32];
    __shared__ long long s_carry;
    __shared__ long long s_stat[3][32];
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    long long nodes = 0, segs = 0;
    int mx = 0;
    if (t == 0) s_carry = 0;
    __syncthreads();
    for (int base = 0; base < n_blk; base += 1024) {
        const int k = base + t;
        const int h = k < n_blk ? hits[k] : 0;
        if (k < n_blk) { nodes += ntot[k]; segs += nseg[k]; mx = max(mx, h); }
        long long inc = h;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += y; }
        if (lane == 31) wsum[warp] = inc;
        __syncthreads();
        if (warp == 0) {
            const long long v = wsum[lane];
            long long x = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { const long long y = __shfl_up_sync(0xffffffffu, x, d); if (lane >= d) x += y; }
            wsum[lane] = x - v;                         // exclusive prefix of the warp totals
            if (lane == 31) s_stat[0][0] = x;           // tile total
        }
        __syncthreads();
        const long long carry = s_carry;
        if (k < n_blk) cellbase[k] = carry + wsum[warp] + inc - h;
        __syncthreads();
        if (t == 0) s_carry = carry + s_stat[0][0];
        __syncthreads();
    }
    // statistics: nodes on the grid, segments, max hits
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        nodes += __shfl_xor_sync(0xffffffffu, nodes, d); segs += __shfl_xor_sync(0xffffffffu, segs, d);
        mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    }
    if (lane == 0) { s_stat[0][warp] = nodes; s_stat[1][warp] = segs; s_stat[2][warp] = mx; }
    __syncthreads();
    if (t == 0) {
        long long a = 0, s2 = 0, m = 0;
        for (int w = 0; w < 32; ++w) { a += s_stat[0][w]; s2 += s_stat[1][w]; m = max(m, s_stat[2][w]); }
        const long long total = s_carry;
        summary[0] = total * L.totcoup;                 // nnz of the block
        summary[1] = m;                                 // max hit cells of any source cell
        summary[2] = a; summary[3] = s2;
        cellbase[n_blk] = total;
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

// Pattern pass, kernel B: column indices, ascending within each row.  The hit cells of a source cell are read
// off its node lists (the target cell at the first sorted position of every rank).  Thread = output (alpha, m-th
// coupled alpha'), looping over the hit cells k: entry k of row alpha sits at row_start + k*nc + m, so the threads
// of a warp write runs of consecutive m and consecutive k fill the gaps (the same store pattern as the fill's rows).
__global__ void __launch_bounds__(1024) k_emit_cols(DevLattice L, NodeLists nl, int hmax,
                                                   const int64_t* __restrict__ rowptr, int32_t* __restrict__ colidx)
{
    extern __shared__ __align__(16) char smem[];
    const int T = blockDim.x, tid = threadIdx.x;
    int* hitcol = (int*)smem;                        // first column of every hit cell: cell * n_ch
    const int H = nl.hits[blockIdx.x], ntot = nl.ntot[blockIdx.x];
    const unsigned short* g_rkpos = nl.rkpos + (size_t)blockIdx.x * L.nnode;
    const unsigned* g_key = nl.key + (size_t)blockIdx.x * L.nnode;
    for (int pos = tid; pos < ntot; pos += T) {
        const int r = g_rkpos[pos];
        if (pos == 0 || g_rkpos[pos - 1] != r) hitcol[r] = (int)(g_key[pos] >> 14) * L.n_ch;
    }
    __syncthreads();
    int32_t* __restrict__ row0 = colidx + rowptr[(int64_t)blockIdx.x * L.n_ch];
    // the block is G groups of `ow` threads: a group covers all outputs (in passes if totcoup > ow) for k = g, g+G, ...
    const int ow = min(T, (L.totcoup + 31) & ~31), G = T / ow, g = tid / ow;
    if (g < G)
        for (int o = tid - g * ow; o < L.totcoup; o += ow) {
            const int al = L.o_alpha[o], off = L.cl_off[al], nc = L.cl_off[al + 1] - off, ap = L.cl[o];
            int32_t* out = row0 + ((size_t)H * off + (o - off));
#pragma unroll 4
            for (int k = g; k < H; k += G) out[(size_t)k * nc] = hitcol[k] + ap;
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
        for (int64_t k = rowptr[r] + lane; k < rowptr[r + 1]; k += 32) s += vals[k] * x[colidx[k]];
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
__global__ void __launch_bounds__(kThreads) k_hit_list(DevLattice L, NodeLists nl, const int64_t* __restrict__ cellbase,
                                                      int* __restrict__ hitlist)
{
    const int ntot = nl.ntot[blockIdx.x];
    const unsigned short* g_rkpos = nl.rkpos + (size_t)blockIdx.x * L.nnode;
    const unsigned* g_key = nl.key + (size_t)blockIdx.x * L.nnode;
    int* out = hitlist + cellbase[blockIdx.x];
    for (int pos = threadIdx.x; pos < ntot; pos += blockDim.x) {
        const int r = g_rkpos[pos];
        if (pos == 0 || g_rkpos[pos - 1] != r) out[r] = (int)(g_key[pos] >> 14);
    }
}

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

cudaError_t launch_map_sort(const DevLattice& L, int cell_begin, int n_blk, const NodeLists& nl, cudaStream_t st)
{
    // per-warp histograms up to this many hit cells per source cell, one warp beyond (PM_HITS_FAST: test hook)
    static const int hits_fast = [] { const char* e = std::getenv("PM_HITS_FAST"); return e ? std::max(1, std::atoi(e)) : kHitsFast; }();
    const size_t sm = map_sort_smem(L, hits_fast);
    cudaError_t e = cudaFuncSetAttribute(k_map_sort, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    k_map_sort<<<n_blk, kThreads, sm, st>>>(L, cell_begin, nl, hits_fast);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_scan_rows(const DevLattice& L, int n_blk, const NodeLists& nl, int64_t* cellbase, int64_t* rowptr,
                             int64_t* summary, cudaStream_t st)
{
    k_scan_cells<<<1, 1024, 0, st>>>(L, n_blk, nl.hits, nl.ntot, nl.nseg, cellbase, summary);
    ++g_launches;
    const int64_t n = (int64_t)n_blk * L.n_ch + 1;
    k_write_rowptr<<<(unsigned)std::min<int64_t>((n + 255) / 256, 148 * 8), 256, 0, st>>>(L, n_blk, nl.hits, cellbase, rowptr);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_emit_cols(const DevLattice& L, int n_blk, const NodeLists& nl, int hmax, const int64_t* rowptr,
                             int32_t* colidx, cudaStream_t st)
{
    const size_t sm = al16(4 * (size_t)std::max(hmax, 1));
    cudaError_t e = cudaFuncSetAttribute(k_emit_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    const int threads = std::min(1024, std::max(128, (L.totcoup + 31) & ~31));
    k_emit_cols<<<n_blk, threads, sm, st>>>(L, nl, hmax, rowptr, colidx);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_hit_list(const DevLattice& L, int n_blk, const NodeLists& nl, const int64_t* cellbase, int* hitlist, cudaStream_t st)
{
    k_hit_list<<<n_blk, kThreads, 0, st>>>(L, nl, cellbase, hitlist);
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
                                                    double* __restrict__ out)
{
    extern __shared__ __align__(16) char smem[];
    const int ld = Np + 1;                                     // padded row length of the B tile
    double* sB = (double*)smem;                                 // [kBlkT][Np + 1]
    double* sX = sB + kBlkT * ld;                               // [Np][kBlkT]
    const int ti = (Np + kBlkT - 1) / kBlkT, tj = (Nq + kBlkT - 1) / kBlkT;
    const int a = blockIdx.x / (ti * tj), rem = blockIdx.x - a * ti * tj, i0 = (rem / tj) * kBlkT, j0 = (rem % tj) * kBlkT;
    const int64_t stride = (int64_t)Nq * n_ch;
    const double* Ba = B + (size_t)a * Np * Np;
    for (int k = threadIdx.x; k < kBlkT * Np; k += blockDim.x) {
        const int r = k / Np, c = k - r * Np;
        sB[r * ld + c] = (i0 + r < Np) ? Ba[(size_t)(i0 + r) * Np + c] : 0.0;
    }
    for (int k = threadIdx.x; k < Np * kBlkT; k += blockDim.x) {
        const int ip = k / kBlkT, jj = k - ip * kBlkT;
        double x = 0.0;
        if (j0 + jj < Nq) { const int64_t c = (int64_t)ip * stride + (int64_t)(j0 + jj) * n_ch + a; x = diag ? diag[c] * in[c] : in[c]; }
        sX[k] = x;
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
                               cudaStream_t st)
{
    const int ti = (Np + kBlkT - 1) / kBlkT, tj = (Nq + kBlkT - 1) / kBlkT;
    const size_t sm = sizeof(double) * ((size_t)kBlkT * (Np + 1) + (size_t)Np * kBlkT);
    if (sm > 227 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(k_block_apply, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    k_block_apply<<<(unsigned)(n_ch * ti * tj), 256, sm, st>>>(Np, Nq, n_ch, B, diag, in, out);
    count_launch();
    return cudaGetLastError();
}

}  // namespace pm
