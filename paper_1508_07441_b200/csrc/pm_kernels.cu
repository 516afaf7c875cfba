// pm_kernels.cu — CUDA kernels of libpm for sm_100a: pattern pass (a6), generic fill pass (a7), SpMV (a9).
// One CTA per source cell D_ij; the node map and location live in pm_device.cuh.
// Paper's prior art: one thread per pre-selected element or per cell pair (L376) with
// constants in global memory (L341) and a CPU repack into CSR (L376).  Here all constants sit in shared
// memory, a source cell's nodes are binned once and serve every channel pair, and the cell-major row order
// makes every row segment contiguous, so no repack exists.
#include "pm_kernels.cuh"

#include "pm_ylm.h"

namespace pm {

// ------------------------------------------------------------------------------------------------
// Shared-memory staging common to pattern and fill: edges, rules, hit bitset.
// ------------------------------------------------------------------------------------------------
struct Stage {
    double *pe, *qe, *tp, *tq, *tx;
    unsigned* bits;      // n_words hit bitset of this source cell
    int* wpre;           // n_words exclusive prefix popcounts
    int* scratch;        // blockDim+1
};

__device__ __forceinline__ char* carve(char*& p, size_t bytes)
{
    char* r = p;
    p += (bytes + 15) & ~size_t(15);
    return r;
}

__device__ inline Stage stage_common(const DevLattice& L, char*& sp)
{
    Stage s;
    s.pe = (double*)carve(sp, sizeof(double) * L.pe_pad);
    s.qe = (double*)carve(sp, sizeof(double) * L.qe_pad);
    s.tp = (double*)carve(sp, sizeof(double) * L.n_p);
    s.tq = (double*)carve(sp, sizeof(double) * L.n_q);
    s.tx = (double*)carve(sp, sizeof(double) * L.n_x);
    s.bits = (unsigned*)carve(sp, sizeof(unsigned) * L.n_words);
    s.wpre = (int*)carve(sp, sizeof(int) * L.n_words);
    s.scratch = (int*)carve(sp, sizeof(int) * (blockDim.x + 1));
    for (int k = threadIdx.x; k < L.pe_pad; k += blockDim.x) s.pe[k] = L.pe[k];
    for (int k = threadIdx.x; k < L.qe_pad; k += blockDim.x) s.qe[k] = L.qe[k];
    for (int k = threadIdx.x; k < L.n_p; k += blockDim.x) s.tp[k] = L.tp[k];
    for (int k = threadIdx.x; k < L.n_q; k += blockDim.x) s.tq[k] = L.tq[k];
    for (int k = threadIdx.x; k < L.n_x; k += blockDim.x) s.tx[k] = L.tx[k];
    for (int k = threadIdx.x; k < L.n_words; k += blockDim.x) s.bits[k] = 0u;
    return s;
}

// size in bytes of what stage_common carves (host mirror)
size_t stage_bytes(const DevLattice& L, int threads)
{
    auto al = [](size_t b) { return (b + 15) & ~size_t(15); };
    return al(8 * (size_t)L.pe_pad) + al(8 * (size_t)L.qe_pad) + al(8 * (size_t)L.n_p) + al(8 * (size_t)L.n_q)
         + al(8 * (size_t)L.n_x) + 2 * al(4 * (size_t)L.n_words) + al(4 * (size_t)(threads + 1));
}

// Map every node of source cell `cell`, mark its target in the bitset and (optionally) record it.
template <bool kRecord>
__device__ inline void map_cell(const DevLattice& L, const Stage& s, int cell, int* tgt)
{
    const int i = cell / L.Nq, j = cell - i * L.Nq;
    const CellGeom g = cell_geom(s.pe, s.qe, i, j);
    const int nqx = L.n_q * L.n_x;
    for (int n = threadIdx.x; n < L.nnode; n += blockDim.x) {
        const int a = n / nqx, r = n - a * nqx, b = r / L.n_x, c = r - b * L.n_x;
        double p, q, pp, qq;
        map_node(g, s.tp[a], s.tq[b], s.tx[c], p, q, pp, qq);
        const int t = target_cell(s.pe, L.pe_pad, L.Np, s.qe, L.qe_pad, L.Nq, pp, qq);
        if (t >= 0) atomicOr(&s.bits[t >> 5], 1u << (t & 31));
        if (kRecord) tgt[n] = t;
    }
}

// popcount prefix over the bitset words; returns the number of hit cells H
__device__ inline int rank_bits(const DevLattice& L, const Stage& s)
{
    for (int k = threadIdx.x; k < L.n_words; k += blockDim.x) s.wpre[k] = __popc(s.bits[k]);
    __syncthreads();
    return block_exclusive_scan(s.wpre, L.n_words, s.scratch);
}

__device__ __forceinline__ int rank_of(const Stage& s, int t)
{
    return s.wpre[t >> 5] + __popc(s.bits[t >> 5] & ((1u << (t & 31)) - 1u));
}

__device__ inline void list_hits(const DevLattice& L, const Stage& s, int* hitcell)
{
    for (int k = threadIdx.x; k < L.n_words; k += blockDim.x) {
        unsigned w = s.bits[k];
        int r = s.wpre[k];
        while (w) { const int b = __ffs(w) - 1; hitcell[r++] = (k << 5) + b; w &= w - 1; }
    }
}

// ------------------------------------------------------------------------------------------------
// Pattern pass, kernel A: number of hit cells per source cell.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) k_count_hits(DevLattice L, int cell_begin, int n_blk, int* __restrict__ hits)
{
    extern __shared__ __align__(16) char smem[];
    char* sp = smem;
    Stage s = stage_common(L, sp);
    __syncthreads();
    map_cell<false>(L, s, cell_begin + blockIdx.x, nullptr);
    __syncthreads();
    const int H = rank_bits(L, s);
    if (threadIdx.x == 0) hits[blockIdx.x] = H;
}

// Pattern pass, kernel S: exclusive scan of hits -> rowptr (block-local), nnz and max hits.  One CTA.
__global__ void __launch_bounds__(1024) k_scan_rows(DevLattice L, int n_blk, const int* __restrict__ hits,
                                                   int64_t* __restrict__ cellbase, int64_t* __restrict__ rowptr,
                                                   int64_t* __restrict__ summary)
{
    __shared__ long long part[1024];
    __shared__ int pmax[1024];
    const int T = blockDim.x, t = threadIdx.x;
    const int chunk = (n_blk + T - 1) / T, b = min(t * chunk, n_blk), e = min(b + chunk, n_blk);
    long long sum = 0; int mx = 0;
    for (int k = b; k < e; ++k) { sum += hits[k]; mx = max(mx, hits[k]); }
    part[t] = sum; pmax[t] = mx;
    __syncthreads();
    if (t == 0) {
        long long run = 0; int m = 0;
        for (int k = 0; k < T; ++k) { long long v = part[k]; part[k] = run; run += v; m = max(m, pmax[k]); }
        summary[0] = run * L.totcoup;      // nnz of the block
        summary[1] = m;                    // max hit cells of any source cell
        rowptr[(int64_t)n_blk * L.n_ch] = run * L.totcoup;
    }
    __syncthreads();
    long long run = part[t];
    for (int k = b; k < e; ++k) {
        cellbase[k] = run;
        const int H = hits[k];
        for (int a = 0; a < L.n_ch; ++a) rowptr[(int64_t)k * L.n_ch + a] = run * L.totcoup + (long long)H * L.cl_off[a];
        run += H;
    }
}

// Pattern pass, kernel B: column indices, ascending within each row.
__global__ void __launch_bounds__(kThreads) k_emit_cols(DevLattice L, int cell_begin, const int64_t* __restrict__ rowptr,
                                                       int32_t* __restrict__ colidx)
{
    extern __shared__ __align__(16) char smem[];
    char* sp = smem;
    Stage s = stage_common(L, sp);
    int* hitcell = (int*)carve(sp, sizeof(int) * min(L.n_cells, L.nnode));
    __syncthreads();
    map_cell<false>(L, s, cell_begin + blockIdx.x, nullptr);
    __syncthreads();
    const int H = rank_bits(L, s);
    list_hits(L, s, hitcell);
    __syncthreads();
    for (int a = 0; a < L.n_ch; ++a) {
        const int off = L.cl_off[a], nc = L.cl_off[a + 1] - off;
        int32_t* out = colidx + rowptr[(int64_t)blockIdx.x * L.n_ch + a];
        const int len = H * nc;
        for (int idx = threadIdx.x; idx < len; idx += blockDim.x) {
            const int k = idx / nc, m = idx - k * nc;
            out[idx] = hitcell[k] * L.n_ch + L.cl[off + m];
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Fill pass, generic (table-driven) kernel: any channel list.  One CTA per source cell.
//   phase 1  map nodes -> target cells, bitset, ranks, hit list
//   phase 2  deterministic counting sort of the node ids by hit rank (stable in node order)
//   phase 3  one warp per hit cell: lanes take that cell's nodes, evaluate the ket harmonics and the
//            n_fun orbital functions, accumulate privately, then a fixed-shape butterfly reduces the lanes
//   phase 4  per hit cell: contract with the channel coefficients c^L and write the row segments
// Node sums are formed in an order fixed by (node id, lane, butterfly): bitwise reproducible.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kThreads) k_fill_generic(DevLattice L, int cell_begin, int hmax,
                                                          const int64_t* __restrict__ rowptr, double* __restrict__ vals)
{
    extern __shared__ __align__(16) char smem[];
    char* sp = smem;
    Stage s = stage_common(L, sp);
    const int nw = blockDim.x >> 5, warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double* s_wp = (double*)carve(sp, sizeof(double) * L.n_p);
    double* s_wq = (double*)carve(sp, sizeof(double) * L.n_q);
    double* s_wx = (double*)carve(sp, sizeof(double) * L.n_x);
    double* s_sx = (double*)carve(sp, sizeof(double) * L.n_x);
    double* s_acc = (double*)carve(sp, sizeof(double) * nw * L.n_fun);
    int* tgt = (int*)carve(sp, sizeof(int) * L.nnode);
    int* sorted = (int*)carve(sp, sizeof(int) * L.nnode);
    int* hitcell = (int*)carve(sp, sizeof(int) * hmax);
    int* start = (int*)carve(sp, sizeof(int) * (hmax + 1));
    int* hist = (int*)carve(sp, sizeof(int) * nw * hmax);
    for (int k = threadIdx.x; k < L.n_p; k += blockDim.x) s_wp[k] = L.wp[k];
    for (int k = threadIdx.x; k < L.n_q; k += blockDim.x) s_wq[k] = L.wq[k];
    for (int k = threadIdx.x; k < L.n_x; k += blockDim.x) { s_wx[k] = L.wx[k]; s_sx[k] = L.sx[k]; }
    for (int k = threadIdx.x; k < nw * hmax; k += blockDim.x) hist[k] = 0;
    __syncthreads();

    // ---- phase 1
    const int cell = cell_begin + blockIdx.x;
    map_cell<true>(L, s, cell, tgt);
    __syncthreads();
    const int H = rank_bits(L, s);
    if (H > hmax) return;                       // cannot happen when hmax comes from pm_pattern of this block
    list_hits(L, s, hitcell);

    // ---- phase 2: each warp owns a contiguous slice of node ids
    const int slice = (((L.nnode + nw - 1) / nw) + 31) & ~31;
    const int nb = warp * slice, ne = min(nb + slice, L.nnode);
    for (int n = nb + lane; n < ne; n += 32) {
        const int t = tgt[n];
        if (t >= 0) atomicAdd(&hist[warp * hmax + rank_of(s, t)], 1);
    }
    __syncthreads();
    for (int k = threadIdx.x; k < H; k += blockDim.x) {
        int tot = 0;
        for (int w = 0; w < nw; ++w) tot += hist[w * hmax + k];
        start[k] = tot;
    }
    if (threadIdx.x == 0) start[H] = 0;
    __syncthreads();
    block_exclusive_scan(start, H + 1, s.scratch);
    for (int k = threadIdx.x; k < H; k += blockDim.x) {
        int run = start[k];
        for (int w = 0; w < nw; ++w) { const int v = hist[w * hmax + k]; hist[w * hmax + k] = run; run += v; }
    }
    __syncthreads();
    for (int n0 = nb; n0 < ne; n0 += 32) {
        const int n = n0 + lane;
        const int t = (n < ne) ? tgt[n] : -1;
        const int key = (t >= 0) ? rank_of(s, t) : -1;
        const unsigned same = __match_any_sync(0xffffffffu, key);
        if (key >= 0) {
            const int pos = hist[warp * hmax + key] + __popc(same & ((1u << lane) - 1u));
            sorted[pos] = n;
        }
        __syncwarp();
        if (key >= 0 && lane == (__ffs(same) - 1)) hist[warp * hmax + key] += __popc(same);
        __syncwarp();
    }
    __syncthreads();

    // ---- phase 3 + 4
    const int i = cell / L.Nq, j = cell - i * L.Nq;
    const CellGeom g = cell_geom(s.pe, s.qe, i, j);
    const double dsrc = (s.pe[i + 1] - s.pe[i]) * (s.qe[j + 1] - s.qe[j]);
    const int nqx = L.n_q * L.n_x;
    double* wacc = s_acc + warp * L.n_fun;
    for (int k = warp; k < H; k += nw) {
        double acc[kMaxFun];
        for (int f = 0; f < L.n_fun; ++f) acc[f] = 0.0;
        for (int sidx = start[k] + lane; sidx < start[k + 1]; sidx += 32) {
            const int n = sorted[sidx];
            const int a = n / nqx, r = n - a * nqx, b = r / L.n_x, c = r - b * L.n_x;
            double p, q, pp, qq;
            const double x = s.tx[c];
            map_node(g, s.tp[a], s.tq[b], x, p, q, pp, qq);
            const double w = __dmul_rn(__dmul_rn(__dmul_rn(g.hp, s_wp[a]), __dmul_rn(g.hq, s_wq[b])), s_wx[c]);
            const double omega = w * ((p * q) / (pp * qq));
            // rotated directions from vector components (frame: q^ = z, p^ = (sx, 0, x))
            const double sx = s_sx[c];
            const double ax = -0.5 * p * sx, az = -0.5 * p * x - 0.75 * q;
            const double bx = p * sx, bz = p * x - 0.5 * q;
            const double ra = rsqrt(ax * ax + az * az), rb = rsqrt(bx * bx + bz * bz);
            double Yp[kMaxY], Yq[kMaxY], K[kMaxSlot];
            ylm_fill(L.lmax, ax * ra, az * ra, L.ya, L.yb, L.ydiag, Yp);
            ylm_fill(L.lmax, bx * rb, bz * rb, L.ya, L.yb, L.ydiag, Yq);
            for (int sl = 0; sl < L.n_slot; ++sl) {
                double v = 0.0;
                for (int t = L.kt_off[sl]; t < L.kt_off[sl + 1]; ++t) v += L.kt_c[t] * Yp[L.kt_ip[t]] * Yq[L.kt_iq[t]];
                K[sl] = v * omega;
            }
            const double* bra = L.bra + (size_t)c * L.n_slot;
            for (int f = 0; f < L.n_fun; ++f) {
                const int4 fn = L.fun[f];
                double v = 0.0;
                for (int m = 0; m < fn.z; ++m) v += bra[fn.x + m] * K[fn.y + m];
                acc[f] += v;
            }
        }
        for (int f = 0; f < L.n_fun; ++f) {
            double v = acc[f];
#pragma unroll
            for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
            if (lane == 0) wacc[f] = v;
        }
        __syncwarp();
        const int hc = hitcell[k], ic = hc / L.Nq, jc = hc - ic * L.Nq;
        const double norm = 1.0 / sqrt(dsrc * ((s.pe[ic + 1] - s.pe[ic]) * (s.qe[jc + 1] - s.qe[jc])));
        for (int o = lane; o < L.totcoup; o += 32) {
            const int a = L.o_alpha[o], off = L.cl_off[a], nc = L.cl_off[a + 1] - off;
            double v = 0.0;
            for (int t = L.ot_off[o]; t < L.ot_off[o + 1]; ++t) v += L.ot_c[t] * wacc[L.ot_f[t]];
            vals[rowptr[(int64_t)blockIdx.x * L.n_ch + a] + (int64_t)k * nc + (o - off)] = v * norm;
        }
        __syncwarp();
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
// Host launchers
// ------------------------------------------------------------------------------------------------
static std::atomic<int64_t> g_launches{0};
int64_t launch_count() { return g_launches.load(); }
void count_launch() { ++g_launches; }

size_t fill_generic_smem(const DevLattice& L, int hmax)
{
    auto al = [](size_t b) { return (b + 15) & ~size_t(15); };
    const int nw = kThreads / 32;
    return stage_bytes(L, kThreads) + al(8 * (size_t)L.n_p) + al(8 * (size_t)L.n_q) + 2 * al(8 * (size_t)L.n_x)
         + al(8 * (size_t)nw * L.n_fun) + 2 * al(4 * (size_t)L.nnode) + al(4 * (size_t)hmax) + al(4 * (size_t)(hmax + 1))
         + al(4 * (size_t)nw * hmax);
}

cudaError_t launch_count_hits(const DevLattice& L, int cell_begin, int n_blk, int* hits, cudaStream_t st)
{
    const size_t sm = stage_bytes(L, kThreads);
    cudaError_t e = cudaFuncSetAttribute(k_count_hits, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    k_count_hits<<<n_blk, kThreads, sm, st>>>(L, cell_begin, n_blk, hits);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_scan_rows(const DevLattice& L, int n_blk, const int* hits, int64_t* cellbase, int64_t* rowptr,
                             int64_t* summary, cudaStream_t st)
{
    k_scan_rows<<<1, 1024, 0, st>>>(L, n_blk, hits, cellbase, rowptr, summary);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_emit_cols(const DevLattice& L, int cell_begin, int n_blk, const int64_t* rowptr, int32_t* colidx,
                             cudaStream_t st)
{
    const size_t sm = stage_bytes(L, kThreads) + 16 + 4 * (size_t)std::min(L.n_cells, L.nnode);
    cudaError_t e = cudaFuncSetAttribute(k_emit_cols, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    k_emit_cols<<<n_blk, kThreads, sm, st>>>(L, cell_begin, rowptr, colidx);
    ++g_launches;
    return cudaGetLastError();
}

cudaError_t launch_fill_generic(const DevLattice& L, int cell_begin, int n_blk, int hmax, const int64_t* rowptr,
                                double* vals, cudaStream_t st)
{
    const size_t sm = fill_generic_smem(L, hmax);
    cudaError_t e = cudaFuncSetAttribute(k_fill_generic, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
    if (e != cudaSuccess) return e;
    k_fill_generic<<<n_blk, kThreads, sm, st>>>(L, cell_begin, hmax, rowptr, vals);
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

}  // namespace pm
