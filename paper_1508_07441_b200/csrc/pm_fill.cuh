// pm_fill.cuh — the fill pass (hot-path step a7; the paper's step 2b).
//
// One persistent CTA per SM slot walks source cells D_ij.  Per source cell:
//   A  map    every node (c-major node ids) -> target cell from p'^2, q'^2 against sqrt-thresholds of the edges
//             (bit-identical decisions to "sqrt, then compare with the edges"), hit bitset
//   B  sort   ranks of the hit cells, stable counting sort of the node ids by rank: the sorted list is ordered by
//             (target t, x-node c, a, b), so the nodes of one (t, c) pair are consecutive
//   C  nodes  lane = node, 32 consecutive sorted nodes per warp step: omega, directions, the ket harmonics K[slot]
//             (Spec::ket — generated straight-line code, registers only), K tile -> shared memory (XOR swizzle)
//   D  sums   lane = slot: walks the 32 nodes of the tile, summing K over each (t, c) segment; at a segment end
//             lane = function: acc_t[f] += sum_M bra[c][sa+M] * S[sb+M] (the bra harmonics depend on c only, so they
//             are applied once per segment, not once per node); at the end of target t the 140 sums go to the
//             CTA's scratch row of t (global memory, L2-resident)
//   E  rows   thread = output (alpha, alpha'): P = norm_t * sum_L c^L_{alpha alpha'} acc_t[f], coalesced CSR writes
// Every sum has a fixed order (sorted node order, fixed warp ranges): bitwise reproducible, no floating atomics.
// Prior art this replaces: one thread per element / per cell pair, constants in global memory, CPU repack
// (PAPER.md:L341, L348-356, L376).
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

#include "pm_device.cuh"
#include "pm_ylm.h"

namespace pm {

constexpr int kFillMaxSlot = 160;      // table-driven fallback: slots / functions it can hold
constexpr int kFillMaxFun = 256;
constexpr int kFillMaxY = 45;

// Table-driven ket code for channel sets without a generated kernel (slow: local arrays, table loads).
struct SpecGeneric {
    static constexpr bool kStatic = false;
    static constexpr int NS = kFillMaxSlot, NF = kFillMaxFun, NCH = kFillMaxFun / 32;
    static constexpr unsigned long long kHash = 0ull;
    static __device__ __noinline__ void ket(const DevLattice& L, double om, double uxa, double uza, double uxb, double uzb,
                                            double (&K)[NS])
    {
        double Yp[kFillMaxY], Yq[kFillMaxY];
        ylm_fill(L.lmax, uxa, uza, L.ya, L.yb, L.ydiag, Yp);
        ylm_fill(L.lmax, uxb, uzb, L.ya, L.yb, L.ydiag, Yq);
        for (int s = 0; s < L.n_slot; ++s) {
            double v = 0.0;
            for (int t = L.kt_off[s]; t < L.kt_off[s + 1]; ++t) v += L.kt_c[t] * Yp[L.kt_ip[t]] * Yq[L.kt_iq[t]];
            K[s] = v * om;
        }
    }
};

struct FillSmem {           // byte offsets into dynamic shared memory, computed on the host
    int thr_p, thr_q, tp, tq, tx, sx, wx, wpa, wqb, bra, bits, wpre, rk, sorted, hitcell, start, hist, scratch,
        tile, sseg, head, normk, k0, total;
};

inline int fill_align16(int b) { return (b + 15) & ~15; }

// shared-memory plan for NW warps; ns = slots, nf = functions
inline FillSmem fill_smem_plan(const DevLattice& L, int hmax, int nw)
{
    FillSmem s{};
    int o = 0;
    auto take = [&](int bytes) { int r = o; o += fill_align16(bytes); return r; };
    s.thr_p = take(8 * L.pe_pad); s.thr_q = take(8 * L.qe_pad);
    s.tp = take(8 * L.n_p); s.tq = take(8 * L.n_q); s.tx = take(8 * L.n_x); s.sx = take(8 * L.n_x); s.wx = take(8 * L.n_x);
    s.wpa = take(8 * L.n_p); s.wqb = take(8 * L.n_q);
    s.bra = take(8 * L.n_x * L.n_slot);
    s.bits = take(4 * L.n_words); s.wpre = take(4 * L.n_words);
    s.rk = take(2 * L.nnode); s.sorted = take(2 * (L.nnode + 1));
    s.hitcell = take(4 * hmax); s.start = take(4 * (hmax + 1)); s.hist = take(4 * nw * hmax);
    s.scratch = take(4 * (nw * 32 + 1));
    const int tile_tgt = 4 * L.nnode, tile_k = 8 * 32 * L.n_slot * nw;       // union: tgt[nnode] (A, B) / K tiles (C, D)
    s.tile = take(tile_tgt > tile_k ? tile_tgt : tile_k);
    s.sseg = take(8 * L.n_slot * nw);
    s.head = take(8 * L.n_fun * nw);
    s.normk = take(8 * hmax);
    s.k0 = take(4 * (2 * nw + 2));
    s.total = o;
    return s;
}

// number of thresholds <= v, minus one, by integer comparison of the bit patterns (valid for v >= +0; a negative
// pattern, i.e. -0.0, sorts below every threshold).  thr has `pad` (power of two) entries, tail = +inf.
__device__ __forceinline__ int locate_bits(const long long* __restrict__ thr, int pad, long long v)
{
    int lo = 0;
#pragma unroll 1
    for (int s = pad >> 1; s > 0; s >>= 1) lo += (thr[lo + s - 1] <= v) ? s : 0;
    lo += (thr[lo] <= v) ? 1 : 0;
    return lo - 1;
}

// exact node map up to p'^2, q'^2 (every operation a single IEEE double operation)
__device__ __forceinline__ void map_node_sq(const CellGeom& g, double ta, double tb, double tc,
                                            double& p, double& q, double& P2, double& Q2)
{
    p = __dadd_rn(g.cp, __dmul_rn(g.hp, ta));
    q = __dadd_rn(g.cq, __dmul_rn(g.hq, tb));
    const double pq = __dmul_rn(p, q), p2 = __dmul_rn(p, p), q2 = __dmul_rn(q, q), pqx = __dmul_rn(pq, tc);
    P2 = __dadd_rn(__dadd_rn(__dmul_rn(0.25, p2), __dmul_rn(0.5625, q2)), __dmul_rn(0.75, pqx));
    Q2 = __dsub_rn(__dadd_rn(p2, __dmul_rn(0.25, q2)), pqx);
    P2 = P2 < 0.0 ? 0.0 : P2;
    Q2 = Q2 < 0.0 ? 0.0 : Q2;
}

__device__ __forceinline__ int target_cell_sq(const long long* thr_p, int pe_pad, int Np, const long long* thr_q, int qe_pad,
                                              int Nq, double P2, double Q2)
{
    const int ic = locate_bits(thr_p, pe_pad, __double_as_longlong(P2)), jc = locate_bits(thr_q, qe_pad, __double_as_longlong(Q2));
    const bool ok = (ic >= 0) & (ic < Np) & (jc >= 0) & (jc < Nq) & (P2 != 0.0) & (Q2 != 0.0);   // sqrt(y) = 0 <=> y = 0
    return ok ? ic * Nq + jc : -1;
}

// hit bitset of one source cell with word-prefix popcounts (ranks of the hit cells)
struct HitSet { unsigned* bits; int* wpre; int* scratch; };

__device__ inline int rank_bits_n(int n_words, const HitSet& s)
{
    for (int k = threadIdx.x; k < n_words; k += blockDim.x) s.wpre[k] = __popc(s.bits[k]);
    __syncthreads();
    return block_exclusive_scan(s.wpre, n_words, s.scratch);
}

__device__ __forceinline__ int rank_of(const HitSet& s, int t)
{
    return s.wpre[t >> 5] + __popc(s.bits[t >> 5] & ((1u << (t & 31)) - 1u));
}

__device__ inline void list_hits_n(int n_words, const HitSet& s, int* hitcell)
{
    for (int k = threadIdx.x; k < n_words; k += blockDim.x) {
        unsigned w = s.bits[k];
        int r = s.wpre[k];
        while (w) { const int b = __ffs(w) - 1; hitcell[r++] = (k << 5) + b; w &= w - 1; }
    }
}

template <class Spec, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_fill_seg(DevLattice L, FillSmem S, int cell_begin, int n_blk, int hmax, const int64_t* __restrict__ rowptr,
           double* __restrict__ vals, double* __restrict__ accG)
{
    constexpr int T = NW * 32;
    constexpr int NSC = (Spec::NS + 31) / 32;           // slot chunks of the lane = slot walk
    constexpr int NCH = Spec::NCH;                      // function chunks of the lane = function stage
    extern __shared__ __align__(16) char smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ns = Spec::kStatic ? Spec::NS : L.n_slot, nf = L.n_fun;
    const int npq = L.n_p * L.n_q;

    long long* s_thr_p = (long long*)(smem + S.thr_p);
    long long* s_thr_q = (long long*)(smem + S.thr_q);
    double* s_tp = (double*)(smem + S.tp);   double* s_tq = (double*)(smem + S.tq);   double* s_tx = (double*)(smem + S.tx);
    double* s_sx = (double*)(smem + S.sx);   double* s_wx = (double*)(smem + S.wx);
    double* s_wpa = (double*)(smem + S.wpa); double* s_wqb = (double*)(smem + S.wqb);
    double* s_bra = (double*)(smem + S.bra);
    unsigned* s_bits = (unsigned*)(smem + S.bits);
    int* s_wpre = (int*)(smem + S.wpre);
    unsigned short* s_rk = (unsigned short*)(smem + S.rk);
    unsigned short* s_sorted = (unsigned short*)(smem + S.sorted);
    int* s_hitcell = (int*)(smem + S.hitcell);
    int* s_start = (int*)(smem + S.start);
    int* s_hist = (int*)(smem + S.hist);
    int* s_scratch = (int*)(smem + S.scratch);
    int* s_tgt = (int*)(smem + S.tile);
    double* s_tile = (double*)(smem + S.tile) + (size_t)warp * 32 * ns;
    double* s_sseg = (double*)(smem + S.sseg) + warp * ns;
    double* s_head = (double*)(smem + S.head);
    double* s_normk = (double*)(smem + S.normk);
    int* s_k0 = (int*)(smem + S.k0);                   // [NW] first target of each warp range, then [NW+1] range starts
    int* s_wbeg = s_k0 + NW;

    // ---- once per CTA: thresholds, rules, bra harmonics, per-lane function descriptors
    for (int k = tid; k < L.pe_pad; k += T) s_thr_p[k] = L.thr_p[k];
    for (int k = tid; k < L.qe_pad; k += T) s_thr_q[k] = L.thr_q[k];
    for (int k = tid; k < L.n_p; k += T) s_tp[k] = L.tp[k];
    for (int k = tid; k < L.n_q; k += T) s_tq[k] = L.tq[k];
    for (int k = tid; k < L.n_x; k += T) { s_tx[k] = L.tx[k]; s_sx[k] = L.sx[k]; s_wx[k] = L.wx[k]; }
    for (int k = tid; k < L.n_x * ns; k += T) s_bra[k] = L.bra[k];
    int fd[NCH];                                        // sa | sb << 8 | nM << 16 of function f = ch*32 + lane
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        const int f = ch * 32 + lane;
        fd[ch] = 0;
        if (f < nf) { const int4 fn = L.fun[f]; fd[ch] = fn.x | (fn.y << 8) | (fn.z << 16); }
    }
    double* accS = accG + (size_t)blockIdx.x * hmax * nf;
    HitSet st;
    st.bits = s_bits; st.wpre = s_wpre; st.scratch = s_scratch;

    for (int cb = blockIdx.x; cb < n_blk; cb += gridDim.x) {
        const int cell = cell_begin + cb;
        const int ci = cell / L.Nq, cj = cell - ci * L.Nq;
        const CellGeom g = cell_geom(L.pe, L.qe, ci, cj);
        __syncthreads();                                // previous cell's phase E is done with shared memory
        for (int k = tid; k < L.n_words; k += T) s_bits[k] = 0u;
        for (int k = tid; k < L.n_p; k += T) s_wpa[k] = __dmul_rn(g.hp, L.wp[k]);
        for (int k = tid; k < L.n_q; k += T) s_wqb[k] = __dmul_rn(g.hq, L.wq[k]);
        for (int k = tid; k < NW * hmax; k += T) s_hist[k] = 0;
        __syncthreads();

        // ---- A: map (node id m = c*npq + a*n_q + b)
        for (int m = tid; m < L.nnode; m += T) {
            const int c = m / npq, ab = m - c * npq, a = ab / L.n_q, b = ab - a * L.n_q;
            double p, q, P2, Q2;
            map_node_sq(g, s_tp[a], s_tq[b], s_tx[c], p, q, P2, Q2);
            const int t = target_cell_sq(s_thr_p, L.pe_pad, L.Np, s_thr_q, L.qe_pad, L.Nq, P2, Q2);
            if (t >= 0) atomicOr(&s_bits[t >> 5], 1u << (t & 31));
            s_tgt[m] = t;
        }
        __syncthreads();
        const int H = rank_bits_n(L.n_words, st);
        if (H > hmax) continue;                         // cannot happen: hmax comes from pm_pattern of this block
        list_hits_n(L.n_words, st, s_hitcell);

        // ---- B: stable counting sort of node ids by rank; each warp owns a contiguous slice of ids
        const int slice = (((L.nnode + NW - 1) / NW) + 31) & ~31;
        const int nb = warp * slice, ne = min(nb + slice, L.nnode);
        for (int m = nb + lane; m < ne; m += 32) {
            const int t = s_tgt[m];
            const int r = (t >= 0) ? rank_of(st, t) : 0xffff;
            s_rk[m] = (unsigned short)r;
            if (t >= 0) atomicAdd(&s_hist[warp * hmax + r], 1);
        }
        __syncthreads();
        for (int k = tid; k < H; k += T) {
            int tot = 0;
            for (int w = 0; w < NW; ++w) tot += s_hist[w * hmax + k];
            s_start[k] = tot;
        }
        if (tid == 0) s_start[H] = 0;
        __syncthreads();
        block_exclusive_scan(s_start, H + 1, s_scratch);
        for (int k = tid; k < H; k += T) {
            int run = s_start[k];
            for (int w = 0; w < NW; ++w) { const int v = s_hist[w * hmax + k]; s_hist[w * hmax + k] = run; run += v; }
        }
        __syncthreads();
        for (int m0 = nb; m0 < ne; m0 += 32) {
            const int m = m0 + lane;
            const int key = (m < ne) ? (int)s_rk[m] : 0xffff;
            const unsigned same = __match_any_sync(0xffffffffu, key);
            if (key != 0xffff) {
                const int pos = s_hist[warp * hmax + key] + __popc(same & ((1u << lane) - 1u));
                s_sorted[pos] = (unsigned short)m;
            }
            __syncwarp();
            if (key != 0xffff && lane == (__ffs(same) - 1)) s_hist[warp * hmax + key] += __popc(same);
            __syncwarp();
        }
        const int ntot = s_start[H];
        // warp ranges over the sorted list, in whole 32-node steps
        if (tid <= NW) { const int G = (ntot + 31) >> 5; s_wbeg[tid] = min(ntot, ((int)(((long long)tid * G) / NW)) << 5); }
        __syncthreads();                                // sorted[], rk[] complete; tgt[] dead from here (tile reuse)
        const int wb = s_wbeg[warp], we = s_wbeg[warp + 1];
        const int k0 = (wb < we) ? (int)s_rk[s_sorted[wb]] : -1;
        if (lane == 0) s_k0[warp] = k0;

        // ---- C + D: 32 sorted nodes per step
        double runT[NCH];
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) runT[ch] = 0.0;
        double runS[NSC];
#pragma unroll
        for (int i = 0; i < NSC; ++i) runS[i] = 0.0;
        for (int base = wb; base < we; base += 32) {
            const int pos = base + lane;
            const bool active = pos < we;
            const int m = s_sorted[active ? pos : wb];
            const int c = m / npq, ab = m - c * npq, a = ab / L.n_q, b = ab - a * L.n_q;
            const int rkv = s_rk[m];
            // segment ends: (t, c) changes after this node, or the tile ends; target ends: t changes / range ends
            bool tend = false, send = false;
            if (active) {
                const bool last = (pos + 1 >= we);
                const int m1 = s_sorted[last ? pos : pos + 1];
                tend = last || ((int)s_rk[m1] != rkv);
                send = tend || (m1 / npq != c) || lane == 31;
            }
            const unsigned tmask = __ballot_sync(0xffffffffu, tend), smask = __ballot_sync(0xffffffffu, send);
            const int cnt = min(32, we - base);
            {
                double p, q, P2, Q2;
                const double x = s_tx[c];
                map_node_sq(g, s_tp[a], s_tq[b], x, p, q, P2, Q2);
                // omega = w * p q / (p' q'),  w = ((hp wp_a)(hq wq_b)) wx_c
                const double w = __dmul_rn(__dmul_rn(s_wpa[a], s_wqb[b]), s_wx[c]);
                const double om = w * (p * q) * rsqrt(P2 * Q2);
                // rotated directions from vector components (frame: q^ = z, p^ = (sx, 0, x)):
                //   p' = -p/2 - 3q/4 ,  q' = p - q/2
                const double sx = s_sx[c], psx = p * sx, px = p * x;
                const double ax = -0.5 * psx, az = fma(-0.5, px, -0.75 * q);
                const double bx = psx, bz = fma(-0.5, q, px);
                const double ra = rsqrt(fma(ax, ax, az * az)), rb = rsqrt(fma(bx, bx, bz * bz));
                double K[Spec::NS];
                Spec::ket(L, om, ax * ra, az * ra, bx * rb, bz * rb, K);
                if (Spec::kStatic) {
#pragma unroll
                    for (int s = 0; s < Spec::NS; ++s) s_tile[s * 32 + (lane ^ (s & 31))] = K[s];
                } else {
                    for (int s = 0; s < ns; ++s) s_tile[s * 32 + (lane ^ (s & 31))] = K[s];
                }
            }
            __syncwarp();
            // lane = slot walk over the tile's nodes
            for (int j = 0; j < cnt; ++j) {
#pragma unroll
                for (int i = 0; i < NSC; ++i) {
                    const int s = i * 32 + lane;
                    if (s < ns) runS[i] += s_tile[s * 32 + (j ^ lane)];
                }
                if ((smask >> j) & 1u) {
#pragma unroll
                    for (int i = 0; i < NSC; ++i) {
                        const int s = i * 32 + lane;
                        if (s < ns) s_sseg[s] = runS[i];
                        runS[i] = 0.0;
                    }
                    __syncwarp();
                    const int cseg = __shfl_sync(0xffffffffu, c, j);
                    const double* bra = s_bra + cseg * ns;
#pragma unroll
                    for (int ch = 0; ch < NCH; ++ch) {
                        const int sa = fd[ch] & 255, sb = (fd[ch] >> 8) & 255, nM = fd[ch] >> 16;
                        double v = 0.0;
                        for (int i = 0; i < nM; ++i) v = fma(bra[sa + i], s_sseg[sb + i], v);
                        runT[ch] += v;
                    }
                    if ((tmask >> j) & 1u) {
                        const int kseg = __shfl_sync(0xffffffffu, rkv, j);
                        double* dst = (kseg == k0) ? (s_head + warp * nf) : (accS + (size_t)kseg * nf);
#pragma unroll
                        for (int ch = 0; ch < NCH; ++ch) {
                            const int f = ch * 32 + lane;
                            if (f < nf) dst[f] = runT[ch];
                            runT[ch] = 0.0;
                        }
                    }
                    __syncwarp();
                }
            }
            __syncwarp();
        }
        __syncthreads();

        // ---- targets shared by several warp ranges: add the range heads in warp order; per-target norms
        {
            const double dsrc = (L.pe[ci + 1] - L.pe[ci]) * (L.qe[cj + 1] - L.qe[cj]);
            for (int k = tid; k < H; k += T) {
                const int hc = s_hitcell[k], ic = hc / L.Nq, jc = hc - ic * L.Nq;
                s_normk[k] = 1.0 / sqrt(dsrc * ((L.pe[ic + 1] - L.pe[ic]) * (L.qe[jc + 1] - L.qe[jc])));
            }
            for (int w = 0; w < NW; ++w) {
                const int k = s_k0[w];
                if (k < 0 || (w > 0 && s_k0[w - 1] == k)) continue;          // empty range, or not the first head of k
                const bool own = s_start[k] < s_wbeg[w];                     // k began in an earlier range: accS[k] was written
                // (k began before range w but is w's first target only if the earlier warp wrote it as a non-head)
                for (int f = tid; f < nf; f += T) {
                    double sum = own ? accS[(size_t)k * nf + f] : 0.0;
                    for (int w2 = w; w2 < NW && s_k0[w2] == k; ++w2) sum += s_head[w2 * nf + f];
                    accS[(size_t)k * nf + f] = sum;
                }
            }
        }
        __syncthreads();

        // ---- E: thread = output o = (alpha, m-th coupled alpha'); P = norm_k * sum_t c_t * acc_k[f_t]
        for (int o = tid; o < L.totcoup; o += T) {
            const int al = L.o_alpha[o], off = L.cl_off[al], nc = L.cl_off[al + 1] - off;
            const int t0 = L.ot_off[o], nt = L.ot_off[o + 1] - t0;
            double* out = vals + rowptr[(int64_t)cb * L.n_ch + al] + (o - off);
            double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
            int f0 = 0, f1 = 0, f2 = 0, f3 = 0;
            if (nt > 0) { c0 = L.ot_c[t0]; f0 = L.ot_f[t0]; }
            if (nt > 1) { c1 = L.ot_c[t0 + 1]; f1 = L.ot_f[t0 + 1]; }
            if (nt > 2) { c2 = L.ot_c[t0 + 2]; f2 = L.ot_f[t0 + 2]; }
            if (nt > 3) { c3 = L.ot_c[t0 + 3]; f3 = L.ot_f[t0 + 3]; }
            for (int k = 0; k < H; ++k) {
                const double* acc = accS + (size_t)k * nf;
                double v = c0 * acc[f0];
                v = fma(c1, acc[f1], v);
                v = fma(c2, acc[f2], v);
                v = fma(c3, acc[f3], v);
                for (int t = 4; t < nt; ++t) v = fma(L.ot_c[t0 + t], acc[L.ot_f[t0 + t]], v);
                out[(size_t)k * nc] = v * s_normk[k];
            }
        }
    }
}

}  // namespace pm
