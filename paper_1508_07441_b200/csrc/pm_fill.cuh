// pm_fill.cuh — the fill pass (hot-path step a7; the paper's step 2b).
//
// One persistent CTA per SM slot walks source cells D_ij.  Per source cell:
//   (the pattern pass has left the cell's node ids sorted by (target t, x-node c, a, b) in NodeLists, so the nodes
//    of one (t, c) pair are consecutive; nothing is mapped or sorted again here)
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
    static constexpr int NS = kFillMaxSlot, NF = kFillMaxFun, NCH = kFillMaxFun / 32, MAXM = 99;
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
    int thr_p, thr_q, tp, tq, tx, sx, wx, wpa, wqb, bra, tile, tile_bytes, sseg, head, normk, k0, total;
};

constexpr int kTileStride = 33;        // double2 per K-tile row: 32 nodes + 1 pad (conflict-free rows and columns)

inline int fill_align16(int b) { return (b + 15) & ~15; }

// shared-memory plan for nw warps
inline FillSmem fill_smem_plan(const DevLattice& L, int hmax, int nw)
{
    FillSmem s{};
    int o = 0;
    auto take = [&](int bytes) { int r = o; o += fill_align16(bytes); return r; };
    s.thr_p = take(8 * L.pe_pad); s.thr_q = take(8 * L.qe_pad);
    s.tp = take(8 * L.n_p); s.tq = take(8 * L.n_q); s.tx = take(8 * L.n_x); s.sx = take(8 * L.n_x); s.wx = take(8 * L.n_x);
    s.wpa = take(8 * L.n_p); s.wqb = take(8 * L.n_q);
    s.bra = take(8 * L.n_x * (L.n_slot + 1));       // rows padded with one zero slot
    const int np = (L.n_slot + 1) / 2;              // slot pairs
    s.tile_bytes = 16 * kTileStride * np * nw;      // K tiles (phases C, D); staging of target sums (phase E)
    if (s.tile_bytes < 8 * L.n_fun) s.tile_bytes = 8 * L.n_fun;
    s.tile = take(s.tile_bytes);
    s.sseg = take(16 * np * nw);
    s.head = take(8 * L.n_fun * nw);
    s.normk = take(8 * hmax);
    s.k0 = take(4 * (2 * nw + 2));
    s.total = o;
    return s;
}

template <class Spec, int NW>
__global__ void __launch_bounds__(NW * 32, 1)
k_fill_seg(DevLattice L, FillSmem S, NodeLists nl, int cell_begin, int n_blk, int hmax, const int64_t* __restrict__ rowptr,
           double* __restrict__ vals, double* __restrict__ accG)
{
    constexpr int T = NW * 32;
    constexpr int NP = (Spec::NS + 1) / 2;              // slot pairs (one double2 per pair and node in the K tile)
    constexpr int NPC = (NP + 31) / 32;                 // pair chunks of the lane = slot-pair walk
    constexpr int NCH = Spec::NCH;                      // function chunks of the lane = function stage
    extern __shared__ __align__(16) char smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ns = Spec::kStatic ? Spec::NS : L.n_slot, nf = L.n_fun, np = (ns + 1) >> 1;

    double* s_thr_p = (double*)(smem + S.thr_p);
    double* s_thr_q = (double*)(smem + S.thr_q);
    double* s_tp = (double*)(smem + S.tp);   double* s_tq = (double*)(smem + S.tq);   double* s_tx = (double*)(smem + S.tx);
    double* s_sx = (double*)(smem + S.sx);   double* s_wx = (double*)(smem + S.wx);
    double* s_wpa = (double*)(smem + S.wpa); double* s_wqb = (double*)(smem + S.wqb);
    double* s_bra = (double*)(smem + S.bra);
    double2* s_tile = (double2*)(smem + S.tile) + (size_t)warp * kTileStride * np;
    double2* s_sseg2 = (double2*)(smem + S.sseg) + warp * np;
    const double* s_sseg = (const double*)s_sseg2;
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
    const int nsb = ns + 1;                             // bra rows carry one trailing zero slot (index ns)
    for (int k = tid; k < L.n_x * nsb; k += T) { const int c = k / nsb, sl = k - c * nsb; s_bra[k] = sl < ns ? L.bra[c * ns + sl] : 0.0; }
    // per-lane descriptors of function f = ch*32 + lane.  kPacked (at most 3 M-terms per function): byte i of fa / fb =
    // bra / ket slot of term i, unused terms point at the zero bra slot; else fa = sa | sb << 8 | nM << 16.
    constexpr bool kPacked = Spec::MAXM <= 3;
    int fa[NCH], fb[NCH];
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
        const int f = ch * 32 + lane;
        fa[ch] = kPacked ? (ns | (ns << 8) | (ns << 16)) : 0;
        fb[ch] = 0;
        if (f < nf) {
            const int4 fn = L.fun[f];
            if (kPacked) {
                fa[ch] = 0;
                for (int i = 0; i < 3; ++i) {
                    fa[ch] |= (i < fn.z ? fn.x + i : ns) << (8 * i);
                    fb[ch] |= (i < fn.z ? fn.y + i : 0) << (8 * i);
                }
            } else fa[ch] = fn.x | (fn.y << 8) | (fn.z << 16);
        }
    }
    double* accS = accG + (size_t)blockIdx.x * hmax * nf;

    for (int cb = blockIdx.x; cb < n_blk; cb += gridDim.x) {
        const int cell = cell_begin + cb;
        const int ci = cell / L.Nq, cj = cell - ci * L.Nq;
        const CellGeom g = cell_geom(L.pe, L.qe, ci, cj);
        const int H = nl.hits[cb], ntot = nl.ntot[cb];
        const unsigned short* __restrict__ g_sorted = nl.sorted + (size_t)cb * L.nnode;
        const unsigned short* __restrict__ g_rkpos = nl.rkpos + (size_t)cb * L.nnode;
        __syncthreads();                                // previous cell's phase E is done with shared memory
        for (int k = tid; k < L.n_p; k += T) s_wpa[k] = __dmul_rn(g.hp, L.wp[k]);
        for (int k = tid; k < L.n_q; k += T) s_wqb[k] = __dmul_rn(g.hq, L.wq[k]);
        // warp ranges over the sorted list, in whole 32-node steps; first target of each range
        if (tid <= NW) { const int G = (ntot + 31) >> 5; s_wbeg[tid] = min(ntot, ((int)(((long long)tid * G) / NW)) << 5); }
        // normalisation of every target: its first node is mapped again (exact arithmetic: the same cell)
        {
            const double dsrc = (L.pe[ci + 1] - L.pe[ci]) * (L.qe[cj + 1] - L.qe[cj]);
            for (int pos = tid; pos < ntot; pos += T) {
                const int r = g_rkpos[pos];
                if (pos > 0 && g_rkpos[pos - 1] == r) continue;
                int c, a, b;
                split_node(L, g_sorted[pos], c, a, b);
                double p, q, P2, Q2;
                map_node_sq(g, s_tp[a], s_tq[b], s_tx[c], p, q, P2, Q2);
                const int hc = target_cell_sq(s_thr_p, L.pe_pad, L.Np, s_thr_q, L.qe_pad, L.Nq, P2, Q2);
                const int ic = hc / L.Nq, jc = hc - ic * L.Nq;
                s_normk[r] = 1.0 / sqrt(dsrc * ((L.pe[ic + 1] - L.pe[ic]) * (L.qe[jc + 1] - L.qe[jc])));
            }
        }
        __syncthreads();
        const int wb = s_wbeg[warp], we = s_wbeg[warp + 1];
        const int k0 = (wb < we) ? (int)g_rkpos[wb] : -1;
        if (lane == 0) s_k0[warp] = k0;

        // ---- C + D: 32 sorted nodes per step; the node ids of the next two steps are already in flight
        double runT[NCH];
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) runT[ch] = 0.0;
        double2 runS[NPC];
#pragma unroll
        for (int i = 0; i < NPC; ++i) runS[i] = make_double2(0.0, 0.0);
        int mC = 0, rC = -1, mN = 0, rN = -1;           // this step's and the next step's node id / target rank (-1: none)
        if (wb + lane < we) { mC = g_sorted[wb + lane]; rC = g_rkpos[wb + lane]; }
        if (wb + 32 + lane < we) { mN = g_sorted[wb + 32 + lane]; rN = g_rkpos[wb + 32 + lane]; }
        for (int base = wb; base < we; base += 32) {
            int mF = 0, rF = -1;
            if (base + 64 + lane < we) { mF = g_sorted[base + 64 + lane]; rF = g_rkpos[base + 64 + lane]; }
            const bool active = rC >= 0;
            int c, a, b;
            split_node(L, mC, c, a, b);
            // the node after this one (next lane, or lane 0 of the next step); rank -1 past the end of the range
            int m1 = __shfl_down_sync(0xffffffffu, mC, 1), r1 = __shfl_down_sync(0xffffffffu, rC, 1);
            const int m1n = __shfl_sync(0xffffffffu, mN, 0), r1n = __shfl_sync(0xffffffffu, rN, 0);
            if (lane == 31) { m1 = m1n; r1 = r1n; }
            const int c1 = L.mg_npq ? (int)__umulhi((unsigned)m1, L.mg_npq) : m1;
            // target ends: t changes after this node (or the range ends); segment ends: (t, c) changes
            const bool tend = active && (r1 != rC);
            const bool send = active && (tend || c1 != c);
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
                    for (int i = 0; i < NP; ++i)
                        s_tile[i * kTileStride + lane] = make_double2(K[2 * i], (2 * i + 1 < Spec::NS) ? K[(2 * i + 1) % Spec::NS] : 0.0);
                } else {
                    for (int i = 0; i < np; ++i)
                        s_tile[i * kTileStride + lane] = make_double2(K[2 * i], (2 * i + 1 < ns) ? K[2 * i + 1] : 0.0);
                }
            }
            __syncwarp();
            // lane = slot pair: walks the tile's nodes, up to 4 per step, never across a segment end
            for (int j = 0; j < cnt;) {
                const int nbnd = __ffs((smask >> j) & 0xfu);             // 1-based offset of the next segment end, 0 = none in 4
                const int step = nbnd ? nbnd : min(4, cnt - j);
                if (step == 4) {
#pragma unroll
                    for (int i = 0; i < NPC; ++i) {
                        const int sp = i * 32 + lane;
                        if (sp < np) {
                            const double2* row = s_tile + sp * kTileStride + j;
                            const double2 d0 = row[0], d1 = row[1], d2 = row[2], d3 = row[3];
                            runS[i].x += (d0.x + d1.x) + (d2.x + d3.x);
                            runS[i].y += (d0.y + d1.y) + (d2.y + d3.y);
                        }
                    }
                } else {
                    for (int r = 0; r < step; ++r) {
#pragma unroll
                        for (int i = 0; i < NPC; ++i) {
                            const int sp = i * 32 + lane;
                            if (sp < np) { const double2 d = s_tile[sp * kTileStride + j + r]; runS[i].x += d.x; runS[i].y += d.y; }
                        }
                    }
                }
                j += step;
                if (nbnd) {                                              // node jb ends a (t, c) segment
                    const int jb = j - 1;
#pragma unroll
                    for (int i = 0; i < NPC; ++i) {
                        const int sp = i * 32 + lane;
                        if (sp < np) s_sseg2[sp] = runS[i];
                        runS[i] = make_double2(0.0, 0.0);
                    }
                    __syncwarp();
                    const int cseg = __shfl_sync(0xffffffffu, c, jb);
                    const double* bra = s_bra + cseg * nsb;
#pragma unroll
                    for (int ch = 0; ch < NCH; ++ch) {
                        if (kPacked) {
                            const int ia = fa[ch], ib = fb[ch];
                            double v = bra[ia & 255] * s_sseg[ib & 255];
                            v = fma(bra[(ia >> 8) & 255], s_sseg[(ib >> 8) & 255], v);
                            v = fma(bra[ia >> 16], s_sseg[ib >> 16], v);
                            runT[ch] += v;
                        } else {
                            const int sa = fa[ch] & 255, sb = (fa[ch] >> 8) & 255, nM = fa[ch] >> 16;
                            double v = 0.0;
                            for (int i = 0; i < nM; ++i) v = fma(bra[sa + i], s_sseg[sb + i], v);
                            runT[ch] += v;
                        }
                    }
                    if ((tmask >> jb) & 1u) {                            // ... and ends target t: its sums are complete
                        const int kseg = __shfl_sync(0xffffffffu, rC, jb);
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
            mC = mN; rC = rN; mN = mF; rN = rF;
        }
        __syncthreads();

        // ---- targets shared by several warp ranges: add the range heads in warp order
        for (int w = 0; w < NW; ++w) {
            const int k = s_k0[w];
            if (k < 0 || (w > 0 && s_k0[w - 1] == k)) continue;              // empty range, or not the first head of k
            // k began in an earlier range (then accS[k] already holds that part) iff the node before this range is in k
            const bool own = s_wbeg[w] > 0 && (int)g_rkpos[s_wbeg[w] - 1] == k;
            for (int f = tid; f < nf; f += T) {
                double sum = own ? accS[(size_t)k * nf + f] : 0.0;
                for (int w2 = w; w2 < NW && s_k0[w2] == k; ++w2) sum += s_head[w2 * nf + f];
                accS[(size_t)k * nf + f] = sum;
            }
        }
        __syncthreads();

        // ---- E: thread = output o = (alpha, m-th coupled alpha'); P = norm_k * sum_t c_t * acc_k[f_t].
        // The sums of a chunk of targets are staged in shared memory (the K-tile area is free here).
        {
            double* s_acc = (double*)(smem + S.tile);
            const int kc = max(1, S.tile_bytes / (8 * nf));
            for (int kb = 0; kb < H; kb += kc) {
                const int ke = min(H, kb + kc), n = (ke - kb) * nf;
                const double* src = accS + (size_t)kb * nf;
                for (int idx = tid; idx < n; idx += T) s_acc[idx] = src[idx];
                __syncthreads();
                for (int o = tid; o < L.totcoup; o += T) {
                    const int al = L.o_alpha[o], off = L.cl_off[al], nc = L.cl_off[al + 1] - off;
                    const int t0 = L.ot_off[o], nt = L.ot_off[o + 1] - t0;
                    double* out = vals + rowptr[(int64_t)cb * L.n_ch + al] + (o - off) + (size_t)kb * nc;
                    double c0 = 0.0, c1 = 0.0, c2 = 0.0;
                    int f0 = 0, f1 = 0, f2 = 0;
                    if (nt > 0) { c0 = L.ot_c[t0]; f0 = L.ot_f[t0]; }
                    if (nt > 1) { c1 = L.ot_c[t0 + 1]; f1 = L.ot_f[t0 + 1]; }
                    if (nt > 2) { c2 = L.ot_c[t0 + 2]; f2 = L.ot_f[t0 + 2]; }
                    if (nt <= 3) {
#pragma unroll 4
                        for (int k = 0; k < ke - kb; ++k) {
                            const double* acc = s_acc + k * nf;
                            const double v = fma(c2, acc[f2], fma(c1, acc[f1], c0 * acc[f0]));
                            out[(size_t)k * nc] = v * s_normk[kb + k];
                        }
                    } else {
                        for (int k = 0; k < ke - kb; ++k) {
                            const double* acc = s_acc + k * nf;
                            double v = fma(c2, acc[f2], fma(c1, acc[f1], c0 * acc[f0]));
                            for (int t = 3; t < nt; ++t) v = fma(L.ot_c[t0 + t], acc[L.ot_f[t0 + t]], v);
                            out[(size_t)k * nc] = v * s_normk[kb + k];
                        }
                    }
                }
                __syncthreads();
            }
        }
    }
}

}  // namespace pm
