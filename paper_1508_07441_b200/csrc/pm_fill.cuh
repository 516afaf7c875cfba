// pm_fill.cuh — the fill pass (hot-path step a7; the paper's step 2b).
//
// One WARP builds all rows of one source cell D_ij; warps take cells from a global counter, so no block-level
// barrier exists after start-up and the warps of an SM drift apart and hide each other's latencies.
// The pattern pass has left the cell's node ids sorted by (target t, x-node c, a, b) with the target cell of
// every sorted position (NodeLists), so the nodes of one (t, c) pair are consecutive; nothing is mapped or sorted here.
//   C  nodes  lane = node, 32 consecutive sorted nodes per step: omega, directions, the ket harmonics K[slot]
//             (Spec::ket — generated straight-line code, registers only); K tile -> shared memory as double2 pairs
//   D  sums   lane = slot pair: walks the tile's nodes, summing K over each (t, c) segment; at a segment end
//             lane = function: acc_t[f] += sum_M bra[c][sa+M] * S[sb+M] (the bra harmonics depend on c only, so they
//             are applied once per segment, not once per node)
//   E  rows   at the end of target t, lane = output (alpha, alpha'): P = norm_t * sum_L c^L_{alpha alpha'} acc_t[f],
//             written straight into the CSR rows (runs of consecutive alpha' are contiguous)
// Every sum has a fixed order (sorted node order): bitwise reproducible, no floating atomics.
// Prior art this replaces: one thread per element / per cell pair, constants in global memory, CPU repack
// (PAPER.md:L341, L348-356, L376).
#pragma once
#include "pm_device.cuh"
#include "pm_ylm.h"

namespace pm {

constexpr int kFillMaxSlot = 96;       // ket slots / orbital functions one kernel launch holds (larger channel sets are
constexpr int kFillMaxFun = 320;       // split into column-channel groups, pm_tables.hpp)
constexpr int kFillMaxOut = 1400;      // outputs (alpha, alpha') per launch of the table-driven kernel (their tables live in shared memory)
constexpr int kFillJitSlot = 40;       // ... and what one SPECIALISED kernel holds: its ket slots are accumulators in registers,
constexpr int kFillJitFun = 160;       // its functions five stage steps, its output tables share the SM's shared memory with
constexpr int kFillJitOut = 700;       // twelve warps' tiles
constexpr int kFillMaxY = 91;          // harmonics per direction up to l = PM_MAX_L = 12

// Table-driven ket code for channel sets without a generated kernel (slow: local arrays, table loads).
struct SpecGeneric {
    static constexpr bool kStatic = false;
    static constexpr int NS = kFillMaxSlot, NF = kFillMaxFun, NCH = kFillMaxFun / 32, MAXM = 99, MAXL1 = 99;
    static constexpr unsigned long long kHash = 0ull;
    static constexpr bool kBraSmem = false;             // (decided at run time for this kernel: FillSmem::bra)
    static constexpr int NOT = 3;                       // terms per output kept in shared memory (more come from the global tables)
    static constexpr bool kOutTail = true;
    static __device__ __forceinline__ constexpr int terms(int) { return 3; }      // (unused: MAXM > 3 loops over the function's own terms)
    // writes the node's column of the K tile directly (no per-thread K array): col = tile + lane, np slot pairs
    static __device__ __noinline__ void ket_tile(const DevLattice& L, double om, double uxa, double uza, double uxb, double uzb,
                                                 double2* __restrict__ col, int stride, int np, int ns, bool first)
    {
        double Yp[kFillMaxY], Yq[kFillMaxY];
        ylm_fill(L.lmax, uxa, uza, L.ya, L.yb, L.ydiag, Yp);
        ylm_fill(L.lmax, uxb, uzb, L.ya, L.yb, L.ydiag, Yq);
        for (int i = 0; i < np; ++i) {
            double v[2] = {0.0, 0.0};
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int s = 2 * i + h;
                if (s < ns) {
                    double a = 0.0;
                    for (int t = L.kt_off[s]; t < L.kt_off[s + 1]; ++t) a += L.kt_c[t] * Yp[L.kt_ip[t]] * Yq[L.kt_iq[t]];
                    v[h] = a * om;
                }
            }
            if (!first) { const double2 o = col[i * stride]; v[0] += o.x; v[1] += o.y; }       // running sum of the lane's chunk
            col[i * stride] = make_double2(v[0], v[1]);
        }
    }
};


constexpr int kTileStride = 33;        // double2 per K-tile row: 32 nodes + 1 pad (conflict-free rows and columns)

// Private shared-memory area of one warp, byte offsets: everything whose size follows from (slot pairs, functions, row
// batch) first, so that a specialised kernel addresses it with compile-time offsets from ONE base register (the kernel
// runs at the register limit); the per-cell node tables (sizes n_p, n_q) come last.
struct WarpLayout { int tile, sseg, acc, hcol, ring, cell, p2, fixed_bytes; };
__host__ __device__ constexpr int fill_al16(int b) { return (b + 15) & ~15; }
__host__ __device__ constexpr WarpLayout warp_layout(int np, int nf, int row_batch)
{
    WarpLayout w{};
    int o = 0;
    w.tile = o; o += fill_al16(16 * kTileStride * np);
    w.sseg = o; o += fill_al16(16 * np);
    w.acc = o;  o += fill_al16(8 * nf * row_batch);      // sums of finished targets waiting for their rows to be written
    w.hcol = o; o += fill_al16(4 * row_batch);
    w.ring = o; o += 2 * 32 * 8;                         // chunk words of two steps
    w.cell = o; o += 32;
    w.p2 = o;                                            // double2 (p_a, hp wp_a) [n_p], then (q_b, hq wq_b) [n_q]
    w.fixed_bytes = o;
    return w;
}

struct FillSmem {           // byte offsets into dynamic shared memory, computed on the host
    int dp, dq, tx, sx, wx, bra, odesc, ofi, oc, fa, fb, fc, warp0, warp_bytes, total;
    WarpLayout w;
};

inline int fill_align16(int b) { return (b + 15) & ~15; }


// shared-memory plan for nw warps: tables shared by the CTA, then one private area per warp
inline FillSmem fill_smem_plan(const DevLattice& L, int nw, int row_batch, int n_oterm, bool bra_in_smem = true, bool generic = false)
{
    const int nfun_pad = generic ? kFillMaxFun : (L.n_fun + 31) & ~31;     // NCH * 32 of the kernel that runs
    FillSmem s{};
    int o = 0;
    auto take = [&](int bytes) { int r = o; o += fill_align16(bytes); return r; };
    // cell norms of both axes: in shared memory when they fit beside everything else (decided below), else read from the edges
    s.dp = s.dq = -1;
    s.tx = take(8 * L.n_x); s.sx = take(8 * L.n_x); s.wx = take(8 * L.n_x);
    s.bra = bra_in_smem ? take(8 * L.n_x * (L.n_bra + 1)) : -1;      // rows end with one zero slot; -1: read from global memory
    s.odesc = take(4 * L.n_out); s.ofi = take(4 * L.n_out); s.oc = take(8 * n_oterm * L.n_out);
    s.fa = take(4 * nfun_pad); s.fb = take(4 * nfun_pad); s.fc = take(4 * nfun_pad);             // (every function chunk of the stage reads its entry)
    const int np = (L.n_slot + 1) / 2;              // slot pairs
    s.w = warp_layout(np, L.n_fun, row_batch);
    const int w = s.w.fixed_bytes + 16 * (L.n_p + L.n_q);
    s.warp_bytes = w;
    s.warp0 = take(w * nw);
    if (o + fill_align16(8 * L.Np) + fill_align16(8 * L.Nq) <= 227 * 1024) { s.dp = take(8 * L.Np); s.dq = take(8 * L.Nq); }
    s.total = o;
    return s;
}

// cell norm B_k: width (reading A) or (e_{k+1}^3 - e_k^3)/3 (reading B, states normalised in the p^2 dp measure)
__device__ __forceinline__ double cell_norm(const double* __restrict__ e, int k, int norm)
{
    const double e0 = e[k], e1 = e[k + 1];
    return norm ? (e1 * e1 * e1 - e0 * e0 * e0) / 3.0 : e1 - e0;
}

// kMode: 0 values, 1 values and column indices, 2 the PER-PAIR SUMS: for every hit cell pair (source cell, k-th hit cell) the
// normalised sums of the group's orbital functions, vals[(cellbase + k) * op_stride + op_off + f] (`rowptr` is then the
// exclusive scan of the hit counts): the operator form of P0 (every nonzero is a combination of at most four of them) that
// k_op_expand turns into CSR rows for channel sets filled group by group.
template <class Spec, int NW, int kRowBatch, int kMode>
__global__ void __launch_bounds__(NW * 32, 1)
k_fill_warp(DevLattice L, FillSmem S, NodeLists nl, int cell_begin, int n_blk, const int64_t* __restrict__ rowptr,
            double* __restrict__ vals, int32_t* __restrict__ colidx, int* __restrict__ counter, const int64_t* __restrict__ guard)
{
    // pm_build launches this kernel before the host has seen nnz: the scan kernel left guard[4] != 0 when the block's
    // nnz exceeds the caller's capacity, and then nothing may be written
    if (guard != nullptr && guard[4] != 0) return;
    constexpr int T = NW * 32;
    constexpr bool kCols = kMode == 1;
    constexpr int NP = (Spec::NS + 1) / 2;              // slot pairs (one double2 per pair and node in the K tile)
    constexpr int NPC = (NP + 31) / 32;                 // pair chunks of the lane = slot-pair walk
    constexpr int NCH = Spec::NCH;                      // function chunks of the lane = function stage
    extern __shared__ __align__(16) char smem[];
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int ns = Spec::kStatic ? Spec::NS : L.n_slot, nf = Spec::kStatic ? Spec::NF : L.n_fun, np = (ns + 1) >> 1;

    double* s_tx = (double*)(smem + S.tx);
    double* s_sx = (double*)(smem + S.sx);   double* s_wx = (double*)(smem + S.wx);
    double* s_bra = (double*)(smem + (S.bra >= 0 ? S.bra : 0));
    int* s_odesc = (int*)(smem + S.odesc);             // per output o: cl_off[alpha] | nc << 12 | m << 19 | alpha' << 25
    int* s_ofi = (int*)(smem + S.ofi);                 // f0 | f1 << 10 | f2 << 20 | (n_terms - 1) << 30, or four f of 8 bits
    double* s_oc = (double*)(smem + S.oc);             // [NOT][n_out] coefficients c^L, term-major: consecutive lanes read consecutive doubles (0 where there is no term)
    char* wsm = smem + S.warp0 + warp * S.warp_bytes;
    // compile-time offsets for a specialised kernel (the host plan computes the same numbers from the lattice's tables)
    constexpr WarpLayout kW = warp_layout(NP, Spec::NF, kRowBatch);
    const WarpLayout W = Spec::kStatic ? kW : S.w;
    double2* s_tile = (double2*)(wsm + W.tile);
    double2* s_sseg2 = (double2*)(wsm + W.sseg);
    const double* s_sseg = (const double*)s_sseg2;
    double* s_acc = (double*)(wsm + W.acc);           // [kRowBatch][nf] sums of finished targets
    int* s_hcol = (int*)(wsm + W.hcol);                 // first column of each finished target: cell * n_ch (kCols)
    double2* s_p2 = (double2*)(wsm + W.p2);             // (p_a, hp wp_a) of the cell's p-nodes, then (q_b, hq wq_b) at s_p2 + n_p
    uint2* s_ring = (uint2*)(wsm + W.ring);             // chunk words of two steps
    struct CellInfo { int64_t rbase; double dsrc; int H; };
    CellInfo* s_cell = (CellInfo*)(wsm + W.cell);

    // ---- once per CTA: widths, rules, bra harmonics, output descriptors
    const double* s_dp = S.dp >= 0 ? (const double*)(smem + S.dp) : nullptr;
    const double* s_dq = S.dq >= 0 ? (const double*)(smem + S.dq) : nullptr;
    if (S.dp >= 0) {
        for (int k = tid; k < L.Np; k += T) ((double*)(smem + S.dp))[k] = cell_norm(L.pe, k, L.norm);
        for (int k = tid; k < L.Nq; k += T) ((double*)(smem + S.dq))[k] = cell_norm(L.qe, k, L.norm);
    }
    for (int k = tid; k < L.n_x; k += T) { s_tx[k] = L.tx[k]; s_sx[k] = L.sx[k]; s_wx[k] = L.wx[k]; }
    const int nb_ = L.n_bra;                            // bra slots (the whole channel set's)
    const int nsb = nb_ + 1;                            // bra rows carry one trailing zero slot (index nb_), in global memory too
    if (S.bra >= 0)
        for (int k = tid; k < L.n_x * nsb; k += T) s_bra[k] = L.bra[k];
    const double* __restrict__ bra_tab = S.bra >= 0 ? s_bra : L.bra;      // big channel sets: the bra table stays in global memory
    const int bra_stride = nsb;
    constexpr int NOT = Spec::NOT;                      // terms per output kept in shared memory: 3 (f in 10 bits each + count) or 4 (8 bits each)
    for (int o = tid; o < L.n_out; o += T) {
        const int al = L.g_alpha[o], off = L.cl_off[al], nc = L.cl_off[al + 1] - off;
        const int t0 = L.ot_off[o], nt = L.ot_off[o + 1] - t0;
        s_odesc[o] = off | (nc << 12) | (L.g_m[o] << 19) | (L.g_ap[o] << 25);
        int fi = NOT == 3 ? (nt > 0 ? nt - 1 : 0) << 30 : 0;
        for (int i = 0; i < NOT; ++i) {
            s_oc[i * L.n_out + o] = i < nt ? L.ot_c[t0 + i] : 0.0;
            fi |= (i < nt ? L.ot_f[t0 + i] : 0) << ((NOT == 3 ? 10 : 8) * i);
        }
        s_ofi[o] = fi;
    }
    // descriptors of function f (lane = f & 31 in the stage), kept in shared memory (registers are what limits the
    // warps per SM here).  kPacked (at most 3 M-terms per function): byte i of fa = bra slot of term i, unused terms point
    // at the zero bra slot; else fa = sa | nM << 16, fb = sb.
    constexpr bool kPacked = Spec::MAXM <= 3;
    int* s_fa = (int*)(smem + S.fa);
    int* s_fb = (int*)(smem + S.fb);
    int* s_fc = (int*)(smem + S.fc);
    // (the ket side is read from the K tile, where the walk leaves a segment's sums in the column of the segment's last
    // chunk: kPacked keeps the byte offset of each term's slot in column 0, 16 bits each, in fb (terms 0, 1) and fc (term 2))
    auto tile_byte = [](int slot) { return (slot >> 1) * (kTileStride * 16) + (slot & 1) * 8; };
    for (int f = tid; f < NCH * 32; f += T) {
        int va = kPacked ? (nb_ | (nb_ << 8) | (nb_ << 16)) : 0, vb = 0, vc = 0;
        if (f < nf) {
            const int4 fn = L.fun[f];
            if (kPacked) {
                va = 0;
                for (int i = 0; i < 3; ++i) va |= (i < fn.z ? fn.x + i : nb_) << (8 * i);
                vb = tile_byte(0 < fn.z ? fn.y : 0) | (tile_byte(1 < fn.z ? fn.y + 1 : 0) << 16);
                vc = tile_byte(2 < fn.z ? fn.y + 2 : 0);
            } else { va = fn.x | (fn.z << 16); vb = fn.y; }
        }
        s_fa[f] = va; s_fb[f] = vb; s_fc[f] = vc;
    }
    __syncthreads();                                    // the only block-level barrier

    for (;;) {
        int cb = 0;
        if (lane == 0) cb = atomicAdd(counter, 1);
        cb = __shfl_sync(0xffffffffu, cb, 0);
        if (cb >= n_blk) break;
        const int cell = cell_begin + cb;
        const int ci = cell / L.Nq, cj = cell - ci * L.Nq;
        const int H = nl.hits[cb], nck = nl.nchunk[cb];
        const uint2* __restrict__ g_chunk = nl.chunk + (size_t)cb * L.nnode;      // NodeLists (pm_device.cuh)
        // what only the row phase and the target ends need of the cell waits in shared memory (registers are the limit here)
        if (lane == 0) { s_cell->rbase = kMode == 2 ? rowptr[cb] : rowptr[(int64_t)cb * L.n_ch]; s_cell->dsrc = cell_norm(L.pe, ci, L.norm) * cell_norm(L.qe, cj, L.norm); s_cell->H = H; }
        {   // the cell's nodes p_a = cp + hp t_a, q_b = cq + hq t_b (the operations of map_node_sq) and weights hp wp_a, hq wq_b
            const CellGeom g = cell_geom(L.pe, L.qe, ci, cj);
            for (int k = lane; k < L.n_p; k += 32) s_p2[k] = make_double2(__dadd_rn(g.cp, __dmul_rn(g.hp, L.tp[k])), __dmul_rn(g.hp, L.wp[k]));
            for (int k = lane; k < L.n_q; k += 32) s_p2[L.n_p + k] = make_double2(__dadd_rn(g.cq, __dmul_rn(g.hq, L.tq[k])), __dmul_rn(g.hq, L.wq[k]));
        }
        __syncwarp();
        int kcur = 0, kdone = 0;                        // targets finished / written; a target's rank is its position in every row
        // ---- E: lane = output (alpha, m-th coupled alpha'): P = norm_t * sum_L c^L acc_t[f] for targets k0 .. k0+nb-1
        // The rows are ordered by the most terms of their outputs (pm_tables.cpp): a 32-output step inside the one-term
        // (two-term) rows loads one (two) sums per target.  The cell normalisation is already in the sums (target end, below).
        auto write_rows_t = [&](int k0, int nb, auto full_tag) {
            constexpr bool kFull = decltype(full_tag)::value;           // all kRowBatch slots hold a target
            int hcl[kRowBatch];
#pragma unroll
            for (int bb = 0; bb < kRowBatch; ++bb) hcl[bb] = kCols ? s_hcol[bb] : 0;
            const int64_t rbase = s_cell->rbase;
            double* __restrict__ row0 = vals + rbase;
            int32_t* __restrict__ col0 = kCols ? colidx + rbase : nullptr;
            const int Hc = s_cell->H;
            auto outputs = [&](int o_begin, int o_end, auto nt_tag) {
                constexpr int NT = decltype(nt_tag)::value;
#pragma unroll 2
                for (int o = o_begin + lane; o < o_end; o += 32) {
                    const int od = s_odesc[o], fi = s_ofi[o];
                    const int clo = od & 4095, nc = (od >> 12) & 127, mm = (od >> 19) & 63, ap = (unsigned)od >> 25;
                    const double c0 = s_oc[o], c1 = NT > 1 ? s_oc[L.n_out + o] : 0.0, c2 = NT > 2 ? s_oc[2 * L.n_out + o] : 0.0,
                                 c3 = NT > 3 ? s_oc[3 * L.n_out + o] : 0.0;
                    constexpr int FB = NOT == 3 ? 10 : 8, FM = (1 << FB) - 1;
                    const int f0 = fi & FM, f1 = (fi >> FB) & FM, f2 = (fi >> (2 * FB)) & FM, f3 = NOT > 3 ? (int)((unsigned)fi >> 24) : 0;
                    // entry of target k0+bb in row alpha: element H*clo + (k0+bb)*nc + m of the cell's block (fits 32 bits)
                    const unsigned idx0 = (unsigned)(Hc * clo + k0 * nc + mm);
                    const char* acc0 = (const char*)s_acc;
                    const unsigned a0 = 8u * f0, a1 = 8u * f1, a2 = 8u * f2, a3 = 8u * f3;
#pragma unroll
                    for (int bb = 0; bb < kRowBatch; ++bb) {
                        if (kFull || bb < nb) {
                            const char* acc = acc0 + bb * (8 * nf);
                            double v = c0 * *(const double*)(acc + a0);
                            if (NT > 1) v = fma(c1, *(const double*)(acc + a1), v);
                            if (NT > 2) v = fma(c2, *(const double*)(acc + a2), v);
                            if (NT > 3) v = fma(c3, *(const double*)(acc + a3), v);
                            if (Spec::kOutTail) {                     // more L values than the shared-memory tables hold: the tail comes from the global ones
                                const int t0 = L.ot_off[o], nt = L.ot_off[o + 1] - t0;
                                for (int t = NOT; t < nt; ++t) v = fma(L.ot_c[t0 + t], ((const double*)acc)[L.ot_f[t0 + t]], v);
                            }
                            const unsigned e = idx0 + (unsigned)(bb * nc);
                            row0[e] = v;
                            if (kCols) col0[e] = hcl[bb] + ap;
                        }
                    }
                }
            };
            if constexpr (kFull) {
                const int e1 = L.n_out1 & ~31, e2 = max(e1, L.n_out2 & ~31), e3 = NOT > 3 ? max(e2, L.n_out3 & ~31) : L.n_out;
                outputs(0, e1, std::integral_constant<int, 1>{});
                outputs(e1, e2, std::integral_constant<int, 2>{});
                outputs(e2, e3, std::integral_constant<int, 3>{});
                if constexpr (NOT > 3) outputs(e3, L.n_out, std::integral_constant<int, 4>{});
            } else {
                outputs(0, L.n_out, std::integral_constant<int, NOT>{});
            }
            __syncwarp();
        };
        auto write_rows = [&](int k0, int nb) {
            if (nb == kRowBatch) write_rows_t(k0, nb, std::true_type{}); else write_rows_t(k0, nb, std::false_type{});
        };

        // ---- C + D: 32 chunks per step, lane = chunk (at most chunk_len consecutive sorted nodes of one (t, c) segment,
        // cut by the pattern pass): the lane sums the ket harmonics of its nodes in registers, so the K tile holds one
        // column per chunk and the shared-memory traffic of the segment sums falls by the chunk length.
        // The chunk words of the next two steps are already in flight.
        // The running sums of the open segment (runS) and of the open target (runT) live in registers only while a step's
        // segment sums are formed; across the ket code of the next step they wait in shared memory (the open target's
        // slot of the row batch and the segment buffer), which is what keeps the ket code's accumulators out of local memory.
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) { const int f = ch * 32 + lane; if (f < nf) s_acc[f] = 0.0; }
#pragma unroll
        for (int i = 0; i < NPC; ++i) { const int sp = i * 32 + lane; if (sp < np) s_sseg2[sp] = make_double2(0.0, 0.0); }
        // The chunk words travel global -> shared memory by cp.async into a per-warp ring of two steps (the words of step
        // s + 2 are requested when step s is finished): no register holds a word in flight across the ket code, and the
        // step's own words stay readable for the segment and target ends behind it.
        const unsigned ring = (unsigned)__cvta_generic_to_shared(s_ring) + 8u * lane;
        auto fetch = [&](int step, int slot) {          // chunk word of this lane in step `step` -> ring slot `slot`
            const int k = step * 32 + lane;
            if (k < nck) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(ring + 256u * slot), "l"(g_chunk + k) : "memory");
            asm volatile("cp.async.commit_group;" ::: "memory");
        };
        fetch(0, 0);
        fetch(1, 1);
        const unsigned abmask = (1u << nl.ab_bits) - 1u;
        for (int base = 0; base < nck; base += 32) {
            asm volatile("cp.async.wait_group 1;" ::: "memory");
            uint2* s_step = s_ring + (base & 32);                           // this step's chunk words
            if (base + lane >= nck) s_step[lane] = make_uint2(0u, 0u);      // (a lane without a chunk)
            __syncwarp();
            const uint2 dC = s_step[lane];
            const int len = base + lane < nck ? (int)((dC.x >> 18) & 15u) + 1 : 0;
            const int c = (int)(dC.x >> 24);                                // the chunk's x-node
            const int maxlen = __reduce_max_sync(0xffffffffu, len);
            {
                double K[Spec::kStatic ? Spec::NS : 1];
                if constexpr (Spec::kStatic) {
#pragma unroll
                    for (int i = 0; i < Spec::NS; ++i) K[i] = 0.0;
                }
                // One node of the chunk: omega and the rotated directions.  Branch-free (a lane whose chunk is shorter
                // runs node 0 again with omega = 0), so the map of node r + 1 can be scheduled into the ket code of node r.
                struct NodeIn { double om, uxa, uza, uxb, uzb; };
                auto node_in = [&](unsigned abw, bool valid) {
                    const int ab = (int)(abw & abmask);
                    const int a = L.mg_nq ? (int)__umulhi((unsigned)ab, L.mg_nq) : ab, b = ab - a * L.n_q;
                    const double x = s_tx[c], sx = s_sx[c];
                    const double2 pw = s_p2[a], qw = s_p2[L.n_p + b];
                    const double p = pw.x, q = qw.x;                        // cp + hp t_a, cq + hq t_b: the node of DESIGN.md sec. 3.1
                    // omega = w * p q / (p' q'),  w = ((hp wp_a)(hq wq_b)) wx_c; |p'| and |q'| are the lengths
                    // of the rotated vectors below (1/(p'q') = ra * rb: no third reciprocal square root, no second node map)
                    const double w = __dmul_rn(__dmul_rn(pw.y, qw.y), s_wx[c]);
                    // rotated directions from vector components (frame: q^ = z, p^ = (sx, 0, x)):
                    //   p' = -p/2 - 3q/4 ,  q' = p - q/2
                    const double psx = p * sx, px = p * x;
                    const double ax = -0.5 * psx, az = fma(-0.5, px, -0.75 * q);
                    const double bx = psx, bz = fma(-0.5, q, px);
                    const double ra = rsqrt(fma(ax, ax, az * az)), rb = rsqrt(fma(bx, bx, bz * bz));
                    // (reading B: omega = w * p^2 q^2, no Jacobian of the delta functions)
                    const double om = L.norm ? w * ((p * q) * (p * q)) : w * (p * q) * (ra * rb);
                    return NodeIn{valid ? om : 0.0, ax * ra, az * ra, bx * rb, bz * rb};
                };
                unsigned abs_ = dC.y;
                NodeIn cur = node_in(abs_, 0 < len);
#pragma unroll 1
                for (int r = 0; r < maxlen; ++r) {
                    abs_ >>= nl.ab_bits;
                    const NodeIn nxt = node_in(abs_, r + 1 < len);      // (peeling the last iteration doubles the ket code: slower)
                    if constexpr (Spec::kStatic) Spec::ket_acc(L, cur.om, cur.uxa, cur.uza, cur.uxb, cur.uzb, K);
                    else Spec::ket_tile(L, cur.om, cur.uxa, cur.uza, cur.uxb, cur.uzb, s_tile + lane, kTileStride, np, ns, r == 0);
                    cur = nxt;
                }
                if constexpr (Spec::kStatic) {
#pragma unroll
                    for (int i = 0; i < NP; ++i)
                        s_tile[i * kTileStride + lane] = make_double2(K[2 * i], (2 * i + 1 < Spec::NS) ? K[(2 * i + 1) % Spec::NS] : 0.0);
                }
            }
            __syncwarp();
            // segment ends: (t, c) changes behind a chunk; target ends: t changes (or the list ends)
            const unsigned dx = s_step[lane].x;
            const unsigned smask = __ballot_sync(0xffffffffu, (dx >> 22) & 1u), tmask = __ballot_sync(0xffffffffu, (dx >> 23) & 1u);
            const int cnt = min(32, nck - base);
            double runT[NCH];
            double2 runS[NPC];
            int fa[NCH], fb[NCH], fc[NCH];              // this lane's function descriptors, for the step's segment ends (the ket
#pragma unroll                                          // code's accumulators are dead here: registers are free)
            for (int ch = 0; ch < NCH; ++ch) { fa[ch] = s_fa[ch * 32 + lane]; fb[ch] = s_fb[ch * 32 + lane]; fc[ch] = kPacked ? s_fc[ch * 32 + lane] : 0; }
            {
                const int slot = kcur - kdone;
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) { const int f = ch * 32 + lane; runT[ch] = f < nf ? s_acc[slot * nf + f] : 0.0; }
#pragma unroll
                for (int i = 0; i < NPC; ++i) { const int sp = i * 32 + lane; runS[i] = sp < np ? s_sseg2[sp] : make_double2(0.0, 0.0); }
            }
            // D1, lane = slot pair: ONE pass over the step's chunk columns (loads in bursts of 16, every branch uniform); at a
            // segment end the segment's sum replaces the column of its last chunk, where the stage below reads it
#pragma unroll
            for (int i = 0; i < NPC; ++i) {
                const int sp = i * 32 + lane;
                if (sp < np) {
                    double2* row = s_tile + sp * kTileStride;
                    double2 r = runS[i];
                    for (int c0 = 0; c0 < cnt; c0 += 16) {
                        double2 d[16];
#pragma unroll
                        for (int k = 0; k < 16; ++k) d[k] = c0 + k < cnt ? row[c0 + k] : make_double2(0.0, 0.0);
#pragma unroll
                        for (int k = 0; k < 16; ++k) {
                            r.x += d[k].x; r.y += d[k].y;
                            if ((smask >> (c0 + k)) & 1u) { row[c0 + k] = r; r = make_double2(0.0, 0.0); }
                        }
                    }
                    runS[i] = r;                                         // the segment that is still open behind the step
                }
            }
            __syncwarp();
            // D2, lane = orbital function, segment end by segment end
            for (unsigned rem = smask; rem; rem &= rem - 1u) {
                const int jb = __ffs(rem) - 1;                           // chunk jb ends a (t, c) segment
                const int cseg = (int)(s_step[jb].x >> 24);
                const double* bra;                                     // (shared-memory loads for the specialised kernels)
                if constexpr (Spec::kStatic) { if (Spec::kBraSmem) bra = s_bra + cseg * nsb; else bra = L.bra + cseg * nsb; }
                else bra = bra_tab + cseg * bra_stride;
                const char* Sb = (const char*)(s_tile + jb);             // column jb of the tile: the segment's sums
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) {
                    if (kPacked) {
                        const int ia = fa[ch], ib = fb[ch];
                        double v = bra[ia & 255] * *(const double*)(Sb + (ib & 65535));
                        if (Spec::terms(ch) > 1) v = fma(bra[(ia >> 8) & 255], *(const double*)(Sb + ((unsigned)ib >> 16)), v);
                        if (Spec::terms(ch) > 2) v = fma(bra[ia >> 16], *(const double*)(Sb + fc[ch]), v);
                        runT[ch] += v;
                    } else {
                        const int fav = fa[ch], sa = fav & 65535, sb = fb[ch], nM = fav >> 16;
                        double v = 0.0;
                        if constexpr (Spec::kStatic && Spec::MAXM <= 12) {
                            // all bra harmonics of the function first (they may come from global memory: one latency, not nM)
                            double bv[Spec::MAXM];
#pragma unroll
                            for (int i = 0; i < Spec::MAXM; ++i) bv[i] = i < nM ? bra[sa + i] : 0.0;
#pragma unroll
                            for (int i = 0; i < Spec::MAXM; ++i) if (i < nM) v = fma(bv[i], *(const double*)(Sb + tile_byte(sb + i)), v);
                        } else {
                            for (int i = 0; i < nM; ++i) v = fma(bra[sa + i], *(const double*)(Sb + tile_byte(sb + i)), v);
                        }
                        runT[ch] += v;
                    }
                }
                if (!((tmask >> jb) & 1u)) continue;
                // node jb also ends target t: its sums are complete; kRowBatch finished targets are written together
                {
                    const int slot = kcur - kdone;
                    const int tcell = (int)(s_step[jb].x & 262143u);
                    const int ic = L.mg_Nq ? (int)__umulhi((unsigned)tcell, L.mg_Nq) : tcell, jc = tcell - ic * L.Nq;
                    // (d_i dbar_j d_i' dbar_j')^(-1/2), folded into the sums; rsqrt is within 2 ulp of the oracle's 1/sqrt
                    const double nrm = rsqrt(s_cell->dsrc * (s_dp ? s_dp[ic] * s_dq[jc] : cell_norm(L.pe, ic, L.norm) * cell_norm(L.qe, jc, L.norm)));
                    if constexpr (kMode == 2) {
                        double* __restrict__ Ah = vals + (s_cell->rbase + kcur) * (int64_t)L.op_stride + L.op_off;
#pragma unroll
                        for (int ch = 0; ch < NCH; ++ch) {
                            const int f = ch * 32 + lane;
                            if (f < nf) Ah[f] = runT[ch] * nrm;
                            runT[ch] = 0.0;
                        }
                        ++kcur; kdone = kcur;                              // (nothing waits in the row batch)
                    } else {
#pragma unroll
                        for (int ch = 0; ch < NCH; ++ch) {
                            const int f = ch * 32 + lane;
                            if (f < nf) s_acc[slot * nf + f] = runT[ch] * nrm;
                            runT[ch] = 0.0;
                        }
                        if (lane == 0) s_hcol[slot] = tcell * L.n_ch;
                        ++kcur;
                        __syncwarp();
                        if (kcur - kdone == kRowBatch) { write_rows(kdone, kRowBatch); kdone = kcur; }
                    }
                }
            }
            {   // park the running sums
                const int slot = kcur - kdone;
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) { const int f = ch * 32 + lane; if (f < nf) s_acc[slot * nf + f] = runT[ch]; }
#pragma unroll
                for (int i = 0; i < NPC; ++i) { const int sp = i * 32 + lane; if (sp < np) s_sseg2[sp] = runS[i]; }
            }
            __syncwarp();
            fetch((base >> 5) + 2, (base >> 5) & 1);
        }
        if (kcur > kdone) write_rows(kdone, kcur - kdone);
    }
}

}  // namespace pm
