// pm_device.cuh — device-side view of a lattice and the primitives every kernel shares:
// node generation (step a3), kinematic map (a4), branch-free cell location (a5), per-source-cell hit
// bitset and ranks (a6).  SURVEY.md sec. 8(a); DESIGN.md sec. 3.1 gives the operation order that
// makes a node land in the same cell as in the CPU oracle: every operation from the Gauss node to
// p'^2, q'^2 is a single IEEE-754 double operation issued through __dadd_rn/__dmul_rn, which the compiler
// never contracts into FMAs (north_star: "FMA contraction off").  The oracle then takes p' = sqrt(p'^2) and
// compares it with the edges; here p'^2 is compared with sqrt_threshold(edge) (pm_tables.hpp), the smallest
// double whose correctly rounded square root reaches the edge — the same decision without the square root.
#pragma once
#ifdef __CUDACC_RTC__                  // compiled at run time by NVRTC (pm_jit.cpp): no host headers there
typedef int int32_t;
typedef unsigned int uint32_t;
typedef long long int64_t;
typedef unsigned long long uint64_t;
typedef unsigned long size_t;
namespace std {
template <bool B> struct pm_bool_constant { static constexpr bool value = B; };
typedef pm_bool_constant<true> true_type;
typedef pm_bool_constant<false> false_type;
template <class T, T v> struct integral_constant { static constexpr T value = v; };
}
#else
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>
#endif

namespace pm {

struct DevLattice {
    int Np, Nq, n_ch, n_p, n_q, n_x, nnode, n_cells, n_words, pe_pad, qe_pad;
    int totcoup, n_slot, n_fun, lmax, ny;       // n_slot / n_fun: ket slots and orbital functions of THIS column-channel group
    int norm;                                   // cell normalisation: 0 reading A (widths), 1 reading B (p^2 dp measure) — DESIGN.md R2
    int n_out, n_bra;                           // outputs (alpha, alpha') of this group; bra slots of the whole channel set
    int op_stride, op_off;                      // per-pair sums form (pm_fill.cuh, mode 2): doubles per hit cell pair, this group's first
    int n_out1, n_out2, n_out3;                       // the group's rows are ordered by the most terms of their outputs: outputs of rows with at most 1 / 2 / 3
    unsigned mg_npq, mg_nq, mg_Nq;              // ceil(2^32 / d) for d = n_p*n_q, n_q, Nq: exact division of node and cell ids (x*d < 2^32)
    const double *pe, *qe;                      // edges, Np+1 / Nq+1 entries (padded with +inf to pe_pad / qe_pad)
    const double *thr_p, *thr_q;                // sqrt_threshold(edge), padded with +inf to a power of two
    const unsigned short *bk_p, *bk_q;          // kBuckets entries each: first threshold a value of that bucket can meet
    int bk_hmin_p, bk_sh_p, bk_hmin_q, bk_sh_q; // bucket(v) = clamp((hi32(v) - hmin) >> sh, 0, kBuckets-1)
    int bk_kmax;                                // most thresholds any bucket of either axis holds
    const double *tp, *wp, *tq, *wq, *tx, *wx;  // Gauss-Legendre rules on [-1,1]
    const double *sx;                           // sqrt(1-x^2) per x-node
    const int *cl_off, *cl, *o_alpha;           // coupled lists of the whole set; o_alpha[o] = alpha of global output o
    const int *g_alpha, *g_m, *g_ap;            // outputs of this group: row channel, position in the row's coupled list, column channel
    const double *bra;                          // [n_x][n_bra + 1], every row ends with a zero slot
    const int *kt_off, *kt_ip, *kt_iq; const double *kt_c;
    const int4 *fun;                            // (sa0, sb0, nM, L)
    const int *ot_off, *ot_f; const double *ot_c;
    const double *ya, *yb, *ydiag;
};

// Per-source-cell node lists written by the pattern pass and read by the fill pass (library-owned scratch), stride
// nnode per source cell: for every node that hit the grid, in the order (target cell, node id),
//   key   = target cell << 14 | node id     (node id m = c*(n_p*n_q) + a*n_q + b < 2^14, cell < 2^18).
// The rank of a target among the source cell's hit cells is the number of target changes before it.
// Chunks: the sorted list cut into runs of at most chunk_len consecutive nodes that never cross a (target, x-node)
// segment; one lane of the fill kernel sums the ket harmonics of one chunk in registers (pm_fill.cuh).  A chunk carries
// the (a, b) indices of its nodes, so the fill reads no node key on its per-node path:
//   chunk.x = target cell | (len - 1) << 18 | ends a segment << 22 | ends a target << 23 | x-node c << 24
//   chunk.y = ab_0 | ab_1 << ab_bits | ...        (ab = a*n_q + b < 2^ab_bits, len * ab_bits <= 32)
// (cell < 2^18, len <= 16, c < PM_MAX_ORDER = 64)
struct NodeLists {
    unsigned* key;              // [n_blk][nnode]
    int* ntot;                  // [n_blk] nodes on the grid
    int* hits;                  // [n_blk] hit cells H
    uint2* chunk;               // [n_blk][nnode] (at most one chunk per node)
    int* nchunk;                // [n_blk]
    int chunk_len;              // longest chunk the pattern pass cuts: min(wanted, 32 / ab_bits)
    int ab_bits;                // bits of one (a, b) index in chunk.y
};
constexpr int kMaxChunkLen = 16;

struct CellGeom { double cp, hp, cq, hq; };

__device__ __forceinline__ CellGeom cell_geom(const double* pe, const double* qe, int i, int j)
{
    CellGeom g;
    g.cp = __dmul_rn(0.5, __dadd_rn(pe[i], pe[i + 1])); g.hp = __dmul_rn(0.5, __dsub_rn(pe[i + 1], pe[i]));
    g.cq = __dmul_rn(0.5, __dadd_rn(qe[j], qe[j + 1])); g.hq = __dmul_rn(0.5, __dsub_rn(qe[j + 1], qe[j]));
    return g;
}

// node id m -> (c, a, b), m = c*npq + a*n_q + b, by multiply-high with precomputed magic numbers (m*d < 2^32)
__device__ __forceinline__ void split_node(const DevLattice& L, int m, int& c, int& a, int& b)
{
    const int npq = L.n_p * L.n_q;
    c = L.mg_npq ? (int)__umulhi((unsigned)m, L.mg_npq) : m;        // magic 0 encodes divisor 1
    const int ab = m - c * npq;
    a = L.mg_nq ? (int)__umulhi((unsigned)ab, L.mg_nq) : ab;
    b = ab - a * L.n_q;
}

// DESIGN.md sec. 3.1, exactly:  p = cp + hp*t_a ; q = cq + hq*t_b ; x = t_c ; pq = p*q
//   P2 = (0.25*(p*p) + 0.5625*(q*q)) + 0.75*(pq*x) ;  Q2 = ((p*p) + 0.25*(q*q)) - pq*x ; clamp at 0
__device__ __forceinline__ void map_pq_sq(double p, double q, double tc, double& P2, double& Q2);
__device__ __forceinline__ void map_node_sq(const CellGeom& g, double ta, double tb, double tc,
                                            double& p, double& q, double& P2, double& Q2)
{
    p = __dadd_rn(g.cp, __dmul_rn(g.hp, ta));
    q = __dadd_rn(g.cq, __dmul_rn(g.hq, tb));
    map_pq_sq(p, q, tc, P2, Q2);
}
// the map from a node's (p, q, x) on
__device__ __forceinline__ void map_pq_sq(double p, double q, double tc, double& P2, double& Q2)
{
    const double pq = __dmul_rn(p, q), p2 = __dmul_rn(p, p), q2 = __dmul_rn(q, q), pqx = __dmul_rn(pq, tc);
    P2 = __dadd_rn(__dadd_rn(__dmul_rn(0.25, p2), __dmul_rn(0.5625, q2)), __dmul_rn(0.75, pqx));
    Q2 = __dsub_rn(__dadd_rn(p2, __dmul_rn(0.25, q2)), pqx);
    P2 = P2 < 0.0 ? 0.0 : P2;
    Q2 = Q2 < 0.0 ? 0.0 : Q2;
}

constexpr int kBuckets = 1024;

// Number of thresholds <= v, minus one.  The upper 32 bits of a non-negative double grow with its value, so
// bucket(v) = clamp((hi32(v) - hmin) >> sh) is monotone: every threshold in a lower bucket is < v and start[bucket]
// counts exactly those; the few thresholds of v's own bucket are compared one by one (thr ends with +inf).
__device__ __forceinline__ int locate(const double* __restrict__ thr, const unsigned short* __restrict__ start, int hmin, int sh,
                                      double v)
{
    const int b = max(0, min(kBuckets - 1, (__double2hiint(v) - hmin) >> sh));
    int i = start[b];
    while (thr[i] <= v) ++i;
    return i - 1;
}

// The same count when no bucket holds more than K thresholds: K independent comparisons instead of a dependent scan
// (the tables carry K entries of +inf behind the last threshold).
template <int K>
__device__ __forceinline__ int locate_k(const double* __restrict__ thr, const unsigned short* __restrict__ start, int hmin, int sh, double v)
{
    const int b = max(0, min(kBuckets - 1, (__double2hiint(v) - hmin) >> sh));
    const int i = start[b];
    int c = 0;
#pragma unroll
    for (int k = 0; k < K; ++k) c += (thr[i + k] <= v) ? 1 : 0;
    return i + c - 1;
}

constexpr int kLocK = 4;

struct Locator { const double *thr_p, *thr_q; const unsigned short *bk_p, *bk_q; int hmin_p, sh_p, hmin_q, sh_q, Np, Nq; };

// target cell of a mapped node, or -1 (outside the grid, or p' = 0 / q' = 0): readings R5, R6.  sqrt(y) = 0 <=> y = 0.
template <bool kFast>
__device__ __forceinline__ int target_cell_sq(const Locator& lc, double P2, double Q2)
{
    const int ic = kFast ? locate_k<kLocK>(lc.thr_p, lc.bk_p, lc.hmin_p, lc.sh_p, P2) : locate(lc.thr_p, lc.bk_p, lc.hmin_p, lc.sh_p, P2);
    const int jc = kFast ? locate_k<kLocK>(lc.thr_q, lc.bk_q, lc.hmin_q, lc.sh_q, Q2) : locate(lc.thr_q, lc.bk_q, lc.hmin_q, lc.sh_q, Q2);
    const bool ok = (ic >= 0) & (ic < lc.Np) & (jc >= 0) & (jc < lc.Nq) & (P2 != 0.0) & (Q2 != 0.0);
    return ok ? ic * lc.Nq + jc : -1;
}

}  // namespace pm
