// pm_device.cuh — device-side view of a lattice and the primitives every kernel shares:
// node generation (step a3), kinematic map (a4), branch-free cell location (a5), per-source-cell hit
// bitset and ranks (a6).  SURVEY.md sec. 8(a); DESIGN.md sec. 3.1 gives the operation order that
// makes a node land in the same cell as in the CPU oracle: every operation from the Gauss node to
// p', q' is a single IEEE-754 double operation issued through __dadd_rn/__dmul_rn/__dsqrt_rn, which
// the compiler never contracts into FMAs (north_star: "FMA contraction off").
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pm {

struct DevLattice {
    int Np, Nq, n_ch, n_p, n_q, n_x, nnode, n_cells, n_words, pe_pad, qe_pad;
    int totcoup, n_slot, n_fun, lmax, ny;
    const double *pe, *qe;                      // edges padded with +inf to pe_pad / qe_pad (powers of two)
    const long long *thr_p, *thr_q;             // bit patterns of sqrt_threshold(edge), same padding (+inf)
    const double *tp, *wp, *tq, *wq, *tx, *wx;  // Gauss-Legendre rules on [-1,1]
    const double *sx;                           // sqrt(1-x^2) per x-node
    const int *cl_off, *cl, *o_alpha;           // coupled lists; o_alpha[o] = alpha of output o
    const double *bra;                          // [n_x][n_slot]
    const int *kt_off, *kt_ip, *kt_iq; const double *kt_c;
    const int4 *fun;                            // (sa0, sb0, nM, L)
    const int *ot_off, *ot_f; const double *ot_c;
    const double *ya, *yb, *ydiag;
};

// number of edges <= v, minus one; e has `pad` (power of two) entries, the tail filled with +inf
__device__ __forceinline__ int locate(const double* __restrict__ e, int pad, double v)
{
    int lo = 0;
#pragma unroll 1
    for (int s = pad >> 1; s > 0; s >>= 1) lo += (e[lo + s - 1] <= v) ? s : 0;
    lo += (e[lo] <= v) ? 1 : 0;          // entries beyond N+1 are +inf, so lo <= N+1
    return lo - 1;
}

struct CellGeom { double cp, hp, cq, hq; };

__device__ __forceinline__ CellGeom cell_geom(const double* pe, const double* qe, int i, int j)
{
    CellGeom g;
    g.cp = __dmul_rn(0.5, __dadd_rn(pe[i], pe[i + 1])); g.hp = __dmul_rn(0.5, __dsub_rn(pe[i + 1], pe[i]));
    g.cq = __dmul_rn(0.5, __dadd_rn(qe[j], qe[j + 1])); g.hq = __dmul_rn(0.5, __dsub_rn(qe[j + 1], qe[j]));
    return g;
}

// DESIGN.md sec. 3.1, exactly:  p = cp + hp*t_a ; q = cq + hq*t_b ; x = t_c ; pq = p*q
//   P2 = (0.25*(p*p) + 0.5625*(q*q)) + 0.75*(pq*x) ;  Q2 = ((p*p) + 0.25*(q*q)) - pq*x ; clamp at 0 ; sqrt
__device__ __forceinline__ void map_node(const CellGeom& g, double ta, double tb, double tc,
                                         double& p, double& q, double& pp, double& qq)
{
    p = __dadd_rn(g.cp, __dmul_rn(g.hp, ta));
    q = __dadd_rn(g.cq, __dmul_rn(g.hq, tb));
    const double pq = __dmul_rn(p, q), p2 = __dmul_rn(p, p), q2 = __dmul_rn(q, q), pqx = __dmul_rn(pq, tc);
    double P2 = __dadd_rn(__dadd_rn(__dmul_rn(0.25, p2), __dmul_rn(0.5625, q2)), __dmul_rn(0.75, pqx));
    double Q2 = __dsub_rn(__dadd_rn(p2, __dmul_rn(0.25, q2)), pqx);
    P2 = P2 < 0.0 ? 0.0 : P2;
    Q2 = Q2 < 0.0 ? 0.0 : Q2;
    pp = __dsqrt_rn(P2);
    qq = __dsqrt_rn(Q2);
}

// target cell of a mapped node, or -1 (outside the grid, or p' = 0 / q' = 0): readings R5, R6
__device__ __forceinline__ int target_cell(const double* s_pe, int pe_pad, int Np, const double* s_qe, int qe_pad, int Nq,
                                           double pp, double qq)
{
    const int ic = locate(s_pe, pe_pad, pp), jc = locate(s_qe, qe_pad, qq);
    const bool ok = (ic >= 0) & (ic < Np) & (jc >= 0) & (jc < Nq) & (pp != 0.0) & (qq != 0.0);
    return ok ? ic * Nq + jc : -1;
}

// In-place exclusive scan of n ints in shared memory by the whole block; returns the total.
// `scratch` holds blockDim.x + 1 ints.  All threads must call.
__device__ inline int block_exclusive_scan(int* data, int n, int* scratch)
{
    const int T = blockDim.x, t = threadIdx.x;
    const int chunk = (n + T - 1) / T;
    const int b = min(t * chunk, n), e = min(b + chunk, n);
    int s = 0;
    for (int k = b; k < e; ++k) s += data[k];
    scratch[t] = s;
    __syncthreads();
    if (t < 32) {
        int carry = 0;
        for (int base = 0; base < T; base += 32) {
            int v = scratch[base + t], x = v;
#pragma unroll
            for (int d = 1; d < 32; d <<= 1) { int y = __shfl_up_sync(0xffffffffu, x, d); if (t >= d) x += y; }
            scratch[base + t] = carry + x - v;
            carry += __shfl_sync(0xffffffffu, x, 31);
        }
        if (t == 0) scratch[T] = carry;
    }
    __syncthreads();
    int run = scratch[t];
    for (int k = b; k < e; ++k) { int v = data[k]; data[k] = run; run += v; }
    const int total = scratch[T];
    __syncthreads();
    return total;
}

}  // namespace pm
