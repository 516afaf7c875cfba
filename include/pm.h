/* pm.h — C ABI of libpm: construction of the sparse particle-permutation matrix P0 of the Faddeev
 * equation in the three-body lattice (free wave-packet) basis on one NVIDIA B200 (sm_100a).
 *
 * What is computed (arXiv:1508.07441; line numbers refer to PAPER.md):
 *   [P0]_{ij alpha, i'j' alpha'} = <X_ij^alpha | P | X_i'j'^alpha'>,  P = P12 P23 + P13 P23   (eq. 18;
 *   eq. 20-21), an integral of the partial-wave kernel  sum g * I  (eq. 22) over the
 *   lattice cells D_ij = D_i x Dbar_j (L154), stored in CSR (arrays B, C, W of L339).
 *   Evaluation scheme (BASELINE.json north_star; written out in DESIGN.md sec. 3): a tensor Gauss-Legendre rule
 *   in (p, q, x = cos(p^,q^)) inside every source cell; each node is mapped by
 *       p'^2 = p^2/4 + 9 q^2/16 + (3/4) p q x ,   q'^2 = p^2 + q^2/4 - p q x ,
 *   located in its target cell (half-open cells [e_k, e_k+1)), and contributes
 *       w * p q/(p' q') * G_{alpha alpha'}(p,q,x) / sqrt(d_i dbar_j d_i' dbar_j').
 *
 * Index convention (part of the contract — the pattern is compared bit-exactly with the oracle):
 *   source cell  cell = i*Nq + j ; row  r = cell*n_ch + alpha ; column c = cell'*n_ch + alpha' ; 0-based ;
 *   columns ascending within a row ; rowptr is standard CSR (int64), colidx int32, values double.
 *   A row (cell, alpha) holds, for every hit cell in ascending order, every alpha' coupled to alpha in ascending
 *   order: the pattern is structural (hit cells x integer channel mask), never thresholded by value.
 *
 * Memory: pointers named d_* are DEVICE pointers on the current CUDA device, h_* / unprefixed are HOST pointers.
 * The library owns only the handle and its small device tables; every output buffer belongs to the caller and is
 * never freed or reallocated here.  All entry points return a status code; none throws or aborts.  There is no
 * CPU fallback: without a usable sm_100 device the compute calls return PM_ERR_DEVICE.
 * Kernels are launched on the caller's stream (`cuda_stream` is a cudaStream_t cast to void*; NULL = default
 * stream) and are asynchronous, except that a call which returns a host scalar (nnz) synchronises that stream.
 */
#ifndef PM_H_
#define PM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pm_lattice pm_lattice;                        /* opaque, owned by the library */

/* A spin-angular channel alpha = {(l s) j t ; (lam 1/2) I} ('Gamma alpha beta').
 * I2 = 2*I.  Spinless bosons: s = t = 0, j = l, I2 = 2*lam. */
typedef struct { int32_t l, s, j, t, lam, I2; } pm_channel;

enum {
    PM_OK = 0, PM_ERR_ARG = -1, PM_ERR_GRID = -2, PM_ERR_CHANNEL = -3, PM_ERR_ORDER = -4, PM_ERR_CUDA = -5,
    PM_ERR_NOMEM = -6, PM_ERR_STATE = -7, PM_ERR_OVERFLOW = -8, PM_ERR_DEVICE = -9
};
enum { PM_FERMION_ISOSPIN = 0, PM_SPINLESS_BOSON = 1 };      /* `statistics` */
enum { PM_NORM_WIDTH = 0, PM_NORM_P2 = 1 };                  /* cell normalisation, pm_lattice_set_normalisation */
enum { PM_MAX_CHANNELS = 64, PM_MAX_ORDER = 64, PM_MAX_L = 12 };
enum { PM_STATIC_MAX_M = 65536 };                            /* largest matrix dimension pm_rotate_apply_static takes */

/* Create a lattice (host work only: validation, Gauss-Legendre rules, recoupling tables — PAPER.md:L247-256
 * step 1, 'calculation of algebraic coefficients g').
 *   p_edges[Np+1], q_edges[Nq+1] : host, finite, strictly increasing, first edge >= 0   (cells D_i, Dbar_j, L146)
 *   ch[n_ch]                     : host, 1 <= n_ch <= PM_MAX_CHANNELS, distinct, each consistent with
 *                                  (J2 = 2J, parity = +-1, T2 = 2T) and, for fermions, (-1)^(l+s+t) = -1
 *   n_p, n_q, n_x                : Gauss-Legendre orders in p, q, x, each 1..PM_MAX_ORDER; n_p*n_q*n_x <= 16384; Np*Nq <= 262144
 * Errors: PM_ERR_ARG (null pointers), PM_ERR_GRID, PM_ERR_CHANNEL, PM_ERR_ORDER, PM_ERR_OVERFLOW (M >= 2^31). */
int32_t pm_lattice_create(const double* p_edges, int32_t Np, const double* q_edges, int32_t Nq,
                          const pm_channel* ch, int32_t n_ch,
                          int32_t J2, int32_t parity, int32_t T2, int32_t statistics,
                          int32_t n_p, int32_t n_q, int32_t n_x, pm_lattice** out);
int32_t pm_lattice_destroy(pm_lattice* lat);

/* A lattice for ANOTHER channel set (another J^pi) on the grids, orders and rules of `base` (
 * PAPER.md:L374 "up to 62 channels", L394 + Table 1 "all states ... up to J_max = 17/2").  The two share, by reference
 * count, everything that does not depend on the channels: device tables of the grids and the node lists of the pattern
 * pass.  pm_build_reuse on any lattice of such a group reuses the node lists the group already holds for that cell
 * range, so a sweep over J^pi maps and sorts the quadrature nodes once.  pm_lattice_set_rule on one member changes the
 * rule of all.  Each member is destroyed with pm_lattice_destroy, in any order.  Errors as pm_lattice_create. */
int32_t pm_lattice_attach(pm_lattice* base, const pm_channel* ch, int32_t n_ch, int32_t J2, int32_t parity, int32_t T2,
                          int32_t statistics, pm_lattice** out);

/* M = n_ch*Np*Nq (matrix dimension) and the number of lattice cells. */
int32_t pm_lattice_dims(const pm_lattice* lat, int64_t* M, int32_t* n_cells);

/* Read / replace the quadrature rule of one axis (0 = p, 1 = q, 2 = x) on [-1,1].  `nodes`, `weights`: host,
 * length = that axis' order.  set_rule lets a caller feed the very arrays it gives to another implementation
 * (reading R12); nodes must be strictly increasing inside (-1,1); the x-rule must be symmetric. */
int32_t pm_lattice_rule(const pm_lattice* lat, int32_t axis, double* nodes, double* weights);
int32_t pm_lattice_set_rule(pm_lattice* lat, int32_t axis, const double* nodes, const double* weights);

/* Normalisation of the lattice states (eq. 21, is garbled there; reading R2):
 *   PM_NORM_WIDTH (default, reading A): radial states normalised to delta(p - p'), cell norm B_k = e_{k+1} - e_k;
 *                 node weight w * pq/(p'q'), prefactor (B_i Bbar_j B_i' Bbar_j')^(-1/2)
 *   PM_NORM_P2    (reading B): states normalised in the p^2 dp measure, B_k = (e_{k+1}^3 - e_k^3)/3; node weight w * p^2 q^2.
 * Both bases are orthonormal; the pattern does not depend on the choice.  Takes effect at the next pm_fill / pm_build. */
int32_t pm_lattice_set_normalisation(pm_lattice* lat, int32_t normalisation);

/* Channel tables (host out): coupled[n_ch*n_ch] (1 iff the integer selection rules couple alpha, alpha');
 * *n_functions = number of distinct orbital functions A^L_{l lam, l' lam'} the fill evaluates per node. */
int32_t pm_lattice_coupling(const pm_lattice* lat, uint8_t* coupled, int32_t* n_functions);

/* Pattern pass (the paper's step 2a 'pre-selection') for the rows of source cells
 * [cell_begin, cell_end):
 * The pass bins every quadrature node of the range once and keeps, in library-owned device memory, the node lists
 * sorted by target cell (about 12 bytes per node: keys and chunk words); pm_fill of the same range reads them.  Calling with d_colidx = NULL
 * (count) and then with d_colidx for the same range maps the nodes only once.
 *   d_rowptr : device, (cell_end-cell_begin)*n_ch + 1 int64, block-local (d_rowptr[0] = 0)
 *   d_colidx : device, nnz int32 GLOBAL column indices — or NULL to count only (d_rowptr is still written)
 *   colidx_capacity : number of int32 d_colidx can hold (ignored when d_colidx is NULL); if nnz exceeds it
 *                     nothing is written to d_colidx and PM_ERR_OVERFLOW is returned (*nnz_host is valid)
 *   nnz_host : host, receives the block's nnz (the stream is synchronised for this)                     */
int32_t pm_pattern(pm_lattice* lat, int32_t cell_begin, int32_t cell_end,
                   int64_t* d_rowptr, int32_t* d_colidx, int64_t colidx_capacity,
                   int64_t* nnz_host, void* cuda_stream);

/* Fill pass (step 2b 'calculation of nonzero elements'): values of the block
 * whose d_rowptr was produced by the LAST pm_pattern call on this lattice, for the same [cell_begin, cell_end)
 * (PM_ERR_STATE otherwise: the fill reads that call's node lists).  d_vals: device, nnz doubles,
 * every entry is written exactly once; sums are formed in a fixed order (bitwise reproducible run to run). */
int32_t pm_fill(pm_lattice* lat, int32_t cell_begin, int32_t cell_end,
                const int64_t* d_rowptr, double* d_vals, void* cuda_stream);

/* Pattern and fill of one block in one call: the pattern pass up to rowptr and nnz, then ONE kernel writes both the
 * column index and the value of every nonzero — the separate column kernel of pm_pattern is not run.  The kernels are
 * queued back to back; the host reads nnz back once, after the fill has been queued (the capacity check runs on the device).  Same results as pm_pattern + pm_fill, bit for bit.
 *   d_rowptr, d_colidx, d_vals : device, as in pm_pattern / pm_fill;  capacity : entries d_colidx and d_vals can hold;
 *   PM_ERR_OVERFLOW (with *nnz_host valid, nothing written to d_colidx / d_vals) if nnz exceeds it. */
int32_t pm_build(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                 int64_t capacity, int64_t* nnz_host, void* cuda_stream);

/* pm_build without any host synchronisation: the pattern pass, the capacity check and the fill are queued on the stream
 * back to back; nnz stays on the device until pm_build_wait.  If the block's nnz exceeds `capacity` the fill kernel
 * writes nothing (checked on the device) and pm_build_wait returns PM_ERR_OVERFLOW.  reuse_lists != 0: as pm_build_reuse.
 * At most one un-waited build per lattice group: the next pattern / build call on the group waits for it first. */
int32_t pm_build_async(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                       int64_t capacity, int32_t reuse_lists, void* cuda_stream);
/* Waits for the pattern pass of the last pm_build_async (not for its fill kernel) and returns the block's nnz. */
int32_t pm_build_wait(pm_lattice* lat, int64_t* nnz_host);

/* pm_build that skips the node map and sort when the lattice group (pm_lattice_attach) already holds the node lists of
 * [cell_begin, cell_end) from its last pattern / build call; otherwise identical to pm_build, bit for bit. */
int32_t pm_build_reuse(pm_lattice* lat, int32_t cell_begin, int32_t cell_end, int64_t* d_rowptr, int32_t* d_colidx, double* d_vals,
                       int64_t capacity, int64_t* nnz_host, void* cuda_stream);

/* ---- Sharded build over several GPUs (the elements are "calculated ... fully
 * independently from each other").  Rows of different source cells are independent, so every rank builds a contiguous
 * range of source cells; the only exchange is one all-gather of the per-rank nnz (8 bytes), done by the caller.
 *   pm_pattern_cell_hits : hit cells of every source cell of the last pm_pattern / pm_build call, h_hits[cell_end-cell_begin] (HOST out)
 *   pm_partition_cells   : host only.  cuts[n_parts+1] with cuts[0] = 0, cuts[n_parts] = n_cells: contiguous ranges of
 *                          (almost) equal weight sum(hits[k] + cell_cost); deterministic, identical on every rank
 *   pm_rowptr_offset     : d_rowptr[0..n) += offset (block-local row pointers -> global ones)                         */
int32_t pm_pattern_cell_hits(pm_lattice* lat, int32_t* h_hits, void* cuda_stream);
int32_t pm_partition_cells(const int32_t* hits, int32_t n_cells, double cell_cost, int32_t n_parts, int32_t* cuts);
int32_t pm_rowptr_offset(int64_t* d_rowptr, int64_t n, int64_t offset, void* cuda_stream);

/* y = P0 x for the WHOLE lattice without reading column indices: the columns of row (cell, alpha) are implied by the
 * hit cells of the source cell and the coupled-channel list, which the lattice keeps from its last pm_pattern /
 * pm_build call over the whole lattice [0, n_cells) (PM_ERR_STATE otherwise).  d_rowptr, d_vals: that call's outputs.
 * Reads 8 instead of 12 bytes per nonzero; the same bits as pm_spmv. */
int32_t pm_spmv_implicit(pm_lattice* lat, const int64_t* d_rowptr, const double* d_vals, const double* d_x, double* d_y,
                         void* cuda_stream);

/* Device time of the last fill kernel launched for this lattice (by pm_fill, pm_build or pm_build_host), from CUDA
 * events recorded around it on its stream; waits for that kernel.  PM_ERR_STATE before the first fill. */
int32_t pm_last_fill_ms(pm_lattice* lat, float* ms);

/* pm_rotate_apply without any allocation, for callers that cannot call cudaMalloc (CUDA graph capture, serving loops,
 * harnesses that forbid it): d_out = O (P0 (O^T x)) as pm_rotate_apply, the two intermediate vectors in a static device
 * array of the library (2 * PM_STATIC_MAX_M doubles = 1 MiB per GPU that loads libpm, held until exit) instead of d_work.
 *   - M = n_ch*Np*Nq <= PM_STATIC_MAX_M, else PM_ERR_OVERFLOW (use pm_rotate_apply with your own d_work);
 *   - d_colidx is required (PM_ERR_ARG if NULL): the column-free SpMV builds library scratch lazily;
 *   - the lattice's device tables must already exist on the current device — any earlier pm_pattern / pm_build /
 *     pm_block_apply call on it creates them — else PM_ERR_STATE: this call never allocates or frees;
 *   - all calls share the array (it keeps the last call's contents; both vectors are overwritten before use): calls that
 *     overlap on the GPU — other streams, other host threads — RACE; serialise them.
 * Asynchronous on `cuda_stream`; the same kernels, hence the same bits, as pm_rotate_apply with a column array. */
int32_t pm_rotate_apply_static(pm_lattice* lat, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                               const double* d_O, const double* d_x, double* d_out, void* cuda_stream);

/* ---- The operator form of P0: the per-pair sums -----------------------------------------------
 * Every nonzero of a hit cell pair (source cell, k-th hit cell) is a combination, with the recoupling coefficients c^L of
 * eq. (22), of at most four of the pair's sums over quadrature nodes of the orbital functions (140 for 26 channels, 546
 * for 62): 8 * n_functions bytes per pair instead of 8 bytes per nonzero (580 / 3694 per pair) — 1.7 GB instead of 7.1 GB
 * on configs[4].  What the paper's iterations need of P0 is its action on a vector.
 *   pm_operator_build : the sums of the WHOLE lattice into library-owned device memory, from the node lists of the last
 *                       pm_pattern / pm_build call over [0, n_cells) (PM_ERR_STATE otherwise; PM_ERR_STATE too when NVRTC
 *                       is unavailable: the sums are written by run-time specialised kernels).  *n_pairs, *bytes (host,
 *                       may be NULL): hit cell pairs and the size of the sums.  Synchronises the stream once.
 *   pm_operator_apply : d_y = P0 d_x (M doubles each, distinct buffers) straight from the sums; asynchronous; agrees with
 *                       pm_spmv on the CSR to rounding (another summation order), bitwise reproducible.
 * A new pattern pass or pm_lattice_set_normalisation invalidates the sums (PM_ERR_STATE from pm_operator_apply). */
int32_t pm_operator_build(pm_lattice* lat, int64_t* n_pairs, int64_t* bytes, void* cuda_stream);
int32_t pm_operator_apply(pm_lattice* lat, const double* d_x, double* d_y, void* cuda_stream);

/* y = A x for a CSR block (convenience check only): n_rows rows, GLOBAL columns. */
int32_t pm_spmv(pm_lattice* lat, int64_t n_rows, const int64_t* d_rowptr, const int32_t* d_colidx,
                const double* d_vals, const double* d_x, double* d_y, void* cuda_stream);

/* ---- The iteration step that consumes P0 (eq. 24) -------------------
 * K = O P0 V~1 G1 : G1 diagonal, P0 "highly sparse" (the CSR built above, whole lattice, global columns), O and
 * V~1 = O^T V1 "block matrices with the block dimension (N x N)": one (Np x Np) block per channel alpha acting on
 * the pair index i for fixed (j, alpha).  The paper keeps the four factors in memory and applies them one after the
 * other (L239-241); its iterations are what remains its bottleneck after P0 moved to the GPU (L408-410).
 *
 * pm_block_apply : d_out[(i,j,a)] = sum_i' B_a[i][i'] * (d_diag ? d_diag[(i',j,a)] : 1) * d_in[(i',j,a)]
 *   d_blocks : device, n_ch*Np*Np doubles, B_a row-major, a-major;  d_diag : device, M doubles, or NULL;
 *   d_in, d_out : device, M doubles in the lattice's row order r = (i*Nq + j)*n_ch + a, distinct buffers.
 * pm_kernel_apply : d_out = O (P0 (V~1 (G1 u))) — three launches; d_work : device scratch of 2*M doubles;
 *   d_colidx may be NULL: the SpMV then takes the columns from the lattice's hit lists (pm_spmv_implicit).
 * Both are asynchronous on `cuda_stream`. */
int32_t pm_block_apply(pm_lattice* lat, const double* d_blocks, const double* d_diag, const double* d_in, double* d_out,
                       void* cuda_stream);
/* the same with the transposed blocks: d_out[(i,j,a)] = sum_i' B_a[i'][i] * d_in[(i',j,a)] */
int32_t pm_block_apply_t(pm_lattice* lat, const double* d_blocks, const double* d_in, double* d_out, void* cuda_stream);
/* Rotation to the channel basis, eq. (20): P = O P0 O^T applied to a vector,
 * d_out = O (P0 (O^T x)); O as in pm_block_apply (one orthogonal (Np x Np) block per channel); d_work: 2*M doubles;
 * d_colidx may be NULL (columns from the hit lists, as pm_spmv_implicit). */
int32_t pm_rotate_apply(pm_lattice* lat, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                        const double* d_O, const double* d_x, double* d_out, double* d_work, void* cuda_stream);
int32_t pm_kernel_apply(pm_lattice* lat, const int64_t* d_rowptr, const int32_t* d_colidx, const double* d_vals,
                        const double* d_O, const double* d_Vt, const double* d_g1, const double* d_u, double* d_out,
                        double* d_work, void* cuda_stream);

/* Whole build with HOST output buffers and row-block streaming: source-cell ranges are
 * chosen so that one block's CSR (12 B per nonzero) fits `device_budget_bytes` (0 = 3/4 of free device memory);
 * each block is built on the device and copied to the host arrays.
 *   pm_build_host_count : *nnz_total and *n_blocks for that budget (pattern counting only)
 *   pm_build_host       : h_rowptr[M+1] (global CSR), h_colidx[nnz_total], h_vals[nnz_total]  (host; pinned or not) */
int32_t pm_build_host_count(pm_lattice* lat, int64_t device_budget_bytes, int64_t* nnz_total, int32_t* n_blocks);
int32_t pm_build_host(pm_lattice* lat, int64_t device_budget_bytes,
                      int64_t* h_rowptr, int32_t* h_colidx, double* h_vals, int64_t capacity,
                      int64_t* nnz_total, int32_t* n_blocks);

/* Algorithmic work of this lattice's formulation (add = mul = div = sqrt = rsqrt = 1 flop, FMA = 2;
 * comparisons and integer work not counted): FP64 flops per quadrature node that lands on the grid, per
 * (target cell, x-node) segment of a source cell's sorted node list (the bra harmonics are applied once per
 * segment), and per hit (source, target) cell pair.  One build =
 *   flop_per_node * nodes_on_grid + flop_per_segment * segments + flop_per_hit_cell * hit_cells,
 * the three counts coming from pm_pattern_counts.  Host only. */
int32_t pm_lattice_work(const pm_lattice* lat, double* flop_per_node, double* flop_per_segment, double* flop_per_hit_cell,
                        int32_t* n_coupled_pairs);

/* Counts of the last pm_pattern call on this lattice (host out): quadrature nodes that landed on the grid,
 * (target cell, x-node) segments, hit (source, target) cell pairs (= nnz / number of coupled channel pairs).
 * PM_ERR_STATE before the first pm_pattern. */
int32_t pm_pattern_counts(const pm_lattice* lat, int64_t* nodes_on_grid, int64_t* segments, int64_t* hit_cells);

/* Chunks of the last pm_pattern call on this lattice (host out): the pattern pass cuts every source cell's sorted node
 * list into runs of at most four nodes of one (target cell, x-node) segment (one lane of the fill kernel sums one chunk in
 * registers) and leaves one 8-byte word per chunk, which the fill reads once: 8 * chunks are the fill's input bytes.
 * PM_ERR_STATE before the first pm_pattern. */
int32_t pm_pattern_chunks(const pm_lattice* lat, int64_t* chunks);

/* Name of the fill kernel this lattice's channel set selects: "Spec_<set>" when csrc/build.py generated straight-line
 * ket code for it at build time (the channel sets of BASELINE.json's configs, in any channel order); "jit" when the same
 * kind of code is generated from the lattice's tables and compiled with NVRTC at the first fill (any other channel set
 * of at most 40 ket slots; needs libnvrtc and the CUDA driver at run time, 2-4 s once per channel set, variant and
 * process); "jit-grouped" for bigger sets (46-62 channels), whose column-channel groups get one such kernel each and
 * whose CSR rows are assembled from the groups' per-pair sums; "generic" / "generic-grouped" for the
 * table-driven kernel used when run-time compilation is switched off or failed.  All give the same pattern and the same
 * results within the value tolerance.  Host only; library-owned string, never NULL. */
const char* pm_lattice_fill_kernel(const pm_lattice* lat);

/* Switches run-time compilation on (default, unless the environment variable PM_NO_JIT is set) or off for lattices
 * that have not run a fill yet. */
int32_t pm_set_jit(int32_t enabled);

/* Diagnostic (host only, no GPU needed): generates this lattice's run-time kernel source and compiles it with NVRTC
 * for sm_100a (every column-channel group of a "jit-grouped" set, one after the other); *cubin_bytes receives the total
 * size of the binaries.  PM_ERR_STATE with the compiler log as message on failure (also when libnvrtc cannot be loaded). */
int32_t pm_diag_jit_compile(const pm_lattice* lat, int64_t* cubin_bytes);

/* Diagnostic (host only): the smallest double y with sqrt(y) >= edge under IEEE round-to-nearest — the threshold
 * the kernels compare p'^2 with instead of taking sqrt(p'^2) and comparing with the edge. */
double pm_diag_sqrt_threshold(double edge);

/* Diagnostic: measured FP64 FMA throughput of the current device in TFLOP/s (a dependent-free DFMA loop on every
 * SM, timed with CUDA events on `cuda_stream`); the roofline denominator is stated beside it in DESIGN.md sec. 7. */
int32_t pm_diag_dfma_tflops(double* tflops, void* cuda_stream);

/* Number of kernels this library has launched so far in the calling process (bench.py `gpu_launches`). */
int64_t pm_launch_count(void);

/* Thread-local message of the last failing call on this thread; library-owned, never NULL. */
const char* pm_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* PM_H_ */
