// pm_kernels.cuh — launcher declarations of libpm's kernels (definitions in pm_kernels.cu, pm_fill.cu).
#pragma once
#include <algorithm>
#include <atomic>
#include <cstddef>
#include <cstdint>
#include <string>
#include <vector>

#include "pm_device.cuh"
#include "pm_fill.cuh"
#include "pm_tables.hpp"

namespace pm {

constexpr int kThreads = 256;
constexpr int kMapSortMaxWarps = 16;  // k_map_sort: warps (= source cells in flight) per CTA, one CTA per SM
constexpr int kHistCap = 512;         // k_map_sort: rank counters per window (one window unless a source cell hits more cells)

// shared-memory plan of k_map_sort: tables shared by the CTA, then one private area per warp (byte offsets)
struct MapSortSmem { int thr_p, thr_q, bk_p, bk_q, tp, tq, tx, warp0, warp_bytes, w_bits, w_wpre, w_hist, nw, ctas, wide, hist_cap, nchunk, total; };
MapSortSmem map_sort_plan(const DevLattice& L, int max_warps);
int64_t launch_count();
void count_launch();

// pattern pass
size_t map_sort_scratch_bytes(const DevLattice& L, int n_sm);      // per-warp target scratch of k_map_sort (global memory)
cudaError_t launch_map_sort(const DevLattice& L, int cell_begin, int n_blk, const NodeLists& nl, int n_sm, int* counter, void* scratch, cudaStream_t st);
// scan of the hit counts + rowptr; summary = {nnz, max hits, nodes on the grid, (segments), overflow flag: nnz > capacity >= 0}
cudaError_t launch_scan_rows(const DevLattice& L, int n_blk, const NodeLists& nl, int64_t* cellbase, int64_t* rowptr,
                             int64_t* summary, int64_t capacity, cudaStream_t st);
cudaError_t launch_emit_cols(const DevLattice& L, int n_blk, const NodeLists& nl, const int64_t* cellbase, const int* hitlist,
                             const int64_t* rowptr, int32_t* colidx, cudaStream_t st);
cudaError_t launch_count_segments(const DevLattice& L, int n_blk, const NodeLists& nl, unsigned long long* total, cudaStream_t st);

// fill pass (pm_fill.cuh): variant selection and launch
struct FillLaunch { const void *fn, *fn_cols, *fn_op; int nw, grid; FillSmem smem; const char* name; bool jit; };   // fn_cols also writes colidx;
                                                      // jit: fn / fn_cols are CUfunction handles of run-time compiled kernels (pm_jit.hpp)
bool fill_has_spec(unsigned long long tables_hash);
const char* fill_variant_name(unsigned long long tables_hash);
cudaError_t fill_plan(const DevLattice& L, unsigned long long tables_hash, int n_sm, FillLaunch* out);
// run-time compiled kernels for the column-channel groups of one lattice (no build-time kernel): false + message when
// NVRTC / the driver API fails
bool fill_plan_jit(const std::vector<DevLattice>& devs, std::vector<KetView> views, int n_sm, int mode, std::vector<FillLaunch>& out, std::string& err);
cudaError_t launch_fill(const DevLattice& L, const FillLaunch& F, int cell_begin, int n_blk, const NodeLists& nl,
                        const int64_t* rowptr, double* vals, int32_t* colidx, int* counter, const int64_t* guard, cudaStream_t st,
                        bool op_mode = false);      // op_mode: the per-pair sums variant (rowptr = scan of the hit counts, vals = the sums)

// CSR rows (values and, if colidx, column indices) from the per-pair sums A of a whole channel set (pm_kernels.cu)
cudaError_t launch_op_expand(const DevLattice& L, int cell_begin, int n_blk, const NodeLists& nl, const int64_t* cellbase, const int* hitlist,
                             const double* A, const unsigned short* xpos, const double* xc, const int64_t* rowptr, double* vals,
                             int32_t* colidx, int* counter, const int64_t* guard, int n_sm, cudaStream_t st);
// y = P0 x from the per-pair sums A of the whole lattice (pm_kernels.cu)
cudaError_t launch_op_apply(const DevLattice& L, int n_blk, int hmax, const NodeLists& nl, const int64_t* cellbase, const int* hitlist, const double* A,
                            const unsigned short* xpos, const double* xc, const double* x, double* y, int* counter, int n_sm, cudaStream_t st);
cudaError_t launch_hit_list(const DevLattice& L, int n_blk, const NodeLists& nl, const int64_t* cellbase, int* hitlist, cudaStream_t st);
cudaError_t launch_spmv_implicit(const DevLattice& L, int64_t n_rows, const int64_t* rowptr, const int* hits, const int64_t* cellbase,
                                 const int* hitlist, const double* vals, const double* x, double* y, cudaStream_t st);
cudaError_t launch_spmv(int64_t n_rows, const int64_t* rowptr, const int32_t* colidx, const double* vals,
                        const double* x, double* y, cudaStream_t st);

// one block-matrix factor of the iteration step (eq. 24) with an optional diagonal factor
cudaError_t launch_block_apply(int Np, int Nq, int n_ch, const double* B, const double* diag, const double* in, double* out,
                               int transpose, cudaStream_t st);
cudaError_t launch_add_offset(int64_t* a, int64_t n, int64_t off, cudaStream_t st);

// dependent-free DFMA loop on every SM: measured FP64 FMA throughput in TFLOP/s (diagnostic)
cudaError_t measure_dfma(int n_sm, double* tflops, cudaStream_t st);

}  // namespace pm
