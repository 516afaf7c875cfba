// pm_stream.cu — row-block streaming build with host outputs (hot-path step a8).
// PAPER.md:L340 "subdivide the whole calculation of this matrix into some blocks using an external CPU cycle",
// L351-354 (copy a block in, launch, copy the block's values back).  Here a block is a contiguous range of
// source cells whose CSR (12 B per nonzero) fits the caller's device budget; two buffer sets on two streams
// let block b's device->host copies overlap block b+1's kernels.
#include <algorithm>
#include <string>
#include <vector>

#include <cuda_runtime.h>

#include "../../include/pm.h"

namespace {

struct Plan { std::vector<int64_t> rowptr; std::vector<int> cuts; int64_t nnz = 0, max_blk = 0; int n_ch = 0; };

struct DevBuf {
    int64_t* rowptr = nullptr; int32_t* col = nullptr; double* val = nullptr; cudaStream_t st = nullptr;
    ~DevBuf() { if (rowptr) cudaFree(rowptr); if (col) cudaFree(col); if (val) cudaFree(val); if (st) cudaStreamDestroy(st); }
};

int32_t make_plan(pm_lattice* lat, int64_t budget, Plan& P)
{
    int64_t M = 0; int32_t n_cells = 0;
    int32_t rc = pm_lattice_dims(lat, &M, &n_cells);
    if (rc) return rc;
    P.n_ch = (int)(M / n_cells);
    if (budget <= 0) {
        size_t fr = 0, tot = 0;
        if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) { cudaGetLastError(); return PM_ERR_DEVICE; }
        budget = (int64_t)(fr / 4) * 3 / 2;            // two buffer sets share 3/4 of the free memory
    }
    int64_t* d_rowptr = nullptr;
    if (cudaMalloc(&d_rowptr, sizeof(int64_t) * (size_t)(M + 1)) != cudaSuccess) { cudaGetLastError(); return PM_ERR_NOMEM; }
    int64_t nnz = 0;
    rc = pm_pattern(lat, 0, n_cells, d_rowptr, nullptr, 0, &nnz, nullptr);
    if (rc == PM_OK) {
        P.rowptr.resize((size_t)M + 1);
        if (cudaMemcpy(P.rowptr.data(), d_rowptr, sizeof(int64_t) * (size_t)(M + 1), cudaMemcpyDeviceToHost) != cudaSuccess) rc = PM_ERR_CUDA;
    }
    cudaFree(d_rowptr);
    if (rc) return rc;
    P.nnz = nnz;
    P.cuts.assign(1, 0);
    int64_t cur = 0;
    for (int c = 0; c < n_cells; ++c) {
        const int64_t nz = P.rowptr[(size_t)(c + 1) * P.n_ch] - P.rowptr[(size_t)c * P.n_ch];
        if (cur > 0 && 12 * (cur + nz) > budget) { P.cuts.push_back(c); P.max_blk = std::max(P.max_blk, cur); cur = 0; }
        cur += nz;
    }
    P.cuts.push_back(n_cells);
    P.max_blk = std::max(P.max_blk, cur);
    return PM_OK;
}

}  // namespace

extern "C" {

int32_t pm_build_host_count(pm_lattice* lat, int64_t device_budget_bytes, int64_t* nnz_total, int32_t* n_blocks)
{
    if (!lat || !nnz_total || !n_blocks) return PM_ERR_ARG;
    Plan P;
    int32_t rc = make_plan(lat, device_budget_bytes, P);
    if (rc) return rc;
    *nnz_total = P.nnz;
    *n_blocks = (int32_t)P.cuts.size() - 1;
    return PM_OK;
}

int32_t pm_build_host(pm_lattice* lat, int64_t device_budget_bytes, int64_t* h_rowptr, int32_t* h_colidx, double* h_vals,
                      int64_t capacity, int64_t* nnz_total, int32_t* n_blocks)
{
    if (!lat || !h_rowptr || !h_colidx || !h_vals || !nnz_total || !n_blocks) return PM_ERR_ARG;
    Plan P;
    int32_t rc = make_plan(lat, device_budget_bytes, P);
    if (rc) return rc;
    *nnz_total = P.nnz;
    *n_blocks = (int32_t)P.cuts.size() - 1;
    if (P.nnz > capacity) return PM_ERR_OVERFLOW;
    std::copy(P.rowptr.begin(), P.rowptr.end(), h_rowptr);
    const int nb = *n_blocks, nset = nb > 1 ? 2 : 1;
    int max_cells = 0;
    for (int b = 0; b < nb; ++b) max_cells = std::max(max_cells, P.cuts[(size_t)b + 1] - P.cuts[(size_t)b]);
    DevBuf buf[2];
    for (int s = 0; s < nset; ++s) {
        if (cudaStreamCreate(&buf[s].st) != cudaSuccess ||
            cudaMalloc(&buf[s].rowptr, sizeof(int64_t) * ((size_t)max_cells * P.n_ch + 1)) != cudaSuccess ||
            cudaMalloc(&buf[s].col, sizeof(int32_t) * (size_t)std::max<int64_t>(P.max_blk, 1)) != cudaSuccess ||
            cudaMalloc(&buf[s].val, sizeof(double) * (size_t)std::max<int64_t>(P.max_blk, 1)) != cudaSuccess) {
            cudaGetLastError();
            return PM_ERR_NOMEM;
        }
    }
    // The lattice's node lists and work counter serve one block at a time: block b+1's kernels wait for block b's
    // fill (event), so only the device->host copies of block b overlap the kernels of block b+1.
    cudaEvent_t filled = nullptr;
    if (cudaEventCreateWithFlags(&filled, cudaEventDisableTiming) != cudaSuccess) { cudaGetLastError(); return PM_ERR_CUDA; }
    for (int b = 0; b < nb && rc == PM_OK; ++b) {
        DevBuf& B = buf[b % nset];
        if (b > 0 && cudaStreamWaitEvent(B.st, filled, 0) != cudaSuccess) { rc = PM_ERR_CUDA; break; }
        const int cb = P.cuts[(size_t)b], ce = P.cuts[(size_t)b + 1];
        const int64_t off = P.rowptr[(size_t)cb * P.n_ch];
        int64_t nnz = 0;
        // the stream of this buffer set is idle here: pm_pattern synchronises it before reusing the buffers
        rc = pm_build(lat, cb, ce, B.rowptr, B.col, B.val, P.max_blk, &nnz, B.st);
        if (rc) break;
        if (nnz != P.rowptr[(size_t)ce * P.n_ch] - off) { rc = PM_ERR_STATE; break; }
        if (cudaEventRecord(filled, B.st) != cudaSuccess) { rc = PM_ERR_CUDA; break; }
        if (cudaMemcpyAsync(h_colidx + off, B.col, sizeof(int32_t) * (size_t)nnz, cudaMemcpyDeviceToHost, B.st) != cudaSuccess ||
            cudaMemcpyAsync(h_vals + off, B.val, sizeof(double) * (size_t)nnz, cudaMemcpyDeviceToHost, B.st) != cudaSuccess)
            rc = PM_ERR_CUDA;
    }
    cudaEventDestroy(filled);
    for (int s = 0; s < nset; ++s)
        if (buf[s].st && cudaStreamSynchronize(buf[s].st) != cudaSuccess && rc == PM_OK) rc = PM_ERR_CUDA;
    return rc;
}

}  // extern "C"
