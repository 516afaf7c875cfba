// pm_jit.hpp — run-time specialisation of the fill kernel for channel sets that have no build-time kernel.
//
// csrc/build.py generates straight-line ket code only for the channel sets of BASELINE.json's configs.  Any other
// channel set (another J^pi, another order) would run the table-driven `SpecGeneric` kernel, 8x slower.  Instead the
// library emits the same kind of struct from the lattice's tables (pm_emit.cpp), compiles `k_fill_warp<Spec_jit, ...>`
// with NVRTC for sm_100a from the very headers nvcc compiled (embedded as text in gen/pm_jit_src.inc) and launches it
// through the driver API.  libnvrtc and libcuda are opened with dlopen on first use, so libpm.so loads on machines
// without them; if either is missing or the compilation fails, pm_fill falls back to the table-driven kernel and
// `pm_lattice_fill_kernel` says so.  Compiled kernels are cached per tables hash for the life of the process.
#pragma once
#include <cstddef>
#include <string>
#include <vector>

#include "pm_tables.hpp"

namespace pm {

struct JitFill {
    void* fn = nullptr;        // CUfunction of k_fill_warp<Spec_jit, nw, rb, 0>, or NULL (compiled when first needed)
    void* fn_cols = nullptr;   // ... <..., 1>: values and column indices
    void* fn_op = nullptr;     // ... <..., 2>: per-pair sums (pm_fill.cuh)
    int nw = 0, rb = 0;
};

// Enables / disables run-time compilation for lattices planned from now on (default: enabled unless PM_NO_JIT is set).
void jit_set_enabled(bool on);
bool jit_enabled();

// Compiles (or fetches from the cache) ONE kernel variant (mode 0 values, 1 values and column indices, 2 per-pair sums;
// the other members of JitFill stay NULL) for the ket tables in V with `nw` warps and row batch `rb`.  Returns false and a message if NVRTC / the driver API is unavailable or the compilation fails.
bool jit_fill(const KetView& V, int nw, int rb, int mode, JitFill* out, std::string& err);
// The same for several kernels at once (the column-channel groups of a big channel set): the NVRTC compilations run
// on one host thread each, the modules are loaded by the caller's thread.
bool jit_fill_many(const std::vector<KetView>& views, int nw, int rb, int mode, std::vector<JitFill>& out, std::string& err);

// NVRTC only, no device needed: does the kernel for V compile for sm_100a?  (diagnostic, CPU tests)
bool jit_compile_check(const KetView& V, int nw, int rb, size_t* cubin_bytes, std::string& err);

// cuFuncSetAttribute(max dynamic shared memory) + occupancy; returns CTAs per SM (0 on error)
int jit_prepare(const JitFill& k, int mode, int smem_bytes);

// Raises (never lowers) the dynamic shared-memory limit of a run-time compiled function to at least `smem_bytes`;
// returns 0 on success.  Called before every launch: the function is shared by all lattices with the same tables.
int jit_prepare_fn(void* fn, int smem_bytes);

// cuLaunchKernel on `stream` (a cudaStream_t); returns 0 on success, else a CUresult value
int jit_launch(void* fn, int grid, int block, int smem_bytes, void* stream, void** args);

}  // namespace pm
