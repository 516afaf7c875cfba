// pm_emit.hpp — CUDA source text of the channel-specialised ket code (`struct Spec_<name>` with `ket()`), emitted
// from the host tables.  Used at build time by pm_codegen (gen/pm_spec_gen.cuh, compiled by nvcc into libpm.so) and at
// run time by pm_jit.cpp (NVRTC) for channel sets that have no build-time kernel.  See pm_codegen.cpp for the why.
#pragma once
#include <string>

#include "pm_tables.hpp"

namespace pm {

struct EmitStats { int n_prod = 0, n_fma = 0, n_mul = 0; };

// `struct Spec_<name> { ... static __device__ void ket_acc(...) }` for the ket tables in V (no namespace around it)
std::string emit_spec(const std::string& name, const KetView& V, EmitStats& st);

}  // namespace pm
