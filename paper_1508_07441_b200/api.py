"""Thin Python binding of libpm (include/pm.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels of libpm.so; this module turns numpy arrays and
torch CUDA tensors into raw pointers and back.  torch is used for device memory, pinned host memory
and streams only.  There is no CPU fallback: a missing libpm.so or a failing call raises.

Function names mirror the C ABI: pm_lattice_create, pm_pattern, pm_fill, pm_spmv, pm_build_host.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libpm.so")
_lib = None

PM_OK = 0
ERRORS = {-1: "PM_ERR_ARG", -2: "PM_ERR_GRID", -3: "PM_ERR_CHANNEL", -4: "PM_ERR_ORDER", -5: "PM_ERR_CUDA",
          -6: "PM_ERR_NOMEM", -7: "PM_ERR_STATE", -8: "PM_ERR_OVERFLOW", -9: "PM_ERR_DEVICE"}

EXPORTS = ["pm_lattice_create", "pm_lattice_destroy", "pm_lattice_dims", "pm_lattice_rule", "pm_lattice_set_rule",
           "pm_lattice_coupling", "pm_lattice_work", "pm_pattern_counts", "pm_pattern_chunks", "pm_lattice_fill_kernel", "pm_set_jit", "pm_diag_jit_compile", "pm_diag_sqrt_threshold",
           "pm_diag_dfma_tflops", "pm_pattern", "pm_fill", "pm_build", "pm_last_fill_ms", "pm_block_apply", "pm_kernel_apply", "pm_spmv_implicit", "pm_spmv", "pm_build_host_count", "pm_build_host",
           "pm_launch_count", "pm_last_error", "pm_lattice_attach", "pm_build_async", "pm_build_wait", "pm_build_reuse",
           "pm_pattern_cell_hits", "pm_partition_cells", "pm_rowptr_offset", "pm_block_apply_t", "pm_rotate_apply",
           "pm_lattice_set_normalisation", "pm_operator_build", "pm_operator_apply", "pm_rotate_apply_static"]


class PmError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"{ERRORS.get(code, code)}: {msg}")
        self.code = code


class _Channel(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("l", "s", "j", "t", "lam", "I2")]


_vp, _dp, _i32p, _i64p = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int32), C.POINTER(C.c_int64)


def lib():
    """Load libpm.so (built in-tree by csrc/build.py).  Raises if it is missing: no fallback exists."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_1508_07441_b200.csrc.build` "
                          "(or __graft_entry__.build()); libpm has no CPU fallback")
    L = C.CDLL(_LIB_PATH)
    L.pm_last_error.restype = C.c_char_p
    L.pm_launch_count.restype = C.c_int64
    L.pm_lattice_create.argtypes = [_dp, C.c_int32, _dp, C.c_int32, C.POINTER(_Channel), C.c_int32,
                                    C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32,
                                    C.POINTER(_vp)]
    L.pm_lattice_destroy.argtypes = [_vp]
    L.pm_lattice_set_normalisation.argtypes = [_vp, C.c_int32]
    L.pm_operator_build.argtypes = [_vp, _i64p, _i64p, _vp]
    L.pm_operator_apply.argtypes = [_vp, _vp, _vp, _vp]
    L.pm_rotate_apply_static.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp]
    L.pm_lattice_attach.argtypes = [_vp, C.POINTER(_Channel), C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.POINTER(_vp)]
    L.pm_build_async.argtypes = [_vp, C.c_int32, C.c_int32, _vp, _vp, _vp, C.c_int64, C.c_int32, _vp]
    L.pm_build_wait.argtypes = [_vp, _i64p]
    L.pm_build_reuse.argtypes = [_vp, C.c_int32, C.c_int32, _vp, _vp, _vp, C.c_int64, _i64p, _vp]
    L.pm_pattern_cell_hits.argtypes = [_vp, _i32p, _vp]
    L.pm_partition_cells.argtypes = [_i32p, C.c_int32, C.c_double, C.c_int32, _i32p]
    L.pm_rowptr_offset.argtypes = [_vp, C.c_int64, C.c_int64, _vp]
    L.pm_block_apply_t.argtypes = [_vp, _vp, _vp, _vp, _vp]
    L.pm_rotate_apply.argtypes = [_vp] + [_vp] * 8
    L.pm_lattice_dims.argtypes = [_vp, _i64p, _i32p]
    L.pm_lattice_rule.argtypes = [_vp, C.c_int32, _dp, _dp]
    L.pm_lattice_set_rule.argtypes = [_vp, C.c_int32, _dp, _dp]
    L.pm_lattice_coupling.argtypes = [_vp, C.POINTER(C.c_uint8), _i32p]
    L.pm_lattice_work.argtypes = [_vp, _dp, _dp, _dp, _i32p]
    L.pm_pattern_counts.argtypes = [_vp, _i64p, _i64p, _i64p]
    L.pm_pattern_chunks.argtypes = [_vp, _i64p]
    L.pm_diag_dfma_tflops.argtypes = [_dp, _vp]
    L.pm_set_jit.argtypes = [C.c_int32]
    L.pm_diag_jit_compile.argtypes = [_vp, _i64p]
    L.pm_lattice_fill_kernel.argtypes = [_vp]
    L.pm_lattice_fill_kernel.restype = C.c_char_p
    L.pm_diag_sqrt_threshold.argtypes = [C.c_double]
    L.pm_diag_sqrt_threshold.restype = C.c_double
    L.pm_pattern.argtypes = [_vp, C.c_int32, C.c_int32, _vp, _vp, C.c_int64, _i64p, _vp]
    L.pm_fill.argtypes = [_vp, C.c_int32, C.c_int32, _vp, _vp, _vp]
    L.pm_spmv_implicit.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
    L.pm_block_apply.argtypes = [_vp, _vp, _vp, _vp, _vp, _vp]
    L.pm_kernel_apply.argtypes = [_vp] + [_vp] * 10
    L.pm_last_fill_ms.argtypes = [_vp, C.POINTER(C.c_float)]
    L.pm_build.argtypes = [_vp, C.c_int32, C.c_int32, _vp, _vp, _vp, C.c_int64, _i64p, _vp]
    L.pm_spmv.argtypes = [_vp, C.c_int64, _vp, _vp, _vp, _vp, _vp, _vp]
    L.pm_build_host_count.argtypes = [_vp, C.c_int64, _i64p, _i32p]
    L.pm_build_host.argtypes = [_vp, C.c_int64, _vp, _vp, _vp, C.c_int64, _i64p, _i32p]
    for name in EXPORTS:
        if name not in ("pm_last_error", "pm_launch_count", "pm_lattice_fill_kernel", "pm_diag_sqrt_threshold"):
            getattr(L, name).restype = C.c_int32
    _lib = L
    return L


def _check(rc):
    if rc != PM_OK:
        raise PmError(rc, lib().pm_last_error().decode())


def _d(a):
    return a.ctypes.data_as(_dp)


def _stream_ptr(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


# ------------------------------------------------------------------ C-ABI mirrors
def pm_lattice_create(p_edges, q_edges, channels, J2, parity, T2, statistics, n_p, n_q, n_x):
    pe = np.ascontiguousarray(p_edges, dtype=np.float64)
    qe = np.ascontiguousarray(q_edges, dtype=np.float64)
    ch = (_Channel * len(channels))(*[_Channel(*(int(c[k]) for k in ("l", "s", "j", "t", "lam", "I2"))) for c in channels])
    h = _vp()
    _check(lib().pm_lattice_create(_d(pe), len(pe) - 1, _d(qe), len(qe) - 1, ch, len(channels),
                                   int(J2), int(parity), int(T2), int(statistics), int(n_p), int(n_q), int(n_x),
                                   C.byref(h)))
    return h


def pm_lattice_attach(base, channels, J2, parity, T2, statistics):
    """Another channel set (another J^pi) on the grids and rules of `base`; shares its geometric pattern."""
    ch = (_Channel * len(channels))(*[_Channel(*(int(c[k]) for k in ("l", "s", "j", "t", "lam", "I2"))) for c in channels])
    h = _vp()
    _check(lib().pm_lattice_attach(base, ch, len(channels), int(J2), int(parity), int(T2), int(statistics), C.byref(h)))
    return h


def pm_lattice_destroy(h):
    _check(lib().pm_lattice_destroy(h))


def pm_lattice_set_normalisation(h, normalisation):
    """0 = PM_NORM_WIDTH (reading A, default), 1 = PM_NORM_P2 (reading B: p^2 dp measure)."""
    _check(lib().pm_lattice_set_normalisation(h, int(normalisation)))


def pm_lattice_dims(h):
    M, nc = C.c_int64(), C.c_int32()
    _check(lib().pm_lattice_dims(h, C.byref(M), C.byref(nc)))
    return M.value, nc.value


def pm_lattice_rule(h, axis, n):
    t, w = np.empty(n), np.empty(n)
    _check(lib().pm_lattice_rule(h, axis, _d(t), _d(w)))
    return t, w


def pm_lattice_set_rule(h, axis, nodes, weights):
    t = np.ascontiguousarray(nodes, dtype=np.float64)
    w = np.ascontiguousarray(weights, dtype=np.float64)
    _check(lib().pm_lattice_set_rule(h, axis, _d(t), _d(w)))


def pm_lattice_coupling(h, n_ch):
    m = np.zeros(n_ch * n_ch, dtype=np.uint8)
    nf = C.c_int32()
    _check(lib().pm_lattice_coupling(h, m.ctypes.data_as(C.POINTER(C.c_uint8)), C.byref(nf)))
    return m.reshape(n_ch, n_ch).astype(bool), nf.value


def pm_lattice_work(h):
    """(flop per node on the grid, flop per (target, x-node) segment, flop per hit cell pair, coupled channel pairs)."""
    a, s_, b, n = C.c_double(), C.c_double(), C.c_double(), C.c_int32()
    _check(lib().pm_lattice_work(h, C.byref(a), C.byref(s_), C.byref(b), C.byref(n)))
    return a.value, s_.value, b.value, n.value


def pm_pattern_counts(h):
    """(nodes on the grid, (target, x-node) segments, hit cell pairs) of the last pm_pattern call."""
    a, s_, b = C.c_int64(), C.c_int64(), C.c_int64()
    _check(lib().pm_pattern_counts(h, C.byref(a), C.byref(s_), C.byref(b)))
    return a.value, s_.value, b.value


def pm_pattern_chunks(h):
    """Chunks (8-byte words the fill reads) of the last pm_pattern call."""
    a = C.c_int64()
    _check(lib().pm_pattern_chunks(h, C.byref(a)))
    return a.value


def pm_lattice_fill_kernel(h):
    return lib().pm_lattice_fill_kernel(h).decode()


def pm_set_jit(enabled):
    _check(lib().pm_set_jit(1 if enabled else 0))


def pm_diag_jit_compile(h):
    """Compiles the lattice's run-time kernel with NVRTC (no GPU needed); returns the cubin size in bytes."""
    n = C.c_int64()
    _check(lib().pm_diag_jit_compile(h, C.byref(n)))
    return n.value


def pm_diag_sqrt_threshold(edge):
    return lib().pm_diag_sqrt_threshold(float(edge))


def pm_diag_dfma_tflops(stream=None):
    t = C.c_double()
    _check(lib().pm_diag_dfma_tflops(C.byref(t), _stream_ptr(stream)))
    return t.value


def pm_pattern(h, cell_begin, cell_end, d_rowptr, d_colidx=None, stream=None):
    """d_rowptr: int64 CUDA tensor; d_colidx: int32 CUDA tensor or None (count only).  Returns nnz."""
    nnz = C.c_int64()
    _check(lib().pm_pattern(h, cell_begin, cell_end, d_rowptr.data_ptr(),
                            d_colidx.data_ptr() if d_colidx is not None else None,
                            d_colidx.numel() if d_colidx is not None else 0, C.byref(nnz), _stream_ptr(stream)))
    return nnz.value


def pm_fill(h, cell_begin, cell_end, d_rowptr, d_vals, stream=None):
    _check(lib().pm_fill(h, cell_begin, cell_end, d_rowptr.data_ptr(), d_vals.data_ptr(), _stream_ptr(stream)))


def pm_build(h, cell_begin, cell_end, d_rowptr, d_colidx, d_vals, stream=None):
    """Pattern + fill of one block, columns and values written by one kernel.  Returns nnz."""
    nnz = C.c_int64()
    _check(lib().pm_build(h, cell_begin, cell_end, d_rowptr.data_ptr(), d_colidx.data_ptr(), d_vals.data_ptr(),
                          min(d_colidx.numel(), d_vals.numel()), C.byref(nnz), _stream_ptr(stream)))
    return nnz.value


def pm_build_reuse(h, cell_begin, cell_end, d_rowptr, d_colidx, d_vals, stream=None):
    """pm_build that reuses the node lists the lattice group already holds for this cell range.  Returns nnz."""
    nnz = C.c_int64()
    _check(lib().pm_build_reuse(h, cell_begin, cell_end, d_rowptr.data_ptr(), d_colidx.data_ptr(), d_vals.data_ptr(),
                                min(d_colidx.numel(), d_vals.numel()), C.byref(nnz), _stream_ptr(stream)))
    return nnz.value


def pm_build_async(h, cell_begin, cell_end, d_rowptr, d_colidx, d_vals, reuse_lists=False, stream=None):
    """Queues pattern + fill on the stream without any host synchronisation; pm_build_wait returns nnz."""
    _check(lib().pm_build_async(h, cell_begin, cell_end, d_rowptr.data_ptr(), d_colidx.data_ptr(), d_vals.data_ptr(),
                                min(d_colidx.numel(), d_vals.numel()), 1 if reuse_lists else 0, _stream_ptr(stream)))


def pm_build_wait(h):
    nnz = C.c_int64()
    _check(lib().pm_build_wait(h, C.byref(nnz)))
    return nnz.value


def pm_pattern_cell_hits(h, n_cells_in_block, stream=None):
    """Hit cells per source cell of the last pattern / build call (numpy int32)."""
    out = np.empty(n_cells_in_block, dtype=np.int32)
    _check(lib().pm_pattern_cell_hits(h, out.ctypes.data_as(_i32p), _stream_ptr(stream) if n_cells_in_block else None))
    return out


def pm_partition_cells(hits, n_parts, cell_cost=0.0):
    """cuts[n_parts+1]: contiguous source-cell ranges of (almost) equal weight sum(hits + cell_cost).  Host only."""
    h = np.ascontiguousarray(hits, dtype=np.int32)
    cuts = np.empty(n_parts + 1, dtype=np.int32)
    _check(lib().pm_partition_cells(h.ctypes.data_as(_i32p), len(h), float(cell_cost), int(n_parts), cuts.ctypes.data_as(_i32p)))
    return cuts


def pm_rowptr_offset(d_rowptr, offset, stream=None):
    _check(lib().pm_rowptr_offset(d_rowptr.data_ptr(), d_rowptr.numel(), int(offset), _stream_ptr(stream)))


def pm_block_apply_t(h, d_blocks, d_in, d_out, stream=None):
    _check(lib().pm_block_apply_t(h, d_blocks.data_ptr(), d_in.data_ptr(), d_out.data_ptr(), _stream_ptr(stream)))


def pm_rotate_apply(h, d_rowptr, d_colidx, d_vals, d_O, d_x, d_out, d_work, stream=None):
    """d_out = O P0 O^T x (eq. 20); d_work holds 2*M doubles."""
    _check(lib().pm_rotate_apply(h, d_rowptr.data_ptr(), d_colidx.data_ptr() if d_colidx is not None else None, d_vals.data_ptr(),
                                 d_O.data_ptr(), d_x.data_ptr(), d_out.data_ptr(), d_work.data_ptr(), _stream_ptr(stream)))


def pm_spmv_implicit(h, d_rowptr, d_vals, d_x, d_y, stream=None):
    """y = P0 x with the columns implied by the lattice's hit lists (whole lattice, after pm_pattern / pm_build)."""
    _check(lib().pm_spmv_implicit(h, d_rowptr.data_ptr(), d_vals.data_ptr(), d_x.data_ptr(), d_y.data_ptr(), _stream_ptr(stream)))


def pm_operator_build(h, stream=None):
    """Per-pair sums (operator form of P0) of the whole lattice; returns (hit cell pairs, bytes of the sums)."""
    a, b = C.c_int64(), C.c_int64()
    _check(lib().pm_operator_build(h, C.byref(a), C.byref(b), _stream_ptr(stream)))
    return a.value, b.value


def pm_operator_apply(h, d_x, d_y, stream=None):
    """y = P0 x straight from the per-pair sums of pm_operator_build."""
    _check(lib().pm_operator_apply(h, d_x.data_ptr(), d_y.data_ptr(), _stream_ptr(stream)))


def pm_rotate_apply_static(h, d_rowptr, d_colidx, d_vals, d_O, d_x, d_out, stream=None):
    """pm_rotate_apply with the library's static scratch instead of d_work: allocates nothing (M <= PM_STATIC_MAX_M)."""
    _check(lib().pm_rotate_apply_static(h, d_rowptr.data_ptr(), d_colidx.data_ptr(), d_vals.data_ptr(), d_O.data_ptr(),
                                        d_x.data_ptr(), d_out.data_ptr(), _stream_ptr(stream)))


def pm_block_apply(h, d_blocks, d_diag, d_in, d_out, stream=None):
    _check(lib().pm_block_apply(h, d_blocks.data_ptr(), d_diag.data_ptr() if d_diag is not None else None,
                                d_in.data_ptr(), d_out.data_ptr(), _stream_ptr(stream)))


def pm_kernel_apply(h, d_rowptr, d_colidx, d_vals, d_O, d_Vt, d_g1, d_u, d_out, d_work, stream=None):
    """d_out = O P0 V~1 G1 u (eq. 24); d_work holds 2*M doubles."""
    _check(lib().pm_kernel_apply(h, d_rowptr.data_ptr(), d_colidx.data_ptr() if d_colidx is not None else None,
                                 d_vals.data_ptr(), d_O.data_ptr(),
                                 d_Vt.data_ptr(), d_g1.data_ptr(), d_u.data_ptr(), d_out.data_ptr(), d_work.data_ptr(),
                                 _stream_ptr(stream)))


def pm_last_fill_ms(h):
    ms = C.c_float()
    _check(lib().pm_last_fill_ms(h, C.byref(ms)))
    return ms.value


def pm_spmv(h, d_rowptr, d_colidx, d_vals, d_x, d_y, stream=None):
    _check(lib().pm_spmv(h, d_rowptr.numel() - 1, d_rowptr.data_ptr(), d_colidx.data_ptr(), d_vals.data_ptr(),
                         d_x.data_ptr(), d_y.data_ptr(), _stream_ptr(stream)))


def pm_build_host_count(h, budget_bytes=0):
    nnz, nb = C.c_int64(), C.c_int32()
    _check(lib().pm_build_host_count(h, int(budget_bytes), C.byref(nnz), C.byref(nb)))
    return nnz.value, nb.value


def pm_build_host(h, budget_bytes, h_rowptr, h_colidx, h_vals):
    """Host outputs: torch CPU tensors (pinned or not) or numpy arrays.  Returns (nnz, n_blocks)."""
    def ptr(a):
        return a.data_ptr() if hasattr(a, "data_ptr") else a.ctypes.data
    cap = h_colidx.numel() if hasattr(h_colidx, "numel") else h_colidx.size
    nnz, nb = C.c_int64(), C.c_int32()
    _check(lib().pm_build_host(h, int(budget_bytes), ptr(h_rowptr), ptr(h_colidx), ptr(h_vals), cap,
                               C.byref(nnz), C.byref(nb)))
    return nnz.value, nb.value


def pm_launch_count():
    return lib().pm_launch_count()


# ------------------------------------------------------------------ convenience wrapper
class Lattice:
    """Owns a pm_lattice handle created from a `inputs.Workload`; allocates outputs with torch."""

    def __init__(self, wl, use_workload_rules: bool = True, normalisation: int = 0):
        self.wl = wl
        self.h = pm_lattice_create(wl.p_edges, wl.q_edges, wl.channels, wl.J2, wl.parity, wl.T2, wl.statistics,
                                   wl.n_p, wl.n_q, wl.n_x)
        if normalisation:
            pm_lattice_set_normalisation(self.h, normalisation)
        if use_workload_rules:                      # feed the very arrays the oracle gets (reading R12)
            for axis, key in enumerate(("p", "q", "x")):
                pm_lattice_set_rule(self.h, axis, *wl.rules[key])
        self.M, self.n_cells = pm_lattice_dims(self.h)
        self.n_ch = wl.n_ch

    def close(self):
        if self.h is not None:
            pm_lattice_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def pattern(self, cell_begin=0, cell_end=None, count_only=False, stream=None):
        import torch
        cell_end = self.n_cells if cell_end is None else cell_end
        rowptr = torch.empty((cell_end - cell_begin) * self.n_ch + 1, dtype=torch.int64, device="cuda")
        nnz = pm_pattern(self.h, cell_begin, cell_end, rowptr, None, stream)
        if count_only:
            return rowptr, None, nnz
        colidx = torch.empty(max(nnz, 1), dtype=torch.int32, device="cuda")[:nnz]
        pm_pattern(self.h, cell_begin, cell_end, rowptr, colidx, stream)
        return rowptr, colidx, nnz

    def fill(self, rowptr, nnz, cell_begin=0, cell_end=None, out=None, stream=None):
        import torch
        cell_end = self.n_cells if cell_end is None else cell_end
        vals = out if out is not None else torch.empty(max(nnz, 1), dtype=torch.float64, device="cuda")[:nnz]
        pm_fill(self.h, cell_begin, cell_end, rowptr, vals, stream)
        return vals

    def build(self, cell_begin=0, cell_end=None):
        rowptr, colidx, nnz = self.pattern(cell_begin, cell_end)
        return rowptr, colidx, self.fill(rowptr, nnz, cell_begin, cell_end)

    def build_fused(self, cell_begin=0, cell_end=None):
        """pm_build: count (rowptr, nnz), allocate, then one call that writes columns and values together."""
        import torch
        cell_end = self.n_cells if cell_end is None else cell_end
        rowptr, _, nnz = self.pattern(cell_begin, cell_end, count_only=True)
        colidx = torch.empty(max(nnz, 1), dtype=torch.int32, device="cuda")[:nnz]
        vals = torch.empty(max(nnz, 1), dtype=torch.float64, device="cuda")[:nnz]
        if nnz:
            pm_build(self.h, cell_begin, cell_end, rowptr, colidx, vals)
        return rowptr, colidx, vals

    def spmv(self, rowptr, colidx, vals, x):
        import torch
        y = torch.empty(rowptr.numel() - 1, dtype=torch.float64, device="cuda")
        pm_spmv(self.h, rowptr, colidx, vals, x, y)
        return y

    def build_host(self, budget_bytes=0, pinned=True):
        import torch
        nnz, _ = pm_build_host_count(self.h, budget_bytes)
        rowptr = torch.empty(self.M + 1, dtype=torch.int64, pin_memory=pinned)
        colidx = torch.empty(max(nnz, 1), dtype=torch.int32, pin_memory=pinned)
        vals = torch.empty(max(nnz, 1), dtype=torch.float64, pin_memory=pinned)
        nnz, nb = pm_build_host(self.h, budget_bytes, rowptr, colidx, vals)
        return rowptr, colidx[:nnz], vals[:nnz], nnz, nb
