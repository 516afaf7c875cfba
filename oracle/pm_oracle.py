"""ctypes loader for the CPU oracle (oracle/pm_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this module; the product (paper_1508_07441_b200) never does, and this module never imports the product's
CUDA binding.  It takes its inputs as plain numpy arrays (the Workload objects of
paper_1508_07441_b200.inputs are only read for their array fields).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pm_oracle.c")
_BUILD = os.path.join(_HERE, "build")
_FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC"]


def build(force: bool = False) -> dict:
    """Compile the double and the long-double instantiation with gcc.  Returns their paths."""
    os.makedirs(_BUILD, exist_ok=True)
    out = {}
    for name, extra in (("libpm_oracle.so", []), ("libpm_oracle_ld.so", ["-DPO_LONG_DOUBLE"])):
        path = os.path.join(_BUILD, name)
        if force or not os.path.exists(path) or os.path.getmtime(path) < os.path.getmtime(_SRC):
            subprocess.check_call(["gcc", *_FLAGS, *extra, "-o", path, _SRC, "-lm"])
        out[name] = path
    return out


class _Channel(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("l", "s", "j", "t", "lam", "I2")]


_dp = C.POINTER(C.c_double)
_i32p = C.POINTER(C.c_int32)
_i64p = C.POINTER(C.c_int64)
_chp = C.POINTER(_Channel)


def _d(a):
    return a.ctypes.data_as(_dp)


class Oracle:
    """One loaded instantiation of the oracle (`long_double=True` -> 80-bit value arithmetic)."""

    def __init__(self, long_double: bool = False):
        paths = build()
        self.lib = lib = C.CDLL(paths["libpm_oracle_ld.so" if long_double else "libpm_oracle.so"])
        lib.po_wigner3j.restype = C.c_double
        lib.po_wigner3j.argtypes = [C.c_int] * 6
        lib.po_cg.restype = C.c_double
        lib.po_cg.argtypes = [C.c_int] * 6
        lib.po_wigner6j.restype = C.c_double
        lib.po_wigner6j.argtypes = [C.c_int] * 6
        lib.po_wigner9j.restype = C.c_double
        lib.po_wigner9j.argtypes = [C.c_int] * 9
        lib.po_ylm.restype = C.c_double
        lib.po_ylm.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double]
        lib.po_recoupling_C.restype = C.c_double
        lib.po_recoupling_C.argtypes = [_chp, C.c_int, C.c_int, C.c_int]
        lib.po_spin_R.restype = C.c_double
        lib.po_spin_R.argtypes = [C.c_int] * 4
        lib.po_coef_L.restype = C.c_double
        lib.po_coef_L.argtypes = [_chp, _chp] + [C.c_int] * 5
        lib.po_coupled.restype = C.c_int
        lib.po_coupled.argtypes = [_chp, _chp, C.c_int, C.c_int]
        lib.po_A.restype = C.c_double
        lib.po_A.argtypes = [C.c_int] * 5 + [C.c_double] * 3 + [C.c_int]
        lib.po_G.restype = C.c_double
        lib.po_G.argtypes = [_chp, _chp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_int]
        lib.po_cell_nodes.restype = C.c_int
        lib.po_cell_nodes.argtypes = [_dp, C.c_int, _dp, C.c_int, C.c_int,
                                      _dp, _dp, C.c_int, _dp, _dp, C.c_int, _dp, _dp, C.c_int,
                                      _dp, _dp, _dp, _dp, _dp, _dp, _i32p]
        lib.po_build.restype = C.c_int
        lib.po_build.argtypes = [_dp, C.c_int, _dp, C.c_int, _chp, C.c_int, C.c_int, C.c_int, C.c_int,
                                 _dp, _dp, C.c_int, _dp, _dp, C.c_int, _dp, _dp, C.c_int,
                                 C.c_int, C.c_int, _i64p, _i32p, _dp, C.c_int64, _i64p]
        for name in ("po_build_norm", "po_build_xo"):
            f = getattr(lib, name)
            f.restype = C.c_int
            f.argtypes = lib.po_build.argtypes + [C.c_int]
        lib.po_hit_cells.restype = C.c_int
        lib.po_hit_cells.argtypes = [_dp, C.c_int, _dp, C.c_int, _dp, _dp, C.c_int, _dp, _dp, C.c_int, _dp, _dp, C.c_int,
                                     C.c_int, C.c_int, _i64p, _i32p, C.c_int64]
        lib.po_threads.restype = C.c_int
        lib.po_set_threads.argtypes = [C.c_int]

    # ---- scalar helpers (arguments of the Wigner symbols are DOUBLED integers) ----
    def wigner3j(self, *a):
        return self.lib.po_wigner3j(*a)

    def cg(self, *a):
        return self.lib.po_cg(*a)

    def wigner6j(self, *a):
        return self.lib.po_wigner6j(*a)

    def wigner9j(self, *a):
        return self.lib.po_wigner9j(*a)

    def ylm(self, l, m, ux, uz):
        return self.lib.po_ylm(l, m, ux, uz)

    @staticmethod
    def _ch(rec):
        return _Channel(*(int(rec[k]) for k in ("l", "s", "j", "t", "lam", "I2")))

    def spin_R(self, s, sp, S2, set_=2):
        return self.lib.po_spin_R(s, sp, S2, set_)

    def recoupling_C(self, ch, L, S2, J2):
        return self.lib.po_recoupling_C(C.byref(self._ch(ch)), L, S2, J2)

    def coef_L(self, cha, chb, L, J2, T2, stat, set_=2):
        return self.lib.po_coef_L(C.byref(self._ch(cha)), C.byref(self._ch(chb)), L, J2, T2, stat, set_)

    def coupled(self, cha, chb, J2, stat):
        return bool(self.lib.po_coupled(C.byref(self._ch(cha)), C.byref(self._ch(chb)), J2, stat))

    def A(self, l, lam, lp, lamp, L, p, q, x, set_=2):
        return self.lib.po_A(l, lam, lp, lamp, L, p, q, x, set_)

    def G(self, cha, chb, J2, T2, stat, p, q, x, set_=2):
        """One cyclic term G^(set); the matrix uses 2*G^(2)."""
        return self.lib.po_G(C.byref(self._ch(cha)), C.byref(self._ch(chb)), J2, T2, stat, p, q, x, set_)

    def threads(self):
        return self.lib.po_threads()

    def set_threads(self, n):
        self.lib.po_set_threads(int(n))

    # ---- per-node table of one source cell ----
    def cell_nodes(self, wl, cell):
        n = wl.nodes_per_cell
        out = {k: np.empty(n, dtype=np.float64) for k in ("p", "q", "x", "w", "pp", "qq")}
        tgt = np.empty(n, dtype=np.int32)
        (tp, wp), (tq, wq), (tx, wx) = wl.rules["p"], wl.rules["q"], wl.rules["x"]
        self.lib.po_cell_nodes(_d(wl.p_edges), wl.Np, _d(wl.q_edges), wl.Nq, int(cell),
                               _d(tp), _d(wp), wl.n_p, _d(tq), _d(wq), wl.n_q, _d(tx), _d(wx), wl.n_x,
                               *(_d(out[k]) for k in ("p", "q", "x", "w", "pp", "qq")), tgt.ctypes.data_as(_i32p))
        out["target"] = tgt
        return out

    # ---- the build ----
    def build_csr(self, wl, cell_begin=0, cell_end=None, values=True, norm=0, exact_overlap=False):
        """CSR block of rows of source cells [cell_begin, cell_end): (rowptr int64, colidx int32, vals f64).
        norm: 0 = reading A (cell widths), 1 = reading B (p^2 dp measure); exact_overlap: the paper's 'double integral
        with variable limits' (po_build_xo) instead of node binning."""
        if cell_end is None:
            cell_end = wl.n_cells
        chs = np.ascontiguousarray(wl.channels)
        chp = chs.ctypes.data_as(_chp)
        (tp, wp), (tq, wq), (tx, wx) = wl.rules["p"], wl.rules["q"], wl.rules["x"]
        nrows = (cell_end - cell_begin) * wl.n_ch
        rowptr = np.zeros(nrows + 1, dtype=np.int64)
        nnz = C.c_int64(0)

        def call(col, val, cap):
            fn = self.lib.po_build_xo if exact_overlap else self.lib.po_build_norm
            rc = fn(_d(wl.p_edges), wl.Np, _d(wl.q_edges), wl.Nq, chp, wl.n_ch,
                    wl.J2, wl.T2, wl.statistics,
                    _d(tp), _d(wp), wl.n_p, _d(tq), _d(wq), wl.n_q, _d(tx), _d(wx), wl.n_x,
                    cell_begin, cell_end, rowptr.ctypes.data_as(_i64p), col, val, cap, C.byref(nnz), int(norm))
            if rc != 0:
                raise RuntimeError(f"po_build failed: {rc}")

        call(None, None, 0)
        if not values:
            return rowptr, None, None
        colidx = np.empty(nnz.value, dtype=np.int32)
        vals = np.empty(nnz.value, dtype=np.float64)
        call(colidx.ctypes.data_as(_i32p), _d(vals), nnz.value)
        return rowptr, colidx, vals

    # ---- the geometric pattern alone ----
    def hit_cells(self, wl, cell_begin=0, cell_end=None):
        """(hitptr int64[n+1], hitcell int32[]) — the ascending hit cells of every source cell of the range (no values)."""
        if cell_end is None:
            cell_end = wl.n_cells
        (tp, wp), (tq, wq), (tx, wx) = wl.rules["p"], wl.rules["q"], wl.rules["x"]
        hitptr = np.zeros(cell_end - cell_begin + 1, dtype=np.int64)

        def call(hc, cap):
            rc = self.lib.po_hit_cells(_d(wl.p_edges), wl.Np, _d(wl.q_edges), wl.Nq, _d(tp), _d(wp), wl.n_p, _d(tq), _d(wq), wl.n_q,
                                       _d(tx), _d(wx), wl.n_x, cell_begin, cell_end, hitptr.ctypes.data_as(_i64p), hc, cap)
            if rc != 0:
                raise RuntimeError(f"po_hit_cells failed: {rc}")

        call(None, 0)
        hitcell = np.empty(int(hitptr[-1]), dtype=np.int32)
        call(hitcell.ctypes.data_as(_i32p), hitcell.size)
        return hitptr, hitcell

    # ---- scattered source cells, one po_build call per cell, several calls at a time ----
    def build_cells(self, wl, cells, workers=None):
        """[(rowptr, colidx, vals)] of the single-cell blocks `cells`.  po_build's OpenMP loop runs over the source cells of
        ONE call, so a one-cell call uses one thread; here `workers` host threads (default: the OpenMP thread count) each
        issue one-cell calls (ctypes releases the GIL), every call single-threaded.  The arithmetic is po_build's, untouched."""
        from concurrent.futures import ThreadPoolExecutor
        workers = workers or self.threads()

        def one(c):
            self.lib.po_set_threads(1)             # the calling thread's own setting
            return self.build_csr(wl, int(c), int(c) + 1)

        if workers <= 1:
            return [one(c) for c in cells]
        with ThreadPoolExecutor(max_workers=workers) as ex:
            return list(ex.map(one, cells))
