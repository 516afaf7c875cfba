"""CPU-only checks of libpm: the C ABI loads, exports every symbol include/pm.h declares, validates its
inputs, and its host precompute (coupling mask, Gauss-Legendre rules) agrees with the oracle / numpy.
No compute entry point is exercised here (there is no GPU); they must fail loudly with PM_ERR_DEVICE."""
import os
import re

import numpy as np
import pytest

from paper_1508_07441_b200 import api, inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    from paper_1508_07441_b200.csrc import build
    build.build()


def _create(wl, **over):
    kw = dict(p_edges=wl.p_edges, q_edges=wl.q_edges, channels=wl.channels, J2=wl.J2, parity=wl.parity, T2=wl.T2,
              statistics=wl.statistics, n_p=wl.n_p, n_q=wl.n_q, n_x=wl.n_x)
    kw.update(over)
    return api.pm_lattice_create(**kw)


def test_every_declared_symbol_is_exported():
    hdr = open(os.path.join(ROOT, "include", "pm.h")).read()
    declared = set(re.findall(r"\b(pm_[a-z_]+)\s*\(", hdr))
    assert declared == set(api.EXPORTS)
    L = api.lib()
    for name in declared:
        assert hasattr(L, name), name


def test_dims_and_coupling_match_oracle(oracle):
    for k in range(5):
        wl = I.config(k)
        h = _create(wl)
        assert api.pm_lattice_dims(h) == (wl.M, wl.n_cells)
        mask, nfun = api.pm_lattice_coupling(h, wl.n_ch)
        ref = np.array([[oracle.coupled(a, b, wl.J2, wl.statistics) for b in wl.channels] for a in wl.channels])
        assert np.array_equal(mask, ref)
        assert nfun == [1, 1, 73, 140, 140][k]       # 74 / 141 of SURVEY.md minus one whose c^L cancels exactly
        api.pm_lattice_destroy(h)


def test_library_gauss_legendre_vs_numpy():
    wl = I.config(0)
    for n in (1, 2, 5, 10, 32, 64):
        h = _create(wl, n_p=1, n_q=2, n_x=n)
        t, w = api.pm_lattice_rule(h, 2, n)
        tr, wr = np.polynomial.legendre.leggauss(n)
        assert np.max(np.abs(t - tr)) < 2e-15 and np.max(np.abs(w - wr)) < 1e-14
        assert np.all(t == -t[::-1])
        api.pm_lattice_destroy(h)


def test_set_rule_validation():
    wl = I.config(0)
    h = _create(wl)
    t, w = wl.rules["x"]
    api.pm_lattice_set_rule(h, 2, t, w)
    with pytest.raises(api.PmError) as e:
        api.pm_lattice_set_rule(h, 2, t + 0.01, w)          # asymmetric x-rule
    assert e.value.code == -4
    with pytest.raises(api.PmError):
        api.pm_lattice_set_rule(h, 0, t[::-1].copy()[: wl.n_p], w[: wl.n_p])   # decreasing nodes
    api.pm_lattice_destroy(h)


@pytest.mark.parametrize("over,code", [
    (dict(p_edges=np.array([0.0, 1.0, 1.0, 2.0])), -2),
    (dict(p_edges=np.array([-0.1, 1.0, 2.0])), -2),
    (dict(q_edges=np.array([0.0, np.nan, 2.0])), -2),
    (dict(n_x=0), -4),
    (dict(n_p=65), -4),
    (dict(n_p=64, n_q=64, n_x=64), -4),
    (dict(parity=-1), -3),
    (dict(channels=np.array([(0, 0, 0, 0, 0, 1)], dtype=I.CH_DTYPE)), -3),       # Pauli-forbidden
    (dict(channels=np.array([(0, 1, 1, 0, 0, 1), (0, 1, 1, 0, 0, 1)], dtype=I.CH_DTYPE)), -3),   # duplicate
    (dict(channels=np.array([(0, 1, 1, 0, 2, 3)], dtype=I.CH_DTYPE), J2=7), -3),  # triangle (j I J)
    (dict(statistics=7), -3),
])
def test_create_rejects_bad_input(over, code):
    wl = I.config(1)
    with pytest.raises(api.PmError) as e:
        _create(wl, **over)
    assert e.value.code == code
    assert str(e.value)


def test_lattice_size_limit():
    g, g2 = I.tan_grid(512, 1.0), I.tan_grid(513, 1.0)
    with pytest.raises(api.PmError) as e:
        api.pm_lattice_create(g2, g, I.boson_channel(), 0, 1, 0, I.PM_SPINLESS_BOSON, 2, 2, 2)
    assert e.value.code == -2
    h = api.pm_lattice_create(g, g, I.boson_channel(), 0, 1, 0, I.PM_SPINLESS_BOSON, 2, 2, 2)
    assert api.pm_lattice_dims(h) == (262144, 262144)
    api.pm_lattice_destroy(h)


def test_compute_calls_fail_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    wl = I.config(0)
    h = _create(wl)

    class Fake:
        def data_ptr(self):
            return 256

        def numel(self):
            return 1
    with pytest.raises(api.PmError) as e:
        api.pm_pattern(h, 0, 1, Fake(), None, stream=0)
    assert e.value.code == -9
    with pytest.raises(api.PmError) as e:
        api.pm_build_host_count(h, 0)
    assert e.value.code in (-9, -6, -5)
    api.pm_lattice_destroy(h)


def test_fill_kernel_selection_and_work_model():
    """configs[0..4] select a generated (channel-specialised) fill kernel, in any channel ORDER (triples and functions
    are numbered canonically, so the ket tables do not depend on it); another channel SET is specialised at run time or,
    with that switched off, runs the table-driven kernel.  The work model is positive and grows with the set."""
    names, work = [], []
    for k in range(5):
        wl = I.config(k)
        h = _create(wl)
        names.append(api.pm_lattice_fill_kernel(h))
        work.append(api.pm_lattice_work(h))
        with pytest.raises(api.PmError) as e:
            api.pm_pattern_counts(h)
        assert e.value.code == -7
        api.pm_lattice_destroy(h)
    assert names == ["Spec_boson_s", "Spec_boson_s", "Spec_nnn_j2", "Spec_nnn_j3", "Spec_nnn_j3"]
    assert all(w[0] > 25 and w[1] > 0 and w[2] > 0 for w in work)                 # (weight 5 + directions 20 + ket code)
    assert work[4][0] > work[2][0] > work[1][0] and work[4][3] == 580 and work[2][3] == 276
    wl = I.config(2)
    h = _create(wl, channels=wl.channels[::-1].copy())
    assert api.pm_lattice_fill_kernel(h) == "Spec_nnn_j2"
    api.pm_lattice_destroy(h)
    h = _create(wl, channels=I.enumerate_3n_channels(1, +1, 1, 1))
    assert api.pm_lattice_fill_kernel(h) == "jit"             # specialised at run time (NVRTC) at the first fill
    api.pm_set_jit(False)
    try:
        assert api.pm_lattice_fill_kernel(h) == "generic"     # table-driven kernel when run-time compilation is off
    finally:
        api.pm_set_jit(True)
    api.pm_lattice_destroy(h)


def test_runtime_kernel_source_compiles_for_sm100a():
    """The source generated at run time for channel sets without a build-time kernel compiles with NVRTC for sm_100a
    (no GPU needed): J = 3/2-, the pair j <= 1 set of J = 1/2+ in reversed order, bosons with d-waves."""
    g7 = I.tan_grid(7, 1.0)
    cases = [
        I.Workload("3N_J3half-", g7, 0.9 * g7, I.enumerate_3n_channels(3, -1, 1, 1), 3, -1, 1, 0, 3, 4, 8),
        I.Workload("boson_dwave", g7, g7, np.concatenate([I.boson_channel(0, 0), I.boson_channel(2, 2)]), 0, +1, 0,
                   I.PM_SPINLESS_BOSON, 5, 5, 9),
    ]
    wl = I.config(2)
    wl.channels = I.enumerate_3n_channels(1, +1, 1, 1)[::-1].copy()
    cases.append(wl)
    for wl in cases:
        h = _create(wl)
        try:
            n = api.pm_diag_jit_compile(h)
        except api.PmError as e:
            if "libnvrtc not found" in str(e):
                pytest.skip("libnvrtc is not installed here")
            raise
        assert n > 10000
        api.pm_lattice_destroy(h)


def test_sqrt_threshold_is_the_exact_boundary():
    """'edge <= sqrt(y)'  <=>  'y >= thr(edge)' for IEEE doubles: checked on the neighbours of thr for every edge of the
    five lattices and for random edges (numpy's sqrt is correctly rounded)."""
    rng = np.random.default_rng(7)
    edges = np.concatenate([I.config(k).p_edges for k in range(5)] + [I.config(2).q_edges, rng.uniform(1e-6, 1e3, 2000),
                           10.0 ** rng.uniform(-12, 12, 2000)])
    for e in edges:
        t = api.pm_diag_sqrt_threshold(e)
        if e == 0.0:
            assert t == 0.0
            continue
        assert np.sqrt(t) >= e
        assert np.sqrt(np.nextafter(t, 0.0)) < e


def test_product_does_not_import_oracle():
    """The product path must never route through the oracle (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1508_07441_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".cpp", ".hpp", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "pm_oracle" not in src and "from oracle" not in src and "import oracle" not in src, f


def test_partition_cells_is_balanced_and_deterministic():
    """pm_partition_cells (host only): contiguous ranges, every cell in exactly one, loads within one cell of the mean,
    degenerate inputs (more parts than cells, zero hits, one part)."""
    rng = np.random.default_rng(5)
    for n, parts, cost in ((22500, 8, 40.0), (100, 3, 0.0), (5, 8, 1.0), (1, 1, 0.0), (0, 4, 1.0), (1000, 7, 0.5)):
        hits = rng.integers(0, 174, size=n).astype(np.int32)
        cuts = api.pm_partition_cells(hits, parts, cost)
        assert len(cuts) == parts + 1 and cuts[0] == 0 and cuts[-1] == n and np.all(np.diff(cuts) >= 0)
        assert np.array_equal(cuts, api.pm_partition_cells(hits.copy(), parts, cost))
        if n:
            w = hits + cost
            loads = np.array([w[cuts[r]:cuts[r + 1]].sum() for r in range(parts)])
            assert loads.sum() == pytest.approx(w.sum()) and loads.max() <= w.sum() / parts + w.max() + 1e-9
    with pytest.raises(api.PmError):
        api.pm_partition_cells(np.zeros(3, np.int32), 0)


def test_failing_calls_leave_a_message():
    """Every failing path across the ABI sets pm_last_error (also the streaming build of pm_stream.cu)."""
    import torch
    wl = I.config(0)
    h = _create(wl)
    L = api.lib()
    for call in (lambda: L.pm_build_host_count(h, 0, None, None),
                 lambda: L.pm_build_host(h, 0, None, None, None, 0, None, None),
                 lambda: L.pm_build_wait(h, None),
                 lambda: L.pm_pattern_cell_hits(h, None, None),
                 lambda: L.pm_rowptr_offset(None, 4, 1, None)):
        L.pm_lattice_dims(h, None, None)               # a succeeding call in between does not clear or set anything
        rc = call()
        assert rc != 0 and L.pm_last_error().decode() != "", rc
    if not torch.cuda.is_available():
        import ctypes as C
        nnz, nb = C.c_int64(), C.c_int32()
        buf = np.zeros(8, dtype=np.int64)
        rc = L.pm_build_host(h, 0, buf.ctypes.data, buf.ctypes.data, buf.ctypes.data, 1, C.byref(nnz), C.byref(nb))
        assert rc in (-9, -6, -5) and "CUDA" in L.pm_last_error().decode() or "device" in L.pm_last_error().decode()
    api.pm_lattice_destroy(h)


def test_attach_validates_like_create():
    wl = I.config(1)
    h = _create(wl)
    other = I.enumerate_3n_channels(3, -1, 1, 1)
    h2 = api.pm_lattice_attach(h, other, 3, -1, 1, 0)
    assert api.pm_lattice_dims(h2) == (wl.n_cells * len(other), wl.n_cells)
    with pytest.raises(api.PmError) as e:
        api.pm_lattice_attach(h, other, 3, +1, 1, 0)          # wrong parity for these channels
    assert e.value.code == -3
    api.pm_lattice_destroy(h)                                  # base first: the group lives on
    t, w = api.pm_lattice_rule(h2, 2, wl.n_x)
    assert len(t) == wl.n_x
    api.pm_lattice_destroy(h2)
