"""GPU parity: libpm (through the C ABI) against the CPU oracle on the same inputs.

Bar (BASELINE.json north_star): rowptr and colidx bit-exact; |dP| <= max(1e-11*|P_ref|, 1e-14*max|P|).
"""
import os

import numpy as np
import pytest

from paper_1508_07441_b200 import inputs as I

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

REL, FLOOR = 1e-11, 1e-14


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1508_07441_b200 import api as a
    a.lib()                                    # fails loudly if libpm.so is missing
    return a


def _assert_values(v_gpu, v_ref, scale=None):
    scale = np.max(np.abs(v_ref)) if scale is None else scale
    tol = np.maximum(REL * np.abs(v_ref), FLOOR * scale)
    bad = np.abs(v_gpu - v_ref) > tol
    assert not bad.any(), (int(bad.sum()), float(np.max(np.abs(v_gpu - v_ref) / tol)))


def _gpu_csr(api, wl, cb=0, ce=None):
    lat = api.Lattice(wl)
    rp, ci, v = lat.build(cb, ce)
    out = rp.cpu().numpy(), ci.cpu().numpy(), v.cpu().numpy()
    lat.close()
    return out


def _small_cases():
    g7 = I.tan_grid(7, 1.0)
    return [
        I.config(0),
        I.config(1),
        I.small_coupled(N=6, jmax=2, orders=(3, 3, 6)),
        I.small_coupled(N=7, jmax=3, orders=(4, 5, 7)),                   # ragged: odd orders, n_p != n_q
        I.Workload("boson_dwave", g7, g7, np.concatenate([I.boson_channel(0, 0), I.boson_channel(2, 2)]),
                   0, +1, 0, I.PM_SPINLESS_BOSON, 5, 5, 9),
        I.Workload("3N_J3half-", g7, 0.9 * g7, I.enumerate_3n_channels(3, -1, 1, 1), 3, -1, 1, 0, 3, 4, 8),
        I.Workload("offset_grid", 0.3 + g7, 0.2 + g7, I.swave_3n_channels(), 1, 1, 1, 0, 4, 4, 8),   # p_edges[0] > 0
        I.boson_lattice(5, 9, orders=(3, 4, 6), cp=1.0, cq=0.6),                                     # Np != Nq
        I.boson_lattice(9, 5, waves=((0, 0), (2, 2)), orders=(4, 3, 6), cp=0.7, cq=1.3),
        I.small_coupled(N=5, jmax=2, orders=(3, 4, 6), Nq=9),                                        # 18 channels, 5 x 9
        I.small_coupled(N=9, jmax=3, orders=(4, 3, 5), Nq=4),                                        # 26 channels, 9 x 4
        I.boson_lattice(6, 5, orders=(1, 4, 8), cq=0.9),                                             # n_p = 1 (reading R1)
        I.small_coupled(N=6, jmax=2, orders=(1, 5, 6), Nq=7),
        # 300 uniform p-cells: more than four sqrt-thresholds per bucket of the location table (the scanning locate path)
        I.Workload("uniform_fine_300x3", np.linspace(0.0, 1.2, 301), I.tan_grid(3, 1.0), I.boson_channel(), 0, +1, 0, I.PM_SPINLESS_BOSON, 2, 3, 4),
    ]


@pytest.mark.parametrize("wl", _small_cases(), ids=lambda w: w.name)
def test_full_parity_small(api, oracle, wl):
    rp, ci, v = _gpu_csr(api, wl)
    rpo, cio, vo = oracle.build_csr(wl)
    assert np.array_equal(rp, rpo)
    assert np.array_equal(ci, cio)
    _assert_values(v, vo)


@pytest.mark.parametrize("wl", [I.config(1), I.small_coupled(N=12, jmax=2, orders=(3, 4, 6), Nq=17)], ids=lambda w: w.name)
def test_block_ranges_and_empty(api, oracle, wl):
    lat = api.Lattice(wl)
    rp, ci, nnz = lat.pattern(7, 7)
    assert nnz == 0 and rp.cpu().tolist() == [0]
    n = wl.n_cells
    for cb, ce in ((0, 1), (17, 130), (n - 1, n), (n // 3, n // 3 + wl.Nq + 2)):
        rp, ci, v = lat.build(cb, ce)
        rpo, cio, vo = oracle.build_csr(wl, cb, ce)
        assert np.array_equal(rp.cpu().numpy(), rpo) and np.array_equal(ci.cpu().numpy(), cio)
        _assert_values(v.cpu().numpy(), vo)
    lat.close()


def test_bitwise_reproducible(api):
    wl = I.small_coupled(N=8, jmax=3, orders=(4, 4, 8))
    a = _gpu_csr(api, wl)
    b = _gpu_csr(api, wl)
    assert all(np.array_equal(x, y) for x, y in zip(a, b))


@pytest.mark.parametrize("jit", [True, False], ids=["jit", "generic"])
def test_kernels_for_channel_sets_without_a_build_time_kernel(api, oracle, jit):
    """A channel set with no build-time kernel (pair j <= 1, in reversed channel order) is specialised at run time
    (NVRTC) or, with that switched off, runs the table-driven fill; same bar for both, and both are what
    pm_lattice_fill_kernel reports."""
    wl = I.small_coupled(N=6, jmax=1, orders=(3, 4, 6))
    wl.channels = wl.channels[::-1].copy()
    api.pm_set_jit(jit)
    try:
        lat = api.Lattice(wl)
        rp, ci, v = lat.build()
        assert api.pm_lattice_fill_kernel(lat.h) == ("jit" if jit else "generic")
        rp2, ci2, v2 = lat.build_fused()
        assert torch_equal(rp, rp2) and torch_equal(ci, ci2) and torch_equal(v, v2)
    finally:
        api.pm_set_jit(True)
    rpo, cio, vo = oracle.build_csr(wl)
    assert np.array_equal(rp.cpu().numpy(), rpo) and np.array_equal(ci.cpu().numpy(), cio)
    _assert_values(v.cpu().numpy(), vo)
    lat.close()


def torch_equal(a, b):
    import torch
    return torch.equal(a, b)


@pytest.mark.parametrize("wl", [I.config(1), I.small_coupled(N=7, jmax=3, orders=(4, 5, 7))], ids=lambda w: w.name)
def test_pm_build_equals_pattern_plus_fill(api, wl):
    """pm_build (columns and values from one kernel) is bit-identical to pm_pattern + pm_fill."""
    lat = api.Lattice(wl)
    a = [t.cpu().numpy() for t in lat.build()]
    b = [t.cpu().numpy() for t in lat.build_fused()]
    assert all(np.array_equal(x, y) for x, y in zip(a, b))
    c = [t.cpu().numpy() for t in lat.build_fused(3, 11)]
    d = [t.cpu().numpy() for t in lat.build(3, 11)]
    assert all(np.array_equal(x, y) for x, y in zip(c, d))
    assert api.pm_last_fill_ms(lat.h) > 0.0
    lat.close()


@pytest.mark.parametrize("env", [{"PM_HIST_CAP": "8"}, {"PM_MAPSORT_WARPS": "1"}, {"PM_HIST_CAP": "5", "PM_MAPSORT_WARPS": "3"}],
                         ids=lambda e: "-".join(f"{k[3:].lower()}{v}" for k, v in e.items()))
def test_sort_windows_and_warp_counts(oracle, env):
    """k_map_sort counts and places the nodes rank window by rank window (512 counters per window: one window on every
    realistic lattice).  The test hook PM_HIST_CAP forces up to 14 windows per source cell of configs[1]; PM_MAPSORT_WARPS
    changes the warps (source cells in flight) per CTA.  Own process: the hooks are read once."""
    import subprocess
    import sys
    import tempfile
    code = (
        "import sys, numpy as np; sys.path.insert(0, %r)\n"
        "from paper_1508_07441_b200 import api, inputs\n"
        "wl = inputs.config(1); lat = api.Lattice(wl); rp, ci, v = lat.build_fused()\n"
        "np.savez(sys.argv[1], rp=rp.cpu().numpy(), ci=ci.cpu().numpy(), v=v.cpu().numpy())\n"
    ) % ROOT
    with tempfile.TemporaryDirectory() as d:
        out = os.path.join(d, "r.npz")
        subprocess.run([sys.executable, "-c", code, out], check=True, env=dict(os.environ, **env), timeout=600)
        r = np.load(out)
        rpo, cio, vo = oracle.build_csr(I.config(1))
        assert np.array_equal(r["rp"], rpo) and np.array_equal(r["ci"], cio)
        _assert_values(r["v"], vo)


def test_values_do_not_depend_on_the_block_shape(api):
    """One warp owns one source cell and sums in sorted node order, so the bits of every value are the same whatever the
    number of warps per block (PM_FILL_WARPS is read once per process: the 4-warp run is a subprocess)."""
    import subprocess
    import sys
    import tempfile
    wl = I.small_coupled(N=7, jmax=3, orders=(4, 5, 7))
    lat = api.Lattice(wl)
    rp, ci, v = (t.cpu().numpy() for t in lat.build_fused())
    lat.close()
    code = (
        "import sys, numpy as np; sys.path.insert(0, %r)\n"
        "from paper_1508_07441_b200 import api, inputs\n"
        "wl = inputs.small_coupled(N=7, jmax=3, orders=(4, 5, 7)); lat = api.Lattice(wl); rp, ci, v = lat.build_fused()\n"
        "np.savez(sys.argv[1], rp=rp.cpu().numpy(), ci=ci.cpu().numpy(), v=v.cpu().numpy())\n"
    ) % ROOT
    with tempfile.TemporaryDirectory() as d:
        out = os.path.join(d, "r.npz")
        subprocess.run([sys.executable, "-c", code, out], check=True, env=dict(os.environ, PM_FILL_WARPS="4"), timeout=600)
        r = np.load(out)
        assert np.array_equal(r["rp"], rp) and np.array_equal(r["ci"], ci) and np.array_equal(r["v"], v)


def test_pattern_counts(api):
    wl = I.config(1)
    lat = api.Lattice(wl)
    rp, ci, nnz = lat.pattern()
    nodes, segs, hits = api.pm_pattern_counts(lat.h)
    assert hits * 4 == nnz and hits <= segs <= nodes <= wl.n_cells * wl.nodes_per_cell
    assert nodes > 0.9 * wl.n_cells * wl.nodes_per_cell          # fewer than 10 % of the nodes leave the grid
    lat.close()


def test_fill_requires_pattern(api):
    import torch
    wl = I.config(0)
    lat = api.Lattice(wl)
    rp = torch.zeros(wl.M + 1, dtype=torch.int64, device="cuda")
    v = torch.zeros(10, dtype=torch.float64, device="cuda")
    with pytest.raises(api.PmError) as e:
        api.pm_fill(lat.h, 0, wl.n_cells, rp, v)
    assert e.value.code == -7
    lat.close()


def _sample_cells(wl, hits, n_total, seed):
    """Deterministic source cells for the full-size value check: the cells with the most and the fewest hit cells, the four
    corners, 24 evenly spaced cells on each edge of the lattice (i = 0 row, j = 0 column, last row, last column), then
    seeded random cells up to n_total."""
    Np, Nq = wl.Np, wl.Nq
    cells = [int(np.argmax(hits)), int(np.argmin(hits)), 0, Nq - 1, (Np - 1) * Nq, Np * Nq - 1]
    jj = np.unique(np.linspace(0, Nq - 1, 24).astype(int)); ii = np.unique(np.linspace(0, Np - 1, 24).astype(int))
    cells += [int(j) for j in jj] + [int(i) * Nq for i in ii] + [(Np - 1) * Nq + int(j) for j in jj] + [int(i) * Nq + Nq - 1 for i in ii]
    seen = sorted(set(cells))
    rng = np.random.default_rng(seed)
    while len(seen) < n_total:
        seen = sorted(set(seen) | set(rng.integers(0, wl.n_cells, size=n_total - len(seen)).tolist()))
    return seen


@pytest.mark.parametrize("k", [2, 3, 4])
def test_full_size_parity(api, oracle, k):
    """BASELINE configs[2..4] at full size, in the launch configuration bench.py times (pm_build, whole lattice, one block).
    Pattern: rowptr AND the whole colidx bit for bit — the expected column of every nonzero is expanded on the device from
    the oracle's hit-cell lists (po_hit_cells), the oracle's rowptr and the oracle's coupled mask.  Values: every entry of
    256 source cells (most / fewest hits, corners, lattice edges, seeded random cells) within the tolerance, with the
    absolute floor taken from the oracle's own values."""
    import torch
    wl = I.config(k)
    nc = wl.n_ch
    lat = api.Lattice(wl)
    rp, ci, v = lat.build_fused()                  # pm_build: the call bench.py times
    # ---- oracle side of the pattern
    hp_o, hc_o = oracle.hit_cells(wl)
    cmask = np.array([[oracle.coupled(a, b, wl.J2, wl.statistics) for b in wl.channels] for a in wl.channels])
    ncoup = cmask.sum(axis=1).astype(np.int64)
    hits = np.diff(hp_o)
    rp_o = np.concatenate([[0], np.cumsum((hits[:, None] * ncoup[None, :]).ravel())]).astype(np.int64)
    assert np.array_equal(rp_o, oracle.build_csr(wl, values=False)[0])            # po_build's own count pass agrees
    assert np.array_equal(rp.cpu().numpy(), rp_o)
    nnz = int(rp_o[-1])
    assert ci.numel() == nnz and v.numel() == nnz
    d = lambda a, dt: torch.from_numpy(np.ascontiguousarray(a)).to(device="cuda", dtype=dt)
    t_rp, t_hp, t_hc = d(rp_o, torch.int64), d(hp_o, torch.int64), d(hc_o, torch.int64)
    t_ncoup = d(ncoup, torch.int64)
    t_cloff = d(np.concatenate([[0], np.cumsum(ncoup)]), torch.int64)
    t_cl = d(np.concatenate([np.nonzero(cmask[a])[0] for a in range(nc)]), torch.int64)
    chunk = 1 << 26
    for e0 in range(0, nnz, chunk):
        e = torch.arange(e0, min(e0 + chunk, nnz), device="cuda", dtype=torch.int64)
        row = torch.searchsorted(t_rp, e, right=True) - 1
        local = e - t_rp[row]
        a = row % nc
        cell = row // nc
        kk = local // t_ncoup[a]
        m = local - kk * t_ncoup[a]
        col = t_hc[t_hp[cell] + kk] * nc + t_cl[t_cloff[a] + m]
        assert torch.equal(col.to(torch.int32), ci[e0:e0 + e.numel()]), (k, e0)
        del e, row, local, a, cell, kk, m, col
    assert bool(torch.isfinite(v).all())
    # ---- values of 256 source cells
    cells = _sample_cells(wl, hits, 256, 100 + k)
    ref = oracle.build_cells(wl, cells)
    scale = max(float(np.abs(vo).max()) for _, _, vo in ref)          # a lower bound of max|P| from the oracle alone: stricter floor
    rp_h = rp_o
    for c, (rpo, cio, vo) in zip(cells, ref):
        r0, r1 = c * nc, (c + 1) * nc
        assert np.array_equal(rp_h[r0:r1 + 1] - rp_h[r0], rpo)
        sl = slice(int(rp_h[r0]), int(rp_h[r1]))
        assert np.array_equal(ci[sl].cpu().numpy(), cio)
        _assert_values(v[sl].cpu().numpy(), vo, scale)
    lat.close()


def test_two_lattices_interleaved(api, oracle):
    """Two live lattices with the same channel set (same kernel function) and different grids, hence different shared-memory
    plans: fill A, then B (smaller), then A again.  The dynamic shared-memory limit is per kernel function."""
    A = I.small_coupled(N=12, jmax=2, orders=(5, 6, 12), Nq=11)
    B = I.small_coupled(N=4, jmax=2, orders=(2, 2, 4))
    la, lb = api.Lattice(A), api.Lattice(B)
    a1 = [t.cpu().numpy() for t in la.build_fused()]
    b1 = [t.cpu().numpy() for t in lb.build_fused()]
    a2 = [t.cpu().numpy() for t in la.build_fused()]
    b2 = [t.cpu().numpy() for t in lb.build()]
    assert all(np.array_equal(x, y) for x, y in zip(a1, a2)) and all(np.array_equal(x, y) for x, y in zip(b1, b2))
    rpo, cio, vo = oracle.build_csr(B)
    assert np.array_equal(b1[0], rpo) and np.array_equal(b1[1], cio)
    _assert_values(b1[2], vo)
    la.close(); lb.close()


def test_spmv_matches_scipy(api):
    import scipy.sparse as sp
    import torch
    wl = I.config(1)
    lat = api.Lattice(wl)
    rp, ci, v = lat.build()
    x = np.random.default_rng(2024).uniform(-1, 1, wl.M)
    y = lat.spmv(rp, ci, v, torch.from_numpy(x).cuda()).cpu().numpy()
    A = sp.csr_matrix((v.cpu().numpy(), ci.cpu().numpy(), rp.cpu().numpy()), shape=(wl.M, wl.M))
    assert np.max(np.abs(y - A @ x)) < 1e-12 * np.max(np.abs(y))
    lat.close()


@pytest.mark.parametrize("wl", [I.config(1), I.small_coupled(N=9, jmax=2, orders=(3, 4, 6), Nq=14)], ids=lambda w: w.name)
@pytest.mark.parametrize("budget_blocks", [1, 3, 17])
def test_streaming_build_identical(api, oracle, budget_blocks, wl):
    """Row-block streaming: identical CSR whatever the number of blocks (s-wave and a coupled-channel
    rectangular lattice)."""
    lat = api.Lattice(wl)
    nnz, _ = api.pm_build_host_count(lat.h, 1 << 40)
    budget = (1 << 40) if budget_blocks == 1 else int((12 * nnz + 4 * wl.nodes_per_cell * wl.n_cells) / budget_blocks) + 1   # CSR + node lists
    rp, ci, v, nnz2, nb = lat.build_host(budget, pinned=(budget_blocks != 3))
    assert nnz2 == nnz and (nb == 1 if budget_blocks == 1 else budget_blocks <= nb <= 2 * budget_blocks + 2)
    rpo, cio, vo = oracle.build_csr(wl)
    assert np.array_equal(rp.numpy(), rpo) and np.array_equal(ci.numpy(), cio)
    _assert_values(v.numpy(), vo)
    lat.close()


@pytest.mark.parametrize("wl", [I.config(1), I.small_coupled(N=6, jmax=2, orders=(3, 3, 6)),
                                I.small_coupled(N=5, jmax=3, orders=(3, 4, 6), Nq=9), I.boson_lattice(9, 5, orders=(4, 3, 6), cq=1.3)],
                         ids=lambda w: w.name)
def test_iteration_step_matches_oracle(api, oracle, wl):
    """K u = O P0 V~1 G1 u (eq. 24): pm_kernel_apply on the GPU-built P0 against the numpy oracle on the
    oracle-built P0, same seeded factors; also each block factor alone."""
    import torch
    from oracle import pm_iter_oracle as it
    O, V1, g1, u = I.iteration_factors(wl, seed=11)
    Vt = it.vtilde(O, V1)                                   # input data of the product path, formed by the caller
    rpo, cio, vo = oracle.build_csr(wl)
    ref = it.kernel_apply(rpo, cio, vo, O, V1, g1, u, wl.Np, wl.Nq, wl.n_ch)
    lat = api.Lattice(wl)
    rp, ci, v = lat.build_fused()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    dO, dVt, dg, du = dev(O), dev(Vt), dev(g1), dev(u)
    out = torch.empty(wl.M, dtype=torch.float64, device="cuda")
    work = torch.empty(2 * wl.M, dtype=torch.float64, device="cuda")
    api.pm_kernel_apply(lat.h, rp, ci, v, dO, dVt, dg, du, out, work)
    got = out.cpu().numpy()
    assert np.max(np.abs(got - ref)) <= 1e-11 * np.max(np.abs(ref))
    out2 = torch.empty_like(out)
    api.pm_kernel_apply(lat.h, rp, None, v, dO, dVt, dg, du, out2, work)     # columns implied by the hit lists
    assert torch.equal(out, out2)
    y1, y2 = torch.empty_like(out), torch.empty_like(out)
    api.pm_spmv(lat.h, rp, ci, v, du, y1)
    api.pm_spmv_implicit(lat.h, rp, v, du, y2)
    assert torch.equal(y1, y2)                                               # same lane striding, same bits
    lat.pattern(0, 3)                                                        # a partial pattern call drops the whole-lattice lists
    with pytest.raises(api.PmError) as e:
        api.pm_spmv_implicit(lat.h, rp, v, du, y2)
    assert e.value.code == -7
    api.pm_block_apply(lat.h, dO, None, du, out)
    assert np.max(np.abs(out.cpu().numpy() - it.block_apply(O, u, wl.Np, wl.Nq, wl.n_ch))) <= 1e-13 * np.max(np.abs(u)) * wl.Np
    api.pm_block_apply(lat.h, dVt, dg, du, out)
    assert np.max(np.abs(out.cpu().numpy() - it.block_apply(Vt, g1 * u, wl.Np, wl.Nq, wl.n_ch))) <= 1e-12 * np.max(np.abs(Vt)) * wl.Np
    lat.close()


def test_build_async_and_device_side_capacity_check(api, oracle):
    """pm_build_async queues pattern + fill without a host synchronisation; pm_build_wait returns nnz.  With a capacity
    below nnz the device-side check stops the fill: nothing is written and the wait reports PM_ERR_OVERFLOW."""
    import torch
    wl = I.small_coupled(N=6, jmax=2, orders=(3, 4, 6), Nq=7)
    lat = api.Lattice(wl)
    rp0, ci0, v0 = lat.build_fused()
    nnz = ci0.numel()
    rp = torch.empty_like(rp0); ci = torch.full_like(ci0, -7); v = torch.full_like(v0, -7.0)
    api.pm_build_async(lat.h, 0, wl.n_cells, rp, ci, v)
    assert api.pm_build_wait(lat.h) == nnz
    assert torch.equal(rp, rp0) and torch.equal(ci, ci0) and torch.equal(v, v0)
    ci_s = torch.full((nnz - 1,), -7, dtype=torch.int32, device="cuda"); v_s = torch.full((nnz - 1,), -7.0, dtype=torch.float64, device="cuda")
    api.pm_build_async(lat.h, 0, wl.n_cells, rp, ci_s, v_s)
    with pytest.raises(api.PmError) as e:
        api.pm_build_wait(lat.h)
    assert e.value.code == -8 and "too small" in str(e.value)
    torch.cuda.synchronize()
    assert bool((ci_s == -7).all()) and bool((v_s == -7.0).all())
    with pytest.raises(api.PmError) as e:                      # the synchronous call reports the same
        api.pm_build(lat.h, 0, wl.n_cells, rp, ci_s, v_s)
    assert e.value.code == -8
    lat.close()


@pytest.mark.parametrize("wl", [I.config(1), I.small_coupled(N=9, jmax=3, orders=(4, 3, 5), Nq=7)], ids=lambda w: w.name)
@pytest.mark.parametrize("world", [2, 3, 8])
def test_shards_concatenate_to_the_whole_build(api, wl, world):
    """contiguous source-cell ranges balanced by hit count, one shard per rank, the per-shard nnz turned
    into global row-pointer offsets.  Here the shards are built one after the other on one GPU and must concatenate, bit
    for bit, to the single-block build."""
    import torch
    lat = api.Lattice(wl)
    rp0, ci0, v0 = lat.build_fused()
    hits = api.pm_pattern_cell_hits(lat.h, wl.n_cells)
    assert hits.sum() * int(api.pm_lattice_coupling(lat.h, wl.n_ch)[0].sum()) == ci0.numel()
    cuts = api.pm_partition_cells(hits, world, cell_cost=2.0)
    assert cuts[0] == 0 and cuts[-1] == wl.n_cells and np.all(np.diff(cuts) >= 0)
    w = hits.astype(np.float64) + 2.0
    loads = np.array([w[cuts[r]:cuts[r + 1]].sum() for r in range(world)])
    assert loads.max() <= w.sum() / world + w.max()                 # balanced to within one cell
    parts, nnz_r = [], []
    for r in range(world):
        rp, ci, v = lat.build_fused(int(cuts[r]), int(cuts[r + 1]))
        parts.append((rp, ci, v)); nnz_r.append(ci.numel())
    offs = np.concatenate([[0], np.cumsum(nnz_r)])                   # what the all-gather of the per-rank nnz yields
    rows = []
    for r, (rp, ci, v) in enumerate(parts):
        api.pm_rowptr_offset(rp, int(offs[r]))
        rows.append(rp[:-1] if r < world - 1 else rp)
    assert torch.equal(torch.cat(rows), rp0)
    assert torch.equal(torch.cat([p[1] for p in parts]), ci0) and torch.equal(torch.cat([p[2] for p in parts]), v0)
    lat.close()


@pytest.mark.parametrize("wl", [I.small_coupled(N=6, jmax=2, orders=(3, 3, 6)), I.small_coupled(N=5, jmax=3, orders=(3, 4, 6), Nq=9)],
                         ids=lambda w: w.name)
def test_rotation_to_the_channel_basis(api, oracle, wl):
    """eq. (20), P = O P0 O^T: pm_rotate_apply on the GPU-built P0 against the numpy oracle on the
    oracle-built P0; the transposed block factor alone; with and without the column array."""
    import torch
    from oracle import pm_iter_oracle as it
    O, _, _, x = I.iteration_factors(wl, seed=23)
    rpo, cio, vo = oracle.build_csr(wl)
    ref = it.rotate_apply(rpo, cio, vo, O, x, wl.Np, wl.Nq, wl.n_ch)
    lat = api.Lattice(wl)
    rp, ci, v = lat.build_fused()
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    dO, dx = dev(O), dev(x)
    out = torch.empty(wl.M, dtype=torch.float64, device="cuda")
    work = torch.empty(2 * wl.M, dtype=torch.float64, device="cuda")
    api.pm_rotate_apply(lat.h, rp, ci, v, dO, dx, out, work)
    assert np.max(np.abs(out.cpu().numpy() - ref)) <= 1e-11 * np.max(np.abs(ref))
    out2 = torch.empty_like(out)
    api.pm_rotate_apply(lat.h, rp, None, v, dO, dx, out2, work)
    assert torch.equal(out, out2)
    api.pm_block_apply_t(lat.h, dO, dx, out)
    assert np.max(np.abs(out.cpu().numpy() - it.block_apply_t(O, x, wl.Np, wl.Nq, wl.n_ch))) <= 1e-13 * np.max(np.abs(x)) * wl.Np
    lat.close()


def test_attached_lattices_share_the_geometric_pattern(api, oracle):
    """several J^pi on one grid.  Lattices attached to a base share its node lists;
    pm_build_reuse maps and sorts the nodes once for the whole group (the launch counter shows it) and every member's CSR
    meets the oracle's."""
    import torch
    base = I.small_coupled(N=6, jmax=2, orders=(3, 4, 6), Nq=7)
    others = [I.small_coupled(N=6, jmax=2, orders=(3, 4, 6), Nq=7, J2=1, parity=-1),
              I.small_coupled(N=6, jmax=1, orders=(3, 4, 6), Nq=7, J2=3, parity=+1),
              I.small_coupled(N=6, jmax=1, orders=(3, 4, 6), Nq=7, J2=3, parity=-1)]
    lat = api.Lattice(base)
    hs = [api.pm_lattice_attach(lat.h, w.channels, w.J2, w.parity, w.T2, w.statistics) for w in others]
    results = []
    l0 = api.pm_launch_count()
    for h, w in zip([lat.h] + hs, [base] + others):
        rp = torch.empty(w.M + 1, dtype=torch.int64, device="cuda")
        nnz = api.pm_pattern(h, 0, w.n_cells, rp, None) if h is lat.h else None     # the base counts (and maps) first
        cap = base.n_cells * base.nodes_per_cell * w.n_ch * w.n_ch                   # an upper bound: no count needed
        ci = torch.empty(min(cap, 1 << 26), dtype=torch.int32, device="cuda"); v = torch.empty(ci.numel(), dtype=torch.float64, device="cuda")
        n = api.pm_build_reuse(h, 0, w.n_cells, rp, ci, v)
        assert nnz is None or nnz == n
        results.append((rp.cpu().numpy(), ci[:n].cpu().numpy(), v[:n].cpu().numpy()))
    launches = api.pm_launch_count() - l0
    # one map_sort in all (the base's count call); per member scan + rowptr + fill, plus the base's own scan + rowptr
    assert launches == 1 + 2 + 3 * 4, launches
    for (rp, ci, v), w in zip(results, [base] + others):
        rpo, cio, vo = oracle.build_csr(w)
        assert np.array_equal(rp, rpo) and np.array_equal(ci, cio)
        _assert_values(v, vo)
    for h in hs:
        api.pm_lattice_destroy(h)
    # the base still works after its group is gone, and pm_build (no reuse) maps afresh
    rp, ci, v = lat.build_fused()
    assert np.array_equal(ci.cpu().numpy(), results[0][1]) and np.array_equal(v.cpu().numpy(), results[0][2])
    lat.close()


JPI = [(3, -1), (17, +1)]                                   # run-time specialised kernels (3 + 13 of them: NVRTC takes a minute)
JPI_GENERIC = [(3, +1), (5, +1), (5, -1), (9, -1), (17, -1)]  # table-driven kernel, group by group


def test_every_Jpi_up_to_17_halves_on_one_grid(api, oracle):
    """SURVEY sec. 8(f) rank 3 ("up to 62 channels", L394 + Table 1 "all states ... up to J_max = 17/2"):
    the j <= 3 channel sets of J^pi = 3/2+- ... 17/2+- attached to one J = 1/2+ base lattice, built with pm_build_reuse
    (the geometric pattern is mapped once), element by element against the oracle.  Sets beyond one kernel's tables
    (up to 422 ket slots, 546 orbital functions, 3694 coupled channel pairs) run column-channel group by group, each group
    through its own run-time specialised kernel or, with that switched off, through the table-driven one."""
    import torch
    base = I.small_coupled(N=4, jmax=3, orders=(3, 2, 5), Nq=5)
    lat = api.Lattice(base)
    rp0, ci0, v0 = lat.build_fused()
    l0 = api.pm_launch_count()
    kinds = {}
    for J2, par in JPI:
        w = I.small_coupled(N=4, jmax=3, orders=(3, 2, 5), Nq=5, J2=J2, parity=par)
        h = api.pm_lattice_attach(lat.h, w.channels, w.J2, w.parity, w.T2, w.statistics)
        rpo, cio, vo = oracle.build_csr(w)
        rp = torch.empty(w.M + 1, dtype=torch.int64, device="cuda")
        ci = torch.empty(len(cio), dtype=torch.int32, device="cuda"); v = torch.empty(len(cio), dtype=torch.float64, device="cuda")
        n = api.pm_build_reuse(h, 0, w.n_cells, rp, ci, v)
        kinds[(J2, par)] = (w.n_ch, api.pm_lattice_fill_kernel(h))
        assert n == len(cio)
        assert np.array_equal(rp.cpu().numpy(), rpo) and np.array_equal(ci.cpu().numpy(), cio), (J2, par)
        _assert_values(v.cpu().numpy(), vo)
        api.pm_lattice_destroy(h)
    assert kinds[(17, +1)] == (62, "jit-grouped") and kinds[(3, -1)] == (46, "jit-grouped"), kinds
    assert max(k[0] for k in kinds.values()) == 62
    # the same with run-time compilation switched off: the table-driven kernel, group by group, same bar
    api.pm_set_jit(False)
    try:
        for J2, par in JPI_GENERIC:
            w = I.small_coupled(N=4, jmax=3, orders=(3, 2, 5), Nq=5, J2=J2, parity=par)
            h = api.pm_lattice_attach(lat.h, w.channels, w.J2, w.parity, w.T2, w.statistics)
            rpo, cio, vo = oracle.build_csr(w)
            rp = torch.empty(w.M + 1, dtype=torch.int64, device="cuda")
            ci = torch.empty(len(cio), dtype=torch.int32, device="cuda"); v = torch.empty(len(cio), dtype=torch.float64, device="cuda")
            assert api.pm_build_reuse(h, 0, w.n_cells, rp, ci, v) == len(cio)
            assert api.pm_lattice_fill_kernel(h) == "generic-grouped"
            assert np.array_equal(rp.cpu().numpy(), rpo) and np.array_equal(ci.cpu().numpy(), cio), (J2, par)
            _assert_values(v.cpu().numpy(), vo)
            api.pm_lattice_destroy(h)
    finally:
        api.pm_set_jit(True)
    lat.close()


@pytest.mark.parametrize("wl", [I.config(1), I.small_coupled(N=7, jmax=3, orders=(4, 5, 7), Nq=5),
                                I.boson_lattice(9, 5, waves=((0, 0), (2, 2)), orders=(4, 3, 6), cp=0.7, cq=1.3)], ids=lambda w: w.name)
def test_reading_B_normalisation(api, oracle, wl):
    """pm_lattice_set_normalisation(PM_NORM_P2): states normalised in the p^2 dp measure (reading R2-B): the same
    pattern, values against po_build_norm(norm = 1); switching back restores reading A bit for bit."""
    lat = api.Lattice(wl)
    a0 = [t.cpu().numpy() for t in lat.build_fused()]
    api.pm_lattice_set_normalisation(lat.h, 1)
    rp, ci, v = (t.cpu().numpy() for t in lat.build_fused())
    rpo, cio, vo = oracle.build_csr(wl, norm=1)
    assert np.array_equal(rp, rpo) and np.array_equal(ci, cio) and np.array_equal(rp, a0[0]) and np.array_equal(ci, a0[1])
    _assert_values(v, vo)
    assert np.max(np.abs(v - a0[2])) > 1e-3 * np.max(np.abs(vo))            # it is a different matrix
    api.pm_lattice_set_normalisation(lat.h, 0)
    a1 = [t.cpu().numpy() for t in lat.build_fused()]
    assert all(np.array_equal(x, y) for x, y in zip(a0, a1))
    with pytest.raises(api.PmError):
        api.pm_lattice_set_normalisation(lat.h, 7)
    lat.close()


@pytest.mark.parametrize("wl", [I.config(1), I.small_coupled(N=6, jmax=3, orders=(3, 4, 6), Nq=9),
                                I.boson_lattice(9, 5, waves=((0, 0), (2, 2)), orders=(4, 3, 6), cp=0.7, cq=1.3),
                                I.small_coupled(N=4, jmax=3, orders=(3, 2, 5), Nq=5, J2=3, parity=-1),
                                I.small_coupled(N=4, jmax=3, orders=(3, 2, 5), Nq=5, J2=17, parity=+1)], ids=lambda w: w.name)
def test_operator_form_applies_P0(api, oracle, wl):
    """The per-pair sums (operator form of P0): pm_operator_apply against y = P0 x with the ORACLE's
    CSR (scipy), for one kernel per set (2, 26 channels, bosons) and for sets built group by group (46 and 62 channels),
    both normalisations; bitwise reproducible; stale sums are refused (PM_ERR_STATE)."""
    import scipy.sparse as sp
    import torch
    lat = api.Lattice(wl)
    x = np.random.default_rng(77).uniform(-1, 1, wl.M)
    dx = torch.from_numpy(x).cuda()
    y = torch.empty(wl.M, dtype=torch.float64, device="cuda")
    with pytest.raises(api.PmError) as e:
        api.pm_operator_build(lat.h)                                    # no node lists yet
    assert e.value.code == -7
    lat.build_fused()
    with pytest.raises(api.PmError) as e:
        api.pm_operator_apply(lat.h, dx, y)                             # no sums yet
    assert e.value.code == -7
    for norm in (0, 1):
        api.pm_lattice_set_normalisation(lat.h, norm)
        if norm:
            with pytest.raises(api.PmError):
                api.pm_operator_apply(lat.h, dx, y)                     # the sums belong to the other normalisation
        pairs, nbytes = api.pm_operator_build(lat.h)
        rpo, cio, vo = oracle.build_csr(wl, norm=norm)
        assert pairs * int(api.pm_lattice_coupling(lat.h, wl.n_ch)[0].sum()) == len(vo) and nbytes >= 8 * pairs
        ref = sp.csr_matrix((vo, cio, rpo), shape=(wl.M, wl.M)) @ x
        api.pm_operator_apply(lat.h, dx, y)
        assert np.max(np.abs(y.cpu().numpy() - ref)) <= 1e-11 * np.max(np.abs(ref))
        y2 = torch.empty_like(y)
        api.pm_operator_apply(lat.h, dx, y2)
        assert torch.equal(y, y2)
    api.pm_lattice_set_normalisation(lat.h, 0)
    lat.build_fused()                                                   # a new pattern pass: the sums are stale
    with pytest.raises(api.PmError) as e:
        api.pm_operator_apply(lat.h, dx, y)
    assert e.value.code == -7
    lat.close()


def test_grouped_set_in_blocks_and_streamed(api, oracle):
    """A channel set filled group by group through the per-pair sums (46 channels, J = 3/2-): block ranges of source cells
    (pm_pattern + pm_fill without columns, pm_build with columns) and the streaming build with several blocks, all against
    the oracle and bit-identical to the whole build."""
    wl = I.small_coupled(N=5, jmax=3, orders=(3, 2, 5), Nq=6, J2=3, parity=-1)
    lat = api.Lattice(wl)
    rpo, cio, vo = oracle.build_csr(wl)
    rp, ci, v = lat.build_fused()
    assert api.pm_lattice_fill_kernel(lat.h) == "jit-grouped"
    assert np.array_equal(rp.cpu().numpy(), rpo) and np.array_equal(ci.cpu().numpy(), cio)
    _assert_values(v.cpu().numpy(), vo)
    whole = v.cpu().numpy()
    n = wl.n_cells
    for cb, ce in ((0, 7), (7, n), (n // 2, n // 2 + 1)):
        for build in (lat.build, lat.build_fused):
            rpb, cib, vb = build(cb, ce)
            rb, cb_, vb_ = oracle.build_csr(wl, cb, ce)
            assert np.array_equal(rpb.cpu().numpy(), rb) and np.array_equal(cib.cpu().numpy(), cb_)
            lo = int(rpo[cb * wl.n_ch])
            assert np.array_equal(vb.cpu().numpy(), whole[lo:lo + len(vb_)])
    for blocks in (1, 4):
        budget = (1 << 40) if blocks == 1 else int((12 * len(vo) + 12 * wl.nodes_per_cell * wl.n_cells) / blocks) + 1
        h_rp, h_ci, h_v, nnz, nb = lat.build_host(budget)
        assert nnz == len(vo) and nb >= blocks
        assert np.array_equal(h_rp.numpy(), rpo) and np.array_equal(h_ci.numpy(), cio) and np.array_equal(h_v.numpy(), whole)
    lat.close()
