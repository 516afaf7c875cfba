"""pm_rotate_apply_static — the one entry point of libpm that allocates nothing (its scratch is a static device array of
2 * PM_STATIC_MAX_M doubles), for callers that cannot call cudaMalloc (CUDA graph capture, serving loops).

Collected last on purpose (the suite runs with pytest -x): a failure here hides no other test.  Checked against the
existing path pm_rotate_apply (caller's d_work) on two calls in a row — the static array keeps the last call's contents —
and against the numpy oracle of eq. (20), at the tolerance the other iteration tests use (1e-11 of the
largest entry).  Runs alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_1508_07441_b200 import inputs as I

pytestmark = pytest.mark.gpu

PM_STATIC_MAX_M = 65536


@pytest.fixture(scope="module")
def api():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1508_07441_b200 import api as a
    a.lib()                                    # fails loudly if libpm.so is missing
    return a


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def test_rotate_apply_static_matches_the_existing_path(api, oracle):
    import torch
    from oracle import pm_iter_oracle as it
    wl = I.small_coupled(N=5, jmax=3, orders=(3, 4, 6), Nq=9)          # rectangular, 26 channels, M = 1170
    assert wl.M <= PM_STATIC_MAX_M
    lat = api.Lattice(wl)
    rp, ci, v = lat.build_fused()                                       # (creates the lattice's device tables)
    rpo, cio, vo = oracle.build_csr(wl)
    work = torch.empty(2 * wl.M, dtype=torch.float64, device="cuda")
    for call, seed in enumerate((23, 24)):                              # two calls in a row, different inputs
        O, _, _, x = I.iteration_factors(wl, seed=seed)
        dO, dx = _dev(O), _dev(x)
        ref_dev = torch.empty(wl.M, dtype=torch.float64, device="cuda")
        api.pm_rotate_apply(lat.h, rp, ci, v, dO, dx, ref_dev, work)    # the existing path
        out = torch.full((wl.M,), float("nan"), dtype=torch.float64, device="cuda")
        mem0 = torch.cuda.mem_get_info()[0]
        api.pm_rotate_apply_static(lat.h, rp, ci, v, dO, dx, out)
        torch.cuda.synchronize()
        assert torch.cuda.mem_get_info()[0] == mem0, "the call changed the free device memory"
        got, ref = out.cpu().numpy(), ref_dev.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert np.max(np.abs(got - ref)) <= 1e-11 * np.max(np.abs(ref)), call
        ora = it.rotate_apply(rpo, cio, vo, O, x, wl.Np, wl.Nq, wl.n_ch)
        assert np.max(np.abs(got - ora)) <= 1e-11 * np.max(np.abs(ora)), call
    lat.close()


def test_rotate_apply_static_rejects_what_it_cannot_take(api):
    import torch
    # no device tables yet: the call must not create them (it allocates nothing)
    wl = I.small_coupled(N=4, jmax=2, orders=(2, 2, 4))
    lat = api.Lattice(wl)
    z = torch.zeros(wl.M, dtype=torch.float64, device="cuda")
    z2 = torch.zeros_like(z)
    rp = torch.zeros(wl.M + 1, dtype=torch.int64, device="cuda")
    ci = torch.zeros(1, dtype=torch.int32, device="cuda")
    O = torch.zeros(wl.n_ch * wl.Np * wl.Np, dtype=torch.float64, device="cuda")
    with pytest.raises(api.PmError) as e:
        api.pm_rotate_apply_static(lat.h, rp, ci, z, O, z, z2)
    assert e.value.code == -7 and "allocates nothing" in str(e.value)
    lat.close()
    # beyond the static scratch: a clear error, nothing launched
    big = I.small_coupled(N=52, jmax=3, orders=(2, 2, 4))               # M = 52*52*26 = 70304 > 65536
    assert big.M > PM_STATIC_MAX_M
    lb = api.Lattice(big)
    lb.pattern(0, 1)                                                    # device tables exist
    zb = torch.zeros(big.M, dtype=torch.float64, device="cuda")
    zb2 = torch.zeros_like(zb)
    rpb = torch.zeros(big.M + 1, dtype=torch.int64, device="cuda")
    Ob = torch.zeros(big.n_ch * big.Np * big.Np, dtype=torch.float64, device="cuda")
    with pytest.raises(api.PmError) as e:
        api.pm_rotate_apply_static(lb.h, rpb, ci, zb, Ob, zb, zb2)
    assert e.value.code == -8 and "PM_STATIC_MAX_M" in str(e.value)
    lb.close()
