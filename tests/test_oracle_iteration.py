"""Pins of the iteration-step oracle (oracle/pm_iter_oracle.py; eq. 24) — CPU only."""
import numpy as np

from oracle import pm_iter_oracle as it
from paper_1508_07441_b200 import inputs as I


def _dense_factors(wl, rp, ci, v, O, V1, g1):
    """K assembled entry by entry from explicit index loops (no reshapes, no einsum): the definition."""
    Np, Nq, nc, M = wl.Np, wl.Nq, wl.n_ch, wl.M
    r = lambda i, j, a: (i * Nq + j) * nc + a
    Of, Vf = np.zeros((M, M)), np.zeros((M, M))
    for a in range(nc):
        for j in range(Nq):
            for i in range(Np):
                for ip in range(Np):
                    Of[r(i, j, a), r(ip, j, a)] = O[a][i][ip]
                    Vf[r(i, j, a), r(ip, j, a)] = V1[a][i][ip]
    P = np.zeros((M, M))
    for row in range(M):
        for k in range(rp[row], rp[row + 1]):
            P[row, ci[k]] = v[k]
    return Of, Vf, P, np.diag(g1)


def test_kernel_apply_equals_dense_product(oracle):
    wl = I.small_coupled(N=4, jmax=1, orders=(2, 2, 4))
    rp, ci, v = oracle.build_csr(wl)
    O, V1, g1, u = I.iteration_factors(wl, seed=7)
    Of, Vf, P, G = _dense_factors(wl, rp, ci, v, O, V1, g1)
    K = Of @ P @ (Of.T @ Vf) @ G                      # eq. (24): K = O P0 (O^T V1) G1
    ref = K @ u
    got = it.kernel_apply(rp, ci, v, O, V1, g1, u, wl.Np, wl.Nq, wl.n_ch)
    assert np.max(np.abs(got - ref)) < 1e-12 * np.max(np.abs(ref))
    # P V1 G1 with P = O P0 O^T (eq. 20): the same operator
    ref2 = (Of @ P @ Of.T) @ Vf @ G @ u
    assert np.max(np.abs(got - ref2)) < 1e-12 * np.max(np.abs(ref))
    # eq. (20) alone: rotate_apply is the dense P = O P0 O^T, which has P0's spectrum (O is orthogonal)
    Pd = Of @ P @ Of.T
    rot = it.rotate_apply(rp, ci, v, O, u, wl.Np, wl.Nq, wl.n_ch)
    assert np.max(np.abs(rot - Pd @ u)) < 1e-12 * np.max(np.abs(Pd @ u))
    assert np.max(np.abs(Of @ Of.T - np.eye(wl.M))) < 1e-12
    e0, e1 = np.sort(np.linalg.eigvals(P).real), np.sort(np.linalg.eigvals(Pd).real)
    assert np.max(np.abs(e0 - e1)) < 1e-9 * np.max(np.abs(e0))
    # transposed blocks: <y, B x> = <B^T y, x>
    y = np.random.default_rng(5).uniform(-1, 1, wl.M)
    lhs = y @ it.block_apply(O, u, wl.Np, wl.Nq, wl.n_ch)
    rhs = it.block_apply_t(O, y, wl.Np, wl.Nq, wl.n_ch) @ u
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)


def test_identity_factors_reduce_to_the_spmv(oracle):
    wl = I.config(0)
    rp, ci, v = oracle.build_csr(wl)
    eye = np.stack([np.eye(wl.Np)] * wl.n_ch)
    u = np.random.default_rng(3).uniform(-1, 1, wl.M)
    got = it.kernel_apply(rp, ci, v, eye, eye, np.ones(wl.M), u, wl.Np, wl.Nq, wl.n_ch)
    import scipy.sparse as sp
    ref = sp.csr_matrix((v, ci, rp), shape=(wl.M, wl.M)) @ u
    assert np.max(np.abs(got - ref)) < 1e-13 * np.max(np.abs(ref))


def test_rotations_are_orthogonal_and_blocks_act_on_the_pair_index():
    wl = I.config(1)
    O, V1, g1, u = I.iteration_factors(wl)
    for a in range(wl.n_ch):
        assert np.max(np.abs(O[a] @ O[a].T - np.eye(wl.Np))) < 1e-13
        assert np.allclose(V1[a], V1[a].T)
    # a vector supported on one (j, alpha) stays on that (j, alpha)
    x = np.zeros(wl.M)
    j, a = 17, 1
    x[(np.arange(wl.Np) * wl.Nq + j) * wl.n_ch + a] = 1.0
    y = it.block_apply(O, x, wl.Np, wl.Nq, wl.n_ch).reshape(wl.Np, wl.Nq, wl.n_ch)
    mask = np.ones_like(y, dtype=bool)
    mask[:, j, a] = False
    assert np.all(y[mask] == 0.0) and np.allclose(y[:, j, a], O[a].sum(axis=1))
