"""Pins of the oracle's node map, binning and matrix build.

Pins 1, 5, 6, 7, 8, 9, 10: phase-space conservation, symmetry convergence, spectrum bounds,
Monte-Carlo brute force, kinematic invariants, the paper's 'double integral with variable limits'
route, and the long-double instantiation.
"""
import math

import numpy as np
import pytest
import scipy.sparse as sp

from paper_1508_07441_b200 import inputs as I


def _csr(wl, oracle, **kw):
    rp, ci, v = oracle.build_csr(wl, **kw)
    return sp.csr_matrix((v, ci, rp), shape=(len(rp) - 1, wl.M))


def _boson(N, orders, c=1.0):
    g = I.tan_grid(N, c)
    return I.Workload(f"boson{N}", g, g, I.boson_channel(), 0, +1, 0, I.PM_SPINLESS_BOSON, *orders)


@pytest.mark.parametrize("k", [0, 1, 3])
def test_measure_conservation(oracle, k):
    """Pin 1 (north_star: 'the unweighted overlap measures of each row sum to the cell's p^2 q^2
    measure'): sum over ALL nodes (binned + escaped) of (1/2) w p^2 q^2 equals
    (p_i^3 - p_{i-1}^3)(q_j^3 - q_{j-1}^3)/9 — Gauss-Legendre is exact for p^2, q^2."""
    wl = I.config(k)
    rng = np.random.default_rng(k)
    cells = set(rng.integers(0, wl.n_cells, size=12).tolist()) | {0, wl.n_cells - 1}
    for cell in cells:
        nd = oracle.cell_nodes(wl, cell)
        i, j = divmod(cell, wl.Nq)
        exact = (wl.p_edges[i + 1] ** 3 - wl.p_edges[i] ** 3) * (wl.q_edges[j + 1] ** 3 - wl.q_edges[j] ** 3) / 9.0
        got = 0.5 * np.sum(nd["w"] * nd["p"] ** 2 * nd["q"] ** 2)
        assert abs(got - exact) <= 1e-13 * exact
        assert np.all((nd["target"] >= -1) & (nd["target"] < wl.n_cells))


def test_nodes_follow_the_stated_operation_order(oracle):
    """Reading R7: the node map re-evaluated here in numpy float64 with the same association
    reproduces the oracle's p', q' bit for bit, and the target cell is the half-open bin (R5)."""
    wl = I.config(1)
    (tp, wp), (tq, wq), (tx, wx) = wl.rules["p"], wl.rules["q"], wl.rules["x"]
    for cell in (0, 37, 1234, 2499):
        nd = oracle.cell_nodes(wl, cell)
        i, j = divmod(cell, wl.Nq)
        cp, hp = 0.5 * (wl.p_edges[i] + wl.p_edges[i + 1]), 0.5 * (wl.p_edges[i + 1] - wl.p_edges[i])
        cq, hq = 0.5 * (wl.q_edges[j] + wl.q_edges[j + 1]), 0.5 * (wl.q_edges[j + 1] - wl.q_edges[j])
        a, b, c = np.meshgrid(np.arange(wl.n_p), np.arange(wl.n_q), np.arange(wl.n_x), indexing="ij")
        p = (cp + hp * tp[a]).ravel(); q = (cq + hq * tq[b]).ravel(); x = tx[c].ravel()
        pq = p * q
        P2 = (0.25 * (p * p) + 0.5625 * (q * q)) + 0.75 * (pq * x)
        Q2 = ((p * p) + 0.25 * (q * q)) - pq * x
        pp, qq = np.sqrt(np.maximum(P2, 0)), np.sqrt(np.maximum(Q2, 0))
        assert np.array_equal(pp, nd["pp"]) and np.array_equal(qq, nd["qq"])
        ic = np.searchsorted(wl.p_edges, pp, side="right") - 1
        jc = np.searchsorted(wl.q_edges, qq, side="right") - 1
        ok = (ic >= 0) & (ic < wl.Np) & (jc >= 0) & (jc < wl.Nq) & (pp > 0) & (qq > 0)
        assert np.array_equal(np.where(ok, ic * wl.Nq + jc, -1), nd["target"])
        w = ((hp * wp[a]) * (hq * wq[b]) * wx[c]).ravel()
        assert np.array_equal(w, nd["w"])


def test_pattern_entries_obey_kinematic_invariants(oracle):
    """Pin 8: p'^2 + (3/4) q'^2 = p^2 + (3/4) q^2 (energy) and the triangle bounds, so every pattern
    entry couples cells whose energy intervals overlap.  Pins the constants 1/4, 9/16, 3/4."""
    wl = I.config(1)
    rp, ci, _ = oracle.build_csr(wl)
    pe, qe = wl.p_edges, wl.q_edges
    rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
    src, dst = rows // wl.n_ch, ci // wl.n_ch
    i, j, ic, jc = src // wl.Nq, src % wl.Nq, dst // wl.Nq, dst % wl.Nq
    Elo, Ehi = pe[i] ** 2 + 0.75 * qe[j] ** 2, pe[i + 1] ** 2 + 0.75 * qe[j + 1] ** 2
    Flo, Fhi = pe[ic] ** 2 + 0.75 * qe[jc] ** 2, pe[ic + 1] ** 2 + 0.75 * qe[jc + 1] ** 2
    assert np.all((Elo <= Fhi * (1 + 1e-14)) & (Flo <= Ehi * (1 + 1e-14)))
    # q' in [|p - q/2|, p + q/2] for some (p,q) of the source cell; p' in [|p/2 - 3q/4|, p/2 + 3q/4]
    assert np.all(qe[jc] <= pe[i + 1] + 0.5 * qe[j + 1])
    assert np.all(pe[ic] <= 0.5 * pe[i + 1] + 0.75 * qe[j + 1])
    # columns ascending within each row, rows of one source cell share the hit cells
    for r in (0, 1, 777, len(rp) - 2):
        cols = ci[rp[r]:rp[r + 1]]
        assert np.all(np.diff(cols) > 0)
    nd = oracle.cell_nodes(wl, 1300)
    hit = np.unique(nd["target"][nd["target"] >= 0])
    r0 = 1300 * wl.n_ch
    assert np.array_equal(np.unique(ci[rp[r0]:rp[r0 + 1]] // wl.n_ch), hit)


def test_block_builds_concatenate(oracle):
    wl = I.config(1)
    rp, ci, v = oracle.build_csr(wl, 100, 160)
    pieces = [oracle.build_csr(wl, a, b) for a, b in ((100, 101), (101, 130), (130, 160))]
    assert np.array_equal(np.concatenate([p[1] for p in pieces]), ci)
    assert np.array_equal(np.concatenate([p[2] for p in pieces]), v)
    assert rp[-1] == sum(p[0][-1] for p in pieces)


def test_long_double_instantiation_agrees(oracle, oracle_ld):
    """Pin 10: 80-bit value arithmetic changes no pattern entry and moves values by < 1e-13 rel."""
    wl = I.small_coupled(N=5, jmax=3, orders=(3, 3, 6))
    rp, ci, v = oracle.build_csr(wl)
    rpl, cil, vl = oracle_ld.build_csr(wl)
    assert np.array_equal(rp, rpl) and np.array_equal(ci, cil)
    assert np.max(np.abs(v - vl)) <= 1e-13 * np.max(np.abs(vl))


def _asym(A):
    A = A.toarray()
    return np.linalg.norm(A - A.T) / np.linalg.norm(A)


def test_symmetry_converges_with_order(oracle):
    """Pin 5: P0 = P0^T only in the limit of many nodes (one-sided quadrature of a discontinuous
    integrand); the asymmetry must fall monotonically.  Pins the Jacobian weight pq/(p'q') and the
    normalisation (d_i dbar_j d_i' dbar_j')^(-1/2) (reading R2-A)."""
    a = [_asym(_csr(_boson(10, o), oracle)) for o in ((4, 4, 8), (8, 8, 16), (16, 16, 32), (32, 32, 64))]
    assert a[0] > a[1] > a[2] > a[3]
    assert a[0] < 0.3 and a[3] < 1e-2 and a[3] < a[0] / 20, a


def test_spectrum_within_bounds(oracle):
    """Pin 6: P = c + c^2 has eigenvalues 2 and -1 only, so its compression to an orthonormal basis
    has spectrum in [-1, 2].  Fails for a wrong overall factor (16 pi^2, the factor 2) and for a
    non-orthonormal reading of eq. (21)."""
    for wl, lo, hi in (
        (_boson(10, (16, 16, 32)), 1.7, 2.05),
        (I.Workload("sw2", I.tan_grid(8, 1.0), I.tan_grid(8, 1.0), I.swave_3n_channels(), 1, 1, 1, 0, 12, 12, 24), 0.6, 2.05),
        (I.small_coupled(N=6, jmax=2, orders=(8, 8, 16)), 0.6, 2.05),
    ):
        A = _csr(wl, oracle).toarray()
        ev = np.linalg.eigvalsh(0.5 * (A + A.T))
        assert ev.min() > -1.05 and lo < ev.max() < hi, (wl.name, ev.min(), ev.max())


# ---- the integral being approximated, computed two other ways on a 4x4 lattice ------------------
def _exact_x_integral(p, q, plo, phi, qlo, qhi):
    """int dx 1/(p'(x) q'(x)) over {x in [-1,1]: p' in [plo,phi), q' in [qlo,qhi)} for fixed (p,q).
    p'^2 = a + b x and q'^2 = c - d x are linear in x, so the set is one interval and the primitive
    is elementary: 2/sqrt(bd) * asin(sqrt((x - al)/(be - al))), al = -a/b, be = c/d."""
    a, b = 0.25 * p * p + 0.5625 * q * q, 0.75 * p * q
    c, d = p * p + 0.25 * q * q, p * q
    x_lo = np.maximum.reduce([np.full_like(p, -1.0), (plo ** 2 - a) / b, (c - qhi ** 2) / d])
    x_hi = np.minimum.reduce([np.full_like(p, 1.0), (phi ** 2 - a) / b, (c - qlo ** 2) / d])
    al, be = -a / b, c / d
    F = lambda x: 2.0 / np.sqrt(b * d) * np.arcsin(np.sqrt(np.clip((x - al) / (be - al), 0.0, 1.0)))
    return np.where(x_hi > x_lo, F(x_hi) - F(x_lo), 0.0)


def _variable_limits_matrix(g, sub=24, order=6):
    """'a double integral with variable limits' — outer (p,q) by composite
    Gauss-Legendre on sub x sub panels per cell, inner x analytic.  s-wave bosons, G = 1."""
    N = len(g) - 1
    t, w = np.polynomial.legendre.leggauss(order)
    P = np.zeros((N * N, N * N))
    for i in range(N):
        for j in range(N):
            ep = np.linspace(g[i], g[i + 1], sub + 1); eq = np.linspace(g[j], g[j + 1], sub + 1)
            pn = (0.5 * (ep[:-1] + ep[1:])[:, None] + 0.5 * np.diff(ep)[:, None] * t[None, :]).ravel()
            pw = (0.5 * np.diff(ep)[:, None] * w[None, :]).ravel()
            qn = (0.5 * (eq[:-1] + eq[1:])[:, None] + 0.5 * np.diff(eq)[:, None] * t[None, :]).ravel()
            qw = (0.5 * np.diff(eq)[:, None] * w[None, :]).ravel()
            pg, qg = np.meshgrid(pn, qn, indexing="ij"); wg = pw[:, None] * qw[None, :]
            for ic in range(N):
                for jc in range(N):
                    val = np.sum(wg * pg * qg * _exact_x_integral(pg, qg, g[ic], g[ic + 1], g[jc], g[jc + 1]))
                    nrm = math.sqrt((g[i + 1] - g[i]) * (g[j + 1] - g[j]) * (g[ic + 1] - g[ic]) * (g[jc + 1] - g[jc]))
                    P[i * N + j, ic * N + jc] = val / nrm
    return P


def _monte_carlo_matrix(g, n_samples, seed):
    N = len(g) - 1
    rng = np.random.default_rng(seed)
    P = np.zeros((N * N, N * N)); E = np.zeros_like(P)
    for i in range(N):
        for j in range(N):
            p = rng.uniform(g[i], g[i + 1], n_samples); q = rng.uniform(g[j], g[j + 1], n_samples)
            x = rng.uniform(-1, 1, n_samples)
            pp = np.sqrt(0.25 * p * p + 0.5625 * q * q + 0.75 * p * q * x)
            qq = np.sqrt(p * p + 0.25 * q * q - p * q * x)
            ic = np.searchsorted(g, pp, side="right") - 1; jc = np.searchsorted(g, qq, side="right") - 1
            ok = (ic < N) & (jc < N)
            f = p * q / (pp * qq) * 2.0 * (g[i + 1] - g[i]) * (g[j + 1] - g[j])     # volume of the sample box
            tgt = (ic * N + jc)[ok]
            s1 = np.bincount(tgt, weights=f[ok], minlength=N * N) / n_samples
            s2 = np.bincount(tgt, weights=f[ok] ** 2, minlength=N * N) / n_samples
            dd = np.sqrt((g[i + 1] - g[i]) * (g[j + 1] - g[j]) * np.outer(np.diff(g), np.diff(g)).ravel())
            P[i * N + j] = s1 / dd
            E[i * N + j] = np.sqrt(np.maximum(s2 - s1 ** 2, 0) / n_samples) / dd
    return P, E


def test_integral_three_ways_on_4x4(oracle):
    """Pins 7 and 9: on a 4x4 lattice the oracle at high orders, a Monte-Carlo brute force
    (seed 12345) and the paper's variable-limits route agree on the integral itself."""
    wl = _boson(4, (48, 48, 96))
    g = wl.p_edges
    A = _csr(wl, oracle).toarray()
    V = _variable_limits_matrix(g)
    mc, err = _monte_carlo_matrix(g, 1_000_000, 12345)
    scale = np.abs(V).max()
    assert np.all(np.abs(mc - V) <= 5 * err + 2e-4 * scale)          # two independent routes to the integral
    assert np.abs(V - V.T).max() < 2e-5 * scale                      # the exact matrix IS symmetric
    assert np.abs(A - V).max() < 3e-3 * scale                        # node binning converges to it
    coarse = _csr(_boson(4, (12, 12, 24)), oracle).toarray()
    assert np.abs(A - V).max() < np.abs(coarse - V).max()
    assert np.array_equal(A != 0, V > 1e-9 * scale) or np.sum((A != 0) != (V > 1e-9 * scale)) <= 4


def test_oracle_reproduces_its_stored_rows(oracle):
    """Regression fixture written by tests/golden/make_cfg0_rows.py (oracle only): the oracle's arithmetic has not moved.
    A deliberate change of the oracle regenerates the file and says why in its commit message."""
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg0_rows.txt")
    stored = {}
    for ln in open(path):
        if ln.startswith("#"):
            continue
        c, col, hx, _ = ln.split()
        stored.setdefault(int(c), []).append((int(col), float.fromhex(hx)))
    wl = I.config(0)
    for c, entries in stored.items():
        rp, ci, v = oracle.build_csr(wl, c, c + 1)
        assert ci.tolist() == [e[0] for e in entries]
        ref = np.array([e[1] for e in entries])
        assert np.max(np.abs(v - ref)) <= 1e-15 * np.max(np.abs(ref))
