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


# ---- po_build's coupled-channel assembly against the pinned coefficient po_G, node by node ---------------------
def _rebuild_from_G(wl, oracle):
    """Every CSR entry from its definition (eq. 21-22):
    P0[(ij a),(i'j' a')] = sum_{nodes of (i,j) landing in (i',j')} w * pq/(p'q') * 2*G2_{a a'}(p,q,x) / sqrt(d_i dbar_j d_i' dbar_j'),
    nodes from po_cell_nodes, the coefficient from po_G (one call per node and channel pair — nothing of po_build's
    own tables is used).  Returns a dict (row, col) -> value."""
    pe, qe, nc = wl.p_edges, wl.q_edges, wl.n_ch
    ch = wl.channels
    coupled = [[oracle.coupled(a, b, wl.J2, wl.statistics) for b in ch] for a in ch]
    out = {}
    for cell in range(wl.n_cells):
        i, j = divmod(cell, wl.Nq)
        nd = oracle.cell_nodes(wl, cell)
        for n in range(wl.nodes_per_cell):
            t = int(nd["target"][n])
            if t < 0:
                continue
            ic, jc = divmod(t, wl.Nq)
            p, q, x = float(nd["p"][n]), float(nd["q"][n]), float(nd["x"][n])
            om = nd["w"][n] * (p * q / (nd["pp"][n] * nd["qq"][n]))
            nrm = math.sqrt((pe[i + 1] - pe[i]) * (qe[j + 1] - qe[j]) * (pe[ic + 1] - pe[ic]) * (qe[jc + 1] - qe[jc]))
            for a in range(nc):
                for b in range(nc):
                    if coupled[a][b]:
                        key = (cell * nc + a, t * nc + b)
                        out[key] = out.get(key, 0.0) + om * 2.0 * oracle.G(ch[a], ch[b], wl.J2, wl.T2, wl.statistics, p, q, x, 2) / nrm
    return out


@pytest.mark.parametrize("wl", [
    I.small_coupled(N=4, jmax=3, orders=(2, 3, 4)),                            # 26 channels, unequal orders
    I.small_coupled(N=3, jmax=2, orders=(2, 2, 4), Nq=5),                      # 18 channels, Np != Nq
    I.small_coupled(N=3, jmax=1, orders=(2, 3, 4), Nq=4, J2=3, parity=-1),     # J = 3/2-, L up to 3
    I.boson_lattice(4, 6, waves=((0, 0), (2, 2)), J=0, orders=(3, 2, 5), cq=0.7),   # bosons with d-waves, Np != Nq
    I.boson_lattice(3, 3, waves=((0, 2), (2, 0), (2, 2)), J=2, orders=(2, 2, 4)),   # J = L = 2
    I.small_coupled(N=3, jmax=1, orders=(2, 2, 3), Nq=2, J2=9, parity=-1),          # J = 9/2-: lambda up to 6, L up to 6
], ids=lambda w: w.name)
def test_build_equals_node_sum_of_pinned_G(oracle, wl):
    """po_build has its own tabulated route to the coefficient (po_tables_init, po_eval_bipolar, tri_of / coef);
    po_G is the function pinned by tests/test_oracle_algebra.py (product-basis construction, sympy, scipy).  Here every
    entry of po_build's CSR is recomputed from po_cell_nodes and po_G alone and must agree to rounding: a swapped
    bra/ket triple, a lost 1/(2L+1), a wrong factor 2 or a transposed (alpha, alpha') in the assembly would fail.
    Cites eq. (21)-(22); DESIGN.md sec. 3.1 / 3.2."""
    rp, ci, v = oracle.build_csr(wl)
    ref = _rebuild_from_G(wl, oracle)
    assert len(ref) == len(v)                                   # same structural pattern: hit cells x coupled mask
    rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
    want = np.array([ref[(int(r), int(c))] for r, c in zip(rows, ci)])
    assert np.max(np.abs(v - want)) <= 1e-14 * np.max(np.abs(want)), np.max(np.abs(v - want)) / np.max(np.abs(want))
    assert np.max(np.abs(want)) > 1e-3


# ---- rectangular lattices (Np != Nq): every index formula that could mix the two axes --------------------------
RECT = [
    I.boson_lattice(5, 9, orders=(3, 4, 6), cp=1.0, cq=0.6),
    I.boson_lattice(9, 5, orders=(4, 3, 6), cp=0.7, cq=1.3),
    I.small_coupled(N=5, jmax=1, orders=(3, 2, 5), Nq=8),
]


@pytest.mark.parametrize("wl", RECT, ids=lambda w: w.name)
def test_rectangular_lattice_pins(oracle, wl):
    """Np != Nq: cell = i*Nq + j on both the source and the target side.  (1) measure conservation per source cell with
    the cell's own (i, j) = divmod(cell, Nq); (2) the target of every node re-derived in numpy with searchsorted on the
    p- and the q-edges separately; (3) the pattern of po_build is exactly {targets of the cell's nodes} x coupled mask,
    with row = cell*n_ch + a and column = target*n_ch + b; (4) energy invariant of every entry."""
    pe, qe, nc = wl.p_edges, wl.q_edges, wl.n_ch
    (tp, wp), (tq, wq), (tx, wx) = wl.rules["p"], wl.rules["q"], wl.rules["x"]
    rp, ci, v = oracle.build_csr(wl)
    assert len(rp) == wl.Np * wl.Nq * nc + 1
    cmask = np.array([[oracle.coupled(a, b, wl.J2, wl.statistics) for b in wl.channels] for a in wl.channels])
    for cell in range(wl.n_cells):
        i, j = divmod(cell, wl.Nq)
        nd = oracle.cell_nodes(wl, cell)
        exact = (pe[i + 1] ** 3 - pe[i] ** 3) * (qe[j + 1] ** 3 - qe[j] ** 3) / 9.0
        assert abs(0.5 * np.sum(nd["w"] * nd["p"] ** 2 * nd["q"] ** 2) - exact) <= 1e-13 * exact
        assert np.all((nd["p"] > pe[i]) & (nd["p"] < pe[i + 1]) & (nd["q"] > qe[j]) & (nd["q"] < qe[j + 1]))
        ic = np.searchsorted(pe, nd["pp"], side="right") - 1
        jc = np.searchsorted(qe, nd["qq"], side="right") - 1
        ok = (ic >= 0) & (ic < wl.Np) & (jc >= 0) & (jc < wl.Nq) & (nd["pp"] > 0) & (nd["qq"] > 0)
        tgt = np.where(ok, ic * wl.Nq + jc, -1)
        assert np.array_equal(tgt, nd["target"])
        hit = np.unique(tgt[tgt >= 0])
        for a in range(nc):
            r = cell * nc + a
            want = (hit[:, None] * nc + np.nonzero(cmask[a])[0][None, :]).ravel()
            assert np.array_equal(ci[rp[r]:rp[r + 1]], want)
    rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
    src, dst = rows // nc, ci // nc
    i, j, ic, jc = src // wl.Nq, src % wl.Nq, dst // wl.Nq, dst % wl.Nq
    assert ic.max() < wl.Np and jc.max() < wl.Nq
    Elo, Ehi = pe[i] ** 2 + 0.75 * qe[j] ** 2, pe[i + 1] ** 2 + 0.75 * qe[j + 1] ** 2
    Flo, Fhi = pe[ic] ** 2 + 0.75 * qe[jc] ** 2, pe[ic + 1] ** 2 + 0.75 * qe[jc + 1] ** 2
    assert np.all((Elo <= Fhi * (1 + 1e-14)) & (Flo <= Ehi * (1 + 1e-14)))


def test_rectangular_transpose_symmetry(oracle):
    """The exact s-wave matrix is symmetric; at high orders the node-binned one on a 4 x 6 lattice approaches its own
    transpose — an (i, j) / (i', j') index mix-up between the axes would not."""
    a = [_asym(_csr(I.boson_lattice(4, 6, orders=o, cq=0.8), oracle)) for o in ((6, 6, 12), (24, 24, 48))]
    assert a[1] < a[0] / 4 and a[1] < 2e-2, a


def test_single_p_node_is_the_two_axis_rule(oracle):
    """Reading R1: n_p = 1 (the midpoint of the p-cell, weight = the cell width) is north_star's literal 'quadrature in q
    and x'.  The node table has p = the cell midpoint for every node, weights (d_i)(hq wq_b) wx_c, and po_build of the
    s-wave boson lattice equals the direct node sum."""
    wl = I.boson_lattice(5, 4, orders=(1, 3, 6), cq=0.9)
    pe, qe = wl.p_edges, wl.q_edges
    (tq, wq), (tx, wx) = wl.rules["q"], wl.rules["x"]
    assert wl.rules["p"][0].tolist() == [0.0] and wl.rules["p"][1].tolist() == [2.0]
    A = _csr(wl, oracle).toarray()
    B = np.zeros_like(A)
    for cell in range(wl.n_cells):
        i, j = divmod(cell, wl.Nq)
        nd = oracle.cell_nodes(wl, cell)
        assert np.all(nd["p"] == 0.5 * (pe[i] + pe[i + 1]))
        b, c = np.meshgrid(np.arange(wl.n_q), np.arange(wl.n_x), indexing="ij")
        w = ((0.5 * (pe[i + 1] - pe[i]) * 2.0) * (0.5 * (qe[j + 1] - qe[j]) * wq[b]) * wx[c]).ravel()
        assert np.array_equal(w, nd["w"])
        for n in np.nonzero(nd["target"] >= 0)[0]:
            t = nd["target"][n]
            ic, jc = divmod(int(t), wl.Nq)
            nrm = math.sqrt((pe[i + 1] - pe[i]) * (qe[j + 1] - qe[j]) * (pe[ic + 1] - pe[ic]) * (qe[jc + 1] - qe[jc]))
            B[cell, t] += nd["w"][n] * nd["p"][n] * nd["q"][n] / (nd["pp"][n] * nd["qq"][n]) / nrm
    assert np.max(np.abs(A - B)) <= 1e-14 * np.max(np.abs(B))


@pytest.mark.parametrize("wl", [I.config(1), RECT[0], RECT[2]], ids=lambda w: w.name)
def test_hit_cells_is_the_geometric_pattern(oracle, wl):
    """po_hit_cells (pattern without values) against the node table (unique targets per source cell) and against the
    column indices of po_build; sub-ranges are slices of the whole."""
    hp, hc = oracle.hit_cells(wl)
    rp, ci, _ = oracle.build_csr(wl)
    nc = wl.n_ch
    assert hp[0] == 0 and len(hp) == wl.n_cells + 1 and hp[-1] == len(hc)
    for cell in range(0, wl.n_cells, max(1, wl.n_cells // 97)):
        t = oracle.cell_nodes(wl, cell)["target"]
        assert np.array_equal(hc[hp[cell]:hp[cell + 1]], np.unique(t[t >= 0]))
        assert np.array_equal(np.unique(ci[rp[cell * nc]:rp[cell * nc + 1]] // nc), hc[hp[cell]:hp[cell + 1]])
    b, e = wl.n_cells // 5, wl.n_cells // 2
    hp2, hc2 = oracle.hit_cells(wl, b, e)
    assert np.array_equal(hp2, hp[b:e + 1] - hp[b]) and np.array_equal(hc2, hc[hp[b]:hp[e]])
    assert oracle.hit_cells(wl, 3, 3)[0].tolist() == [0]


def test_build_cells_is_build_csr_per_cell(oracle):
    wl = I.small_coupled(N=5, jmax=2, orders=(3, 3, 5), Nq=6)
    cells = [0, 7, 29, 13]
    for (rp, ci, v), c in zip(oracle.build_cells(wl, cells, workers=3), cells):
        rp2, ci2, v2 = oracle.build_csr(wl, c, c + 1)
        assert np.array_equal(rp, rp2) and np.array_equal(ci, ci2) and np.array_equal(v, v2)


# ---- reading-B normalisation and the exact-overlap ("variable limits") evaluation ------
def _variable_limits_matrix_B(g, sub=16, order=6):
    """Reading B for s-wave bosons (G = 1): P = int p^2 dp q^2 dq (length of the x-interval landing in the target cell)
    / sqrt(B_i B_j B_i' B_j'), B_k = (g[k+1]^3 - g[k]^3)/3.  Outer composite Gauss-Legendre, inner x exact."""
    N = len(g) - 1
    t, w = np.polynomial.legendre.leggauss(order)
    Bk = (g[1:] ** 3 - g[:-1] ** 3) / 3.0
    P = np.zeros((N * N, N * N))
    for i in range(N):
        for j in range(N):
            ep = np.linspace(g[i], g[i + 1], sub + 1); eq = np.linspace(g[j], g[j + 1], sub + 1)
            pn = (0.5 * (ep[:-1] + ep[1:])[:, None] + 0.5 * np.diff(ep)[:, None] * t[None, :]).ravel()
            pw = (0.5 * np.diff(ep)[:, None] * w[None, :]).ravel()
            qn = (0.5 * (eq[:-1] + eq[1:])[:, None] + 0.5 * np.diff(eq)[:, None] * t[None, :]).ravel()
            qw = (0.5 * np.diff(eq)[:, None] * w[None, :]).ravel()
            pg, qg = np.meshgrid(pn, qn, indexing="ij"); wg = pw[:, None] * qw[None, :]
            a, b = 0.25 * pg * pg + 0.5625 * qg * qg, 0.75 * pg * qg
            c, d = pg * pg + 0.25 * qg * qg, pg * qg
            for ic in range(N):
                for jc in range(N):
                    lo = np.maximum.reduce([np.full_like(pg, -1.0), (g[ic] ** 2 - a) / b, (c - g[jc + 1] ** 2) / d])
                    hi = np.minimum.reduce([np.full_like(pg, 1.0), (g[ic + 1] ** 2 - a) / b, (c - g[jc] ** 2) / d])
                    val = np.sum(wg * pg ** 2 * qg ** 2 * np.maximum(hi - lo, 0.0))
                    P[i * N + j, ic * N + jc] = val / math.sqrt(Bk[i] * Bk[j] * Bk[ic] * Bk[jc])
    return P


def test_reading_B_and_exact_overlap_on_4x4(oracle):
    """Pins of po_build_norm(norm = 1) and po_build_xo (PAPER.md:L215 'double integral with variable limits') on the 4x4
    s-wave lattice, against numpy routes that share nothing with the oracle:
    * reading A, exact overlap  vs  the variable-limits matrix (inner x analytic) of test_integral_three_ways_on_4x4;
    * reading B, exact overlap  vs  the same route with weight p^2 q^2 (inner x exact: the interval length);
    * node binning in reading B converges to it; both readings give spectra inside [-1, 2];
    * at equal orders the exact-overlap matrix is far more symmetric than the node-binned one."""
    g = I.tan_grid(4, 1.0)
    VA, VB = _variable_limits_matrix(g), _variable_limits_matrix_B(g)
    xo = I.boson_lattice(4, 4, orders=(48, 48, 32))
    XA = _csr(xo, oracle, exact_overlap=True).toarray()
    XB = _csr(xo, oracle, exact_overlap=True, norm=1).toarray()
    # (the interval length is only piecewise smooth in (p, q): the outer rule converges algebraically; 3.5e-4 / 8e-5 observed)
    assert np.abs(XA - VA).max() < 1e-3 * np.abs(VA).max()
    assert np.abs(XB - VB).max() < 2.5e-4 * np.abs(VB).max()
    coarse = I.boson_lattice(4, 4, orders=(24, 24, 16))
    assert np.abs(XB - VB).max() < np.abs(_csr(coarse, oracle, exact_overlap=True, norm=1).toarray() - VB).max()
    assert np.abs(VB - VB.T).max() < 1e-4 * np.abs(VB).max()                 # the exact reading-B matrix is symmetric too
    hi = I.boson_lattice(4, 4, orders=(48, 48, 96))
    BB = _csr(hi, oracle, norm=1).toarray()
    assert np.abs(BB - VB).max() < 3e-3 * np.abs(VB).max()
    for M in (XA, XB, BB):
        ev = np.linalg.eigvalsh(0.5 * (M + M.T))
        assert ev.min() > -1.05 and 1.2 < ev.max() < 2.05
    lo_orders = I.boson_lattice(4, 4, orders=(8, 8, 8))
    assert _asym(_csr(lo_orders, oracle, exact_overlap=True)) < 0.2 * _asym(_csr(lo_orders, oracle))
    # patterns: every node-binned entry lies inside the exact-overlap pattern (a node that lands in a cell proves the overlap)
    pa = _csr(I.boson_lattice(4, 4, orders=(8, 8, 8)), oracle).toarray() != 0
    px = _csr(I.boson_lattice(4, 4, orders=(8, 8, 8)), oracle, exact_overlap=True).toarray() != 0
    assert np.all(px[pa])


def _rebuild_xo_from_G(wl, oracle, norm):
    """Every entry of the exact-overlap matrix from its definition: outer nodes (p, q) of the source cell, the x-interval
    landing in the target cell from the two linear maps p'^2 = A + Bx, q'^2 = C - Dx, the n_x-point rule mapped to it,
    the coefficient from po_G.  numpy + po_G only."""
    pe, qe, nc = wl.p_edges, wl.q_edges, wl.n_ch
    (tp, wp), (tq, wq), (tx, wx) = wl.rules["p"], wl.rules["q"], wl.rules["x"]
    ch = wl.channels
    coupled = [[oracle.coupled(a, b, wl.J2, wl.statistics) for b in ch] for a in ch]
    nk = (lambda e, k: (e[k + 1] ** 3 - e[k] ** 3) / 3.0) if norm else (lambda e, k: e[k + 1] - e[k])
    out = {}
    for cell in range(wl.n_cells):
        i, j = divmod(cell, wl.Nq)
        for a in range(wl.n_p):
            for b in range(wl.n_q):
                p = 0.5 * (pe[i] + pe[i + 1]) + 0.5 * (pe[i + 1] - pe[i]) * tp[a]
                q = 0.5 * (qe[j] + qe[j + 1]) + 0.5 * (qe[j + 1] - qe[j]) * tq[b]
                wab = (0.5 * (pe[i + 1] - pe[i]) * wp[a]) * (0.5 * (qe[j + 1] - qe[j]) * wq[b])
                A, B, Cc, D = 0.25 * p * p + 0.5625 * q * q, 0.75 * p * q, p * p + 0.25 * q * q, p * q
                for t in range(wl.n_cells):
                    ic, jc = divmod(t, wl.Nq)
                    lo = max(-1.0, (pe[ic] ** 2 - A) / B, (Cc - qe[jc + 1] ** 2) / D)
                    hi = min(1.0, (pe[ic + 1] ** 2 - A) / B, (Cc - qe[jc] ** 2) / D)
                    if not hi > lo:
                        continue
                    nrm = math.sqrt(nk(pe, i) * nk(qe, j) * nk(pe, ic) * nk(qe, jc))
                    for c in range(wl.n_x):
                        x = 0.5 * (lo + hi) + 0.5 * (hi - lo) * tx[c]
                        w = wab * 0.5 * (hi - lo) * wx[c]
                        om = w * (p * q) ** 2 if norm else w * p * q / math.sqrt((A + B * x) * (Cc - D * x))
                        for al in range(nc):
                            for be in range(nc):
                                if coupled[al][be]:
                                    key = (cell * nc + al, t * nc + be)
                                    out[key] = out.get(key, 0.0) + om * 2.0 * oracle.G(ch[al], ch[be], wl.J2, wl.T2, wl.statistics, p, q, float(x), 2) / nrm
    return out


@pytest.mark.parametrize("norm", [0, 1])
@pytest.mark.parametrize("wl", [I.small_coupled(N=3, jmax=1, orders=(2, 2, 3), Nq=4),
                                I.boson_lattice(4, 3, waves=((0, 0), (2, 2)), J=0, orders=(2, 3, 3), cq=0.7)], ids=lambda w: w.name)
def test_exact_overlap_build_equals_its_definition(oracle, wl, norm):
    """po_build_xo and po_build_norm entry by entry from numpy + the pinned po_G: intervals, mapped rule, weights, the two
    normalisations, the coupled-channel assembly, the pattern (readings R2, R17)."""
    rp, ci, v = oracle.build_csr(wl, norm=norm, exact_overlap=True)
    ref = _rebuild_xo_from_G(wl, oracle, norm)
    assert len(ref) == len(v)
    rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
    want = np.array([ref[(int(r), int(c))] for r, c in zip(rows, ci)])
    assert np.max(np.abs(v - want)) <= 1e-13 * np.max(np.abs(want))
    if norm:                                               # node binning in reading B: the same check through po_build's node table
        rp, ci, v = oracle.build_csr(wl, norm=1)
        rpA, ciA, vA = oracle.build_csr(wl, norm=0)
        assert np.array_equal(rp, rpA) and np.array_equal(ci, ciA)       # the normalisation does not touch the pattern
        pe, qe = wl.p_edges, wl.q_edges
        Bn = lambda e, k: (e[k + 1] ** 3 - e[k] ** 3) / 3.0
        rows = np.repeat(np.arange(len(rp) - 1), np.diff(rp))
        got = {}
        for cell in range(wl.n_cells):
            i, j = divmod(cell, wl.Nq)
            nd = oracle.cell_nodes(wl, cell)
            for n in np.nonzero(nd["target"] >= 0)[0]:
                t = int(nd["target"][n]); ic, jc = divmod(t, wl.Nq)
                om = nd["w"][n] * (nd["p"][n] * nd["q"][n]) ** 2 / math.sqrt(Bn(pe, i) * Bn(qe, j) * Bn(pe, ic) * Bn(qe, jc))
                for al in range(wl.n_ch):
                    for be in range(wl.n_ch):
                        if oracle.coupled(wl.channels[al], wl.channels[be], wl.J2, wl.statistics):
                            key = (cell * wl.n_ch + al, t * wl.n_ch + be)
                            got[key] = got.get(key, 0.0) + om * 2.0 * oracle.G(wl.channels[al], wl.channels[be], wl.J2, wl.T2, wl.statistics,
                                                                                float(nd["p"][n]), float(nd["q"][n]), float(nd["x"][n]), 2)
        want = np.array([got[(int(r), int(c))] for r, c in zip(rows, ci)])
        assert np.max(np.abs(v - want)) <= 1e-13 * np.max(np.abs(want))
