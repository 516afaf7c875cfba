"""Pins of the oracle's angular-momentum algebra and of the coefficient G.

Nothing here re-types the oracle's formulas: Wigner symbols are compared with sympy's library
routines, harmonics with scipy's, the spin-isospin matrix with the textbook triton values, and the
full coupled-channel G with an explicit construction of the three-particle states in the product
basis |sigma1 sigma2 sigma3> x |tau1 tau2 tau3> on which the cyclic permutation is a relabelling of
particles (no recoupling coefficient is used on that side).
"""
import functools
import itertools
import math

import numpy as np
import pytest
from scipy.special import sph_harm_y
from sympy import Rational
from sympy.physics.quantum.cg import CG
from sympy.physics.wigner import wigner_3j, wigner_6j, wigner_9j

from paper_1508_07441_b200 import inputs as I


def _r(x2):
    return Rational(x2, 2)


def test_wigner3j_cg_vs_sympy(oracle):
    rng = np.random.default_rng(1)
    n = 0
    for j1, j2 in itertools.product(range(0, 9), repeat=2):
        for j3 in range(abs(j1 - j2), j1 + j2 + 1, 2):
            m1 = int(rng.integers(0, j1 + 1)) * 2 - j1
            m2 = int(rng.integers(0, j2 + 1)) * 2 - j2
            m3 = -(m1 + m2)
            ref = float(wigner_3j(_r(j1), _r(j2), _r(j3), _r(m1), _r(m2), _r(m3))) if abs(m3) <= j3 else 0.0
            assert abs(oracle.wigner3j(j1, j2, j3, m1, m2, m3) - ref) < 1e-14
            if abs(m3) <= j3:
                refc = float(CG(_r(j1), _r(m1), _r(j2), _r(m2), _r(j3), _r(-m3)).doit())
                assert abs(oracle.cg(j1, m1, j2, m2, j3, -m3) - refc) < 1e-14
            n += 1
    assert n > 200


def test_wigner6j_9j_vs_sympy(oracle):
    rng = np.random.default_rng(2)
    hits = 0
    for _ in range(400):
        j1, j2, j4, j5 = (int(v) for v in rng.integers(0, 7, size=4))
        j3 = abs(j1 - j2) + 2 * int(rng.integers(0, min(j1, j2) + 1))      # triangle (j1 j2 j3) holds
        lo, hi = max(abs(j1 - j5), abs(j4 - j2)), min(j1 + j5, j4 + j2)
        j6 = lo + 2 * int(rng.integers(0, max(1, (hi - lo) // 2 + 1))) if hi >= lo else lo
        a = [j1, j2, j3, j4, j5, j6]
        try:
            ref = float(wigner_6j(*[_r(v) for v in a]))
        except ValueError:
            ref = 0.0
        assert abs(oracle.wigner6j(*a) - ref) < 1e-14
        hits += ref != 0.0
    assert hits > 40
    # the 9j symbols that actually occur: { l s j ; lam 1/2 I ; L S J }
    n = 0
    for ch in I.enumerate_3n_channels(1, +1, 1, 3).tolist() + I.enumerate_3n_channels(5, -1, 1, 3).tolist()[:12]:
        l, s, j, t, lam, I2 = ch
        for L in range(abs(l - lam), l + lam + 1):
            for S2 in (1, 3):
                for J2 in (1, 5):
                    got = oracle.wigner9j(2 * l, 2 * s, 2 * j, 2 * lam, 1, I2, 2 * L, S2, J2)
                    try:
                        ref = float(wigner_9j(l, s, j, lam, Rational(1, 2), _r(I2), L, _r(S2), _r(J2)))
                    except ValueError:
                        ref = 0.0
                    assert abs(got - ref) < 1e-14
                    n += ref != 0.0
    assert n > 40


def test_ylm_vs_scipy(oracle):
    rng = np.random.default_rng(3)
    for _ in range(40):
        th = rng.uniform(0, math.pi)
        for phi, sgn in ((0.0, 1.0), (math.pi, -1.0)):
            ux, uz = sgn * math.sin(th), math.cos(th)
            for l in range(0, 13):                       # up to l = 12: lambda of the j <= 3 channels at J = 17/2
                for m in range(-l, l + 1):
                    ref = complex(sph_harm_y(l, m, th, phi))
                    assert abs(ref.imag) < 1e-13
                    assert abs(oracle.ylm(l, m, ux, uz) - ref.real) < 1e-13


def test_triton_spin_isospin_matrix(oracle):
    """Two-channel s-wave 3N, S = T = 1/2: the textbook matrix [[1/4,-3/4],[-3/4,1/4]]
    (SURVEY.md sec. 8(c.4) pin 2); spin quartet: -1/2.  G includes both cyclic terms."""
    ch = I.swave_3n_channels()
    G = np.array([[2 * oracle.G(a, b, 1, 1, I.PM_FERMION_ISOSPIN, 0.7, 1.3, 0.2) for b in ch] for a in ch])
    assert np.allclose(G, [[0.25, -0.75], [-0.75, 0.25]], atol=1e-14)
    quartet = np.array([(0, 1, 1, 0, 0, 1)], dtype=I.CH_DTYPE)[0]
    assert abs(2 * oracle.G(quartet, quartet, 3, 1, I.PM_FERMION_ISOSPIN, 0.4, 0.9, -0.6) - (-0.5)) < 1e-14
    b = I.boson_channel()[0]
    assert abs(2 * oracle.G(b, b, 0, 0, I.PM_SPINLESS_BOSON, 0.3, 2.0, 0.9) - 1.0) < 1e-14


# --------------------------------------------------------------------------------------------
# explicit product-basis construction of <p q alpha | P_cyclic | p' q' alpha'>
# --------------------------------------------------------------------------------------------
@functools.lru_cache(maxsize=None)
def _cg(j1, m1, j2, m2, j3, m3):          # doubled arguments, sympy's library routine
    if m1 + m2 != m3 or abs(m3) > j3 or j3 < abs(j1 - j2) or j3 > j1 + j2:
        return 0.0
    return float(CG(_r(j1), _r(m1), _r(j2), _r(m2), _r(j3), _r(m3)).doit())


def _Y(l, m, v):
    r = np.linalg.norm(v)
    return complex(sph_harm_y(l, m, math.acos(max(-1.0, min(1.0, v[2] / r))), math.atan2(v[1], v[0])))


_SIG = (1, -1)      # doubled projections of a spin-1/2; array index 0 <-> +1/2, 1 <-> -1/2


def _three_spin_state(s_pair, S2_list, pair, spect):
    """dict (s ms2, sigma_spect) -> array[s1,s2,s3] of the state chi^{s ms}(pair) |sigma_spect>."""
    out = {}
    a, b = pair
    for ms in range(-2 * s_pair, 2 * s_pair + 1, 2):
        for ic, sc in enumerate(_SIG):
            arr = np.zeros((2, 2, 2))
            for ia, sa in enumerate(_SIG):
                for ib, sb in enumerate(_SIG):
                    idx = [0, 0, 0]
                    idx[a - 1], idx[b - 1], idx[spect - 1] = ia, ib, ic
                    arr[tuple(idx)] += _cg(1, sa, 1, sb, 2 * s_pair, ms)
            out[(ms, sc)] = arr
    return out


def _wavefunction(ch, J2, M2, pvec, qvec, pair, spect):
    """Phi^{JM}_alpha(p^, q^)[s1,s2,s3]: ((l s)j (lam 1/2)I) J M with the pair spin built from `pair`."""
    l, s, j, t, lam, I2 = ch
    spin = _three_spin_state(s, None, pair, spect)
    phi = np.zeros((2, 2, 2), dtype=complex)
    for mj in range(-2 * j, 2 * j + 1, 2):
        mI = M2 - mj
        cJ = _cg(2 * j, mj, I2, mI, J2, M2)
        if cJ == 0.0:
            continue
        for ml in range(-l, l + 1):
            ms = mj - 2 * ml
            c1 = _cg(2 * l, 2 * ml, 2 * s, ms, 2 * j, mj)
            if c1 == 0.0:
                continue
            for mlam in range(-lam, lam + 1):
                sc = mI - 2 * mlam
                if abs(sc) != 1:
                    continue
                c2 = _cg(2 * lam, 2 * mlam, 1, sc, I2, mI)
                if c2 == 0.0:
                    continue
                phi += cJ * c1 * c2 * _Y(l, ml, pvec) * _Y(lam, mlam, qvec) * spin[(ms, sc)]
    return phi


def _isospin_state(t, T2, MT2, pair, spect):
    st = _three_spin_state(t, None, pair, spect)
    eta = np.zeros((2, 2, 2))
    for mt in range(-2 * t, 2 * t + 1, 2):
        tc = MT2 - mt
        if abs(tc) != 1:
            continue
        eta += _cg(2 * t, mt, 1, tc, T2, MT2) * st[(mt, tc)]
    return eta


_SETS = {1: ((2, 3), 1), 2: ((3, 1), 2), 3: ((1, 2), 3)}


def _G_product_basis(cha, chb, J2, T2, p, q, x, set_, rot):
    sx = math.sqrt(1 - x * x)
    pv = rot @ np.array([p * sx, 0.0, p * x])
    qv = rot @ np.array([0.0, 0.0, q])
    if set_ == 2:      # p2 = (k3-k1)/2, q2 = k2 with k1 = q, k2 = p - q/2, k3 = -p - q/2
        ppv, qpv = -0.5 * pv - 0.75 * qv, pv - 0.5 * qv
    else:              # p3 = (k1-k2)/2, q3 = k3
        ppv, qpv = -0.5 * pv + 0.75 * qv, -pv - 0.5 * qv
    tot = 0.0
    for M2 in range(-J2, J2 + 1, 2):
        bra = _wavefunction(cha, J2, M2, pv, qv, *_SETS[1])
        ket = _wavefunction(chb, J2, M2, ppv, qpv, *_SETS[set_])
        tot += np.vdot(bra, ket)
    iso = float(np.sum(_isospin_state(cha[3], T2, 1, *_SETS[1]) * _isospin_state(chb[3], T2, 1, *_SETS[set_])))
    val = 8 * math.pi ** 2 * tot * iso / (J2 + 1)
    assert abs(val.imag) < 1e-12
    return val.real


def _random_rotation(rng):
    qmat, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(qmat) < 0:
        qmat[:, 0] = -qmat[:, 0]
    return qmat


@pytest.mark.parametrize("J2,par,jmax", [(1, +1, 3), (3, -1, 2), (9, -1, 3), (17, +1, 3)])
def test_G_vs_product_basis(oracle, J2, par, jmax):
    """SURVEY.md sec. 8(c.4) pins 2-4 in their strongest form: the oracle's recoupling formula for G
    (9j, 6j, bipolar harmonics, phases) equals the permutation acting on explicit product states,
    for both cyclic terms, at random points and random overall orientation."""
    chs = I.enumerate_3n_channels(J2, par, 1, jmax)
    rng = np.random.default_rng(11 + J2)
    checked = nonzero = 0
    n_samples = 60 if J2 <= 3 else 14               # J up to 17/2 (lambda up to 12, L up to 10): the paper's full channel sets
    for _ in range(n_samples):
        a, b = chs[rng.integers(len(chs))], chs[rng.integers(len(chs))]
        if J2 > 3 and not oracle.coupled(a, b, J2, I.PM_FERMION_ISOSPIN):
            b = a                                    # diagonal pairs are always coupled: keep the few samples informative
        p, q, x = rng.uniform(0.1, 3.0), rng.uniform(0.1, 3.0), rng.uniform(-0.98, 0.98)
        rot = _random_rotation(rng)
        for set_ in (2, 3):
            ref = _G_product_basis(tuple(a.tolist()), tuple(b.tolist()), J2, 1, p, q, x, set_, rot)
            got = oracle.G(a, b, J2, 1, I.PM_FERMION_ISOSPIN, p, q, x, set_)
            assert abs(got - ref) < 2e-12, (a, b, set_, got, ref)
            checked += 1
            nonzero += abs(ref) > 1e-6
        if not oracle.coupled(a, b, J2, I.PM_FERMION_ISOSPIN):
            assert abs(ref) < 1e-12
    assert nonzero > (40 if J2 <= 3 else 12)


def test_two_cyclic_terms_equal_under_x_reflection(oracle):
    """G^(2)(p,q,x) = G^(3)(p,q,-x) for Pauli-allowed pair states: legitimises 'map set 2, times 2'
    with an x-rule symmetric under x -> -x (reading R4)."""
    chs = I.enumerate_3n_channels(1, +1, 1, 3)
    rng = np.random.default_rng(5)
    for _ in range(300):
        a, b = chs[rng.integers(26)], chs[rng.integers(26)]
        p, q, x = rng.uniform(0.05, 4), rng.uniform(0.05, 4), rng.uniform(-1, 1)
        g2 = oracle.G(a, b, 1, 1, 0, p, q, x, 2)
        g3 = oracle.G(a, b, 1, 1, 0, p, q, -x, 3)
        assert abs(g2 - g3) < 1e-13


def test_pointwise_exchange_symmetry(oracle):
    """Hermiticity of P = c + c^2: G2_{ab}(p,q,x) = G3_{ba}(p',q',x') with (p',q',x') the set-2 image."""
    chs = I.enumerate_3n_channels(1, +1, 1, 3)
    rng = np.random.default_rng(6)
    for _ in range(300):
        a, b = chs[rng.integers(26)], chs[rng.integers(26)]
        p, q, x = rng.uniform(0.1, 3), rng.uniform(0.1, 3), rng.uniform(-0.99, 0.99)
        sx = math.sqrt(1 - x * x)
        pv, qv = np.array([p * sx, p * x]), np.array([0.0, q])
        ppv, qpv = -0.5 * pv - 0.75 * qv, pv - 0.5 * qv
        pp, qq = np.linalg.norm(ppv), np.linalg.norm(qpv)
        xp = float(ppv @ qpv) / (pp * qq)
        lhs = oracle.G(a, b, 1, 1, 0, p, q, x, 2)
        rhs = oracle.G(b, a, 1, 1, 0, pp, qq, xp, 3)
        assert abs(lhs - rhs) < 1e-12


def test_coupled_mask_predicts_zeros(oracle):
    """coupled(a,b) is integer logic; wherever it is false G vanishes identically (reading R8)."""
    chs = I.enumerate_3n_channels(1, +1, 1, 3)
    n_c = 0
    for a in chs:
        for b in chs:
            c = oracle.coupled(a, b, 1, 0)
            n_c += c
            if not c:
                assert abs(oracle.G(a, b, 1, 1, 0, 0.8, 1.7, 0.3)) < 1e-14
    assert n_c == 580                       # SURVEY.md size table: 580 of 676 coupled at 26 channels
    chs18 = I.enumerate_3n_channels(1, +1, 1, 2)
    assert sum(oracle.coupled(a, b, 1, 0) for a in chs18 for b in chs18) == 276
