"""Deterministic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic: it only produces the *inputs* of the
permutation-matrix build — momentum-cell edges, the list of spin-angular channels (pure integer
enumeration of quantum numbers), Gauss-Legendre rules (numpy's library routine) and the five
workloads of BASELINE.json `configs`.  Both `oracle/` (through the tests) and the CUDA library
(through `paper_1508_07441_b200.api`) are fed the very same arrays, so a node lands in the same
cell on both sides by construction of the inputs, never by shared code.

Citations: cells D_i, D-bar_j PAPER.md:L146 (sec. 2.4); lattice cells D_ij PAPER.md:L154;
spin-angular channels alpha, beta, Gamma PAPER.md:L148-152 (eq. 15); sizes N~100-150 and up to
62 channels PAPER.md:L231, L374; grid formulas: BASELINE.json configs[0..4] and DESIGN.md
reading R10.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

PM_FERMION_ISOSPIN = 0
PM_SPINLESS_BOSON = 1


# --------------------------------------------------------------------------- grids
def tan_grid(N: int, c: float) -> np.ndarray:
    """Edges p_k = c*tan(pi*k/(2N+2)), k = 0..N (BASELINE.json configs[0]; R10)."""
    k = np.arange(N + 1, dtype=np.float64)
    return c * np.tan(math.pi * k / (2.0 * N + 2.0))


def split_grid(n_low: int = 20, p_low: float = 0.5, n_high: int = 80, p_max: float = 30.0) -> np.ndarray:
    """configs[3]: `n_low` uniform cells on [0, p_low], then `n_high` tangent-mapped cells up to
    p_max: p_{n_low+m} = p_low + (p_max-p_low)*tan(pi*m/(2*n_high+2))/tan(pi*n_high/(2*n_high+2))."""
    lo = p_low * np.arange(n_low + 1, dtype=np.float64) / n_low
    m = np.arange(1, n_high + 1, dtype=np.float64)
    den = math.tan(math.pi * n_high / (2.0 * n_high + 2.0))
    hi = p_low + (p_max - p_low) * np.tan(math.pi * m / (2.0 * n_high + 2.0)) / den
    e = np.concatenate([lo, hi])
    e[-1] = p_max
    return e


def gauss_legendre(n: int) -> tuple[np.ndarray, np.ndarray]:
    """Gauss-Legendre nodes/weights on [-1, 1] (numpy library routine), ascending nodes.
    The arrays are passed as DATA to both the oracle and the CUDA library (R12)."""
    t, w = np.polynomial.legendre.leggauss(n)
    # symmetrise exactly so that the x-rule is invariant under x -> -x (used by reading R4)
    t = 0.5 * (t - t[::-1])
    w = 0.5 * (w + w[::-1])
    return np.ascontiguousarray(t, dtype=np.float64), np.ascontiguousarray(w, dtype=np.float64)


# --------------------------------------------------------------------------- channels
CH_DTYPE = np.dtype([("l", "<i4"), ("s", "<i4"), ("j", "<i4"), ("t", "<i4"), ("lam", "<i4"), ("I2", "<i4")])


def enumerate_3n_channels(J2: int, parity: int, T2: int, jmax: int) -> np.ndarray:
    """All three-nucleon channels alpha = (l, s, j, t; lam, I) for total (J, parity, T).

    Pure integer logic (PAPER.md:L148-152 names the quantum numbers; L374/L378 give the counts 62
    and 18 that tests/test_inputs.py checks):
      pair:      |l-s| <= j <= l+s, j <= jmax, s,t in {0,1}, (-1)^(l+s+t) = -1 (Pauli)
      spectator: 2I = 2*lam +- 1 (I >= 1/2), |j-I| <= J <= j+I
      total:     (-1)^(l+lam) = parity, |t-1/2| <= T <= t+1/2
    Order: by j, then l, s, t, I, lam ascending (R15).
    """
    out = []
    for j in range(0, jmax + 1):
        for l in range(0, j + 2):
            for s in (0, 1):
                if not (abs(l - s) <= j <= l + s):
                    continue
                for t in (0, 1):
                    if (l + s + t) % 2 == 0:
                        continue
                    if not (abs(2 * t - 1) <= T2 <= 2 * t + 1):
                        continue
                    I2lo, I2hi = abs(2 * j - J2), 2 * j + J2
                    for I2 in range(I2lo, I2hi + 1, 2):
                        if I2 < 1:
                            continue
                        for lam in sorted({(I2 - 1) // 2, (I2 + 1) // 2}):
                            if lam < 0 or abs(2 * lam - I2) != 1:
                                continue
                            if (-1) ** (l + lam) != parity:
                                continue
                            out.append((l, s, j, t, lam, I2))
    return np.array(out, dtype=CH_DTYPE)


def boson_channel(l: int = 0, lam: int = 0) -> np.ndarray:
    """Spinless channel: s = t = 0, j = l, I = lam (SURVEY.md sec. 8(b) convention)."""
    return np.array([(l, 0, l, 0, lam, 2 * lam)], dtype=CH_DTYPE)


def swave_3n_channels() -> np.ndarray:
    """configs[1]: the two s-wave 3N channels (s=0,t=1) and (s=1,t=0), l = lam = 0, I = 1/2."""
    return np.array([(0, 0, 0, 1, 0, 1), (0, 1, 1, 0, 0, 1)], dtype=CH_DTYPE)


# --------------------------------------------------------------------------- workloads
@dataclass
class Workload:
    name: str
    p_edges: np.ndarray
    q_edges: np.ndarray
    channels: np.ndarray
    J2: int
    parity: int
    T2: int
    statistics: int
    n_p: int
    n_q: int
    n_x: int
    rules: dict = field(default_factory=dict)

    def __post_init__(self):
        self.p_edges = np.ascontiguousarray(self.p_edges, dtype=np.float64)
        self.q_edges = np.ascontiguousarray(self.q_edges, dtype=np.float64)
        if not self.rules:
            self.rules = {
                "p": gauss_legendre(self.n_p),
                "q": gauss_legendre(self.n_q),
                "x": gauss_legendre(self.n_x),
            }

    @property
    def Np(self) -> int:
        return len(self.p_edges) - 1

    @property
    def Nq(self) -> int:
        return len(self.q_edges) - 1

    @property
    def n_ch(self) -> int:
        return len(self.channels)

    @property
    def n_cells(self) -> int:
        return self.Np * self.Nq

    @property
    def M(self) -> int:
        return self.n_cells * self.n_ch

    @property
    def nodes_per_cell(self) -> int:
        return self.n_p * self.n_q * self.n_x


def config(k: int) -> Workload:
    """The five synthetic lattices of BASELINE.json `configs`.
    Reading R1: the rule is a tensor rule n_p x n_q x n_x with n_p = n_q."""
    if k == 0:
        g = tan_grid(10, 1.0)
        return Workload("cfg0_boson_swave_10x10", g, g, boson_channel(0, 0), 0, +1, 0, PM_SPINLESS_BOSON, 4, 4, 8)
    if k == 1:
        g = tan_grid(50, 1.0)
        return Workload("cfg1_3N_swave_2ch_50x50", g, g, swave_3n_channels(), 1, +1, 1, PM_FERMION_ISOSPIN, 6, 6, 16)
    if k == 2:
        return Workload("cfg2_3N_Jhalf+_jle2_18ch_100x100", tan_grid(100, 1.0), tan_grid(100, 0.8),
                        enumerate_3n_channels(1, +1, 1, 2), 1, +1, 1, PM_FERMION_ISOSPIN, 8, 8, 24)
    if k == 3:
        g = split_grid()
        return Workload("cfg3_3N_Jhalf+_jle3_26ch_100x100_split", g, g,
                        enumerate_3n_channels(1, +1, 1, 3), 1, +1, 1, PM_FERMION_ISOSPIN, 8, 8, 32)
    if k == 4:
        g = tan_grid(150, 1.0)
        return Workload("cfg4_3N_Jhalf+_jle3_26ch_150x150", g, g,
                        enumerate_3n_channels(1, +1, 1, 3), 1, +1, 1, PM_FERMION_ISOSPIN, 10, 10, 32)
    raise ValueError(f"no config {k}")


def small_coupled(N: int = 6, jmax: int = 2, orders=(3, 3, 6), c: float = 1.0, Nq: int | None = None,
                  J2: int = 1, parity: int = +1) -> Workload:
    """A reduced coupled-channel lattice for element-by-element parity tests (same channel
    structure as configs[2]/[3], small grids so that the oracle runs in seconds).  `Nq` (default N) gives a
    rectangular lattice with N cells in p and Nq cells in q; (J2, parity) selects another J^pi."""
    Nq = N if Nq is None else Nq
    tag = "" if (J2, parity) == (1, +1) else f"_J{J2}half{'+' if parity > 0 else '-'}"
    return Workload(f"small_3N_jle{jmax}{tag}_{N}x{Nq}", tan_grid(N, c), tan_grid(Nq, 0.8 * c),
                    enumerate_3n_channels(J2, parity, 1, jmax), J2, parity, 1, PM_FERMION_ISOSPIN, *orders)


def boson_lattice(Np: int, Nq: int, waves=((0, 0),), J: int = 0, orders=(4, 4, 8), cp: float = 1.0, cq: float = 1.0) -> Workload:
    """Spinless-boson lattice with Np x Nq cells (tangent-mapped grids with scales cp, cq) and the channels
    (l, lam) in `waves` coupled to total J = L."""
    ch = np.concatenate([boson_channel(l, lam) for l, lam in waves])
    w = "".join(f"{l}{lam}" for l, lam in waves)
    return Workload(f"boson_w{w}_J{J}_{Np}x{Nq}", tan_grid(Np, cp), tan_grid(Nq, cq), ch, 2 * J, +1 if all((l + lam) % 2 == 0 for l, lam in waves) else -1,
                    0, PM_SPINLESS_BOSON, *orders)


# --------------------------------------------------------------------------- iteration-step inputs (eq. 24)
def iteration_factors(wl: Workload, seed: int = 2025):
    """Seeded synthetic factors of K = O P0 V~1 G1 (eq. 24), standing in for the pair-interaction data that is
    not in the container: per channel an orthogonal (Np x Np) rotation O_a (QR of a Gaussian matrix), a symmetric
    short-ranged V1_a, a diagonal G1 in [-1, 1] and a start vector u.  Data only — V~1 = O^T V1 is formed by whoever
    uses them."""
    rng = np.random.default_rng(seed)
    Np = wl.Np
    O = np.stack([np.linalg.qr(rng.standard_normal((Np, Np)))[0] for _ in range(wl.n_ch)])
    idx = np.arange(Np)
    decay = np.exp(-0.15 * np.abs(idx[:, None] - idx[None, :]))
    V1 = np.stack([(lambda A: 0.5 * (A + A.T) * decay)(rng.standard_normal((Np, Np))) for _ in range(wl.n_ch)])
    g1 = rng.uniform(-1.0, 1.0, wl.M)
    u = rng.uniform(-1.0, 1.0, wl.M)
    return np.ascontiguousarray(O), np.ascontiguousarray(V1), g1, u
