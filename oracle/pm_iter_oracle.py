"""CPU ORACLE for the iteration step that consumes P0.  TEST INFRASTRUCTURE ONLY (tests/, bench.py's cpu legs).

PAPER.md:L235-241, eq. (24):  K = P V1 G1 = O P0 V~1 G1,  V~1 = O^T V1,  "G1 is a diagonal matrix, P0 is a highly
sparse permutation matrix, while V~1 and O are block matrices with the block dimension (N x N)".  A block acts on
the pair index i for fixed spectator index j and channel alpha (the rotation O diagonalises the pair sub-Hamiltonian
in the free wave-packet basis).  Vectors use the lattice's row order r = (i*Nq + j)*n_ch + a.

Plain numpy in fp64, factor by factor in the paper's order; shares no code with the CUDA path.  Pinned in
tests/test_oracle_iteration.py against a dense K assembled entry by entry, and against special cases.
"""
from __future__ import annotations

import numpy as np


def vtilde(O: np.ndarray, V1: np.ndarray) -> np.ndarray:
    """V~1 = O^T V1, block by block (eq. 24).  O, V1: [n_ch][Np][Np]."""
    return np.stack([O[a].T @ V1[a] for a in range(O.shape[0])])


def block_apply(B: np.ndarray, x: np.ndarray, Np: int, Nq: int, n_ch: int) -> np.ndarray:
    """y[(i,j,a)] = sum_i' B[a][i][i'] x[(i',j,a)]."""
    x3 = x.reshape(Np, Nq, n_ch)
    y3 = np.empty_like(x3)
    for a in range(n_ch):
        y3[:, :, a] = B[a] @ x3[:, :, a]
    return y3.reshape(-1)


def csr_matvec(rowptr: np.ndarray, colidx: np.ndarray, vals: np.ndarray, x: np.ndarray) -> np.ndarray:
    y = np.zeros(len(rowptr) - 1)
    for r in range(len(y)):
        s = slice(rowptr[r], rowptr[r + 1])
        y[r] = np.dot(vals[s], x[colidx[s]])
    return y


def kernel_apply(rowptr, colidx, vals, O, V1, g1, u, Np, Nq, n_ch) -> np.ndarray:
    """K u = O (P0 (V~1 (G1 u)))  — the four factors of eq. (24), applied right to left."""
    y = g1 * u
    y = block_apply(vtilde(O, V1), y, Np, Nq, n_ch)
    y = csr_matvec(rowptr, colidx, vals, y)
    return block_apply(O, y, Np, Nq, n_ch)


def block_apply_t(B: np.ndarray, x: np.ndarray, Np: int, Nq: int, n_ch: int) -> np.ndarray:
    """y[(i,j,a)] = sum_i' B[a][i'][i] x[(i',j,a)] — the transposed blocks."""
    x3 = x.reshape(Np, Nq, n_ch)
    y3 = np.empty_like(x3)
    for a in range(n_ch):
        y3[:, :, a] = B[a].T @ x3[:, :, a]
    return y3.reshape(-1)


def rotate_apply(rowptr, colidx, vals, O, x, Np, Nq, n_ch) -> np.ndarray:
    """P x with P = O P0 O^T, eq. (20): the permutation matrix rotated from the lattice (free
    wave-packet) basis to the channel basis, applied factor by factor, right to left."""
    y = block_apply_t(O, x, Np, Nq, n_ch)
    y = csr_matvec(rowptr, colidx, vals, y)
    return block_apply(O, y, Np, Nq, n_ch)
