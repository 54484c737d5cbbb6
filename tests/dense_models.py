"""Independent dense constructions of the three models from Kronecker products of
2x2 operators -- used ONLY to pin the oracle (and, through it, the term lists).

Nothing here is shared with oracle/ or the CUDA library: no term list, no basis
ranking.  Site i is bit i of the basis index, bit 1 = spin up = occupied, so in
``np.kron`` order site 0 is the LAST factor.
"""
from __future__ import annotations

import numpy as np

I2 = np.eye(2)
SZ = np.diag([-0.5, 0.5])                   # index 0 = bit 0 = down
SP = np.array([[0.0, 0.0], [1.0, 0.0]])     # |down> -> |up>
SM = SP.T
SX = 0.5 * (SP + SM)
NOP = np.diag([0.0, 1.0])
PAR = np.diag([1.0, -1.0])                  # (-1)^n


def site_op(op: np.ndarray, i: int, L: int) -> np.ndarray:
    out = np.array([[1.0]])
    for site in range(L - 1, -1, -1):       # site L-1 first factor ... site 0 last
        out = np.kron(out, op if site == i else I2)
    return out


def sector_indices(L: int, n_up: int) -> np.ndarray:
    return np.array([x for x in range(1 << L) if bin(x).count("1") == n_up])


def xxz_dense(L: int, J: float, Delta: float, h, periodic: bool = True) -> np.ndarray:
    """Eq. (54) with S^y S^y written through S^+ S^-: SxSx + SySy = (S+S- + S-S+)/2."""
    H = np.zeros((1 << L, 1 << L))
    nb = L if periodic else L - 1
    for i in range(nb):
        j = (i + 1) % L
        H += J * 0.5 * (site_op(SP, i, L) @ site_op(SM, j, L) + site_op(SM, i, L) @ site_op(SP, j, L))
        H += J * Delta * site_op(SZ, i, L) @ site_op(SZ, j, L)
    for i in range(L):
        H += h[i] * site_op(SZ, i, L)
    return H


def jw_annihilator(j: int, L: int) -> np.ndarray:
    """c_j = (prod_{l<j} (-1)^{n_l}) sigma^-_j."""
    out = site_op(SM, j, L)
    for l in range(j):
        out = site_op(PAR, l, L) @ out
    return out


def fermion_dense(L: int, t: float, t2: float, V: float, eps) -> np.ndarray:
    c = [jw_annihilator(j, L) for j in range(L)]
    H = np.zeros((1 << L, 1 << L))
    for i in range(L - 1):
        H += t * (c[i].T @ c[i + 1] + c[i + 1].T @ c[i])
    for i in range(L - 2):
        H += t2 * (c[i].T @ c[i + 2] + c[i + 2].T @ c[i])
    for i in range(L - 1):
        H += V * site_op(NOP, i, L) @ site_op(NOP, i + 1, L)
    for i in range(L):
        H += eps[i] * site_op(NOP, i, L)
    return H


def quantum_sun_dense(N: int, L: int, dot: np.ndarray, g0: float, alpha: float, u, n_of_j, h):
    """Eq. (67): H_dot (x) 1 + g0 sum alpha^{u_j} Sx_{n(j)} Sx_{N+j} + sum h_j Sz_{N+j}."""
    n = N + L
    H = np.kron(np.eye(1 << L), dot)        # dot acts on bits 0..N-1 (last factors)
    for j in range(L):
        H += g0 * alpha ** u[j] * site_op(SX, int(n_of_j[j]), n) @ site_op(SX, N + j, n)
        H += h[j] * site_op(SZ, N + j, n)
    return H
