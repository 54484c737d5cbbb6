"""The five BASELINE.json workloads as seeded parameter arrays and term lists.

A *term* is a tuple ``(kind, i, j, amp)`` with ``kind`` one of the strings below;
bit ``i`` of a basis state is site ``i`` (0-based), bit value 1 = spin up
(S^z = +1/2) = occupied (reading R12/R13).

    "ZZ"     amp * S^z_i S^z_j                      (diagonal)
    "Z"      amp * S^z_i                            (diagonal, j ignored)
    "NN"     amp * n_i n_j                          (diagonal)
    "N"      amp * n_i                              (diagonal, j ignored)
    "EXCH"   amp * (S^+_i S^-_j + h.c.)             (off-diagonal, no sign)
    "HOPJW"  amp * (c^dag_i c_j + h.c.), Jordan-Wigner sign
             (-1)^{# occupied sites strictly between i and j}
    "XX"     amp * 4 S^x_i S^x_j  = amp * (flip bit i and bit j)

Model definitions: XXZ chain PAPER.md:858-863 (Eq. 54); quantum sun
PAPER.md:939-946 (Eq. 67); the spinless-fermion chain is defined by
BASELINE.json config 5 only (reading R15).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

Term = Tuple[str, int, int, float]


@dataclass
class Workload:
    name: str
    config: int
    n_sites: int
    n_up: int                      # < 0: full 2^n_sites space
    terms: List[Term]
    dot_bits: int = 0              # dense block acts on bits 0..dot_bits-1
    dot_dense: Optional[np.ndarray] = None   # (2^dot_bits, 2^dot_bits) fp64, symmetric
    s: int = 1                     # block size
    nev: int = 1
    target_kind: str = "rescaled"  # "rescaled" (lambda~ given) | "unrescaled" (sigma given)
    target: float = 0.0
    K_fixed: Optional[int] = None  # config 1 fixes K=200; others use the DOS rule
    params: dict = field(default_factory=dict)


def xxz_terms(L: int, J: float, Delta: float, h: np.ndarray, periodic: bool = True) -> List[Term]:
    """Eq. (54): J sum (SxSx + SySy + Delta SzSz) + sum h_i Sz_i.

    SxSx + SySy = (S+S- + h.c.)/2, hence EXCH amplitude J/2 (reading R13)."""
    terms: List[Term] = []
    n_bonds = L if periodic else L - 1
    for i in range(n_bonds):
        j = (i + 1) % L
        terms.append(("EXCH", i, j, 0.5 * J))
        terms.append(("ZZ", i, j, J * Delta))
    for i in range(L):
        terms.append(("Z", i, i, float(h[i])))
    return terms


def fermion_terms(L: int, t: float, t2: float, V: float, eps: np.ndarray) -> List[Term]:
    """BASELINE config 5 (reading R15): open chain,
    H = t sum (c+_i c_{i+1} + h.c.) + t' sum (c+_i c_{i+2} + h.c.)
        + V sum n_i n_{i+1} + sum eps_i n_i."""
    terms: List[Term] = []
    for i in range(L - 1):
        terms.append(("HOPJW", i, i + 1, t))
    for i in range(L - 2):
        terms.append(("HOPJW", i, i + 2, t2))
    for i in range(L - 1):
        terms.append(("NN", i, i + 1, V))
    for i in range(L):
        terms.append(("N", i, i, float(eps[i])))
    return terms


def quantum_sun_terms(N: int, L: int, g0: float, alpha: float, u: np.ndarray,
                      n_of_j: np.ndarray, h: np.ndarray) -> List[Term]:
    """Eq. (67) without H_dot: g0 sum alpha^{u_j} S^x_{n(j)} S^x_j + sum h_j S^z_j.
    Outer spin j lives on bit N + j (reading R14). "XX" amp multiplies 4 SxSx."""
    terms: List[Term] = []
    for j in range(L):
        terms.append(("XX", int(n_of_j[j]), N + j, g0 * float(alpha ** u[j]) / 4.0))
    for j in range(L):
        terms.append(("Z", N + j, N + j, float(h[j])))
    return terms


def goe_dot_block(rng: np.random.Generator, N: int, gamma: float) -> np.ndarray:
    """A iid normal, R' = (A + A^T)/sqrt(2), H_dot = gamma R'/sqrt(2^N + 1)."""
    d = 1 << N
    A = rng.standard_normal((d, d))
    Rp = (A + A.T) / np.sqrt(2.0)
    return np.ascontiguousarray(gamma * Rp / np.sqrt(d + 1.0))


def _xxz_workload(config: int, L: int, W: float, s: int, nev: int, target_kind: str,
                  target: float, K_fixed: Optional[int], seed: int) -> Workload:
    rng = np.random.Generator(np.random.PCG64(seed))
    h = rng.uniform(-W, W, size=L)
    return Workload(name=f"xxz_L{L}", config=config, n_sites=L, n_up=L // 2,
                    terms=xxz_terms(L, 1.0, 1.0, h, periodic=True), s=s, nev=nev,
                    target_kind=target_kind, target=target, K_fixed=K_fixed,
                    params={"J": 1.0, "Delta": 1.0, "W": W, "h": h, "seed": seed})


def make_workload(config: int, *, L_override: Optional[int] = None,
                  seed: Optional[int] = None) -> Workload:
    """Build workload ``config`` in 1..5 (BASELINE.json configs[config-1]).

    ``L_override`` shrinks the system (same model, same distributions) for
    tests; the outer-spin count for config 4, the chain length otherwise."""
    if seed is None:
        seed = 1000 + config
    if config == 1:
        return _xxz_workload(1, L_override or 12, 5.0, 1, 20, "unrescaled", 0.0, 200, seed)
    if config == 2:
        return _xxz_workload(2, L_override or 16, 5.0, 8, 50, "rescaled", 0.0, None, seed)
    if config == 3:
        return _xxz_workload(3, L_override or 20, 3.0, 16, 100, "rescaled", 0.0, None, seed)
    if config == 4:
        N, L = 3, (L_override or 17)
        rng = np.random.Generator(np.random.PCG64(seed))
        dot = goe_dot_block(rng, N, 1.0)
        zeta = rng.uniform(-0.2, 0.2, size=L)
        u = np.arange(L, dtype=np.float64) + zeta
        n_of_j = rng.integers(0, N, size=L)
        h = rng.uniform(0.5, 1.5, size=L)
        return Workload(name=f"qsun_N{N}_L{L}", config=4, n_sites=N + L, n_up=-1,
                        terms=quantum_sun_terms(N, L, 1.0, 0.75, u, n_of_j, h),
                        dot_bits=N, dot_dense=dot, s=16, nev=100,
                        target_kind="unrescaled", target=0.0,
                        params={"alpha": 0.75, "gamma": 1.0, "g0": 1.0, "u": u,
                                "n_of_j": n_of_j, "h": h, "seed": seed})
    if config == 5:
        L = L_override or 26
        rng = np.random.Generator(np.random.PCG64(seed))
        eps = rng.uniform(-2.0, 2.0, size=L)
        return Workload(name=f"fermion_L{L}", config=5, n_sites=L, n_up=L // 2,
                        terms=fermion_terms(L, 1.0, 0.5, 1.0, eps), s=32, nev=200,
                        target_kind="rescaled", target=0.0,
                        params={"t": 1.0, "t2": 0.5, "V": 1.0, "eps": eps, "seed": seed})
    raise ValueError(f"config must be 1..5, got {config}")


CONFIGS = (1, 2, 3, 4, 5)


def start_block(n: int, s: int, seed: int, orthonormal: bool = False) -> np.ndarray:
    """Standard-normal n x s block, row-major fp64 (reading R16).  With
    ``orthonormal`` the block is replaced by the Q factor of its Householder QR
    (numpy/LAPACK), the paper's recommended start."""
    rng = np.random.Generator(np.random.PCG64(seed))
    V = rng.standard_normal((n, s))
    if orthonormal:
        V, _ = np.linalg.qr(V)
    return np.ascontiguousarray(V, dtype=np.float64)
