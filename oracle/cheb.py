"""Scalar side of the oracle: filter coefficients, the filter as a function,
the order rule, density-of-states estimates -- TEST INFRASTRUCTURE ONLY.

Every function is the paper's formula written out (PAPER.md line cited).
"""
from __future__ import annotations

import numpy as np

from . import core

# Cutoff implied by Eq. (42): P(lambda +- delta) -> sin(y)/y at y = 2.655 (reading R4).
OMEGA = float(np.sin(2.655) / 2.655)


def rescale_params(e_min: float, e_max: float, margin: float = 0.0):
    """Eq. (31): E_c = (E_max+E_min)/2, Delta E = (E_max-E_min)/2; reading R5 widens
    Delta E by (1+margin) because Lanczos bounds lie inside the spectrum."""
    a = 0.5 * (e_max + e_min)
    b = 0.5 * (e_max - e_min) * (1.0 + margin)
    return a, b


def filter_coeffs(lam: float, K: int) -> np.ndarray:
    """Eq. (32)-(33): c_n = sqrt(4 - 3 delta_{0n}) cos(n arccos lam), divided by chi
    with chi fixed by P(lam) = 1, i.e. chi = sum_n c_n T_n(lam)."""
    if not (-1.0 < lam < 1.0):
        raise ValueError("rescaled target must lie in (-1, 1)")
    n = np.arange(K + 1)
    Tn = np.cos(n * np.arccos(lam))
    c = np.sqrt(4.0 - 3.0 * (n == 0)) * Tn
    chi = float(np.sum(c * Tn))
    return c / chi


def filter_value(coeffs: np.ndarray, x) -> np.ndarray:
    """P(x) = sum_n coeffs[n] T_n(x) with T_n(x) = cos(n arccos x) (Eq. 32-33), |x| <= 1."""
    x = np.atleast_1d(np.asarray(x, dtype=np.float64))
    n = np.arange(coeffs.shape[0])
    theta = np.arccos(np.clip(x, -1.0, 1.0))
    out = np.empty_like(x)
    chunk = max(1, 4_000_000 // max(1, n.size))
    for lo in range(0, x.size, chunk):
        th = theta[lo:lo + chunk]
        out[lo:lo + chunk] = np.cos(np.outer(th, n)) @ coeffs
    return out


def window_half_width(nev: int, rho: float) -> float:
    """Eq. (40): delta = N_ev / (2 rho(lam))."""
    return nev / (2.0 * rho)


def order_eq42(nev: int, rho: float, lam: float) -> int:
    """Eq. (42): K = 2.655 sqrt(1 - lam^2) / delta, rounded up (reading R4)."""
    return int(np.ceil(2.655 * np.sqrt(1.0 - lam * lam) / window_half_width(nev, rho)))


def order_bisect(nev: int, rho: float, lam: float, omega: float = OMEGA) -> int:
    """Eq. (41) solved by bisection in [K42/2, 2 K42]: the smallest K
    in the bracket with max(P(lam+delta), P(lam-delta)) <= omega."""
    delta = window_half_width(nev, rho)
    K42 = order_eq42(nev, rho, lam)

    def edge(K):
        c = filter_coeffs(lam, K)
        return float(np.max(filter_value(c, [lam - delta, lam + delta])))

    lo, hi = max(1, K42 // 2), 2 * K42
    if edge(lo) <= omega:
        return lo
    if edge(hi) > omega:
        return hi
    while hi - lo > 1:
        mid = (lo + hi) // 2
        if edge(mid) <= omega:
            hi = mid
        else:
            lo = mid
    return hi


# ---- density of states -------------------------------------------------------

def spectral_mean_width(H: core.CSR):
    """mu = Tr H / D and Gamma^2 = Tr H^2 / D - mu^2 (exact from CSR; H symmetric so
    Tr H^2 = sum of squared entries).  Feeds Eq. (34) (reading R7)."""
    n = H.n
    rows = np.repeat(np.arange(n), np.diff(H.row_ptr))
    tr = float(np.sum(H.val[rows == H.col]))
    tr2 = float(np.sum(H.val * H.val))
    mu = tr / n
    return mu, float(np.sqrt(tr2 / n - mu * mu))


def gaussian_dos(E, D: float, mu: float, Gamma: float):
    """Eq. (34)."""
    E = np.asarray(E, dtype=np.float64)
    return D / (np.sqrt(2.0 * np.pi) * Gamma) * np.exp(-(E - mu) ** 2 / (2.0 * Gamma ** 2))


def jackson_kernel(N: int) -> np.ndarray:
    """Eq. (39)/(84), n = 0..N-1."""
    n = np.arange(N)
    q = np.pi / (N + 1)
    return ((N - n + 1) * np.cos(q * n) + np.sin(q * n) / np.tan(q)) / (N + 1)


def kpm_moments(H: core.CSR, a: float, b: float, N: int, R_vectors: np.ndarray) -> np.ndarray:
    """Eq. (37)-(38): mu_n = (1/R) sum_r <r|T_n(H~)|r>, T_n by Eq. (28)-(30).
    R_vectors: D x R block of iid zero-mean unit-variance entries."""
    R = R_vectors.shape[1]
    mu = np.zeros(N)
    T0 = np.ascontiguousarray(R_vectors, dtype=np.float64)
    mu[0] = np.sum(T0 * T0) / R
    if N == 1:
        return mu
    T1 = core.rescaled_apply(H, a, b, T0)
    mu[1] = np.sum(T0 * T1) / R
    Tm, Tc = T0, T1
    for n in range(2, N):
        Tn = 2.0 * core.rescaled_apply(H, a, b, Tc) - Tm
        mu[n] = np.sum(T0 * Tn) / R
        Tm, Tc = Tc, Tn
    return mu


def kpm_dos(E, moments: np.ndarray, g: np.ndarray):
    """Eq. (36): rho(E~) = [mu_0 g_0 + 2 sum_{n>=1} mu_n g_n T_n(E~)] / (pi sqrt(1-E~^2))."""
    E = np.atleast_1d(np.asarray(E, dtype=np.float64))
    n = np.arange(moments.shape[0])
    Tn = np.cos(np.outer(np.arccos(E), n))
    w = moments * g
    series = w[0] + 2.0 * (Tn[:, 1:] @ w[1:])
    return series / (np.pi * np.sqrt(1.0 - E * E))
