"""Textbook Lanczos / block Lanczos / POLFED driver -- TEST INFRASTRUCTURE ONLY.

Follows PAPER.md Sec. 2.1 (Eq. 1-6), Sec. 2.2 (Eq. 7-17) and Sec. 4.3/4.6 (Fig. 4)
in the paper's order and notation; dense pieces are numpy/LAPACK calls.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, List, Optional

import numpy as np

from . import cheb, core


# ---- Sec. 2.1: scalar Lanczos with full reorthogonalisation -----------------

def lanczos_tridiag(apply_H: Callable[[np.ndarray], np.ndarray], v0: np.ndarray, m: int):
    """Eq. (2)-(4): H phi_i = b_i phi_{i-1} + a_i phi_i + b_{i+1} phi_{i+1}.
    Returns (alpha[0:m'], beta[0:m'] with beta[i] = b_{i+2}, Phi n x m')."""
    n = v0.shape[0]
    phi = v0 / np.linalg.norm(v0)
    Phi = np.zeros((n, m))
    alpha, beta = [], []
    for i in range(m):
        Phi[:, i] = phi
        w = apply_H(phi.reshape(-1, 1)).reshape(-1)
        a_i = float(phi @ w)
        alpha.append(a_i)
        w = w - Phi[:, :i + 1] @ (Phi[:, :i + 1].T @ w)     # full reorthogonalisation
        w = w - Phi[:, :i + 1] @ (Phi[:, :i + 1].T @ w)
        b_next = float(np.linalg.norm(w))
        beta.append(b_next)
        if b_next < 1e-14 * max(1.0, abs(a_i)):
            break
        phi = w / b_next
    k = len(alpha)
    return np.array(alpha), np.array(beta), Phi[:, :k]


def lanczos_extrema(H: core.CSR, v0: np.ndarray, m: int = 60):
    """E_min, E_max as extremal Ritz values of the Lanczos matrix."""
    alpha, beta, _ = lanczos_tridiag(lambda X: core.spmm(H, X), v0, min(m, H.n))
    k = alpha.shape[0]
    T = np.diag(alpha) + np.diag(beta[:k - 1], 1) + np.diag(beta[:k - 1], -1)
    ev = np.linalg.eigvalsh(T)
    return float(ev[0]), float(ev[-1])


def lanczos_extrema_residuals(H: core.CSR, v0: np.ndarray, m: int = 60):
    """(E_min, E_max, r_min, r_max): the extremal Ritz values and their residual norms
    ||H y - theta y|| = b_{m+1} |z_m| (Eq. 6; the scalar case of Eq. 16), z the eigenvector of
    the Lanczos matrix and b_{m+1} the norm of the last residual vector."""
    alpha, beta, _ = lanczos_tridiag(lambda X: core.spmm(H, X), v0, min(m, H.n))
    k = alpha.shape[0]
    T = np.diag(alpha) + np.diag(beta[:k - 1], 1) + np.diag(beta[:k - 1], -1)
    ev, Z = np.linalg.eigh(T)
    b_last = float(beta[k - 1])
    return float(ev[0]), float(ev[-1]), b_last * abs(float(Z[k - 1, 0])), b_last * abs(float(Z[k - 1, -1]))


def spectrum_bounds(H: core.CSR, v0: np.ndarray, m: int = 60, margin: float = 0.01):
    """(E_min, E_max, a, b): the extremal Ritz values, and a, b of Eq. (31) computed from the
    Ritz values moved outwards by their residual norms and widened by the margin (reading R5:
    Ritz values lie inside the spectrum)."""
    e_min, e_max, r_min, r_max = lanczos_extrema_residuals(H, v0, m)
    a, b = cheb.rescale_params(e_min - r_min, e_max + r_max, margin)
    return e_min, e_max, a, b


# ---- Sec. 2.2 / 4.3: block Lanczos -------------------------------------------

@dataclass
class BlockLanczosState:
    s: int
    Q: List[np.ndarray] = field(default_factory=list)      # V_1 .. V_{k+1}
    A: List[np.ndarray] = field(default_factory=list)      # A_1 .. A_k
    B: List[np.ndarray] = field(default_factory=list)      # B_2 .. B_{k+1}

    @property
    def steps(self) -> int:
        return len(self.A)

    def lanczos_matrix(self) -> np.ndarray:
        """H_L (M x M, M = k s) filled as Eq. (10), (13), (14)."""
        k, s = self.steps, self.s
        HL = np.zeros((k * s, k * s))
        for i in range(k):
            HL[i * s:(i + 1) * s, i * s:(i + 1) * s] = self.A[i]
            if i + 1 < k:
                HL[(i + 1) * s:(i + 2) * s, i * s:(i + 1) * s] = self.B[i]
                HL[i * s:(i + 1) * s, (i + 1) * s:(i + 2) * s] = self.B[i].T
        return HL

    def basis(self) -> np.ndarray:
        return np.concatenate(self.Q[:self.steps], axis=1)


def block_lanczos_step(st: BlockLanczosState, apply_op: Callable[[np.ndarray], np.ndarray]):
    """One step k of Fig. 4: W = Op V_k; A_k = V_k^T W (Eq. 9); full reorthogonalisation
    against V_1..V_k, done twice (Eq. 11); Householder QR W = V_{k+1} B_{k+1} (Eq. 12)."""
    k = st.steps
    Vk = st.Q[k]
    W = apply_op(Vk)
    st.A.append(Vk.T @ W)
    for _ in range(2):
        for Vi in st.Q[:k + 1]:
            W = W - Vi @ (Vi.T @ W)
    Vn, Bn = np.linalg.qr(W)
    st.Q.append(Vn)
    st.B.append(Bn)


def ritz_pairs(st: BlockLanczosState):
    """eigh(H_L), eigenvalues descending, and the residual estimates
    ||B_{m+1} tau_{mj}|| of Eq. (16)-(17)."""
    HL = st.lanczos_matrix()
    theta, T = np.linalg.eigh(0.5 * (HL + HL.T))
    order = np.argsort(-theta)
    theta, T = theta[order], T[:, order]
    tau_m = T[-st.s:, :]
    est = np.linalg.norm(st.B[-1] @ tau_m, axis=0)
    return theta, T, est


@dataclass
class EigResult:
    evals: np.ndarray
    evecs: np.ndarray
    residuals: np.ndarray
    K: int
    a: float
    b: float
    lam: float
    block_steps: int
    krylov_dim: int
    converged: bool


def h_rayleigh_ritz(H: core.CSR, U: np.ndarray):
    """Rayleigh-Ritz of H itself in span(U) (reading R21): E, X = U Z, ||H x - E x||."""
    U, _ = np.linalg.qr(U)
    HU = core.spmm(H, U)
    G = U.T @ HU
    E, Z = np.linalg.eigh(0.5 * (G + G.T))
    X = U @ Z
    R = HU @ Z - X * E
    return E, X, np.linalg.norm(R, axis=0)


def polfed_eigs(H: core.CSR, a: float, b: float, lam: float, K: int, nev: int,
                V1: np.ndarray, tol: float, max_steps: Optional[int] = None,
                guard: Optional[int] = None, check_every: int = 1) -> EigResult:
    """Sec. 4.6 steps 4-6 with given (a, b, lam, K): block Lanczos on P(H~) with the
    filter applied by Clenshaw, periodic check, back-map Eq. (43), Rayleigh quotients and
    residuals with H itself.  tol is absolute (caller passes 1e-8 ||H||)."""
    n, s = V1.shape
    coeffs = cheb.filter_coeffs(lam, K)
    sigma = a + b * lam
    guard = s if guard is None else guard
    if max_steps is None:
        max_steps = max(4, (n // s) - 1)
    st = BlockLanczosState(s=s, Q=[np.ascontiguousarray(V1)])
    want = min(nev + guard, n)
    best = None
    for k in range(1, max_steps + 1):
        block_lanczos_step(st, lambda X: core.clenshaw(H, a, b, coeffs, X))
        M = k * s
        if M < want or (k % check_every) != 0 and k != max_steps:
            continue
        theta, T, est = ritz_pairs(st)
        U = st.basis() @ T[:, :want]                 # Eq. (43), the `want` largest theta
        E, X, res = h_rayleigh_ritz(H, U)
        order = np.argsort(np.abs(E - sigma))
        good = [j for j in order if res[j] <= tol]
        best = (E, X, res, order)
        if len(good) >= nev:
            sel = np.sort(np.array(good[:nev]))
            return EigResult(E[sel], X[:, sel], res[sel], K, a, b, lam, k, M, True)
    E, X, res, order = best
    sel = np.sort(order[:nev])
    return EigResult(E[sel], X[:, sel], res[sel], K, a, b, lam, st.steps, st.steps * s, False)
