"""ctypes front end of the C oracle -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
legs may import this.  Nothing here touches the CUDA library.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional, Sequence, Tuple

import numpy as np

from . import build as _build

_KIND = {"ZZ": 0, "Z": 1, "NN": 2, "N": 3, "EXCH": 4, "HOPJW": 5, "XX": 6}


class _Term(C.Structure):
    _fields_ = [("kind", C.c_int32), ("i", C.c_int32), ("j", C.c_int32), ("amp", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        p = C.c_void_p
        L.orc_basis_enumerate.restype = C.c_int64
        L.orc_basis_enumerate.argtypes = [C.c_int, C.c_int, p]
        L.orc_basis_rank.restype = C.c_int64
        L.orc_basis_rank.argtypes = [p, C.c_int64, C.c_uint64]
        L.orc_build_csr.restype = C.c_int64
        L.orc_build_csr.argtypes = [p, C.c_int64, p, C.c_int, C.c_int, p, p, p, p]
        L.orc_build_csr_rows.restype = C.c_int64
        L.orc_build_csr_rows.argtypes = [p, C.c_int64, p, C.c_int64, p, C.c_int, C.c_int, p, p, p, p]
        L.orc_spmm.restype = None
        L.orc_spmm.argtypes = [C.c_int64, p, p, p, C.c_int, p, p]
        L.orc_rescale.restype = None
        L.orc_rescale.argtypes = [C.c_int64, C.c_int, C.c_double, C.c_double, p, p]
        L.orc_clenshaw.restype = C.c_int
        L.orc_clenshaw.argtypes = [C.c_int64, p, p, p, C.c_int, C.c_double, C.c_double,
                                   C.c_int, p, p, p, p]
        L.orc_clenshaw_step.restype = None
        L.orc_clenshaw_step.argtypes = [C.c_int64, p, p, p, C.c_int, C.c_double, C.c_double,
                                        C.c_double, p, p, p, p]
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _ptr(a: Optional[np.ndarray]):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def num_threads() -> int:
    return int(lib().orc_num_threads())


# ---- O1 ---------------------------------------------------------------------

def basis_states(n_sites: int, n_up: int) -> np.ndarray:
    """Ascending integers with popcount n_up (n_up < 0: the full space)."""
    dim = lib().orc_basis_enumerate(n_sites, n_up, None)
    states = np.empty(dim, dtype=np.uint64)
    got = lib().orc_basis_enumerate(n_sites, n_up, _ptr(states))
    assert got == dim
    return states


def basis_rank(states: np.ndarray, x: int) -> int:
    return int(lib().orc_basis_rank(_ptr(states), states.shape[0], C.c_uint64(int(x))))


# ---- O2 ---------------------------------------------------------------------

@dataclass
class CSR:
    n: int
    row_ptr: np.ndarray   # int32[n+1]
    col: np.ndarray       # int32[nnz]
    val: np.ndarray       # float64[nnz]

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    def to_dense(self) -> np.ndarray:
        A = np.zeros((self.n, self.n))
        for i in range(self.n):
            for e in range(self.row_ptr[i], self.row_ptr[i + 1]):
                A[i, self.col[e]] += self.val[e]
        return A


def _terms_array(terms: Sequence[Tuple[str, int, int, float]]):
    arr = (_Term * max(1, len(terms)))()
    for k, (kind, i, j, amp) in enumerate(terms):
        arr[k].kind = _KIND[kind]
        arr[k].i = int(i)
        arr[k].j = int(j)
        arr[k].amp = float(amp)
    return arr


def build_csr(states: np.ndarray, terms, dot_bits: int = 0,
              dot_dense: Optional[np.ndarray] = None) -> CSR:
    dim = int(states.shape[0])
    tarr = _terms_array(terms)
    dd = None
    if dot_bits > 0:
        dd = np.ascontiguousarray(dot_dense, dtype=np.float64)
        assert dd.shape == (1 << dot_bits, 1 << dot_bits)
    row_ptr = np.zeros(dim + 1, dtype=np.int32)
    nnz = lib().orc_build_csr(_ptr(states), dim, tarr, len(terms), dot_bits, _ptr(dd),
                              _ptr(row_ptr), None, None)
    if nnz < 0:
        raise ValueError("oracle CSR build failed (a term leaves the basis?)")
    col = np.empty(nnz, dtype=np.int32)
    val = np.empty(nnz, dtype=np.float64)
    got = lib().orc_build_csr(_ptr(states), dim, tarr, len(terms), dot_bits, _ptr(dd),
                              _ptr(row_ptr), _ptr(col), _ptr(val))
    if got != nnz:
        raise ValueError("oracle CSR fill failed")
    return CSR(dim, row_ptr, col, val)


def build_csr_rows(states: np.ndarray, rows: np.ndarray, terms, dot_bits: int = 0,
                   dot_dense: Optional[np.ndarray] = None) -> CSR:
    """Mini-CSR holding only the matrix rows ``rows`` (columns index the full dimension);
    ``spmm`` on it returns (H X)[rows, :].  For spot checks at full BASELINE sizes."""
    dim = int(states.shape[0])
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    tarr = _terms_array(terms)
    dd = None
    if dot_bits > 0:
        dd = np.ascontiguousarray(dot_dense, dtype=np.float64)
    row_ptr = np.zeros(rows.shape[0] + 1, dtype=np.int32)
    nnz = lib().orc_build_csr_rows(_ptr(states), dim, _ptr(rows), rows.shape[0], tarr, len(terms),
                                   dot_bits, _ptr(dd), _ptr(row_ptr), None, None)
    if nnz < 0:
        raise ValueError("oracle CSR build failed (a term leaves the basis?)")
    col = np.empty(nnz, dtype=np.int32)
    val = np.empty(nnz, dtype=np.float64)
    lib().orc_build_csr_rows(_ptr(states), dim, _ptr(rows), rows.shape[0], tarr, len(terms),
                             dot_bits, _ptr(dd), _ptr(row_ptr), _ptr(col), _ptr(val))
    return CSR(int(rows.shape[0]), row_ptr, col, val)


def hamiltonian(workload) -> Tuple[np.ndarray, CSR]:
    """(states, CSR) of a workloads.Workload."""
    states = basis_states(workload.n_sites, workload.n_up)
    return states, build_csr(states, workload.terms, workload.dot_bits, workload.dot_dense)


# ---- O3 / O4 / O6 -------------------------------------------------------------

def _block(X: np.ndarray) -> Tuple[np.ndarray, int]:
    X = np.ascontiguousarray(X, dtype=np.float64)
    if X.ndim == 1:
        X = X.reshape(-1, 1)
    return X, X.shape[1]


def spmm(H: CSR, X: np.ndarray) -> np.ndarray:
    X, s = _block(X)
    assert H.col.size == 0 or int(H.col.max()) < X.shape[0]
    Y = np.empty((H.n, s), dtype=np.float64)
    lib().orc_spmm(H.n, _ptr(H.row_ptr), _ptr(H.col), _ptr(H.val), s, _ptr(X), _ptr(Y))
    return Y


def rescaled_apply(H: CSR, a: float, b: float, X: np.ndarray) -> np.ndarray:
    """H~ X = (H X - a X)/b, Eq. (31)."""
    X, s = _block(X)
    T = spmm(H, X)
    lib().orc_rescale(H.n, s, a, b, _ptr(X), _ptr(T))
    return T


def clenshaw(H: CSR, a: float, b: float, coeffs: np.ndarray, V: np.ndarray) -> np.ndarray:
    """W = sum_{k=0..K} coeffs[k] T_k(H~) V by Eq. (51)."""
    V, s = _block(V)
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    K = c.shape[0] - 1
    W = np.empty_like(V)
    work = np.empty(3 * V.size, dtype=np.float64)
    products = lib().orc_clenshaw(H.n, _ptr(H.row_ptr), _ptr(H.col), _ptr(H.val), s, a, b,
                                  K, _ptr(c), _ptr(V), _ptr(W), _ptr(work))
    assert products == K            # "only K sparse matrix-block multiplications"
    return W


def clenshaw_step(H: CSR, a: float, b: float, ck: float, V, B1, B2, T) -> None:
    """In place B2 <- ck V + 2 H~ B1 - B2 (one recurrence step; timing helper)."""
    s = V.shape[1]
    lib().orc_clenshaw_step(H.n, _ptr(H.row_ptr), _ptr(H.col), _ptr(H.val), s, a, b, ck,
                            _ptr(V), _ptr(B1), _ptr(B2), _ptr(T))
