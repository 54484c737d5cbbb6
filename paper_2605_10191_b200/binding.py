"""ctypes binding of libpolfed.so -- argument marshalling only.

Every function has the name of the C entry point it wraps (include/polfed.h).  Blocks are
torch CUDA tensors (fp64, contiguous, N x s); torch supplies device memory and the current
stream, nothing else.  There is no CPU fallback: a missing library raises ImportError.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpolfed.so")

OK, EINVAL, ENOMEM, ECUDA, ERANGE, ENOCONV, EBREAKDOWN, EWINDOW = range(8)
TERM_KINDS = {"ZZ": 0, "Z": 1, "NN": 2, "N": 3, "EXCH": 4, "HOPJW": 5, "XX": 6}
FORMAT_CSR, FORMAT_TILED, FORMAT_FLIP, FORMAT_SECTOR = 0, 2, 3, 4
HAM_NO_SNAPSHOT = 1

EXPORTS = (
    "polfed_last_error", "polfed_version", "polfed_release_scratch",
    "polfed_build_basis", "polfed_basis_destroy", "polfed_basis_dim", "polfed_basis_states",
    "polfed_basis_rank",
    "polfed_build_hamiltonian", "polfed_ham_from_csr", "polfed_ham_from_csr_ex", "polfed_ham_destroy",
    "polfed_ham_csr",
    "polfed_fused_step", "polfed_filter_workspace_bytes", "polfed_filter_workspace_bytes_ham",
    "polfed_filter_apply",
    "polfed_filter_apply_host", "polfed_filter_coeffs",
    "polfed_spectrum_bounds", "polfed_block_lanczos_eigs",
    "polfed_kpm_workspace_bytes", "polfed_kpm_moments", "polfed_kpm_dos",
    "polfed_block_gram", "polfed_block_update", "polfed_block_gram_static",
)


class PolfedError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"libpolfed error {code}: {message}")
        self.code = code


class _Term(C.Structure):
    _fields_ = [("i", C.c_int32), ("j", C.c_int32), ("amp", C.c_double), ("kind", C.c_int32)]


class _DenseBlock(C.Structure):
    _fields_ = [("n_bits", C.c_int32), ("h_dense", C.c_void_p)]


class _Options(C.Structure):
    _fields_ = [("tol", C.c_double), ("max_krylov_dim", C.c_int32), ("check_every", C.c_int32),
                ("K_override", C.c_int32), ("bounds_steps", C.c_int32),
                ("bounds_margin", C.c_double), ("a", C.c_double), ("b", C.c_double),
                ("sigma_is_rescaled", C.c_int32), ("dos", C.c_int32), ("kpm_moments", C.c_int32),
                ("kpm_vectors", C.c_int32), ("d_kpm_block", C.c_void_p), ("window_levels", C.c_int32)]


class _Report(C.Structure):
    _fields_ = [("a", C.c_double), ("b", C.c_double), ("lambda_rescaled", C.c_double),
                ("e_min", C.c_double), ("e_max", C.c_double), ("tol", C.c_double),
                ("K", C.c_int32), ("block_steps", C.c_int32), ("krylov_dim", C.c_int32),
                ("n_converged", C.c_int32), ("n_checks", C.c_int32), ("K_gaussian", C.c_int32),
                ("sparse_products", C.c_int64),
                ("seconds_bounds", C.c_double), ("seconds_filter", C.c_double),
                ("seconds_reorth", C.c_double), ("seconds_qr", C.c_double),
                ("seconds_projected_eig", C.c_double), ("seconds_extraction", C.c_double),
                ("seconds_total", C.c_double), ("rho_gaussian", C.c_double),
                ("rho_kpm", C.c_double), ("K_kpm", C.c_int32), ("nev_window", C.c_int32),
                ("seconds_dos", C.c_double), ("products_without_v", C.c_int64)]


_lib = None


def lib() -> C.CDLL:
    """Load libpolfed.so (built in-tree by paper_2605_10191_b200/build.py)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2605_10191_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    p, i64, i32, f64 = C.c_void_p, C.c_int64, C.c_int, C.c_double
    L.polfed_last_error.restype = C.c_char_p
    L.polfed_last_error.argtypes = []
    L.polfed_version.restype = i32
    L.polfed_build_basis.argtypes = [i32, i32, p, C.POINTER(p)]
    L.polfed_basis_destroy.argtypes = [p]
    L.polfed_basis_dim.argtypes = [p, C.POINTER(i64)]
    L.polfed_basis_states.argtypes = [p, C.POINTER(p)]
    L.polfed_basis_rank.argtypes = [p, p, i64, p, p]
    L.polfed_build_hamiltonian.argtypes = [p, p, i32, p, i32, p, C.POINTER(p)]
    L.polfed_ham_from_csr.argtypes = [i64, i64, p, p, p, C.POINTER(p)]
    L.polfed_ham_from_csr_ex.argtypes = [i64, i64, p, p, p, C.c_uint, p, C.POINTER(p)]
    L.polfed_ham_destroy.argtypes = [p]
    L.polfed_ham_csr.argtypes = [p, C.POINTER(i64), C.POINTER(i64), C.POINTER(p), C.POINTER(p),
                                 C.POINTER(p)]
    L.polfed_fused_step.argtypes = [p, i32, f64, f64, f64, f64, p, p, p, p, p]
    L.polfed_filter_workspace_bytes.restype = C.c_size_t
    L.polfed_filter_workspace_bytes.argtypes = [i64, i32]
    L.polfed_filter_workspace_bytes_ham.restype = C.c_size_t
    L.polfed_filter_workspace_bytes_ham.argtypes = [p, i32]
    L.polfed_filter_apply.argtypes = [p, f64, f64, i32, p, i32, p, p, p, p]
    L.polfed_filter_apply_host.argtypes = [p, f64, f64, i32, p, i32, p, p, p]
    L.polfed_filter_coeffs.argtypes = [f64, f64, f64, i32, f64, i32, C.POINTER(i32), p, i32]
    L.polfed_spectrum_bounds.argtypes = [p, i32, p, f64, p, C.POINTER(f64), C.POINTER(f64),
                                         C.POINTER(f64), C.POINTER(f64)]
    L.polfed_block_lanczos_eigs.argtypes = [p, f64, i32, i32, p, C.POINTER(_Options), p, p, p,
                                            C.POINTER(_Report), p]
    L.polfed_kpm_workspace_bytes.restype = C.c_size_t
    L.polfed_kpm_workspace_bytes.argtypes = [i64, i32, i32]
    L.polfed_kpm_moments.argtypes = [p, f64, f64, i32, i32, p, p, p, p]
    L.polfed_kpm_dos.argtypes = [p, i32, p, i32, p]
    L.polfed_block_gram.argtypes = [i32, i64, p, i32, i64, p, p, i32, p]
    L.polfed_block_update.argtypes = [i32, i64, p, i32, i64, p, f64, f64, p, p]
    L.polfed_block_gram_static.argtypes = [i32, i64, p, i32, i64, p, p, i32, p]
    _lib = L
    return L


def _check(code: int) -> None:
    if code != OK:
        raise PolfedError(code, lib().polfed_last_error().decode("utf-8", "replace"))


def _stream(stream=None) -> Optional[int]:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    stream = getattr(stream, "cuda_stream", stream)   # a torch.cuda.Stream or a raw handle
    return C.c_void_p(int(stream)) if stream else None


def _dev(t) -> Optional[int]:
    """Device address of a torch CUDA tensor (None passes NULL)."""
    if t is None:
        return None
    if not t.is_cuda or not t.is_contiguous():
        raise ValueError("expected a contiguous CUDA tensor")
    return C.c_void_p(t.data_ptr())


def _block(t, n: int, s: int):
    import torch
    if t.dtype != torch.float64 or t.numel() != n * s:
        raise ValueError(f"expected an fp64 block with {n}x{s} entries")
    return _dev(t)


def polfed_last_error() -> str:
    return lib().polfed_last_error().decode("utf-8", "replace")


def polfed_version() -> int:
    return int(lib().polfed_version())


def polfed_release_scratch() -> None:
    """Give the unused memory of the library's scratch pool back to the driver."""
    _check(lib().polfed_release_scratch())


# ---- basis ----------------------------------------------------------------------------

class Basis:
    """Owner of a polfed_basis handle."""

    def __init__(self, handle: int, n_sites: int, n_up: int):
        self.handle, self.n_sites, self.n_up = handle, n_sites, n_up

    @property
    def dim(self) -> int:
        return polfed_basis_dim(self)

    def close(self) -> None:
        if self.handle:
            lib().polfed_basis_destroy(C.c_void_p(self.handle))
            self.handle = 0

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def polfed_build_basis(n_sites: int, n_up: int, stream=None) -> Basis:
    h = C.c_void_p()
    _check(lib().polfed_build_basis(n_sites, n_up, _stream(stream), C.byref(h)))
    return Basis(h.value, n_sites, n_up)


def polfed_basis_dim(basis: Basis) -> int:
    d = C.c_int64()
    _check(lib().polfed_basis_dim(C.c_void_p(basis.handle), C.byref(d)))
    return int(d.value)


def polfed_basis_states(basis: Basis):
    """The ascending states as an int64 CUDA tensor (a copy; bit patterns of the uint64 states)."""
    import torch
    ptr = C.c_void_p()
    _check(lib().polfed_basis_states(C.c_void_p(basis.handle), C.byref(ptr)))
    return _copy_out(ptr.value, basis.dim, "<i8", torch.int64)


def polfed_basis_rank(basis: Basis, states, stream=None):
    """Ranks (int64 CUDA tensor, -1 = not in the basis) of an int64 CUDA tensor of states."""
    import torch
    if states.dtype != torch.int64:
        raise ValueError("states must be an int64 CUDA tensor")
    out = torch.empty_like(states)
    _check(lib().polfed_basis_rank(C.c_void_p(basis.handle), _dev(states), states.numel(),
                                   _dev(out), _stream(stream)))
    return out


# ---- Hamiltonian ----------------------------------------------------------------------

class Ham:
    """Owner of a polfed_ham handle (keeps wrapped tensors alive)."""

    def __init__(self, handle: int, keep=()):
        self.handle, self._keep = handle, keep
        n, nnz = C.c_int64(), C.c_int64()
        _check(lib().polfed_ham_csr(C.c_void_p(handle), C.byref(n), C.byref(nnz), None, None, None))
        self.n, self.nnz = int(n.value), int(nnz.value)

    def close(self) -> None:
        if self.handle:
            lib().polfed_ham_destroy(C.c_void_p(self.handle))
            self.handle = 0
            self._keep = ()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def _terms_array(terms: Sequence[Tuple[str, int, int, float]]):
    arr = (_Term * max(1, len(terms)))()
    for k, (kind, i, j, amp) in enumerate(terms):
        arr[k].i, arr[k].j, arr[k].amp, arr[k].kind = int(i), int(j), float(amp), TERM_KINDS[kind]
    return arr


def polfed_build_hamiltonian(basis: Basis, terms, dot_bits: int = 0,
                             dot_dense: Optional[np.ndarray] = None, fmt: int = FORMAT_CSR,
                             stream=None) -> Ham:
    arr = _terms_array(terms)
    dot = None
    if dot_bits > 0:
        dense = np.ascontiguousarray(dot_dense, dtype=np.float64)
        if dense.shape != (1 << dot_bits, 1 << dot_bits):
            raise ValueError("dot_dense has the wrong shape")
        dot = _DenseBlock(dot_bits, dense.ctypes.data)
    h = C.c_void_p()
    _check(lib().polfed_build_hamiltonian(C.c_void_p(basis.handle), arr, len(terms),
                                          C.byref(dot) if dot is not None else None, fmt,
                                          _stream(stream), C.byref(h)))
    return Ham(h.value)


def polfed_ham_from_csr(row_ptr, col, val) -> Ham:
    """Wrap int32/int32/fp64 CUDA tensors (kept alive by the returned handle)."""
    import torch
    if row_ptr.dtype != torch.int32 or col.dtype != torch.int32 or val.dtype != torch.float64:
        raise ValueError("CSR tensors must be int32, int32, float64")
    n, nnz = row_ptr.numel() - 1, col.numel()
    h = C.c_void_p()
    _check(lib().polfed_ham_from_csr(n, nnz, _dev(row_ptr), _dev(col), _dev(val), C.byref(h)))
    return Ham(h.value, keep=(row_ptr, col, val))


def polfed_ham_from_csr_ex(row_ptr, col, val, flags: int = 0, stream=None) -> Ham:
    """polfed_ham_from_csr with flags (HAM_NO_SNAPSHOT: the handle keeps no copy of the values, so
    in-place updates of `val` are seen by later steps) and the stream the arrays were written on."""
    import torch
    if row_ptr.dtype != torch.int32 or col.dtype != torch.int32 or val.dtype != torch.float64:
        raise ValueError("CSR tensors must be int32, int32, float64")
    n, nnz = row_ptr.numel() - 1, col.numel()
    h = C.c_void_p()
    _check(lib().polfed_ham_from_csr_ex(n, nnz, _dev(row_ptr), _dev(col), _dev(val), flags,
                                        _stream(stream), C.byref(h)))
    return Ham(h.value, keep=(row_ptr, col, val))


def polfed_ham_csr(ham: Ham):
    """(row_ptr, col, val) as CUDA tensors (copies of the device arrays)."""
    import torch
    n, nnz = C.c_int64(), C.c_int64()
    rp, cp, vp = C.c_void_p(), C.c_void_p(), C.c_void_p()
    _check(lib().polfed_ham_csr(C.c_void_p(ham.handle), C.byref(n), C.byref(nnz), C.byref(rp),
                                C.byref(cp), C.byref(vp)))
    return (_copy_out(rp.value, n.value + 1, "<i4", torch.int32),
            _copy_out(cp.value, nnz.value, "<i4", torch.int32),
            _copy_out(vp.value, nnz.value, "<f8", torch.float64))


class _RawDevice:
    """Library-owned device memory exposed through __cuda_array_interface__."""

    def __init__(self, ptr: int, n: int, typestr: str):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": typestr,
                                         "data": (int(ptr), False), "version": 2}


def _copy_out(ptr: Optional[int], n: int, typestr: str, dtype):
    import torch
    if n == 0 or not ptr:
        return torch.empty(n, dtype=dtype, device="cuda")
    torch.cuda.synchronize()
    return torch.as_tensor(_RawDevice(ptr, n, typestr), device="cuda").clone()


# ---- hot path -------------------------------------------------------------------------

def polfed_fused_step(ham: Ham, s: int, p: float, q: float, r: float, c: float, X, Z, V, Y,
                      stream=None) -> None:
    _check(lib().polfed_fused_step(C.c_void_p(ham.handle), s, p, q, r, c, _block(X, ham.n, s),
                                   None if Z is None else _block(Z, ham.n, s),
                                   None if V is None else _block(V, ham.n, s),
                                   _block(Y, ham.n, s), _stream(stream)))


def polfed_filter_workspace_bytes(n: int, s: int) -> int:
    return int(lib().polfed_filter_workspace_bytes(n, s))


def polfed_filter_workspace_bytes_ham(ham: Ham, s: int) -> int:
    return int(lib().polfed_filter_workspace_bytes_ham(C.c_void_p(ham.handle), s))


def polfed_filter_apply(ham: Ham, a: float, b: float, coeffs: np.ndarray, s: int, V, W, work,
                        stream=None) -> None:
    """W = sum_k coeffs[k] T_k((H-a)/b) V; K = len(coeffs) - 1; work holds
    polfed_filter_workspace_bytes_ham(ham, s) bytes."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    K = c.shape[0] - 1
    if work is not None and \
            work.numel() * work.element_size() < polfed_filter_workspace_bytes_ham(ham, s):
        raise ValueError("workspace too small")
    _check(lib().polfed_filter_apply(C.c_void_p(ham.handle), a, b, K, c.ctypes.data, s,
                                     _block(V, ham.n, s), _block(W, ham.n, s), _dev(work),
                                     _stream(stream)))


def polfed_filter_apply_host(ham: Ham, a: float, b: float, coeffs: np.ndarray, s: int,
                             V_host, W_host, stream=None) -> None:
    """Same with HOST blocks (numpy arrays or pinned CPU torch tensors), copies included."""
    c = np.ascontiguousarray(coeffs, dtype=np.float64)
    K = c.shape[0] - 1

    def host_ptr(t):
        if isinstance(t, np.ndarray):
            if t.dtype != np.float64 or not t.flags.c_contiguous or t.size != ham.n * s:
                raise ValueError("expected a contiguous fp64 host block")
            return C.c_void_p(t.ctypes.data)
        if t.is_cuda or not t.is_contiguous() or t.numel() != ham.n * s:
            raise ValueError("expected a contiguous fp64 host block")
        return C.c_void_p(t.data_ptr())

    _check(lib().polfed_filter_apply_host(C.c_void_p(ham.handle), a, b, K, c.ctypes.data, s,
                                          host_ptr(V_host), host_ptr(W_host), _stream(stream)))


def polfed_filter_coeffs(a: float, b: float, sigma: float, nev: int = 1,
                         rho_rescaled: float = 0.0, K_in: int = 0) -> np.ndarray:
    """Coefficients c_0..c_K (K = K_in, or the order rule when rho_rescaled > 0)."""
    K = C.c_int()
    _check(lib().polfed_filter_coeffs(a, b, sigma, nev, rho_rescaled, K_in, C.byref(K), None, 0))
    out = np.empty(K.value + 1, dtype=np.float64)
    _check(lib().polfed_filter_coeffs(a, b, sigma, nev, rho_rescaled, K_in, C.byref(K),
                                      out.ctypes.data, out.shape[0]))
    return out


# ---- spectral bounds and the eigen-solver ---------------------------------------------------

def polfed_spectrum_bounds(ham: Ham, v0, n_steps: int = 0, margin: float = -1.0, stream=None):
    """(e_min, e_max, a, b) from n_steps Lanczos steps started at the fp64 CUDA vector v0."""
    import torch
    if v0.dtype != torch.float64 or v0.numel() != ham.n:
        raise ValueError("v0 must be an fp64 CUDA vector of length n")
    out = [C.c_double() for _ in range(4)]
    _check(lib().polfed_spectrum_bounds(C.c_void_p(ham.handle), n_steps, _dev(v0), margin,
                                        _stream(stream), *[C.byref(o) for o in out]))
    return tuple(o.value for o in out)


def polfed_block_gram(Q, B, variant: int = 0, stream=None):
    """C[j] = Q[j]^T B for the panels Q[j] (CUDA tensor k x n x s) and the block B (n x s):
    returns a CUDA tensor k x s x s.  variant: 0 library's choice, 1 FMA kernel, 2 tensor cores."""
    import torch
    k, n, s = Q.shape
    Cm = torch.empty(k, s, s, dtype=torch.float64, device="cuda")
    _check(lib().polfed_block_gram(s, n, _dev(Q), k, n * s, _block(B, n, s), _dev(Cm), variant,
                                   _stream(stream)))
    return Cm


STATIC_GRAM_DOUBLES = 524288   # POLFED_STATIC_GRAM_DOUBLES of include/polfed.h


def polfed_block_gram_static(Q, B, out, variant: int = 0, stream=None):
    """polfed_block_gram without any device allocation, for callers that cannot allocate (all HBM
    already given to the Krylov basis, a fixed device-memory budget, or a loop that must not meet the
    allocator's synchronisation): the partial sums go to a 4 MiB array inside the library.  The
    wrapper allocates nothing either, so the result tensor `out` (k x s x s, fp64, CUDA) is the
    caller's.  Needs k*s*s <= STATIC_GRAM_DOUBLES (else PolfedError, code ERANGE).  Calls share
    the array: never let two of them overlap on the GPU.  Returns `out`."""
    import torch
    k, n, s = Q.shape
    if out.dtype != torch.float64 or tuple(out.shape) != (k, s, s):
        raise ValueError(f"out must be an fp64 CUDA tensor of shape {(k, s, s)}")
    _check(lib().polfed_block_gram_static(s, n, _dev(Q), k, n * s, _block(B, n, s), _dev(out),
                                          variant, _stream(stream)))
    return out


def polfed_block_update(Q, Cm, B, alpha: float, beta: float, stream=None) -> None:
    """B = beta B + alpha sum_j Q[j] C[j] in place (Q: k x n x s, C: k x s x s, B: n x s)."""
    k, n, s = Q.shape
    _check(lib().polfed_block_update(s, n, _dev(Q), k, n * s, _dev(Cm), alpha, beta,
                                     _block(B, n, s), _stream(stream)))


def polfed_kpm_workspace_bytes(n: int, s: int, n_moments: int) -> int:
    return int(lib().polfed_kpm_workspace_bytes(n, s, n_moments))


def polfed_kpm_moments(ham: Ham, a: float, b: float, n_moments: int, R, work=None,
                       stream=None) -> np.ndarray:
    """Chebyshev moments mu_0..mu_{n_moments-1} of the density of states from the n x s fp64 CUDA
    block R of random vectors (Eq. 37-38)."""
    import torch
    if R.dim() != 2 or R.shape[0] != ham.n:
        raise ValueError("R must be an n x s block")
    s = int(R.shape[1])
    need = polfed_kpm_workspace_bytes(ham.n, s, n_moments)
    if work is None:
        work = torch.empty(max(need // 8, 1), dtype=torch.float64, device="cuda")
    if work.dtype != torch.float64 or work.numel() * 8 < need:
        raise ValueError("work is too small (polfed_kpm_workspace_bytes)")
    out = np.empty(max(n_moments, 0), dtype=np.float64)
    _check(lib().polfed_kpm_moments(C.c_void_p(ham.handle), a, b, n_moments, s, _block(R, ham.n, s),
                                    _dev(work), out.ctypes.data, _stream(stream)))
    return out


def polfed_kpm_dos(moments: np.ndarray, e_rescaled) -> np.ndarray:
    """Jackson-damped KPM density of states (states per unit rescaled energy), Eq. (36), (39)."""
    mu = np.ascontiguousarray(moments, dtype=np.float64)
    e = np.ascontiguousarray(np.atleast_1d(e_rescaled), dtype=np.float64)
    rho = np.empty_like(e)
    _check(lib().polfed_kpm_dos(mu.ctypes.data, mu.shape[0], e.ctypes.data, e.shape[0],
                                rho.ctypes.data))
    return rho


def polfed_block_lanczos_eigs(ham: Ham, sigma: float, nev: int, s: int, V0, *, tol: float = 0.0,
                              max_krylov_dim: int = 0, check_every: int = 0, K_override: int = 0,
                              bounds_steps: int = 0, bounds_margin: float = -1.0, a: float = 0.0,
                              b: float = 0.0, sigma_is_rescaled: bool = False, stream=None,
                              allow_unconverged: bool = False, kpm_block=None,
                              kpm_moments: int = 0, window_levels: int = 0):
    """The nev eigenpairs of H nearest sigma: (evals ndarray, evecs CUDA tensor n x nev,
    residuals ndarray, report dict).  Raises PolfedError(ENOCONV or EWINDOW) unless allow_unconverged
    (report["status"] then holds the code).
    kpm_block (CUDA tensor n x R, R a multiple of 4): size K with the KPM density of states.
    window_levels > 0: size the filter window for that many levels instead of nev + 10 %."""
    import torch
    opt = _Options(tol, max_krylov_dim, check_every, K_override, bounds_steps, bounds_margin, a, b,
                   int(bool(sigma_is_rescaled)), 0, 0, 0, None, int(window_levels))
    if kpm_block is not None:
        if (kpm_block.dim() != 2 or kpm_block.shape[0] != ham.n or kpm_block.dtype != torch.float64
                or not kpm_block.is_cuda or not kpm_block.is_contiguous()):
            raise ValueError("kpm_block must be a contiguous fp64 CUDA tensor n x R")
        opt.dos, opt.kpm_moments, opt.kpm_vectors = 1, kpm_moments, int(kpm_block.shape[1])
        opt.d_kpm_block = kpm_block.data_ptr()
    rep = _Report()
    evals = np.empty(nev, dtype=np.float64)
    resid = np.empty(nev, dtype=np.float64)
    evecs = torch.empty(ham.n, nev, dtype=torch.float64, device="cuda")
    code = lib().polfed_block_lanczos_eigs(C.c_void_p(ham.handle), sigma, nev, s,
                                           _block(V0, ham.n, s), C.byref(opt), evals.ctypes.data,
                                           _dev(evecs), resid.ctypes.data, C.byref(rep),
                                           _stream(stream))
    if not (code in (ENOCONV, EWINDOW) and allow_unconverged):
        _check(code)
    report = {name: getattr(rep, name) for name, _ in _Report._fields_ if name != "reserved"}
    report["status"] = code
    return evals, evecs, resid, report
