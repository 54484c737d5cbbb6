"""CPU-only checks of the C-ABI library: it loads, exports every symbol include/polfed.h
declares, and its host-only entry points agree with the oracle.  No GPU compute is called."""
from __future__ import annotations

import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2605_10191_b200 as P
from paper_2605_10191_b200 import build as libbuild
from oracle import cheb

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "polfed.h")


@pytest.fixture(scope="module")
def lib():
    libbuild.build()
    return P.lib()


def declared_symbols():
    text = open(HEADER).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(polfed_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(lib):
    names = declared_symbols()
    assert len(names) >= 16
    for name in names:
        assert hasattr(lib, name), f"{name} declared in polfed.h but not exported"
    assert set(P.EXPORTS) == set(names)


def test_binding_has_a_wrapper_for_every_entry_point():
    for name in declared_symbols():
        if name.endswith("_destroy"):
            continue          # owned by the Basis / Ham wrappers
        assert callable(getattr(P, name)), name


def test_product_package_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2605_10191_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert "oracle" not in open(os.path.join(dirpath, f)).read().lower(), f


@pytest.mark.parametrize("lam,K", [(0.0, 0), (0.0, 1), (0.3, 50), (-0.61, 777), (0.0, 5000),
                                   (0.07, 20000)])
def test_filter_coeffs_match_oracle(lib, lam, K):
    a, b = 0.4, 3.0
    got = P.polfed_filter_coeffs(a, b, a + b * lam, K_in=K)
    want = cheb.filter_coeffs(lam, K)
    assert got.shape == (K + 1,)
    # T_n = cos(n theta): an ulp of theta (or of lambda = (sigma-a)/b) moves T_n by ~ n * eps
    eps = np.finfo(np.float64).eps
    assert np.max(np.abs(got - want)) <= (4 + 4 * K) * eps * np.max(np.abs(want))
    # P(lambda) = 1 for the library's own coefficients
    assert abs(cheb.filter_value(got, [lam])[0] - 1.0) < 1e-12


def test_filter_coeffs_at_mid_spectrum_have_exact_zeros(lib):
    """Eq. (33): c_n is proportional to T_n(lambda~), and T_n(0) = 0 exactly for odd
    n.  The library must return exact zeros there at every order (R22: a zero coefficient lets the
    fused step skip its V read) -- K = 13 422 is config 3's order -- and +-2/chi at the even ones."""
    a, b, K = -0.7, 2.5, 13422
    got = P.polfed_filter_coeffs(a, b, a, K_in=K)           # sigma = a: lambda~ = 0 exactly
    assert np.count_nonzero(got[1::2]) == 0 and got[1::2].size == 6711
    chi = 1.0 + 2.0 * (K // 2)                               # 1 + 2 * #(even n in 1..K)
    n_even = np.arange(2, K + 1, 2)
    assert got[0] == 1.0 / chi
    assert np.array_equal(got[2::2], np.where(n_even % 4 == 0, 2.0, -2.0) / chi)
    want = cheb.filter_coeffs(0.0, K)
    eps = np.finfo(np.float64).eps
    assert np.max(np.abs(got - want)) <= (4 + 4 * K) * eps * np.max(np.abs(want))


@pytest.mark.parametrize("lam,nev,rho", [(0.0, 50, 20000.0), (0.1, 50, 20000.0),
                                         (-0.3, 20, 900.0), (0.45, 100, 3.0e5)])
def test_order_rule_matches_oracle(lib, lam, nev, rho):
    got = P.polfed_filter_coeffs(0.0, 1.0, lam, nev=nev, rho_rescaled=rho)
    K = got.shape[0] - 1
    K_or = cheb.order_bisect(nev, rho, lam)
    assert abs(K - K_or) <= 1          # both bisect Eq. (41); allow a rounding tie at the edge
    K42 = cheb.order_eq42(nev, rho, lam)
    assert K42 // 2 <= K <= 2 * K42    # the bracket of PAPER.md:362


def test_host_argument_errors(lib):
    K = C.c_int()
    assert lib.polfed_filter_coeffs(0.0, 1.0, 2.0, 1, 0.0, 10, C.byref(K), None, 0) == P.binding.ERANGE
    assert "outside" in P.polfed_last_error()
    assert lib.polfed_filter_coeffs(0.0, -1.0, 0.0, 1, 0.0, 10, C.byref(K), None, 0) == P.binding.ERANGE
    buf = (C.c_double * 4)()
    assert lib.polfed_filter_coeffs(0.0, 1.0, 0.0, 1, 0.0, 10, C.byref(K), buf, 4) == P.binding.EINVAL
    assert K.value == 10
    assert lib.polfed_filter_workspace_bytes(1000, 8) == 2 * 1000 * 8 * 8
    h = C.c_void_p()
    assert lib.polfed_ham_from_csr(-1, 0, None, None, None, C.byref(h)) == P.binding.EINVAL
    assert lib.polfed_ham_destroy(None) == 0 and lib.polfed_basis_destroy(None) == 0


def test_kpm_dos_host_series_matches_oracle(lib):
    """polfed_kpm_dos is host-only (Eq. 36 with the Jackson kernel Eq. 39): same numbers as the
    oracle's series for arbitrary moments; energies outside (-1, 1) are a range error."""
    from oracle import cheb
    rng = np.random.default_rng(9)
    mu = rng.standard_normal(75)
    mu[0] = 100.0
    e = np.linspace(-0.95, 0.95, 41)
    want = cheb.kpm_dos(e, mu, cheb.jackson_kernel(75))
    got = P.polfed_kpm_dos(mu, e)
    assert np.max(np.abs(got - want)) <= 1e-11 * np.max(np.abs(want))
    with pytest.raises(P.PolfedError):
        P.polfed_kpm_dos(mu, [1.0])
    assert lib.polfed_kpm_workspace_bytes(1000, 8, 75) >= (2 * 1000 * 8 + 75) * 8
