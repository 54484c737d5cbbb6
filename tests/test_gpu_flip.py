"""Parity of the flip format (POLFED_FORMAT_FLIP: matrix-free rows for full-space models with a
dense block on bits 0-2 and uniform two-bit flips, include/polfed.h) against the CPU oracle's CSR
SpMM and textbook Clenshaw (Eq. 31, 51 PAPER.md:274-276, 427-431) on the same seeded inputs.
The flip path differs from the oracle only in summation order."""
from __future__ import annotations

import numpy as np
import pytest

import workloads
from oracle import cheb, core, lanczos

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import paper_2605_10191_b200 as pkg
    pkg.lib()
    return pkg


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def rel_l2(got, want):
    return float(np.linalg.norm(got - want) / max(np.linalg.norm(want), 1e-300))


def build(P, n_sites, terms, dot_bits=0, dot_dense=None):
    basis = P.polfed_build_basis(n_sites, -1)
    return P.polfed_build_hamiltonian(basis, terms, dot_bits, dot_dense, fmt=P.FORMAT_FLIP)


def oracle_csr(n_sites, terms, dot_bits=0, dot_dense=None):
    return core.build_csr(core.basis_states(n_sites, -1), terms, dot_bits, dot_dense)


@pytest.mark.parametrize("s", (8, 16, 32))
@pytest.mark.parametrize("L_outer", (2, 6, 9))
def test_flip_fused_step_matches_oracle_on_quantum_sun(P, s, L_outer):
    w = workloads.make_workload(4, L_override=L_outer)
    _, H = core.hamiltonian(w)
    ham = build(P, w.n_sites, w.terms, w.dot_bits, w.dot_dense)
    rng = np.random.default_rng(10 * L_outer + s)
    X, Z, V = (rng.standard_normal((H.n, s)) for _ in range(3))
    p, q, r, c = 0.13, -0.7, -1.0, 0.45
    want = p * core.spmm(H, X) + q * X + r * Z + c * V
    scale = np.abs(p) * core.spmm(core.CSR(H.n, H.row_ptr, H.col, np.abs(H.val)), np.abs(X)) \
        + np.abs(q * X) + np.abs(r * Z) + np.abs(c * V)
    Y = torch.full((H.n, s), float("nan"), dtype=torch.float64, device="cuda")
    P.polfed_fused_step(ham, s, p, q, r, c, dev(X), dev(Z), dev(V), Y)
    assert np.all(np.abs(Y.cpu().numpy() - want) <= 1e-13 * scale)
    Zd = dev(Z)                                   # in place over Z, and the r = c = 0 variant
    P.polfed_fused_step(ham, s, p, q, r, c, dev(X), Zd, dev(V), Zd)
    assert np.all(np.abs(Zd.cpu().numpy() - want) <= 1e-13 * scale)
    P.polfed_fused_step(ham, s, 1.0, 0.0, 0.0, 0.0, dev(X), None, None, Y)
    assert np.all(np.abs(Y.cpu().numpy() - core.spmm(H, X)) <= 1e-13 * scale / abs(p))


def test_flip_general_terms(P):
    """Flips inside the low three bits, outside them, across; duplicates; negative amplitudes;
    a dense block on two bits only; diagonal kinds; no dense block at all."""
    n_sites, s = 9, 16
    rng = np.random.default_rng(77)
    A = rng.standard_normal((4, 4))
    dot = (A + A.T) / 2
    terms = [("XX", 0, 1, 0.3), ("XX", 2, 0, -0.2), ("XX", 1, 5, 0.7), ("XX", 1, 5, 0.1),
             ("XX", 4, 8, -0.9), ("XX", 3, 7, 0.25), ("XX", 2, 8, 0.6),
             ("Z", 3, 3, 0.8), ("ZZ", 0, 6, -0.5), ("Z", 0, 0, 0.3)]
    for dot_bits, dd in ((2, dot), (0, None)):
        H = oracle_csr(n_sites, terms, dot_bits, dd)
        ham = build(P, n_sites, terms, dot_bits, dd)
        X = rng.standard_normal((H.n, s))
        Y = torch.empty(H.n, s, dtype=torch.float64, device="cuda")
        P.polfed_fused_step(ham, s, 1.0, 0.0, 0.0, 0.0, dev(X), None, None, Y)
        want = core.spmm(H, X)
        assert np.max(np.abs(Y.cpu().numpy() - want)) <= 1e-13 * np.abs(want).max() * 10


@pytest.mark.parametrize("L_outer,K", [(7, 300), (9, 1000)])
def test_flip_filter_matches_oracle(P, L_outer, K):
    w = workloads.make_workload(4, L_override=L_outer)
    _, H = core.hamiltonian(w)
    v0 = workloads.start_block(H.n, 1, seed=3004)[:, 0]
    _, _, a, b = lanczos.spectrum_bounds(H, v0, m=60, margin=0.01)
    lam = (w.target - a) / b
    coeffs = cheb.filter_coeffs(lam, K)
    V = workloads.start_block(H.n, w.s, seed=2004, orthonormal=True)
    want = core.clenshaw(H, a, b, coeffs, V)
    ham = build(P, w.n_sites, w.terms, w.dot_bits, w.dot_dense)
    W = torch.empty(H.n, w.s, dtype=torch.float64, device="cuda")
    work = torch.empty(P.polfed_filter_workspace_bytes_ham(ham, w.s) // 8, dtype=torch.float64,
                       device="cuda")
    P.polfed_filter_apply(ham, a, b, coeffs, w.s, dev(V), W, work)
    assert rel_l2(W.cpu().numpy(), want) <= 1e-9


def test_flip_filter_with_the_librarys_exact_zero_coefficients(P):
    """R22 / VERDICT r2: target in the middle of the interval (lambda~ = 0), the library's
    coefficients (odd ones exactly 0, Eq. 33) on both sides: the flip steps without a V read."""
    w = workloads.make_workload(4, L_override=9)
    _, H = core.hamiltonian(w)
    v0 = workloads.start_block(H.n, 1, seed=3004)[:, 0]
    _, _, a, b = lanczos.spectrum_bounds(H, v0, m=60, margin=0.01)
    K = 640
    coeffs = P.polfed_filter_coeffs(a, b, a, K_in=K)
    assert np.count_nonzero(coeffs[1::2]) == 0 and np.count_nonzero(coeffs[0::2]) == K // 2 + 1
    V = workloads.start_block(H.n, w.s, seed=2004, orthonormal=True)
    want = core.clenshaw(H, a, b, coeffs, V)
    ham = build(P, w.n_sites, w.terms, w.dot_bits, w.dot_dense)
    W = torch.empty(H.n, w.s, dtype=torch.float64, device="cuda")
    work = torch.empty(P.polfed_filter_workspace_bytes_ham(ham, w.s) // 8, dtype=torch.float64,
                       device="cuda")
    P.polfed_filter_apply(ham, a, b, coeffs, w.s, dev(V), W, work)
    assert rel_l2(W.cpu().numpy(), want) <= 1e-9


def test_flip_eigensolver_and_small_block_sizes(P):
    """The eigen-solver on a flip handle (every fused step goes through the flip kernel) returns
    true eigenpairs; block sizes the flip kernel does not cover use the CSR of the same handle."""
    w = workloads.make_workload(4, L_override=8)
    _, H = core.hamiltonian(w)
    ham = build(P, w.n_sites, w.terms, w.dot_bits, w.dot_dense)
    V0 = dev(workloads.start_block(H.n, 16, seed=2004))
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(ham, w.target, 12, 16, V0)
    U = evecs.cpu().numpy()
    hnorm = max(abs(rep["e_min"]), abs(rep["e_max"]))
    R = core.spmm(H, U) - U * evals
    assert np.max(np.linalg.norm(R, axis=0)) <= 1e-8 * hnorm
    dense = np.linalg.eigvalsh(np.asarray(
        __import__("scipy.sparse", fromlist=["csr_matrix"]).csr_matrix(
            (H.val, H.col, H.row_ptr), shape=(H.n, H.n)).todense()))
    nearest = dense[np.argsort(np.abs(dense - w.target))[:12]]
    assert np.max(np.abs(np.sort(nearest) - np.sort(evals))) <= 1e-9 * hnorm
    X = np.random.default_rng(3).standard_normal((H.n, 4))
    Y = torch.empty(H.n, 4, dtype=torch.float64, device="cuda")
    P.polfed_fused_step(ham, 4, 1.0, 0.0, 0.0, 0.0, dev(X), None, None, Y)
    assert np.max(np.abs(Y.cpu().numpy() - core.spmm(H, X))) <= 1e-12


def test_flip_ineligible_requests_fail_loudly(P):
    cases = [(8, 4, [("XX", 0, 1, 1.0)], 0, None),                          # fixed n_up
             (8, -1, [("EXCH", 0, 1, 1.0)], 0, None),                       # state-dependent hop
             (2, -1, [("XX", 0, 1, 1.0)], 0, None),                         # fewer than 3 sites
             (8, -1, [("XX", 0, 5, 1.0)], 4, np.eye(16))]                   # dense block too wide
    for n_sites, n_up, terms, db, dd in cases:
        basis = P.polfed_build_basis(n_sites, n_up)
        with pytest.raises(P.PolfedError):
            P.polfed_build_hamiltonian(basis, terms, db, dd, fmt=P.FORMAT_FLIP)


def test_flip_full_size_config4_sampled_rows(P):
    """Config 4 at full size (D = 2^20, s = 16) in bench.py's launch configuration: one recurrence
    step on sampled rows the oracle computes one by one, plus agreement with the CSR kernel."""
    w = workloads.make_workload(4)
    states = core.basis_states(w.n_sites, w.n_up)
    n, s = int(states.shape[0]), w.s
    ham = build(P, w.n_sites, w.terms, w.dot_bits, w.dot_dense)
    assert ham.n == n == 1 << 20 and ham.nnz == 26_214_400
    gen = torch.Generator(device="cuda").manual_seed(5004)
    B1, B2, V = (torch.randn(n, s, dtype=torch.float64, device="cuda", generator=gen)
                 for _ in range(3))
    a, b, ck = 0.3, 9.0, 0.123
    Y = torch.empty_like(B1)
    P.polfed_fused_step(ham, s, 2.0 / b, -2.0 * a / b, -1.0, ck, B1, B2, V, Y)
    rng = np.random.default_rng(4004)
    rows = np.unique(np.concatenate([[0, 1, 7, 8, n // 2, n - 2, n - 1], rng.integers(0, n, 3000)]))
    mini = core.build_csr_rows(states, rows, w.terms, w.dot_bits, w.dot_dense)
    B1h = B1.cpu().numpy()
    rows_d = torch.from_numpy(rows).cuda()
    T = (core.spmm(mini, B1h) - a * B1h[rows]) / b
    want = ck * V[rows_d].cpu().numpy() + 2.0 * T - B2[rows_d].cpu().numpy()
    assert np.max(np.abs(Y[rows_d].cpu().numpy() - want)) <= 1e-12
    basis = P.polfed_build_basis(w.n_sites, -1)
    csr = P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense)
    Y2 = torch.empty_like(B1)
    P.polfed_fused_step(csr, s, 2.0 / b, -2.0 * a / b, -1.0, ck, B1, B2, V, Y2)
    assert float((Y - Y2).norm() / Y2.norm()) <= 1e-14


def test_flip_full_size_config4_filter_K1000_whole_block_against_oracle(P):
    """Config 4 at full size (quantum sun, D = 2^20, s = 16), K = 1000 (SURVEY 8(d)'s K_par), every
    element judged by the ORACLE: its CSR of the whole matrix, its textbook Clenshaw (Eq. 51
    PAPER.md:427-431) on the whole block, against polfed_filter_apply on the flip handle (the path
    bench.py times) and on the CSR handle.  rel l2 <= 1e-9 (north_star)."""
    w = workloads.make_workload(4)
    _, H = core.hamiltonian(w)
    n, s, K = H.n, w.s, 1000
    assert n == 1 << 20 and H.nnz == 26_214_400
    v0 = workloads.start_block(n, 1, seed=3004)[:, 0]
    _, _, a, b = lanczos.spectrum_bounds(H, v0, m=60, margin=0.01)
    lam = (w.target - a) / b
    coeffs = cheb.filter_coeffs(lam, K)
    V = workloads.start_block(n, s, seed=2004, orthonormal=True)
    want = core.clenshaw(H, a, b, coeffs, V)
    del H
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    for fmt in (P.FORMAT_FLIP, P.FORMAT_CSR):
        ham = P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense, fmt=fmt)
        W = torch.full((n, s), float("nan"), dtype=torch.float64, device="cuda")
        work = torch.empty(P.polfed_filter_workspace_bytes_ham(ham, s) // 8, dtype=torch.float64,
                           device="cuda")
        P.polfed_filter_apply(ham, a, b, coeffs, s, dev(V), W, work)
        got = W.cpu().numpy()
        assert np.all(np.isfinite(got)), fmt
        assert rel_l2(got, want) <= 1e-9, fmt
        assert np.max(np.abs(got - want)) <= 1e-11 * np.abs(want).max(), fmt
