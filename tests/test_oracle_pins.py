"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these re-type an oracle formula: each compares the oracle with an
independent object (a closed form, a library routine, a dense Kronecker-product
construction, brute force, or an invariant).  CPU only.
"""
from __future__ import annotations

import math
import os

import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb

import workloads
from oracle import cheb, core, lanczos
from tests import dense_models as dm

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_closed_forms.txt")


def golden():
    out = {}
    with open(GOLDEN) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if line:
                out.setdefault(line[0], []).append([float(t) for t in line[1:]])
    return out


def random_symmetric_csr(n, density, seed):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((n, n)) * (rng.random((n, n)) < density)
    A = np.triu(A, 1)
    A = A + A.T + np.diag(rng.standard_normal(n))
    row_ptr, col, val = [0], [], []
    for i in range(n):
        for j in range(n):
            if A[i, j] != 0.0 or i == j:
                col.append(j)
                val.append(A[i, j])
        row_ptr.append(len(col))
    H = core.CSR(n, np.array(row_ptr, np.int32), np.array(col, np.int32), np.array(val))
    return A, H


# ---- basis (O1) ---------------------------------------------------------------

@pytest.mark.parametrize("L,n_up", [(4, 2), (10, 5), (12, 6), (9, 3), (7, 0), (7, 7)])
def test_basis_dimension_order_and_combinadic_rank(L, n_up):
    st = core.basis_states(L, n_up)
    assert st.shape[0] == math.comb(L, n_up)
    assert np.all(np.diff(st.astype(np.int64)) > 0)
    assert all(bin(int(x)).count("1") == n_up for x in st)
    # combinatorial number system: rank(x) = sum_k C(p_k, k), p_1 < ... < p_k set bits
    for r, x in enumerate(st[:: max(1, st.shape[0] // 97)]):
        pos = [p for p in range(L) if (int(x) >> p) & 1]
        rank = sum(math.comb(p, k + 1) for k, p in enumerate(pos))
        assert core.basis_rank(st, int(x)) == rank
    assert core.basis_rank(st, (1 << L) + 1) == -1


def test_basis_dims_match_paper_closed_form():
    for L, D in golden()["u1_dim"]:
        if L <= 20:
            assert core.basis_states(int(L), int(L) // 2).shape[0] == int(D)
        assert math.comb(int(L), int(L) // 2) == int(D)


def test_full_space_basis_is_identity():
    st = core.basis_states(6, -1)
    assert np.array_equal(st, np.arange(64, dtype=np.uint64))


# ---- CSR assembly (O2) against independent dense constructions -------------------

@pytest.mark.parametrize("L,periodic", [(6, True), (8, True), (7, False)])
def test_xxz_csr_equals_kron_construction(L, periodic):
    rng = np.random.default_rng(7)
    h = rng.uniform(-2, 2, L)
    J, Delta = 1.22, 0.55                                     # the paper's values
    n_up = L // 2
    idx = dm.sector_indices(L, n_up)
    Hd = dm.xxz_dense(L, J, Delta, h, periodic)[np.ix_(idx, idx)]
    st = core.basis_states(L, n_up)
    H = core.build_csr(st, workloads.xxz_terms(L, J, Delta, h, periodic))
    assert np.allclose(H.to_dense(), Hd, atol=1e-14, rtol=0)


@pytest.mark.parametrize("L,N", [(6, 3), (8, 4), (7, 2)])
def test_fermion_csr_equals_jordan_wigner_construction(L, N):
    rng = np.random.default_rng(11)
    eps = rng.uniform(-2, 2, L)
    idx = dm.sector_indices(L, N)
    Hd = dm.fermion_dense(L, 1.0, 0.5, 1.0, eps)[np.ix_(idx, idx)]
    st = core.basis_states(L, N)
    H = core.build_csr(st, workloads.fermion_terms(L, 1.0, 0.5, 1.0, eps))
    assert np.allclose(H.to_dense(), Hd, atol=1e-14, rtol=0)
    # the next-nearest hop must carry minus signs somewhere (Jordan-Wigner), else the pin is blind
    assert (H.val < 0).any()


@pytest.mark.parametrize("N,L", [(2, 3), (3, 4)])
def test_quantum_sun_csr_equals_kron_construction(N, L):
    rng = np.random.default_rng(5)
    dot = workloads.configs.goe_dot_block(rng, N, 1.0)
    u = np.arange(L) + rng.uniform(-0.2, 0.2, L)
    n_of_j = rng.integers(0, N, L)
    h = rng.uniform(0.5, 1.5, L)
    Hd = dm.quantum_sun_dense(N, L, dot, 1.0, 0.75, u, n_of_j, h)
    st = core.basis_states(N + L, -1)
    H = core.build_csr(st, workloads.quantum_sun_terms(N, L, 1.0, 0.75, u, n_of_j, h), N, dot)
    assert np.allclose(H.to_dense(), Hd, atol=1e-14, rtol=0)
    # exactly 2^N dot entries (diagonal included) + L double flips per row (reading R14)
    assert np.all(np.diff(H.row_ptr) == (1 << N) + L)


def test_xxz_offdiagonal_count_matches_eq63_and_trace_closed_form():
    g = golden()
    for L, total in g["xxz_offdiag_total"]:
        L, total = int(L), int(total)
        if L > 16:
            continue
        w = workloads.make_workload(1, L_override=L)
        st, H = core.hamiltonian(w)
        D = st.shape[0]
        assert H.nnz - D == total                               # Eq. (63)
        # columns ascending, diagonal always stored
        for i in range(0, D, max(1, D // 50)):
            c = H.col[H.row_ptr[i]:H.row_ptr[i + 1]]
            assert np.all(np.diff(c) > 0) and i in c
        # Tr H / D = -J Delta L / (4 (L-1)) in the S_z = 0 sector (reading R13); fields average out
        rows = np.repeat(np.arange(D), np.diff(H.row_ptr))
        tr = H.val[rows == H.col].sum()
        assert abs(tr / D - (-L / (4.0 * (L - 1)))) < 1e-12


def test_xxz_L20_count_matches_eq63():
    total = [int(t) for L, t in golden()["xxz_offdiag_total"] if int(L) == 20][0]
    st, H = core.hamiltonian(workloads.make_workload(3))
    assert st.shape[0] == 184756 and H.nnz - st.shape[0] == total


def test_fermion_nnz_closed_form_and_symmetry():
    # open chain, L sites, N particles: each of the (L-1)+(L-2) bonds connects
    # 2 C(L-2, N-1) ordered pairs of basis states.
    L, N = 12, 6
    w = workloads.make_workload(5, L_override=L)
    st, H = core.hamiltonian(w)
    D = st.shape[0]
    assert H.nnz == (2 * L - 3) * 2 * math.comb(L - 2, N - 1) + D
    A = H.to_dense()
    assert np.array_equal(A, A.T)
    assert (2 * 26 - 3) * 2 * math.comb(24, 12) + math.comb(26, 13) == 275_407_888


def test_goe_block_normalisation():
    exp = golden()["goe_trace_expectation"][0][1]
    rng = np.random.Generator(np.random.PCG64(3))
    tr = np.mean([np.trace(np.linalg.matrix_power(
        workloads.configs.goe_dot_block(rng, 3, 1.0) * 3.0, 2)) for _ in range(4000)])
    assert abs(tr - exp) / exp < 0.02


def test_csr_symmetry_and_conservation_config2_size():
    st, H = core.hamiltonian(workloads.make_workload(2, L_override=12))
    A = H.to_dense()
    assert np.array_equal(A, A.T)
    assert H.col.min() >= 0 and H.col.max() < st.shape[0]


# ---- SpMM (O3) and rescaling (O4) ------------------------------------------------

def test_spmm_equals_dense_matmul_and_is_linear_and_symmetric():
    A, H = random_symmetric_csr(83, 0.15, 1)
    rng = np.random.default_rng(2)
    for s in (1, 3, 8):
        X = rng.standard_normal((83, s))
        assert np.allclose(core.spmm(H, X), A @ X, atol=1e-13)
    x, y = rng.standard_normal((83, 1)), rng.standard_normal((83, 1))
    assert np.allclose(core.spmm(H, 2 * x - 3 * y), 2 * core.spmm(H, x) - 3 * core.spmm(H, y), atol=1e-12)
    assert abs(float(x.T @ core.spmm(H, y)) - float(y.T @ core.spmm(H, x))) < 1e-11
    a, b = 0.3, 2.5
    assert np.allclose(core.rescaled_apply(H, a, b, x), (A - a * np.eye(83)) @ x / b, atol=1e-13)


def test_spmm_transpose_symmetry_at_large_size():
    st, H = core.hamiltonian(workloads.make_workload(2))          # D = 12 870
    rng = np.random.default_rng(4)
    x, y = rng.standard_normal((H.n, 2)), rng.standard_normal((H.n, 2))
    lhs = np.sum(x * core.spmm(H, y))
    rhs = np.sum(y * core.spmm(H, x))
    assert abs(lhs - rhs) <= 1e-10 * abs(lhs)


# ---- coefficients and the filter as a function -----------------------------------

@pytest.mark.parametrize("lam", [0.0, 0.37, -0.61])
@pytest.mark.parametrize("K", [1, 7, 200, 1001])
def test_filter_is_one_at_target_and_matches_dirichlet_closed_form(lam, K):
    c = cheb.filter_coeffs(lam, K)
    assert abs(cheb.filter_value(c, [lam])[0] - 1.0) < 1e-12       # P(lam) = 1
    # closed form: P(cos th) = [D_K(th-ph) + D_K(th+ph)] / (2 chi), D_K(u) = sin((K+1/2)u)/sin(u/2)
    ph = math.acos(lam)
    dk = lambda u: math.sin((K + 0.5) * u) / math.sin(0.5 * u) if abs(math.sin(0.5 * u)) > 1e-300 else 2 * K + 1
    chi = 0.5 * ((2 * K + 1) + dk(2 * ph))
    for x in (-0.93, -0.2, 0.111, 0.5, 0.99):
        th = math.acos(x)
        closed = (dk(th - ph) + dk(th + ph)) / (2 * chi)
        assert abs(cheb.filter_value(c, [x])[0] - closed) < 1e-11
    assert abs(c[0] - 1.0 / chi) < 1e-13 / chi
    if lam == 0.0:
        assert abs(1.0 / c[0] - (1 + 2 * (K // 2))) < 1e-9           # chi = 1 + 2 floor(K/2)


def test_filter_value_equals_numpy_chebval():
    c = cheb.filter_coeffs(0.23, 300)
    x = np.linspace(-1, 1, 41)
    assert np.allclose(cheb.filter_value(c, x), npcheb.chebval(x, c), atol=1e-12)


# ---- Clenshaw (O6) ---------------------------------------------------------------

@pytest.mark.parametrize("k", [0, 1, 2, 5, 40])
def test_clenshaw_single_coefficient_gives_cos_k_theta(k):
    # T_k(cos th) = cos(k th) (inside Eq. 33): a 1x1 "Hamiltonian" [x], coefficient e_k
    for th in (0.3, 1.1, 2.9):
        x = math.cos(th)
        H = core.CSR(1, np.array([0, 1], np.int32), np.array([0], np.int32), np.array([x]))
        c = np.zeros(k + 1)
        c[k] = 1.0
        W = core.clenshaw(H, 0.0, 1.0, c, np.array([[1.0]]))
        assert abs(W[0, 0] - math.cos(k * th)) < 1e-12


@pytest.mark.parametrize("K", [0, 1, 2, 3, 50, 300])
def test_matrix_clenshaw_equals_spectral_definition(K):
    # Eq. (27): f(H) = U f(Lambda) U^T, so P(H~) V = U diag(P(lam~_i)) U^T V
    A, H = random_symmetric_csr(60, 0.2, K + 1)
    ev, U = np.linalg.eigh(A)
    a, b = cheb.rescale_params(ev[0], ev[-1], 0.01)
    rng = np.random.default_rng(9)
    c = rng.standard_normal(K + 1)                                    # arbitrary coefficients
    V = rng.standard_normal((60, 4))
    P = npcheb.chebval((ev - a) / b, c)
    truth = U @ (P[:, None] * (U.T @ V))
    W = core.clenshaw(H, a, b, c, V)
    assert np.linalg.norm(W - truth) <= 1e-12 * max(1.0, np.linalg.norm(truth)) * (K + 1)


def test_clenshaw_on_config1_equals_dense_diagonalisation():
    w = workloads.make_workload(1)
    st, H = core.hamiltonian(w)
    A = H.to_dense()
    ev, U = np.linalg.eigh(A)
    a, b = cheb.rescale_params(ev[0], ev[-1], 0.01)
    lam = (w.target - a) / b
    c = cheb.filter_coeffs(lam, w.K_fixed)
    V = workloads.start_block(H.n, 3, 2001)
    truth = U @ (cheb.filter_value(c, (ev - a) / b)[:, None] * (U.T @ V))
    W = core.clenshaw(H, a, b, c, V)
    assert np.linalg.norm(W - truth) <= 1e-11 * np.linalg.norm(truth)


def test_clenshaw_column_independence_and_linearity():
    A, H = random_symmetric_csr(40, 0.3, 3)
    c = cheb.filter_coeffs(0.1, 25)
    rng = np.random.default_rng(1)
    V = rng.standard_normal((40, 5))
    W = core.clenshaw(H, 0.2, 9.0, c, V)
    for j in range(5):
        assert np.array_equal(core.clenshaw(H, 0.2, 9.0, c, V[:, j:j + 1])[:, 0], W[:, j])


# ---- sampled-row builder and single-step helper (full-size spot checks, cpu_baseline) ----

@pytest.mark.parametrize("config,L", [(3, 14), (4, 9), (5, 14)])
def test_build_csr_rows_equals_the_same_rows_of_build_csr(config, L):
    # orc_build_csr_rows carries the full-size parity checks of configs 4-5 (tests/test_gpu_*.py)
    # and bench.py's cpu_baseline: it must return exactly the rows of the full assembly (O2,
    # PAPER.md:858-861 Eq. 54, 939-946 Eq. 67), whatever the order of the requested rows.
    w = workloads.make_workload(config, L_override=L)
    st, H = core.hamiltonian(w)
    D = H.n
    rng = np.random.default_rng(17 + config)
    rows = np.concatenate([[0, D - 1, D - 1, 0, D // 2], rng.integers(0, D, 400),
                           np.arange(D - 5, D), np.arange(7)[::-1]]).astype(np.int64)
    sub = core.build_csr_rows(st, rows, w.terms, w.dot_bits, w.dot_dense)
    assert sub.n == rows.size and sub.row_ptr[0] == 0
    assert np.array_equal(np.diff(sub.row_ptr), np.diff(H.row_ptr)[rows])
    assert sub.nnz == int(np.diff(H.row_ptr)[rows].sum())
    for k, r in enumerate(rows):
        lo, hi = H.row_ptr[r], H.row_ptr[r + 1]
        slo, shi = sub.row_ptr[k], sub.row_ptr[k + 1]
        assert np.array_equal(sub.col[slo:shi], H.col[lo:hi])
        assert np.array_equal(sub.val[slo:shi].view(np.int64), H.val[lo:hi].view(np.int64))
    # and the product on the mini-CSR is the corresponding rows of the full product
    X = rng.standard_normal((D, 3))
    assert np.array_equal(core.spmm(sub, X), core.spmm(H, X)[rows])


def test_build_csr_rows_empty_selection():
    w = workloads.make_workload(5, L_override=10)
    st, _ = core.hamiltonian(w)
    sub = core.build_csr_rows(st, np.zeros(0, np.int64), w.terms)
    assert sub.n == 0 and sub.nnz == 0 and sub.row_ptr.tolist() == [0]


@pytest.mark.parametrize("K", [1, 2, 3, 17, 120])
def test_clenshaw_step_chain_reproduces_clenshaw(K):
    # the timed cpu_baseline calls orc_clenshaw_step; K-1 of them with the buffer swap of Fig. 5
    # must give the b_1, b_2 of orc_clenshaw (Eq. 51) to the last bit, and the
    # final line W = c_0 V + H~ b_1 - b_2 must then reproduce its W.
    A, H = random_symmetric_csr(60, 0.2, 40 + K)
    ev = np.linalg.eigvalsh(A)
    a, b = cheb.rescale_params(ev[0], ev[-1], 0.01)
    rng = np.random.default_rng(K)
    c = rng.standard_normal(K + 1)
    V = rng.standard_normal((60, 4))
    B1 = c[K] * V                      # b_K = c_K V (b_{K+1} = b_{K+2} = 0)
    B2 = np.zeros_like(V)
    T = np.empty_like(V)
    for k in range(K - 1, 0, -1):
        core.clenshaw_step(H, a, b, float(c[k]), V, B1, B2, T)   # B2 <- c_k V + 2 H~ B1 - B2
        B1, B2 = B2, B1
    W = c[0] * V + core.rescaled_apply(H, a, b, B1) - B2
    want = core.clenshaw(H, a, b, c, V)
    assert np.array_equal(W.view(np.int64), want.view(np.int64))
    # and against the spectral definition, so that the chain is pinned to something else too
    evv, U = np.linalg.eigh(A)
    truth = U @ (npcheb.chebval((evv - a) / b, c)[:, None] * (U.T @ V))
    assert np.linalg.norm(W - truth) <= 1e-12 * max(1.0, np.linalg.norm(truth)) * (K + 1)


# ---- order rule (Eq. 40-42) ------------------------------------------------------

def test_order_rule_constant_and_cutoff():
    g = golden()
    assert abs(cheb.OMEGA - g["omega_cutoff"][0][0]) < 5e-6
    # Eq. (42) and the bisection of Eq. (41) agree to O(1/K) for |lam| <= 0.5
    for lam in (0.0, 0.3, -0.5):
        for nev, rho in ((50, 4000.0), (100, 30000.0)):
            k42 = cheb.order_eq42(nev, rho, lam)
            kb = cheb.order_bisect(nev, rho, lam)
            assert abs(kb - k42) <= 0.03 * k42 + 2
            delta = cheb.window_half_width(nev, rho)
            assert abs(k42 * delta / math.sqrt(1 - lam * lam) - g["eq42_constant"][0][0]) < 2 * delta


def test_window_contains_about_nev_levels_on_config2_size():
    # Fig. 1(b): with K from the rule, about N_ev transformed eigenvalues lie above Omega
    w = workloads.make_workload(2, L_override=12)
    st, H = core.hamiltonian(w)
    ev = np.linalg.eigvalsh(H.to_dense())
    a, b = cheb.rescale_params(ev[0], ev[-1], 0.01)
    evt = (ev - a) / b
    nev = 30
    # exact DOS at the target from the level spacing around it
    mid = np.searchsorted(evt, 0.0)
    rho = 60 / (evt[mid + 30] - evt[mid - 30])
    K = cheb.order_bisect(nev, rho, 0.0)
    above = int(np.sum(cheb.filter_value(cheb.filter_coeffs(0.0, K), evt) > cheb.OMEGA))
    assert abs(above - nev) <= 6


# ---- DOS ----------------------------------------------------------------------------

def test_gaussian_and_kpm_dos_integrate_to_dimension_and_track_histogram():
    assert abs(cheb.jackson_kernel(75)[0] - golden()["jackson_g0"][0][0]) < 1e-15
    w = workloads.make_workload(2, L_override=12)
    st, H = core.hamiltonian(w)
    D = H.n
    ev = np.linalg.eigvalsh(H.to_dense())
    a, b = cheb.rescale_params(ev[0], ev[-1], 0.01)
    mu, Gamma = cheb.spectral_mean_width(H)
    assert abs(mu - ev.mean()) < 1e-10 and abs(Gamma - ev.std()) < 1e-10
    E = np.linspace(-0.999, 0.999, 4001)
    dE = E[1] - E[0]
    gauss = cheb.gaussian_dos(E, D, (mu - a) / b, Gamma / b)
    assert abs(gauss.sum() * dE - D) < 0.02 * D
    rng = np.random.default_rng(0)
    mom = cheb.kpm_moments(H, a, b, 75, rng.standard_normal((D, 40)))
    assert abs(mom[0] - D) < 0.05 * D
    # moments are traces of T_n(H~): compare with the exact spectrum (Eq. 37)
    exact = np.array([np.cos(n * np.arccos((ev - a) / b)).sum() for n in range(75)])
    assert np.max(np.abs(mom - exact)) < 0.08 * D
    kpm = cheb.kpm_dos(E, exact, cheb.jackson_kernel(75))
    assert abs(kpm.sum() * dE - D) < 0.02 * D
    hist, edges = np.histogram((ev - a) / b, bins=20, range=(-1, 1))
    centers = 0.5 * (edges[1:] + edges[:-1])
    kc = cheb.kpm_dos(centers, exact, cheb.jackson_kernel(75)) * (edges[1] - edges[0])
    assert np.max(np.abs(kc - hist)) < 0.25 * hist.max()


@pytest.mark.parametrize("N", [8, 75, 200])
def test_jackson_kernel_is_the_autocorrelation_of_its_optimal_weights(N):
    # Eq. (39)/(84).  The Jackson kernel is the solution of a
    # variational problem (narrowest positive kernel): g_n = sum_{v=0}^{N-1-n} a_v a_{v+n} with
    # a_v proportional to sin(pi (v+1)/(N+1)), normalised to g_0 = 1.  That sum is an object
    # independent of the closed form the oracle types in.
    g = cheb.jackson_kernel(N)
    assert g.shape == (N,)
    a = np.sin(np.pi * (np.arange(N) + 1) / (N + 1))
    a /= np.sqrt(np.sum(a * a))
    want = np.array([np.dot(a[:N - n], a[n:]) for n in range(N)])
    assert np.max(np.abs(g - want)) < 1e-13
    assert abs(g[0] - 1.0) < 1e-15 and np.all(np.diff(g) < 0) and 0 < g[-1] < 2.0 / N
    # positivity of the kernel polynomial (a delta function smeared with g_n stays >= 0)
    x = np.cos(np.linspace(0.0, np.pi, 4001))
    n = np.arange(N)
    for y in (0.0, 0.37, -0.9):
        Ty = np.cos(n * np.arccos(y))
        series = g[0] + 2.0 * (np.cos(np.outer(np.arccos(x), n[1:])) @ (g[1:] * Ty[1:]))
        assert series.min() > -1e-10


def test_gaussian_dos_is_centred_at_mu_with_width_gamma():
    # Eq. (34): maximum D/(sqrt(2 pi) Gamma) at E = mu, symmetric about it,
    # full width at half maximum 2 sqrt(2 ln 2) Gamma.
    D, mu, Gamma = 924.0, 0.31, 0.27
    E = np.linspace(mu - 2.0, mu + 2.0, 400001)
    rho = cheb.gaussian_dos(E, D, mu, Gamma)
    assert abs(E[np.argmax(rho)] - mu) < 2e-5
    assert abs(rho.max() - D / (math.sqrt(2 * math.pi) * Gamma)) < 1e-9 * D
    assert np.allclose(cheb.gaussian_dos(mu + 0.4, D, mu, Gamma), cheb.gaussian_dos(mu - 0.4, D, mu, Gamma),
                       rtol=1e-14)
    above = E[rho >= 0.5 * rho.max()]
    assert abs((above[-1] - above[0]) - 2.0 * math.sqrt(2.0 * math.log(2.0)) * Gamma) < 5e-5
    assert abs(np.sum(rho) * (E[1] - E[0]) - D) < 1e-6 * D


# ---- Lanczos ----------------------------------------------------------------------

def test_lanczos_extrema_converge_to_spectrum_edges():
    st, H = core.hamiltonian(workloads.make_workload(1))
    ev = np.linalg.eigvalsh(H.to_dense())
    v0 = workloads.start_block(H.n, 1, 5)[:, 0]
    e_min, e_max = lanczos.lanczos_extrema(H, v0, 60)
    assert ev[0] - 1e-9 <= e_min <= ev[0] + 1e-3 * (ev[-1] - ev[0])
    assert ev[-1] + 1e-9 >= e_max >= ev[-1] - 1e-3 * (ev[-1] - ev[0])
    e_min, e_max, a, b = lanczos.spectrum_bounds(H, v0, 60, 0.01)
    assert (ev[0] - a) / b > -1.0 and (ev[-1] - a) / b < 1.0


def test_lanczos_residual_norm_identity_and_widened_bounds():
    """Eq. (6) / (16) for the scalar recurrence: ||H y - theta y|| = b_{m+1} |z_m| for a Ritz pair
    (y = Phi z); spectrum_bounds (reading R5) moves the extremal Ritz values outwards by it, so an
    unconverged run (m = 8) still has a true eigenvalue inside each widened end."""
    st, H = core.hamiltonian(workloads.make_workload(1))
    v0 = workloads.start_block(H.n, 1, 6)[:, 0]
    m = 8
    alpha, beta, Phi = lanczos.lanczos_tridiag(lambda X: core.spmm(H, X), v0, m)
    T = np.diag(alpha) + np.diag(beta[:m - 1], 1) + np.diag(beta[:m - 1], -1)
    th, Z = np.linalg.eigh(T)
    e_min, e_max, r_min, r_max = lanczos.lanczos_extrema_residuals(H, v0, m)
    for j, r in ((0, r_min), (m - 1, r_max)):
        y = Phi @ Z[:, j]
        direct = np.linalg.norm(core.spmm(H, y.reshape(-1, 1)).reshape(-1) - th[j] * y)
        assert abs(direct - r) <= 1e-10 * max(1.0, abs(th[j]))
    assert r_min > 1e-3 and r_max > 1e-3                      # not converged after 8 steps
    ev = np.linalg.eigvalsh(H.to_dense())
    assert np.min(np.abs(ev - e_min)) <= r_min + 1e-12        # an eigenvalue within the residual
    assert np.min(np.abs(ev - e_max)) <= r_max + 1e-12
    g_min, g_max, a, b = lanczos.spectrum_bounds(H, v0, m, 0.0)
    assert (g_min, g_max) == (e_min, e_max)
    assert abs((a - b) - (e_min - r_min)) <= 1e-12 and abs((a + b) - (e_max + r_max)) <= 1e-12


def test_block_lanczos_invariants():
    A, H = random_symmetric_csr(96, 0.2, 21)
    s, m = 4, 8
    V1 = workloads.start_block(96, s, 3, orthonormal=True)
    st = lanczos.BlockLanczosState(s=s, Q=[V1])
    for _ in range(m):
        lanczos.block_lanczos_step(st, lambda X: core.spmm(H, X))
    Q = st.basis()
    M = m * s
    assert np.linalg.norm(Q.T @ Q - np.eye(M)) < 1e-12
    HL = st.lanczos_matrix()
    assert np.linalg.norm(Q.T @ A @ Q - HL) < 1e-11 * np.linalg.norm(A)   # block tridiagonal projection
    # Eq. (15)/(16): A Q = Q H_L + V_{m+1} B_{m+1} E_m^T
    R = A @ Q - Q @ HL
    R[:, -s:] -= st.Q[m] @ st.B[m - 1]
    assert np.linalg.norm(R) < 1e-11 * np.linalg.norm(A)
    theta, T, est = lanczos.ritz_pairs(st)
    true_res = np.linalg.norm(A @ (Q @ T) - (Q @ T) * theta, axis=0)
    assert np.allclose(est, true_res, atol=1e-10 * np.linalg.norm(A))       # Eq. (16)-(17)
    # B_k upper triangular
    assert all(np.allclose(B, np.triu(B)) for B in st.B)


def test_block_lanczos_full_dimension_reproduces_filtered_spectrum():
    A, H = random_symmetric_csr(48, 0.3, 8)
    ev = np.linalg.eigvalsh(A)
    a, b = cheb.rescale_params(ev[0], ev[-1], 0.01)
    c = cheb.filter_coeffs(0.05, 12)
    s = 4
    st = lanczos.BlockLanczosState(s=s, Q=[workloads.start_block(48, s, 2, orthonormal=True)])
    for _ in range(48 // s):
        lanczos.block_lanczos_step(st, lambda X: core.clenshaw(H, a, b, c, X))
    theta = np.linalg.eigvalsh(st.lanczos_matrix())
    assert np.allclose(np.sort(theta), np.sort(cheb.filter_value(c, (ev - a) / b)), atol=1e-10)


def test_polfed_eigs_matches_dense_eigh_on_config1():
    w = workloads.make_workload(1)
    st, H = core.hamiltonian(w)
    ev, U = np.linalg.eigh(H.to_dense())
    norm_H = max(abs(ev[0]), abs(ev[-1]))
    v0 = workloads.start_block(H.n, 1, 77)[:, 0]
    _, _, a, b = lanczos.spectrum_bounds(H, v0, 60, 0.01)
    lam = (w.target - a) / b
    V1 = workloads.start_block(H.n, 4, 2001, orthonormal=True)
    res = lanczos.polfed_eigs(H, a, b, lam, w.K_fixed, w.nev, V1, tol=1e-8 * norm_H)
    assert res.converged
    assert np.all(res.residuals <= 1e-8 * norm_H)
    nearest = np.sort(ev[np.argsort(np.abs(ev - w.target))[:w.nev]])
    # same set except possibly the window edge members (reading R11)
    common = sum(np.min(np.abs(ev_i - nearest)) < 1e-9 * norm_H for ev_i in res.evals)
    assert common >= w.nev - 2
    for e in res.evals:
        assert np.min(np.abs(ev - e)) <= 1e-9 * norm_H
    # contiguous in the spectrum: no level skipped between the smallest and largest returned
    inside = ev[(ev >= res.evals[0] - 1e-9) & (ev <= res.evals[-1] + 1e-9)]
    assert inside.shape[0] == w.nev
