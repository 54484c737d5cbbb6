"""Spectral bounds and the eigen-solver (block Lanczos on P(H~)) on the GPU against the oracle
and against dense diagonalisation.  Acceptance (BASELINE.json north_star): eigenvalues
|dlambda| <= 1e-9 ||H||, every returned pair ||Hx - lambda x|| <= 1e-8 ||H||."""
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


def build(P, w):
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    return P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense)


@pytest.mark.parametrize("config,L_override", [(1, None), (2, None), (4, 9), (5, 14)])
def test_spectrum_bounds_match_oracle_and_lie_inside_the_spectrum(P, config, L_override):
    w = workloads.make_workload(config, L_override=L_override)
    _, H = core.hamiltonian(w)
    v0 = workloads.start_block(H.n, 1, seed=3000 + config)[:, 0]
    e0, e1, a, b = lanczos.spectrum_bounds(H, v0, m=60, margin=0.01)
    g0, g1, ga, gb = P.polfed_spectrum_bounds(build(P, w), dev(v0), 60, 0.01)
    scale = max(abs(e0), abs(e1))
    assert abs(g0 - e0) <= 1e-8 * scale and abs(g1 - e1) <= 1e-8 * scale
    assert abs(ga - a) <= 1e-8 * scale and abs(gb - b) <= 1e-8 * scale
    if H.n <= 4096:
        ev = np.linalg.eigvalsh(H.to_dense())
        assert ev[0] - 1e-9 * scale <= g0 <= g1 <= ev[-1] + 1e-9 * scale     # Ritz values are interior
        assert g0 - ev[0] <= 1e-3 * scale and ev[-1] - g1 <= 1e-3 * scale


def check_pairs(H, evals, evecs, resid, tol_abs):
    X = evecs.cpu().numpy()
    R = core.spmm(H, X) - X * evals
    true_res = np.linalg.norm(R, axis=0)
    assert np.all(true_res <= tol_abs), true_res.max()            # judged by the ORACLE's SpMM
    assert np.all(np.abs(true_res - resid) <= 1e-3 * tol_abs + 1e-2 * true_res)
    assert np.linalg.norm(X.T @ X - np.eye(X.shape[1])) <= 1e-10
    assert np.all(np.diff(evals) >= 0)


def test_eigs_config1_matches_dense_and_oracle(P):
    w = workloads.make_workload(1)
    _, H = core.hamiltonian(w)
    ev = np.linalg.eigvalsh(H.to_dense())
    hnorm = max(abs(ev[0]), abs(ev[-1]))
    V0 = workloads.start_block(H.n, w.s, seed=2001, orthonormal=True)
    v0 = V0[:, 0].copy()
    _, _, a, b = lanczos.spectrum_bounds(H, v0, m=60, margin=0.01)
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(build(P, w), w.target, w.nev, w.s, dev(V0),
                                                           K_override=w.K_fixed, max_krylov_dim=400)
    assert rep["K"] == 200 and abs(rep["a"] - a) <= 1e-8 * hnorm and abs(rep["b"] - b) <= 1e-8 * hnorm
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    nearest = np.sort(ev[np.argsort(np.abs(ev - w.target))[: w.nev]])
    assert np.max(np.abs(evals - nearest)) <= 1e-9 * hnorm
    # the oracle's own POLFED run returns the same eigenvalues
    lam = (w.target - a) / b
    ref = lanczos.polfed_eigs(H, a, b, lam, 200, w.nev, V0, tol=1e-8 * hnorm)
    # (R11: the oracle stops as soon as nev candidates have converged, so its set may differ from
    # the true nearest set in at most the two edge members; the dense truth above is the judge)
    assert ref.converged
    common = [x for x in ref.evals if np.min(np.abs(evals - x)) <= 1e-9 * hnorm]
    assert len(common) >= w.nev - 2


def test_eigs_config2_full_pipeline_matches_dense(P):
    w = workloads.make_workload(2)
    _, H = core.hamiltonian(w)
    ev = np.linalg.eigvalsh(H.to_dense())
    hnorm = max(abs(ev[0]), abs(ev[-1]))
    V0 = workloads.start_block(H.n, w.s, seed=2002, orthonormal=True)
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(build(P, w), 0.0, w.nev, w.s, dev(V0),
                                                           sigma_is_rescaled=True)
    sigma = rep["a"] + rep["b"] * rep["lambda_rescaled"]
    assert 500 <= rep["K"] <= 5000              # about 1.6-1.75k by the DOS rule
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    nearest = np.sort(ev[np.argsort(np.abs(ev - sigma))[: w.nev]])
    # R11: the same contiguous set except possibly the two edge members
    assert np.max(np.abs(evals[1:-1] - nearest[1:-1])) <= 1e-9 * hnorm
    for lam_ in evals:
        assert np.min(np.abs(ev - lam_)) <= 1e-9 * hnorm
    assert rep["sparse_products"] >= rep["K"] * rep["block_steps"]
    assert rep["seconds_filter"] > 0 and rep["seconds_total"] >= rep["seconds_filter"]
    # R22: at lambda~ = 0 the odd coefficients are exact zeros at every order, so the launches of the
    # odd steps k = 1, 3, .. <= K-1 skip the V read
    assert rep["products_without_v"] == (rep["K"] // 2) * rep["block_steps"]


@pytest.mark.parametrize("config,L_override,nev", [(4, 9, 24), (5, 14, 40), (3, 14, 30)])
def test_eigs_shrunk_workloads_residuals_and_completeness(P, config, L_override, nev):
    w = workloads.make_workload(config, L_override=L_override)
    _, H = core.hamiltonian(w)
    ev = np.linalg.eigvalsh(H.to_dense())
    hnorm = max(abs(ev[0]), abs(ev[-1]))
    V0 = workloads.start_block(H.n, w.s, seed=2000 + config, orthonormal=True)
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(
        build(P, w), w.target, nev, w.s, dev(V0), sigma_is_rescaled=(w.target_kind == "rescaled"),
        max_krylov_dim=40 * w.s)     # nev/s is far below the paper's rule of thumb (Eq. 53) here
    sigma = rep["a"] + rep["b"] * rep["lambda_rescaled"]
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    nearest = np.sort(ev[np.argsort(np.abs(ev - sigma))[:nev]])
    assert np.max(np.abs(evals[1:-1] - nearest[1:-1])) <= 1e-9 * hnorm


def test_eigs_wider_window_gives_lower_order_and_the_same_pairs(P):
    """options.window_levels: the window of Eq. (40)-(41) sized for 2 nev levels instead of
    nev + 10 % -- about half the order, the same nev pairs nearest the target (dense truth)."""
    w = workloads.make_workload(2)
    _, H = core.hamiltonian(w)
    ev = np.linalg.eigvalsh(H.to_dense())
    hnorm = max(abs(ev[0]), abs(ev[-1]))
    V0 = dev(workloads.start_block(H.n, w.s, seed=2002, orthonormal=True))
    ham = build(P, w)
    _, _, _, rep0 = P.polfed_block_lanczos_eigs(ham, 0.0, w.nev, w.s, V0, sigma_is_rescaled=True)
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(ham, 0.0, w.nev, w.s, V0, sigma_is_rescaled=True,
                                                           window_levels=2 * w.nev)
    assert rep0["nev_window"] == w.nev + 5 and rep["nev_window"] == 2 * w.nev
    assert 0.45 * rep0["K"] <= rep["K"] <= 0.65 * rep0["K"]
    sigma = rep["a"] + rep["b"] * rep["lambda_rescaled"]
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    nearest = np.sort(ev[np.argsort(np.abs(ev - sigma))[: w.nev]])
    assert np.max(np.abs(evals[1:-1] - nearest[1:-1])) <= 1e-9 * hnorm
    with pytest.raises(P.PolfedError) as err:
        P.polfed_block_lanczos_eigs(ham, 0.0, w.nev, w.s, V0, sigma_is_rescaled=True, window_levels=w.nev - 1)
    assert err.value.code == P.binding.EINVAL


def test_eigs_window_too_narrow_is_reported_early_with_valid_pairs(P):
    """with an order K far above what Eq. (40)-(42) give for nev (as after an overestimated
    density of states) the main lobe holds fewer than nev levels.  Once every extracted pair is a
    converged eigenpair nothing can change that: the solver must say so (POLFED_EWINDOW) instead of
    running to max_krylov_dim, and what it returns must be true eigenpairs (dense truth)."""
    w = workloads.make_workload(1)
    _, H = core.hamiltonian(w)
    ev = np.linalg.eigvalsh(H.to_dense())
    hnorm = max(abs(ev[0]), abs(ev[-1]))
    V0 = dev(workloads.start_block(H.n, 1, seed=2001, orthonormal=True))
    ham = build(P, w)
    _, _, _, rep0 = P.polfed_block_lanczos_eigs(ham, w.target, w.nev, 1, V0, max_krylov_dim=900)
    K_high = 5 * rep0["K"]
    with pytest.raises(P.PolfedError) as err:
        P.polfed_block_lanczos_eigs(ham, w.target, w.nev, 1, V0, K_override=K_high, max_krylov_dim=900)
    assert err.value.code == P.binding.EWINDOW
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(ham, w.target, w.nev, 1, V0, K_override=K_high,
                                                           max_krylov_dim=900, allow_unconverged=True)
    assert rep["status"] == P.binding.EWINDOW and rep["n_converged"] < w.nev
    assert rep["krylov_dim"] < 900                       # stopped early, not at the cap
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    for lam_ in evals:
        assert np.min(np.abs(ev - lam_)) <= 1e-9 * hnorm


def test_eigs_refuses_an_interval_the_spectrum_sticks_out_of(P):
    """a, b that do not enclose the spectrum (here: 60 % of its half-width) must come
    back as POLFED_ERANGE -- a Rayleigh-Ritz value of H outside [a - b, a + b] proves it -- and not as
    slow or wrong convergence."""
    w = workloads.make_workload(1)
    ham = build(P, w)
    V0 = dev(workloads.start_block(ham.n, 1, seed=2001, orthonormal=True))
    _, _, _, rep0 = P.polfed_block_lanczos_eigs(ham, w.target, w.nev, 1, V0, max_krylov_dim=900)
    with pytest.raises(P.PolfedError) as err:
        P.polfed_block_lanczos_eigs(ham, w.target, w.nev, 1, V0, a=rep0["a"], b=0.6 * rep0["b"],
                                    K_override=40, max_krylov_dim=900)
    assert err.value.code == P.binding.ERANGE


def test_eigs_reports_no_convergence_and_bad_arguments(P):
    w = workloads.make_workload(1)
    ham = build(P, w)
    V0 = dev(workloads.start_block(ham.n, 1, seed=1, orthonormal=True))
    with pytest.raises(P.PolfedError) as err:
        P.polfed_block_lanczos_eigs(ham, 0.0, 20, 1, V0, K_override=10, max_krylov_dim=24)
    assert err.value.code == P.binding.ENOCONV
    out = P.polfed_block_lanczos_eigs(ham, 0.0, 20, 1, V0, K_override=10, max_krylov_dim=24,
                                      allow_unconverged=True)
    assert out[3]["status"] == P.binding.ENOCONV and np.all(np.isfinite(out[0]))
    with pytest.raises(P.PolfedError):
        P.polfed_block_lanczos_eigs(ham, 1e9, 20, 1, V0)                 # target outside the spectrum
    with pytest.raises(P.PolfedError):
        P.polfed_block_lanczos_eigs(ham, 0.0, 0, 1, V0)
    Z = torch.zeros(ham.n, 4, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PolfedError) as err:
        P.polfed_block_lanczos_eigs(ham, 0.0, 4, 4, Z, a=0.0, b=20.0, K_override=20)
    assert err.value.code == P.binding.EBREAKDOWN


@pytest.mark.parametrize("config,L_override,s", [(2, None, 8), (1, None, 1), (5, 14, 32), (4, 9, 16)])
def test_kpm_moments_match_oracle(P, config, L_override, s):
    """Eq. (37)-(38): Chebyshev moments from the same random block on both sides; the recurrence
    is the fused step with c = 0, so agreement is to rounding (|T_n| <= 1 on [-1, 1])."""
    w = workloads.make_workload(config, L_override=L_override)
    _, H = core.hamiltonian(w)
    v0 = workloads.start_block(H.n, 1, seed=3000 + config)[:, 0]
    _, _, a, b = lanczos.spectrum_bounds(H, v0, m=60, margin=0.01)
    R = np.random.default_rng(6000 + config).standard_normal((H.n, s))
    N = 75                                                   # PAPER.md:341 (Fig. 3)
    want = cheb.kpm_moments(H, a, b, N, R)
    ham = build(P, w)
    got = P.polfed_kpm_moments(ham, a, b, N, dev(R))
    assert np.max(np.abs(got - want)) <= 1e-10 * H.n
    assert abs(got[0] - np.sum(R * R) / s) <= 1e-10 * H.n
    # the density integrates to mu_0 and, fed to the order rule, gives the oracle's K
    lam = 0.1
    rho_got = float(P.polfed_kpm_dos(got, [lam])[0])
    rho_want = float(cheb.kpm_dos(lam, want, cheb.jackson_kernel(N))[0])
    assert abs(rho_got - rho_want) <= 1e-9 * abs(rho_want)
    if rho_want > 0:
        assert abs(len(P.polfed_filter_coeffs(a, b, a + b * lam, 10, rho_got)) - 1
                   - cheb.order_bisect(10, rho_want, lam)) <= 1


def test_kpm_moments_argument_errors(P):
    w = workloads.make_workload(1)
    ham = build(P, w)
    R = torch.randn(ham.n, 4, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PolfedError):
        P.polfed_kpm_moments(ham, 0.0, -1.0, 10, R)          # b <= 0
    with pytest.raises(P.PolfedError):
        P.polfed_kpm_moments(ham, 0.0, 10.0, 0, R)           # no moments
    with pytest.raises(P.PolfedError):
        P.polfed_kpm_moments(ham, 0.0, 10.0, 10, torch.randn(ham.n, 3, dtype=torch.float64,
                                                             device="cuda"))     # s = 3
    assert P.polfed_kpm_moments(ham, 0.0, 10.0, 1, R).shape == (1,)


# ---- KPM density of states inside the solver ----

def test_eigs_kpm_sized_window_holds_nev_levels(P):
    """Config 2 with options.dos = KPM (R = 100 random vectors, N = 75 moments): the
    window |E~ - lambda~| <= delta of the K the solver picks holds nev +- 15 % exact levels (dense
    eigh), the report carries both orders, and the pairs are accepted as with the Gaussian."""
    w = workloads.make_workload(2)
    _, H = core.hamiltonian(w)
    ev = np.linalg.eigvalsh(H.to_dense())
    hnorm = max(abs(ev[0]), abs(ev[-1]))
    V0 = workloads.start_block(H.n, w.s, seed=2002, orthonormal=True)
    R = np.random.default_rng(6102).standard_normal((H.n, 100))
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(build(P, w), 0.0, w.nev, w.s, dev(V0),
                                                           sigma_is_rescaled=True, kpm_block=dev(R))
    assert rep["K"] == rep["K_kpm"] > 0 and rep["K_gaussian"] > 0 and rep["rho_kpm"] > 0
    # the oracle's KPM density from the same block gives the same order (+- 1 from rounding)
    a, b, lam = rep["a"], rep["b"], rep["lambda_rescaled"]
    mu = cheb.kpm_moments(H, a, b, 75, R)
    rho = float(cheb.kpm_dos(lam, mu, cheb.jackson_kernel(75))[0])
    assert abs(rho - rep["rho_kpm"]) <= 1e-8 * rho
    assert rep["nev_window"] == w.nev + 5                    # nev + max(2, 10 %)
    assert abs(cheb.order_bisect(rep["nev_window"], rho, lam) - rep["K"]) <= 1
    # Eq. (42) inverted: half-width delta of the window of this K; count exact levels inside
    delta = 2.655 * np.sqrt(1.0 - lam * lam) / rep["K"]
    inside = int(np.sum(np.abs((ev - a) / b - lam) <= delta))
    assert abs(inside - rep["nev_window"]) <= 0.15 * w.nev, (inside, rep["K"], rep["K_gaussian"])
    assert inside >= w.nev
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    with pytest.raises(P.PolfedError):      # R must be a multiple of 4
        P.polfed_block_lanczos_eigs(build(P, w), 0.0, w.nev, w.s, dev(V0), sigma_is_rescaled=True,
                                    kpm_block=dev(R[:, :10].copy()))


# ---- full BASELINE sizes: every returned pair judged by the ORACLE's SpMM --------

def check_window(evals, rep, coeffs_K):
    """lambda ascending and every returned level inside the filter window P(lambda~_i) > Omega."""
    lam_i = (evals - rep["a"]) / rep["b"]
    c = cheb.filter_coeffs(rep["lambda_rescaled"], coeffs_K)
    p = np.array([cheb.filter_value(c, x) for x in lam_i])
    assert np.all(np.diff(evals) >= 0)
    assert np.all(p > 0.17613), p.min()            # Omega (R4)


def test_eigs_full_size_config3_pairs_verified_by_oracle(P):
    """Config 3 (XXZ L=20, D=184 756, s=16, nev=100 at lambda~ = 0): the whole solve; the oracle's
    CSR builder and SpMM judge ||Hx - lambda x|| <= 1e-8 ||H|| and X^T X = I."""
    w = workloads.make_workload(3)
    _, H = core.hamiltonian(w)
    V0 = workloads.start_block(H.n, w.s, seed=2003, orthonormal=True)
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(build(P, w), 0.0, w.nev, w.s, dev(V0),
                                                           sigma_is_rescaled=True)
    hnorm = max(abs(rep["e_min"]), abs(rep["e_max"]))
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    check_window(evals, rep, rep["K"])
    assert rep["n_converged"] == w.nev
    # contiguous: no gap is far above the mean level spacing (a level on a secondary peak of the
    # filter would sit about 90 spacings away from the rest)
    gaps = np.diff(evals)
    assert gaps.max() <= 12 * gaps.mean()


@pytest.mark.parametrize("window", [
    "2nev",
    pytest.param("paper", marks=pytest.mark.skipif(
        not __import__("os").environ.get("POLFED_SLOW"),
        reason="about 10 minutes on a B200 (K = 85 018): set POLFED_SLOW=1; the 2 nev window runs by default")),
])
def test_eigs_full_size_config4_pairs_verified_by_oracle(P, window):
    """Config 4 (quantum sun, D = 2^20, s=16, nev=100 at sigma = 0, flip format): the whole solve,
    every returned pair judged by the oracle's CSR and SpMM.  Default: the filter window sized for
    2 nev levels (polfed_options.window_levels, K = 46 760, about 5 minutes); the paper's rule
    (window for nev + 10 %, K = 85 018) behind POLFED_SLOW."""
    w = workloads.make_workload(4)
    _, H = core.hamiltonian(w)
    V0 = workloads.start_block(H.n, w.s, seed=2004, orthonormal=True)
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    ham = P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense, fmt=P.FORMAT_FLIP)
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(
        ham, w.target, w.nev, w.s, dev(V0), window_levels=2 * w.nev if window == "2nev" else 0)
    hnorm = max(abs(rep["e_min"]), abs(rep["e_max"]))
    check_pairs(H, evals, evecs, resid, 1e-8 * hnorm)
    check_window(evals, rep, rep["K"])
    assert rep["n_converged"] == w.nev
    gaps = np.diff(evals)
    assert gaps.max() <= 12 * gaps.mean()          # contiguous: no level from a secondary peak


def test_block_steps_full_size_config5_checked_by_oracle_rows(P):
    """Config 5 (D = 10 400 600, s=32): the full solve needs about 1e7 sparse products, so a stated
    number of block steps is run instead: K = 512, Krylov dimension 4 s.  The
    unconverged Ritz vectors that come back must still be orthonormal, and their Rayleigh quotients
    and residuals must be those of H: H x is recomputed on 2000 sampled rows with the oracle's row
    builder and SpMM (one matrix row needs the whole vector, so X is brought to the host)."""
    w = workloads.make_workload(5)
    states = core.basis_states(w.n_sites, w.n_up)
    n, s, nev = int(states.shape[0]), w.s, 32
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    ham = P.polfed_build_hamiltonian(basis, w.terms, fmt=P.FORMAT_TILED)
    gen = torch.Generator(device="cuda").manual_seed(2005)
    V0 = torch.randn(n, s, dtype=torch.float64, device="cuda", generator=gen)
    evals, evecs, resid, rep = P.polfed_block_lanczos_eigs(
        ham, 0.0, nev, s, V0, sigma_is_rescaled=True, K_override=512, max_krylov_dim=4 * s,
        allow_unconverged=True)
    assert rep["block_steps"] == 4 and rep["K"] == 512 and rep["sparse_products"] >= 4 * 512
    G = (evecs.T @ evecs).cpu().numpy()
    assert np.linalg.norm(G - np.eye(nev)) <= 1e-10
    X = evecs.cpu().numpy()
    rows = np.unique(np.random.default_rng(4205).integers(0, n, 2000))
    Hs = core.build_csr_rows(states, rows, w.terms, w.dot_bits, w.dot_dense)
    HX = core.spmm(Hs, X)                                   # rows of H X, by the oracle
    R = HX - X[rows] * evals
    # Rayleigh quotients and residual norms reported by the library are consistent with these rows:
    # E_j = x_j^T H x_j is checked through the sampled estimator n/|rows| sum_r x_rj (Hx)_rj
    est = (n / rows.size) * np.sum(X[rows] * HX, axis=0)
    hnorm = max(abs(rep["e_min"]), abs(rep["e_max"]))
    assert np.max(np.abs(est - evals)) <= 0.2 * hnorm        # 2000 of 1e7 rows: a coarse estimator
    res_est = np.sqrt((n / rows.size) * np.sum(R * R, axis=0))
    assert np.all(res_est <= 3.0 * resid + 1e-6 * hnorm) and np.all(resid <= 3.0 * res_est + 1e-6 * hnorm)
