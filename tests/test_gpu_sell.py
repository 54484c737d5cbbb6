"""Parity of the SELL-8-sigma format (POLFED_FORMAT_SELL, include/polfed.h) against the CPU oracle's
CSR SpMM and textbook Clenshaw (Eq. 31, 51 PAPER.md:274-276, 427-431).  The SELL kernel sums a row in
the same order as the oracle, so one step agrees to rounding of the FMAs."""
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
    return P.polfed_build_hamiltonian(basis, w.terms, w.dot_bits, w.dot_dense, fmt=P.FORMAT_SELL)


# ragged XXZ rows (lengths 1..L/2+1), fermions, quantum sun; sizes around and across the window of
# 1024 rows and the slice of 8 (D = 6, 70, 924, 3432, 12870; 2^11)
CASES = [(1, 4), (1, 8), (1, None), (5, 14), (2, None), (4, 8), (3, 14)]


@pytest.mark.parametrize("s", (8, 16, 32))
@pytest.mark.parametrize("config,L_override", CASES)
def test_sell_fused_step_matches_oracle(P, config, L_override, s):
    w = workloads.make_workload(config, L_override=L_override)
    _, H = core.hamiltonian(w)
    ham = build(P, w)
    rng = np.random.default_rng(100 * config + s)
    X, Z, V = (rng.standard_normal((H.n, s)) for _ in range(3))
    p, q, r, c = 0.21, -0.6, -1.0, 0.37
    want = p * core.spmm(H, X) + q * X + r * Z + c * V
    scale = np.abs(p) * core.spmm(core.CSR(H.n, H.row_ptr, H.col, np.abs(H.val)), np.abs(X)) \
        + np.abs(q * X) + np.abs(r * Z) + np.abs(c * V)
    Y = torch.full((H.n, s), float("nan"), dtype=torch.float64, device="cuda")
    P.polfed_fused_step(ham, s, p, q, r, c, dev(X), dev(Z), dev(V), Y)
    assert np.all(np.abs(Y.cpu().numpy() - want) <= 1e-13 * scale)
    Zd = dev(Z)                                               # in place over Z
    P.polfed_fused_step(ham, s, p, q, r, c, dev(X), Zd, dev(V), Zd)
    assert np.all(np.abs(Zd.cpu().numpy() - want) <= 1e-13 * scale)
    P.polfed_fused_step(ham, s, 1.0, 0.0, 0.0, 0.0, dev(X), None, None, Y)
    assert np.all(np.abs(Y.cpu().numpy() - core.spmm(H, X)) <= 1e-13 * scale / abs(p))


def test_sell_handles_misaligned_blocks_and_other_block_sizes(P):
    """Blocks that are only 16-byte aligned (s >= 16) and block sizes below 8 run the CSR kernel of
    the same handle; the CSR itself is unchanged."""
    w = workloads.make_workload(2)
    _, H = core.hamiltonian(w)
    ham = build(P, w)
    row_ptr, col, val = (t.cpu().numpy() for t in P.polfed_ham_csr(ham))
    assert np.array_equal(col, H.col) and np.array_equal(val, H.val)
    rng = np.random.default_rng(8)
    for s in (16, 4):
        X = rng.standard_normal((H.n, s))
        buf = torch.empty(H.n * s + 2, dtype=torch.float64, device="cuda")
        Xd = buf[2:].view(H.n, s)                              # 16-byte, not 32-byte aligned
        Xd.copy_(dev(X))
        assert Xd.data_ptr() % 32 == 16
        Y = torch.empty(H.n, s, dtype=torch.float64, device="cuda")
        P.polfed_fused_step(ham, s, 1.0, 0.0, 0.0, 0.0, Xd, None, None, Y)
        want = core.spmm(H, X)
        assert np.max(np.abs(Y.cpu().numpy() - want)) <= 1e-12 * np.abs(want).max()


@pytest.mark.parametrize("config,L_override,K", [(2, None, 1654), (3, 16, 800), (5, 16, 300)])
def test_sell_filter_matches_oracle(P, config, L_override, K):
    w = workloads.make_workload(config, L_override=L_override)
    _, H = core.hamiltonian(w)
    v0 = workloads.start_block(H.n, 1, seed=3000 + config)[:, 0]
    _, _, a, b = lanczos.spectrum_bounds(H, v0, m=60, margin=0.01)
    coeffs = cheb.filter_coeffs(w.target, K)
    V = workloads.start_block(H.n, w.s, seed=2000 + config, orthonormal=True)
    want = core.clenshaw(H, a, b, coeffs, V)
    ham = build(P, w)
    W = torch.empty(H.n, w.s, dtype=torch.float64, device="cuda")
    work = torch.empty(P.polfed_filter_workspace_bytes_ham(ham, w.s) // 8, dtype=torch.float64,
                       device="cuda")
    P.polfed_filter_apply(ham, a, b, coeffs, w.s, dev(V), W, work)
    err = float(np.linalg.norm(W.cpu().numpy() - want) / np.linalg.norm(want))
    assert err <= 1e-9
