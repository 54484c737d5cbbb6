"""The tall-skinny products of the full reorthogonalisation (Eq. 9, 11 PAPER.md:147-153):
C_j = Q_j^T B and B -= sum_j Q_j C_j, against numpy in fp64 on the same seeded blocks, for both
Gram variants (shared-memory FMA kernel, fp64 tensor-core mma), and bit-reproducibility of the
reductions (H_L must not vary from run to run)."""
from __future__ import annotations

import numpy as np
import pytest

import workloads

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import paper_2605_10191_b200 as pkg
    pkg.lib()
    return pkg


@pytest.mark.parametrize("variant", (1, 2))
@pytest.mark.parametrize("s", (1, 2, 4, 8, 16, 32))
@pytest.mark.parametrize("n,k", [(1, 1), (3, 2), (37, 3), (4099, 5), (50001, 2)])
def test_block_gram_and_update_match_numpy(P, n, k, s, variant):
    rng = np.random.default_rng(1000 * n + 10 * s + k)
    Q = rng.standard_normal((k, n, s))
    B = rng.standard_normal((n, s))
    want = np.einsum("jra,rb->jab", Q, B)
    dQ, dB = torch.from_numpy(Q).cuda(), torch.from_numpy(B).cuda()
    got = P.polfed_block_gram(dQ, dB, variant=variant).cpu().numpy()
    scale = np.sqrt(n) * 4.0
    assert np.max(np.abs(got - want)) <= 1e-13 * scale * max(1.0, np.sqrt(n))
    P.polfed_block_update(dQ, torch.from_numpy(want).cuda(), dB, -1.0, 1.0)
    want_B = B - np.einsum("jra,jab->rb", Q, want)
    assert np.max(np.abs(dB.cpu().numpy() - want_B)) <= 1e-12 * np.abs(want_B).max()


def test_block_products_reject_misaligned_and_overlapping_blocks(P):
    """the header promises 16-byte aligned pointers; the tensor-core update moves B in
    16-byte pieces, so an 8-byte aligned B must come back as POLFED_EINVAL, not as a device fault."""
    import ctypes as C
    n, s, k = 64, 16, 2
    buf = torch.zeros(k * n * s + n * s + k * s * s + 8, dtype=torch.float64, device="cuda")
    q, b, c = buf.data_ptr(), buf.data_ptr() + 8 * k * n * s, buf.data_ptr() + 8 * (k + 1) * n * s
    L, vp = P.lib(), C.c_void_p
    ok = lambda rc: rc == 0
    assert ok(L.polfed_block_gram(s, n, vp(q), k, n * s, vp(b), vp(c), 0, None))
    assert ok(L.polfed_block_update(s, n, vp(q), k, n * s, vp(c), -1.0, 1.0, vp(b), None))
    for args in ((q + 8, b, c), (q, b + 8, c), (q, b, c + 8)):
        assert L.polfed_block_gram(s, n, vp(args[0]), k, n * s, vp(args[1]), vp(args[2]), 0, None) == 1
        assert L.polfed_block_gram_static(s, n, vp(args[0]), k, n * s, vp(args[1]), vp(args[2]), 0, None) == 1
        assert L.polfed_block_update(s, n, vp(args[0]), k, n * s, vp(args[2]), -1.0, 1.0, vp(args[1]), None) == 1
    # overlapping panels
    assert L.polfed_block_gram(s, n, vp(q), k, n * s - 2, vp(b), vp(c), 0, None) == 1
    assert L.polfed_block_update(s, n, vp(q), k, n * s - 2, vp(c), -1.0, 1.0, vp(b), None) == 1
    torch.cuda.synchronize()                      # and the context is still healthy
    assert float(buf.sum()) == 0.0


@pytest.mark.parametrize("variant", (0, 1, 2))
def test_block_gram_is_bit_reproducible(P, variant):
    gen = torch.Generator(device="cuda").manual_seed(7)
    Q = torch.randn(6, 300_007, 16, dtype=torch.float64, device="cuda", generator=gen)
    B = torch.randn(300_007, 16, dtype=torch.float64, device="cuda", generator=gen)
    first = P.polfed_block_gram(Q, B, variant=variant)
    for _ in range(5):
        assert torch.equal(P.polfed_block_gram(Q, B, variant=variant), first)


def test_eigen_solver_is_bit_reproducible(P):
    """Same inputs, same eigenvalues, residuals and iteration counts, bit for bit."""
    w = workloads.make_workload(2)
    basis = P.polfed_build_basis(w.n_sites, w.n_up)
    ham = P.polfed_build_hamiltonian(basis, w.terms)
    V0 = torch.from_numpy(workloads.start_block(ham.n, w.s, seed=2002, orthonormal=True)).cuda()
    runs = [P.polfed_block_lanczos_eigs(ham, 0.0, w.nev, w.s, V0, sigma_is_rescaled=True)
            for _ in range(3)]
    for ev, X, res, rep in runs[1:]:
        assert np.array_equal(ev, runs[0][0]) and np.array_equal(res, runs[0][2])
        assert torch.equal(X, runs[0][1])
        assert rep["block_steps"] == runs[0][3]["block_steps"] and rep["K"] == runs[0][3]["K"]
