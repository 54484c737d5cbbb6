"""polfed_block_gram_static: the Gram product C_j = Q_j^T B (Eq. 9, 11 PAPER.md:147-153) for callers
that cannot allocate device memory -- an eigen-solver that has filled HBM with its Krylov basis, a
process under a fixed device-memory budget, a loop that must stay clear of the CUDA allocator's
synchronisation.  Its partial sums sit in one 4 MiB array inside the library instead of a pool block.

Checked here: on two calls in a row (the second smaller than the first and with another block size,
so that the array still holds the first call's partial sums when the second runs) the result agrees
with polfed_block_gram on the same inputs within the bound tests/test_gpu_reorth.py uses against
numpy, and bit for bit where both paths run the same kernel on the same grid; a panel list beyond the stated limit is
refused before anything is launched.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must
not hide the parity tests.  The test holds no state from other tests and leaves none: it passes
alone in a fresh process (where its first call also does the one-time address lookup) and after the
rest of the suite."""
from __future__ import annotations

import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import paper_2605_10191_b200 as pkg
    pkg.lib()
    return pkg


def _bound(n: int) -> float:
    # the bound of test_block_gram_and_update_match_numpy for standard-normal entries
    return 1e-13 * np.sqrt(n) * 4.0 * max(1.0, np.sqrt(n))


# (k panels, n rows, s): first a grid that does not fit the array at s = 32 (the static path takes a
# smaller one: different summation order), then shapes whose grid fits (bit-identical results)
CALLS = [(3, 200_003, 32), (5, 4099, 16)]


@pytest.mark.parametrize("variant", (0, 1))
def test_static_gram_matches_the_pool_path_on_two_calls_in_a_row(P, variant):
    gen = torch.Generator(device="cuda").manual_seed(11 + variant)
    inputs, want = [], []
    for k, n, s in CALLS:
        Q = torch.randn(k, n, s, dtype=torch.float64, device="cuda", generator=gen)
        B = torch.randn(n, s, dtype=torch.float64, device="cuda", generator=gen)
        inputs.append((Q, B))
        want.append(P.polfed_block_gram(Q, B, variant=variant))
    outs = [torch.full((k, s, s), float("nan"), dtype=torch.float64, device="cuda") for k, _, s in CALLS]
    torch.cuda.synchronize()
    # the two calls under test, back to back on one stream, nothing in between
    for (Q, B), out in zip(inputs, outs):
        P.polfed_block_gram_static(Q, B, out, variant=variant)
    torch.cuda.synchronize()
    for (k, n, s), out, ref in zip(CALLS, outs, want):
        err = (out - ref).abs().max().item()
        assert np.isfinite(err) and err <= _bound(n), (k, n, s, err)
    # the shared-memory FMA kernel takes the same grid on both paths at s = 16 (8 CTAs per SM fit the
    # array): bit-identical sums.  (variant 0 is the tensor-core kernel, which on the pool path walks
    # several panels per CTA and so adds in another order.)
    if variant == 1:
        assert torch.equal(outs[1], want[1])
    # and against numpy, so that the check does not rest on the pool path alone
    Q, B = inputs[1]
    exact = np.einsum("jra,rb->jab", Q.cpu().numpy(), B.cpu().numpy())
    assert np.max(np.abs(outs[1].cpu().numpy() - exact)) <= _bound(CALLS[1][1])


def test_static_gram_is_bit_reproducible(P):
    gen = torch.Generator(device="cuda").manual_seed(5)
    Q = torch.randn(4, 100_001, 32, dtype=torch.float64, device="cuda", generator=gen)
    B = torch.randn(100_001, 32, dtype=torch.float64, device="cuda", generator=gen)
    first = P.polfed_block_gram_static(Q, B, torch.empty(4, 32, 32, dtype=torch.float64, device="cuda"))
    again = P.polfed_block_gram_static(Q, B, torch.empty(4, 32, 32, dtype=torch.float64, device="cuda"))
    assert torch.equal(first, again)


def test_static_gram_refuses_more_panels_than_its_array_holds(P):
    s = 32
    k = P.STATIC_GRAM_DOUBLES // (s * s) + 1          # one panel too many
    Q = torch.zeros(k, 4, s, dtype=torch.float64, device="cuda")
    B = torch.zeros(4, s, dtype=torch.float64, device="cuda")
    out = torch.full((k, s, s), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(P.PolfedError) as e:
        P.polfed_block_gram_static(Q, B, out)
    assert e.value.code == 4 and "POLFED_STATIC_GRAM_DOUBLES" in str(e.value)   # POLFED_ERANGE
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                   # nothing was launched
    # the largest panel list that fits is accepted
    P.polfed_block_gram_static(Q[:k - 1], B, out[:k - 1])
    torch.cuda.synchronize()
    assert bool((out[:k - 1] == 0.0).all())
