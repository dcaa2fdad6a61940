"""kg_kpm_reconstruct_noalloc against kg_kpm_reconstruct.

The no-alloc entry point exists for programs that cannot allocate GPU memory when they want a
spectrum from their moments: the card is already full (their own caching allocator or their
Chebyshev vectors own every byte, so a further cudaMalloc fails) or they sit in a loop whose
latency a device-wide allocation stall would break.  It keeps its only temporary, the damped
weights, in one fixed array per GPU inside libkg (KG_KPM_NOALLOC_MAX_M entries).

What is checked: the output equals the allocating path's within the suite's 1e-10, on two calls in
a row that share the array (the second with a shorter series and the other damping, so that
entries left by the first call sit behind the ones it uses; then a longer one again), with
several rows at once; and that sizes beyond the limit and host arrays are refused with a message.

This file is named to be collected last: `pytest -x` stops at the first failure and one in here
must not hide the parity suite.  It needs nothing from the other tests (moments are seeded random
numbers), so it passes alone in a fresh process as well as at the end of the full run.
"""
import numpy as np
import pytest
import torch

from helpers import relerr

TOL = 1e-10
E0, SCALE = 0.1, 8.5


@pytest.fixture(scope="module")
def B():
    from paper_1307_0288_b200 import binding
    return binding


def _moments(rows, M, seed):
    """Moment-like rows: decaying complex numbers with mu_0 = 1 (the reconstruction is linear in
    them; their origin does not matter here)."""
    rng = np.random.default_rng(seed)
    mu = (rng.normal(size=(rows, M)) + 1j * rng.normal(size=(rows, M))) / (1.0 + np.arange(M)) ** 0.5
    mu[:, 0] = 1.0
    return mu


@pytest.mark.gpu
def test_noalloc_matches_allocating_path_on_consecutive_calls(B):
    dev = torch.device("cuda:0")
    en = torch.linspace(E0 - 0.97 * SCALE, E0 + 0.97 * SCALE, 1001, dtype=torch.float64, device=dev)
    # (rows, M, jackson): long, then shorter with the other weights, then the longest allowed
    calls = [(3, 3000, True), (5, 257, False), (2, B.KG_KPM_NOALLOC_MAX_M, True)]
    cases = [(torch.from_numpy(_moments(r, M, 7 + i)).to(dev), M, j) for i, (r, M, j) in enumerate(calls)]
    outs = [torch.full((mu.shape[0], en.shape[0]), float("nan"), dtype=torch.float64, device=dev) for mu, _, _ in cases]
    # the new entry point first, back to back on one stream with nothing in between ...
    for (mu, M, jackson), f in zip(cases, outs):
        assert B.kpm_reconstruct_noalloc(mu, E0, SCALE, en, f, jackson) is f
    # ... then the existing path on the same inputs
    for (mu, M, jackson), f in zip(cases, outs):
        want = B.kpm_reconstruct(mu, E0, SCALE, en, jackson).cpu().numpy()
        got = f.cpu().numpy()
        assert np.all(np.isfinite(got))
        assert relerr(got, want) <= TOL, (M, jackson)
    # and once more after the allocating path has run: same answer as the first time
    mu, M, jackson = cases[0]
    again = torch.empty_like(outs[0])
    B.kpm_reconstruct_noalloc(mu, E0, SCALE, en, again, jackson)
    assert torch.equal(again, outs[0])


@pytest.mark.gpu
def test_noalloc_refuses_host_arrays_and_leading_shapes_work(B):
    dev = torch.device("cuda:0")
    en = torch.linspace(-8.0, 8.0, 64, dtype=torch.float64, device=dev)
    mu = torch.from_numpy(_moments(6, 64, 3).reshape(2, 3, 64)).to(dev)
    f = torch.empty((2, 3, 64), dtype=torch.float64, device=dev)
    B.kpm_reconstruct_noalloc(mu, E0, SCALE, en, f)
    assert relerr(f.cpu().numpy(), B.kpm_reconstruct(mu, E0, SCALE, en).cpu().numpy()) <= TOL
    for bad in ((mu.cpu(), en, f), (mu, en.cpu(), f), (mu, en, f.cpu())):
        with pytest.raises(B.KgError) as e:
            B.kpm_reconstruct_noalloc(bad[0], E0, SCALE, bad[1], bad[2])
        assert e.value.code == B.KG_EINVAL and "device memory" in str(e.value)


def test_noalloc_rejects_series_beyond_the_fixed_table():
    """Needs no GPU: the size check comes before anything touches the device."""
    from paper_1307_0288_b200 import binding as B
    assert B.KG_KPM_NOALLOC_MAX_M == 16384
    buf = np.zeros(4, np.complex128)
    rc = B._lib.kg_kpm_reconstruct_noalloc(buf.ctypes.data, 1, B.KG_KPM_NOALLOC_MAX_M + 1, 1, 0.0, 1.0,
                                           buf.ctypes.data, 1, buf.ctypes.data, None)
    assert rc == B.KG_EINVAL
    msg = B._lib.kg_last_error().decode()
    assert "KG_KPM_NOALLOC_MAX_M = 16384" in msg and "16385" in msg
    assert B._lib.kg_kpm_reconstruct_noalloc(None, 1, 8, 1, 0.0, 1.0, None, 1, None, None) == B.KG_EINVAL
