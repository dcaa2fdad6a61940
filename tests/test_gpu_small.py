"""The single-launch moment loop for launch-bound sizes (kg_small.cuh, KG_OPT_ONE_LAUNCH): one thread-
block cluster keeps the vectors and matrix rows of all tiles in distributed shared memory and runs every
Chebyshev step after the first on the device.  Bitwise equal to the one-launch-per-step path (plain
launches, programmatic dependent launches, or CUDA-graph replay), and within 1e-10 of the oracle."""
import numpy as np
import pytest

from helpers import relerr, ring, to_oracle_lattice
from paper_1307_0288_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1307_0288_b200 import binding
    return binding


def dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.cpu().numpy()


def case(kind):
    if kind == "config1":
        cfg = W.make_config(1)
        return cfg.lattice, cfg.scale
    if kind == "ragged+onsite":                               # 13 x 11 cells minus vacancies = 535 sites
        full = W.honeycomb(13, 11)
        lat = W.remove_sites(full, W.vacancy_mask(full.n, 37, 5))
        lat.onsite = W.anderson(lat.n, 2.7, 6)
        return lat, (3 * 2.7 + 1.35) * 1.05
    if kind == "open-ribbon":
        lat = W.honeycomb(9, 40, periodic_x=False, periodic_y=True)
        return lat, 3 * 2.7 * 1.05
    raise ValueError(kind)


@pytest.mark.parametrize("kind", ["config1", "ragged+onsite", "open-ribbon"])
@pytest.mark.parametrize("R", [1, 2, 4, 8])
def test_one_launch_equals_per_step_launches_bitwise(B, kgo, kind, R):
    import torch
    lat, s = case(kind)
    if lat.n * R > 16384:
        pytest.skip("batch does not fit one cluster")
    olat = to_oracle_lattice(kgo, lat)
    phi = W.random_phase_vectors(lat.n, R, 3)
    L = W.random_phase_vectors(lat.n, R, 4)
    M, nt, dt = 37, 3, 0.7
    res = {}
    stream = torch.cuda.Stream()
    for one in (1, 0):
        h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
        h.set_option(B.KG_OPT_ONE_LAUNCH, one)
        with torch.cuda.stream(stream):
            l0 = h.launch_count
            dos = B.dos_moments(h, dev(phi), M)
            n_dos = h.launch_count - l0
            out = [dos, B.moments(h, dev(L), dev(phi), M), B.msd(h, dev(phi), M, nt, dt)]
            if R <= 4:
                out.append(B.vac(h, dev(phi), M, nt, dt))        # 2R columns in the batch
        stream.synchronize()
        res[one] = [host(o) for o in out]
        if one:
            assert n_dos == 3                                   # first step + the cluster kernel + the reduction
        else:
            assert n_dos == M // 2 + 1
    for a, b in zip(res[1], res[0]):
        assert a.tobytes() == b.tobytes()
    for r in sorted({0, R - 1}):
        v = phi[:, r].copy()
        assert relerr(res[1][0][r], kgo.dos_moments(olat, 0.0, s, v, M)) <= TOL
        assert relerr(res[1][1][r], kgo.moments(olat, 0.0, s, L[:, r].copy(), v, M)) <= TOL
        assert relerr(res[1][2][r], kgo.msd(olat, olat.x, olat.period_x, 0.0, s, v, M, nt, dt)) <= TOL
        if R <= 4:
            assert relerr(res[1][3][r], kgo.vac(olat, olat.x, olat.period_x, 0.0, s, v, M, nt, dt)) <= TOL


def test_one_launch_literal_alg5_and_chain(B, kgo):
    """Literal Alg. 5 (doubling off) and a K = 2 chain through the cluster kernel."""
    lat = ring(kgo, 3000)
    wl = W.Lattice(lat.n, 2, lat.nn, lat.nl, lat.hop, None, lat.x, lat.y, lat.period_x, 0.0)
    s = 2 * 2.7 * 1.05
    phi = W.random_phase_vectors(lat.n, 2, 3)
    M = 50
    want = np.stack([kgo.dos_moments(lat, 0.0, s, phi[:, r].copy(), M) for r in range(2)])
    for doubling in (1, 0):
        h = B.from_lattice(wl, wl.x, wl.period_x, 0.0, s)
        h.set_option(B.KG_OPT_DOUBLING, doubling)
        l0 = h.launch_count
        got = host(B.dos_moments(h, dev(phi), M))
        assert h.launch_count - l0 == 3
        assert relerr(got, want) <= TOL


def test_config1_step_time(B):
    """Config 1 (4096 sites): time per Chebyshev step of the moment loop, one launch vs one launch per step."""
    import torch
    cfg = W.make_config(1)
    lat = cfg.lattice
    phi = dev(W.random_phase_vectors(lat.n, 1, cfg.seed))
    M = 2000
    stream = torch.cuda.Stream()
    times = {}
    for one in (1, 0):
        h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
        h.set_option(B.KG_OPT_ONE_LAUNCH, one)
        with torch.cuda.stream(stream):
            B.dos_moments(h, phi, M)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            for _ in range(5):
                B.dos_moments(h, phi, M)
            e1.record(stream)
        stream.synchronize()
        times[one] = e0.elapsed_time(e1) * 1e3 / (5 * (M // 2))
    print(f"config 1: {times[1]:.2f} us per Chebyshev step in one launch, {times[0]:.2f} us with one launch per step")
    # a report, not a pass / fail criterion of the parity suite: a busy or down-clocked box must not turn it red
    # (measured on an idle B200: 0.83 us against 2.7 us)
    if not (times[1] < 1.0 and times[1] < 0.5 * times[0]):
        import warnings
        warnings.warn(f"config 1 one-launch loop slower than expected: {times[1]:.2f} us per step (per-step launches: {times[0]:.2f} us)")
