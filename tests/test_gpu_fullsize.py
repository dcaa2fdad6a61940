"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(default options: staged kernel, dictionary, alternating sweep, 3 CTAs/SM).

The single-threaded oracle cannot run the full jobs (1e11-2e13 site-updates), so
each config is compared on what the oracle can compute in seconds, chosen so that every kernel
mode runs at full size:

  * Chebyshev moments do not depend on M (only the Jackson damping does), so a PREFIX of
    M' moments of the full job is a sampled output: DOS moments, and VAC / MSD rows
    k = 0..n_t' for a few time steps, compared entry by entry (tolerance 1e-10, max-norm
    relative, BASELINE.json);
  * properties that hold at any size for the full-M run: mu_0 = 1, |mu_m| <= 1, the first M'
    moments of the M = 3000 run equal the M' run bit for bit, MSD row 0 is exactly 0.
"""
import numpy as np
import pytest

from helpers import relerr, to_oracle_lattice
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


@pytest.mark.parametrize("idx,Mp,ntp", [(2, 24, 2), (3, 16, 2), (4, 16, 1)])
def test_config_prefix_parity(B, kgo, idx, Mp, ntp):
    cfg = W.make_config(idx)
    lat = cfg.lattice
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    R = cfg.R
    phi = W.random_phase_vectors(lat.n, R, cfg.seed)
    dphi = dev(phi)
    dos = host(B.dos_moments(h, dphi, Mp))
    vac = host(B.vac(h, dphi, Mp, ntp, cfg.dt_fs))
    msd = host(B.msd(h, dphi, Mp, ntp, cfg.dt_fs))
    assert np.all(msd[:, 0, :] == 0)
    for r in sorted({0, R - 1}):
        v = phi[:, r].copy()
        assert relerr(dos[r], kgo.dos_moments(olat, cfg.e0, cfg.scale, v, Mp)) <= TOL
        assert relerr(vac[r], kgo.vac(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, Mp, ntp, cfg.dt_fs)) <= TOL
        assert relerr(msd[r], kgo.msd(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, Mp, ntp, cfg.dt_fs)) <= TOL


def test_config4_full_M_properties(B):
    """The exact call bench.py times: config 4, kg_dos_moments with M = 3000."""
    cfg = W.make_config(4)
    lat = cfg.lattice
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    dphi = dev(W.random_phase_vectors(lat.n, 1, cfg.seed))
    full = host(B.dos_moments(h, dphi, cfg.M))[0]
    head = host(B.dos_moments(h, dphi, 16))[0]
    assert abs(full[0] - 1.0) < 1e-12
    assert np.max(np.abs(full)) <= 1.0 + 1e-12            # |<phi|T_m|phi>| <= 1 for a unit vector
    assert np.max(np.abs(full.imag)) < 1e-12              # <phi|T_m(H~)|phi> is real (T_m Hermitian)
    assert full[:16].tobytes() == head.tobytes()
    again = host(B.dos_moments(h, dphi, cfg.M))[0]
    assert full.tobytes() == again.tobytes()              # bitwise reproducible at full size


def test_config5_batched_prefix_parity(B, kgo):
    """16 M sites x 8 vectors in one SpMM batch (2 GB per state set); vectors 0 and 7 against
    the oracle on an 8-moment prefix of DOS and on MSD rows 0..1."""
    cfg = W.make_config(5)
    lat = cfg.lattice
    assert lat.n == 15_984_000
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    phi = W.random_phase_vectors(lat.n, cfg.R, cfg.seed)
    dphi = dev(phi)
    Mp = 8
    dos = host(B.dos_moments(h, dphi, Mp))
    msd = host(B.msd(h, dphi, 4, 1, cfg.dt_fs))
    assert np.allclose(dos[:, 0], 1.0, atol=1e-12)
    for r in (0, 7):
        v = phi[:, r].copy()
        assert relerr(dos[r], kgo.dos_moments(olat, cfg.e0, cfg.scale, v, Mp)) <= TOL
        assert relerr(msd[r], kgo.msd(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, 4, 1, cfg.dt_fs)) <= TOL


def test_full_recursion_depth_M3000(B, kgo):
    """Rounding-error growth over the FULL recursion depth of configs 4-5 (M = 3000) on a lattice the
    oracle can finish (160 x 160 cells = 102 400 sites, Anderson W = |t|, config 4's scale): all three
    moment kernels — literal Alg. 5 (phi_L != phi_R), doubling (DOS) and cross-doubling (VAC, t = 0) —
    against the oracle's literal recursion, every one of the 3000 moments, tolerance 1e-10."""
    lat = W.honeycomb(160, 160)
    lat.onsite = W.anderson(lat.n, 2.7, 2)
    s = (3 * 2.7 + 1.35) * 1.05
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    M = 3000
    phi = W.random_phase_vectors(lat.n, 2, 7)
    a, b = phi[:, 0].copy(), phi[:, 1].copy()
    dos = host(B.dos_moments(h, dev(a), M))[0]
    assert relerr(dos, kgo.dos_moments(olat, 0.0, s, a, M)) <= TOL
    mom = host(B.moments(h, dev(b), dev(a), M))[0]
    assert relerr(mom, kgo.moments(olat, 0.0, s, b, a, M)) <= TOL
    vac = host(B.vac(h, dev(a), M, 0, 1.0))[0]
    assert relerr(vac, kgo.vac(olat, olat.x, olat.period_x, 0.0, s, a, M, 0, 1.0)) <= TOL
