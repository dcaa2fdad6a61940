"""Wide stencil in the tuned kernels ("more complicated tight-binding models ... denser
Hamiltonian"): next-nearest-neighbour graphene, row width K = 9, two hopping values (hopping
dictionary ids 1 and 2), E0 = 3 t' != 0 (the Dirac-point energy; exercises the shift in the matrix, in
the evolution phase and in the reconstruction).  Every call against the oracle at R = 1 and 4, with the
TMA-staged kernels (K = 9 instantiation) and, as a cross-check, the one-thread-per-element kernels."""
import numpy as np
import pytest

from helpers import relerr, to_oracle_lattice
from paper_1307_0288_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-10
T, T2 = 2.7, 0.27


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


@pytest.mark.parametrize("R", [1, 4])
@pytest.mark.parametrize("open_x", [False, True])
@pytest.mark.parametrize("onsite", [False, True])
def test_nnn_every_call(B, kgo, R, open_x, onsite):
    lat = W.honeycomb_nnn(37, 23, periodic_x=not open_x, periodic_y=True)        # 3404 sites: 7 tiles of 512, ragged
    if onsite:
        lat.onsite = W.anderson(lat.n, 2.7, 3)
    e0 = 3 * T2
    s = (abs(e0) + 3 * T + 6 * T2 + (1.35 if onsite else 0.0)) * 1.05
    period = 0.0 if open_x else lat.period_x
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, period, e0, s)
    phi = W.random_phase_vectors(lat.n, R, 6)
    L = W.random_phase_vectors(lat.n, R, 7)
    M, nt, dt = 40, 2, 0.9
    got = {"dos": host(B.dos_moments(h, dev(phi), M)), "mom": host(B.moments(h, dev(L), dev(phi), M)),
           "vac": host(B.vac(h, dev(phi), M, nt, dt)), "msd": host(B.msd(h, dev(phi), M, nt, dt)),
           "evo": host(B.evolve(h, dev(phi), -dt)), "vel": host(B.apply_velocity(h, dev(phi)))}
    for r in sorted({0, R - 1}):
        v, l = phi[:, r].copy(), L[:, r].copy()
        assert relerr(got["dos"][r], kgo.dos_moments(olat, e0, s, v, M)) <= TOL
        assert relerr(got["mom"][r], kgo.moments(olat, e0, s, l, v, M)) <= TOL
        assert relerr(got["vac"][r], kgo.vac(olat, olat.x, period, e0, s, v, M, nt, dt)) <= TOL
        assert relerr(got["msd"][r], kgo.msd(olat, olat.x, period, e0, s, v, M, nt, dt)) <= TOL
        assert relerr(got["evo"][:, r], kgo.evolve(olat, e0, s, v, -dt)) <= 1e-12
        assert relerr(got["vel"][:, r], kgo.apply_velocity(olat, olat.x, period, v)) <= 1e-12
    # the same through the one-thread-per-element kernels
    l0 = h.launch_count
    h.set_option(B.KG_OPT_STAGED, 0)
    assert relerr(host(B.vac(h, dev(phi), M, nt, dt)), got["vac"]) <= 1e-12
    assert relerr(host(B.msd(h, dev(phi), M, nt, dt)), got["msd"]) <= 1e-12
    assert relerr(host(B.dos_moments(h, dev(phi), M)), got["dos"]) <= 1e-12
    assert h.launch_count > l0


def test_nnn_dos_shows_electron_hole_asymmetry(B):
    """Physics of the t' term on the GPU path: the Dirac point moves to E = 3 t' and the band becomes
    asymmetric ([-3|t| - 6 t', +3|t| + 3 t']); KPM DOS of a 90 000-site sheet, 4 random vectors."""
    import torch
    lat = W.honeycomb_nnn(150, 150)
    e0 = 3 * T2
    s = (abs(e0) + 3 * T + 6 * T2) * 1.05
    h = B.from_lattice(lat, lat.x, lat.period_x, e0, s)
    phi = dev(W.random_phase_vectors(lat.n, 4, 1))
    en = torch.linspace(-10.2, 9.5, 395, dtype=torch.float64).cuda()
    rho = host(B.kpm_reconstruct(B.dos_moments(h, phi, 600), e0, s, en)).mean(axis=0)
    e = host(en)
    assert abs(np.trapezoid(rho, e) - 1.0) < 5e-3
    dirac = e[np.argmin(np.where(np.abs(e - e0) < 1.0, rho, np.inf))]
    assert abs(dirac - e0) < 0.1                                  # DOS minimum at the shifted Dirac point
    assert rho[e < -3 * T - 6 * T2 - 0.3].max() < 2e-3 and rho[e > 3 * T + 3 * T2 + 0.3].max() < 2e-3
    assert rho[(e > -9.5) & (e < -9.0)].mean() > 0.01             # states below -3|t|: the asymmetry
