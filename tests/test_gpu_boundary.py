"""GPU tests of the boundary's edges (include/kg.h): R = 16 wherever the kernels take it, the opt-in
non-finite input check, the post-processing calls with device grids, and the local density of
states (unit vectors instead of random-phase vectors) as one R = 8 batch."""
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


def lattice():
    full = W.honeycomb(14, 12)
    lat = W.remove_sites(full, W.vacancy_mask(full.n, 20, 4))
    lat.onsite = W.anderson(lat.n, 2.7, 5)
    return lat, (3 * 2.7 + 1.35) * 1.05


def test_sixteen_vectors_per_batch(B, kgo):
    """R = 16 in kg_moments / kg_dos_moments / kg_msd / kg_evolve_x / kg_fourier_moments (kg_evolve and
    kg_apply_velocity are covered in test_gpu_parity.py); kg_vac advances 2R columns and stops at R = 8."""
    lat, s = lattice()
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    R = 16
    phi = W.random_phase_vectors(lat.n, R, 2)
    L = W.random_phase_vectors(lat.n, R, 3)
    M, nt, dt = 24, 2, 0.6
    dos = host(B.dos_moments(h, dev(phi), M))
    mom = host(B.moments(h, dev(L), dev(phi), M))
    msd = host(B.msd(h, dev(phi), M, nt, dt))
    F = host(B.fourier_moments(h, dev(L), dev(phi), 2, 0.3))
    psi, psix = dev(phi.copy()), dev(np.zeros_like(phi))
    B.evolve_x(h, psi, psix, dt)
    psi, psix = host(psi), host(psix)
    for r in (0, 7, 15):
        v, l = phi[:, r].copy(), L[:, r].copy()
        assert relerr(dos[r], kgo.dos_moments(olat, 0.0, s, v, M)) <= TOL
        assert relerr(mom[r], kgo.moments(olat, 0.0, s, l, v, M)) <= TOL
        assert relerr(msd[r], kgo.msd(olat, olat.x, olat.period_x, 0.0, s, v, M, nt, dt)) <= TOL
        assert relerr(F[r], kgo.fourier_moments(olat, 0.0, s, l, v, 2, 0.3)) <= TOL
        assert relerr(psi[:, r], kgo.evolve(olat, 0.0, s, v, dt)) <= 1e-12
        assert relerr(psix[:, r], kgo.comm_evolve(olat, olat.x, olat.period_x, 0.0, s, v, dt)) <= 1e-12
    with pytest.raises(B.KgError) as e:
        B.vac(h, dev(phi), M, 1, dt)
    assert e.value.code == B.KG_EUNSUPPORTED
    for bad_R in (3, 32):
        with pytest.raises(B.KgError) as e:
            B.dos_moments(h, dev(W.random_phase_vectors(lat.n, bad_R, 1)), M)
        assert e.value.code == B.KG_EUNSUPPORTED


def test_non_finite_input_check_is_opt_in(B):
    lat, s = lattice()
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, 2, 2)
    phi[17, 1] = complex(np.nan, 0.0)
    out = host(B.dos_moments(h, dev(phi), 8))                   # default: not checked, NaN propagates
    assert np.all(np.isfinite(out[0])) and np.any(np.isnan(out[1]))
    h.set_option(B.KG_OPT_CHECK_INPUT, 1)
    for call in (lambda: B.dos_moments(h, dev(phi), 8), lambda: B.evolve(h, dev(phi), 0.5), lambda: B.apply_velocity(h, dev(phi)),
                 lambda: B.msd(h, dev(phi), 8, 1, 0.5), lambda: B.vac(h, phi, 8, 1, 0.5)):
        with pytest.raises(B.KgError) as e:
            call()
        assert e.value.code == B.KG_EINVAL
    phi[17, 1] = complex(0.0, np.inf)
    with pytest.raises(B.KgError):
        B.dos_moments(h, dev(phi), 8)
    good = W.random_phase_vectors(lat.n, 2, 2)
    assert np.all(np.isfinite(host(B.dos_moments(h, dev(good), 8))))


def test_post_processing_with_device_grids(B, kgo):
    """kg_kpm_reconstruct / kg_transport take every array as a device pointer and then neither allocate
    with cudaMalloc nor synchronise; an energy outside (E0 - s, E0 + s) on a DEVICE grid gives NaN, on a
    host grid KG_EINVAL."""
    import torch
    lat, s = lattice()
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = dev(W.random_phase_vectors(lat.n, 2, 2))
    M, nt, dt = 48, 4, 0.7
    en = np.linspace(-6.0, 6.0, 41)
    mu = B.msd(h, phi, M, nt, dt)
    dos = B.dos_moments(h, phi, M)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        stream.wait_stream(torch.cuda.default_stream())
        for _ in range(3):                                       # warm pool: later rounds re-use it
            rho = B.kpm_reconstruct(dos, 0.0, s, dev(en)).mean(dim=0).contiguous()
            f = B.kpm_reconstruct(mu, 0.0, s, dev(en)).mean(dim=0).contiguous()
            tr = B.transport(rho, None, f, dt, 1.0, 1.0)
    stream.synchronize()
    fh, rh = host(f), host(rho)
    want = kgo.transport(rh, None, fh, dt, 1.0, 1.0)
    for key in ("sigma_e1", "sigma_e2", "length_nm", "conductance"):
        assert relerr(host(tr[key]), want[key]) <= 1e-12
    bad = np.array([0.0, s, 1.0])
    out = host(B.kpm_reconstruct(dos, 0.0, s, dev(bad)))
    assert np.all(np.isnan(out[:, 1])) and np.all(np.isfinite(out[:, [0, 2]]))
    with pytest.raises(B.KgError) as e:
        B.kpm_reconstruct(dos, 0.0, s, bad)
    assert e.value.code == B.KG_EINVAL


def test_local_density_of_states_batch(B, kgo):
    """Local DOS: <i| delta(E - H) |i> from unit vectors |i>, R = 8 sites as ONE batch through
    kg_dos_moments -> kg_kpm_reconstruct, against the oracle: the three neighbours of a single vacancy,
    one site a few bonds away and four sites far from it.  The vacancy's zero mode (one state at E = 0 on
    the sublattice of its neighbours) shows as the local-DOS peak at E = 0 on the neighbours only."""
    full = W.honeycomb(40, 36)
    vacant = np.zeros(full.n, np.uint8)
    vacant[4 * (18 * 40 + 20) + 1] = 1
    lat = W.remove_sites(full, vacant)
    s = 3 * 2.7 * 1.05
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    near = np.nonzero(lat.nn == 2)[0]
    assert len(near) == 3
    d = np.hypot(lat.x[:, None] - lat.x[near][None, :], lat.y[:, None] - lat.y[near][None, :]).min(axis=1)
    mid_range = np.nonzero((d > 0.5) & (d < 0.6))[0][:1]
    far = np.nonzero(d > 3.0)[0][:4]
    sites = np.concatenate([near, mid_range, far])
    assert len(sites) == 8
    phi = np.zeros((lat.n, 8), complex)
    phi[sites, np.arange(8)] = 1.0
    M = 400
    en = np.linspace(-8.4, 8.4, 337)
    mu = B.dos_moments(h, dev(phi), M)
    ldos = host(B.kpm_reconstruct(mu, 0.0, s, dev(en)))
    muh = host(mu)
    for r in range(8):
        want_mu = kgo.dos_moments(olat, 0.0, s, phi[:, r].copy(), M)
        assert relerr(muh[r], want_mu) <= TOL
        assert relerr(ldos[r], kgo.kpm_reconstruct(want_mu, 0.0, s, en)) <= TOL
        assert abs(np.trapezoid(ldos[r], en) - 1.0) < 1e-2      # each local DOS integrates to 1
    zero = np.argmin(np.abs(en))
    assert ldos[:3, zero].min() > 10 * ldos[4:, zero].max()
