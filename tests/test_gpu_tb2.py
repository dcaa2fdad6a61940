"""GPU parity of the site re-ordering done at create (kg_partition.h) and of the two-step
(temporally blocked) moment kernel (kg_tb2.cuh), against the CPU oracle.

Both are automatic only on large systems (n >= 65536; >= 2 tiles per SM), so the tests force
them on small lattices with kg_set_default_option(KG_OPT_REORDER, 1) and
kg_set_option(KG_OPT_TWO_STEP, 1).  Sizes span several 1024-element tiles with a ragged last
tile; the halo rings H1 / H2 of a tile then reach into several other tiles and across the
periodic boundary.  Edge cases: M from 6 (one single-step pass) upwards, odd and even, so that
the last pass is a two-step or a one-step one; R = 1, 2 for DOS / MSD, R = 1 for VAC (two
columns in the batch); with / without on-site energies; row widths K = 2, 3, 4, 6; vacancies
(rows with 0-3 neighbours); several hopping values (dictionary ids).
Tolerance 1e-10 (BASELINE.json) on moments, 1e-12 on state vectors."""
import numpy as np
import pytest

from helpers import relerr, to_oracle_lattice
from paper_1307_0288_b200 import workloads as W
from test_gpu_staged import grid_lattice

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1307_0288_b200 import binding
    return binding


@pytest.fixture()
def reordered(B):
    """Handles created inside the test have their sites re-ordered whatever their size."""
    B.set_default_option(B.KG_OPT_REORDER, 1)
    yield
    B.set_default_option(B.KG_OPT_REORDER, -1)


def dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.cpu().numpy()


def sheet(onsite, nvac=40, three_hops=False):
    """31 x 27 cells = 3348 sites minus vacancies: 4 tiles of 1024 sites (7 of 512), ragged tail."""
    full = W.honeycomb(31, 27)
    lat = W.remove_sites(full, W.vacancy_mask(full.n, nvac, 5)) if nvac else full
    if onsite:
        lat.onsite = W.anderson(lat.n, 2.7, 6)
    if three_hops:
        # symmetric bond-dependent hoppings from three values (dictionary ids 1..3)
        nl = lat.nl.reshape(3, lat.n)
        i = np.arange(lat.n)[None, :]
        key = (np.minimum(i, nl) * 7 + np.maximum(i, nl) * 13) % 3
        lat.hop = (np.where(np.arange(3)[:, None] < lat.nn[None, :], np.array([-2.7, -2.4, -3.0])[key], 0.0)).reshape(-1)
    s = (3 * 3.0 + (1.35 if onsite else 0.0)) * 1.05
    return lat, s


@pytest.mark.parametrize("M", [6, 7, 8, 9, 10, 64, 65])
@pytest.mark.parametrize("R", [1, 2])
@pytest.mark.parametrize("onsite", [False, True])
def test_two_step_dos_moments(B, kgo, reordered, M, R, onsite):
    lat, s = sheet(onsite, three_hops=(M == 65))
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_TWO_STEP, 1)
    phi = W.random_phase_vectors(lat.n, R, 3)
    B.dos_moments(h, dev(phi), M)                      # builds the per-tile plan
    l0 = h.launch_count
    mu = host(B.dos_moments(h, dev(phi), M))
    # the two-step passes really ran: first step + ceil((M/2 - 1)/2) passes + permutation + reduction
    assert h.launch_count - l0 == 1 + (M // 2 - 1 + 1) // 2 + 1 + 1
    for r in range(R):
        assert relerr(mu[r], kgo.dos_moments(olat, 0.0, s, phi[:, r].copy(), M)) <= TOL
    # and equal the one-step kernels up to rounding
    h.set_option(B.KG_OPT_TWO_STEP, 0)
    assert relerr(host(B.dos_moments(h, dev(phi), M)), mu) <= 1e-12


@pytest.mark.parametrize("M", [6, 9, 48])
@pytest.mark.parametrize("onsite", [False, True])
def test_two_step_vac_and_msd(B, kgo, reordered, M, onsite):
    """kg_vac (cross-doubling on the batch [V psi | chi]: two columns) and kg_msd with R = 1 and 2 over
    several time steps, two-step kernel forced."""
    lat, s = sheet(onsite)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_TWO_STEP, 1)
    nt, dt = 3, 0.7
    phi = W.random_phase_vectors(lat.n, 2, 4)
    vac = host(B.vac(h, dev(phi[:, :1]), M, nt, dt))
    msd = host(B.msd(h, dev(phi), M, nt, dt))
    v0 = phi[:, 0].copy()
    assert relerr(vac[0], kgo.vac(olat, olat.x, olat.period_x, 0.0, s, v0, M, nt, dt)) <= TOL
    for r in range(2):
        assert relerr(msd[r], kgo.msd(olat, olat.x, olat.period_x, 0.0, s, phi[:, r].copy(), M, nt, dt)) <= TOL


@pytest.mark.parametrize("shape", [(5000,), (90, 70), (22, 18, 16)])
def test_two_step_other_row_widths(B, kgo, reordered, shape):
    """K = 2, 4, 6 (chain, square, cubic Anderson models)."""
    lat = grid_lattice(shape, onsite_w=1.0)
    s = (lat.kmax * 1.0 + 0.5) * 1.05
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_TWO_STEP, 1)
    phi = W.random_phase_vectors(lat.n, 2, 9)
    M = 31
    dos = host(B.dos_moments(h, dev(phi), M))
    vac = host(B.vac(h, dev(phi[:, :1]), M, 1, 0.9))
    for r in range(2):
        assert relerr(dos[r], kgo.dos_moments(olat, 0.0, s, phi[:, r].copy(), M)) <= TOL
    assert relerr(vac[0], kgo.vac(olat, olat.x, olat.period_x, 0.0, s, phi[:, 0].copy(), M, 1, 0.9)) <= TOL


def test_two_step_bitwise_reproducible(B, reordered):
    lat, s = sheet(True)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_TWO_STEP, 1)
    phi = dev(W.random_phase_vectors(lat.n, 1, 3))
    a = host(B.dos_moments(h, phi, 100)).tobytes()
    v = host(B.vac(h, phi, 50, 2, 0.5)).tobytes()
    for _ in range(3):
        assert host(B.dos_moments(h, phi, 100)).tobytes() == a
        assert host(B.vac(h, phi, 50, 2, 0.5)).tobytes() == v


@pytest.mark.parametrize("open_x", [False, True])
@pytest.mark.parametrize("host_ptrs", [False, True])
def test_every_call_with_reordered_sites(B, kgo, reordered, open_x, host_ptrs):
    """Site vectors cross the boundary in the CALLER's order whatever the internal order: every call
    that takes or returns a vector, with device and with host pointers, against the oracle."""
    full = W.honeycomb(23, 19, periodic_x=not open_x, periodic_y=True)
    lat = W.remove_sites(full, W.vacancy_mask(full.n, 30, 2))
    lat.onsite = W.anderson(lat.n, 2.7, 3)
    s = (3 * 2.7 + 1.35 + 0.2) * 1.05
    e0 = 0.2
    olat = to_oracle_lattice(kgo, lat)
    period = 0.0 if open_x else lat.period_x
    h = B.from_lattice(lat, lat.x, period, e0, s)
    R = 2
    rng = np.random.default_rng(8)
    phi = rng.normal(size=(lat.n, R)) + 1j * rng.normal(size=(lat.n, R))
    phi /= np.linalg.norm(phi, axis=0)
    L = W.random_phase_vectors(lat.n, R, 1)
    put = (lambda x: np.ascontiguousarray(x)) if host_ptrs else dev
    get = (lambda x: x) if host_ptrs else host
    M, nt, dt = 20, 2, 0.8
    evo = get(B.evolve(h, put(phi), -dt))
    vel = get(B.apply_velocity(h, put(phi)))
    mom = get(B.moments(h, put(L), put(phi), M))
    vac = get(B.vac(h, put(phi), M, nt, dt))
    msd = get(B.msd(h, put(phi), M, nt, dt))
    psi, psix = put(phi.copy()), put(np.zeros_like(phi))
    B.evolve_x(h, psi, psix, dt)
    B.evolve_x(h, psi, psix, dt)
    if not host_ptrs:
        import torch
        torch.cuda.synchronize()
    psi, psix = get(psi), get(psix)
    F = get(B.fourier_moments(h, put(L), put(phi), 3, 0.4))
    for r in range(R):
        v, l = phi[:, r].copy(), L[:, r].copy()
        assert relerr(evo[:, r], kgo.evolve(olat, e0, s, v, -dt)) <= 1e-12
        assert relerr(vel[:, r], kgo.apply_velocity(olat, olat.x, period, v)) <= 1e-12
        assert relerr(mom[r], kgo.moments(olat, e0, s, l, v, M)) <= TOL
        assert relerr(vac[r], kgo.vac(olat, olat.x, period, e0, s, v, M, nt, dt)) <= TOL
        assert relerr(msd[r], kgo.msd(olat, olat.x, period, e0, s, v, M, nt, dt)) <= TOL
        u1 = kgo.evolve(olat, e0, s, v, dt)
        x1 = kgo.comm_evolve(olat, olat.x, period, e0, s, v, dt)
        u2 = kgo.evolve(olat, e0, s, u1, dt)
        x2 = kgo.evolve(olat, e0, s, x1, dt) + kgo.comm_evolve(olat, olat.x, period, e0, s, u1, dt)
        assert relerr(psi[:, r], u2) <= 1e-12 and relerr(psix[:, r], x2) <= 1e-12
        assert relerr(F[r], kgo.fourier_moments(olat, e0, s, l, v, 3, 0.4)) <= TOL


def test_reordering_is_a_permutation_and_keeps_results(B, reordered):
    """Same handle data with and without re-ordering: moments agree to rounding, vectors bit for bit
    where the arithmetic per site does not depend on the order (velocity)."""
    lat, s = sheet(True)
    phi = dev(W.random_phase_vectors(lat.n, 2, 3))
    h1 = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    B.set_default_option(B.KG_OPT_REORDER, 0)
    h0 = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    assert host(B.apply_velocity(h1, phi)).tobytes() == host(B.apply_velocity(h0, phi)).tobytes()
    assert relerr(host(B.dos_moments(h1, phi, 40)), host(B.dos_moments(h0, phi, 40))) <= 1e-13
    assert relerr(host(B.evolve(h1, phi, 1.3)), host(B.evolve(h0, phi, 1.3))) <= 1e-14


@pytest.mark.parametrize("R", [4, 8])
def test_two_step_wider_batches_as_column_pair_planes(B, kgo, reordered, R):
    """R = 4, 8: the doubling moment loops run the two-column two-step kernel on column-pair planes, all planes in
    one launch per pass (DOS and MSD: pairs (0,1), (2,3), ...; VAC: the pair [V psi_r | chi_r] of every vector);
    every vector against the oracle, and the launch count shows that no one-step sweep ran."""
    lat, s = sheet(True)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_TWO_STEP, 1)
    M, nt, dt = 21, 2, 0.6
    phi = W.random_phase_vectors(lat.n, R, 5)
    B.dos_moments(h, dev(phi), M)                      # builds the per-tile plan
    l0 = h.launch_count
    dos = host(B.dos_moments(h, dev(phi), M))
    passes = (M // 2 - 1 + 1) // 2
    assert h.launch_count - l0 == 1 + 1 + R + passes + 1      # permutation, first step, T_0 / T_1 into R/2 planes, passes, reduction
    vac = host(B.vac(h, dev(phi), M, nt, dt))
    msd = host(B.msd(h, dev(phi), M, nt, dt))
    for r in range(R):
        v = phi[:, r].copy()
        assert relerr(dos[r], kgo.dos_moments(olat, 0.0, s, v, M)) <= TOL
        assert relerr(vac[r], kgo.vac(olat, olat.x, olat.period_x, 0.0, s, v, M, nt, dt)) <= TOL
        assert relerr(msd[r], kgo.msd(olat, olat.x, olat.period_x, 0.0, s, v, M, nt, dt)) <= TOL
    h.set_option(B.KG_OPT_TWO_STEP, 0)
    assert relerr(host(B.dos_moments(h, dev(phi), M)), dos) <= 1e-12
    assert relerr(host(B.vac(h, dev(phi), M, nt, dt)), vac) <= 1e-12


def test_tile_plans_are_built_at_create_on_auto_handles(B):
    """A handle on which the two-step kernel is chosen automatically (re-ordered sites, >= 4 tiles per SM: here
    config 3's 1.2 M-site ribbon) gets its tile plans inside kg_create_hamiltonian, so the FIRST moments call
    enqueues exactly the launches of the second one (the plan builder's own kernel is not among them) and is
    bitwise equal to it; the two-step passes really run (fewer launches than Chebyshev steps)."""
    cfg = W.make_config(3)
    lat = cfg.lattice
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    phi = dev(W.random_phase_vectors(lat.n, 1, cfg.seed))
    M = 40
    l0 = h.launch_count
    mu1 = host(B.dos_moments(h, phi, M))
    l1 = h.launch_count
    mu2 = host(B.dos_moments(h, phi, M))
    l2 = h.launch_count
    assert l1 - l0 == l2 - l1
    assert l2 - l1 < M // 2                        # M/2 - 1 = 19 steps in 10 passes + first step, permutation, reduction
    assert mu1.tobytes() == mu2.tobytes()
    assert abs(mu1[0, 0] - 1.0) < 1e-12
