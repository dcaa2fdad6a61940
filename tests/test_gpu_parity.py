"""GPU parity: every C-ABI call of libkg against the CPU oracle, element by element, on the
same seeded inputs.  Sizes span several 256-thread tiles with a ragged tail; edge cases:
R in {1,2,4,8}, with / without on-site terms, kmax = 2 (generic-width kernel), rows with 0-3
neighbours (vacancies), open and periodic transport axis, E0 != 0, host-pointer arguments.

Tolerance (BASELINE.json north_star): max-norm relative error <= 1e-10 on moments / VAC / MSD,
normalised by the largest magnitude of the array.  State vectors (evolve, velocity) are held to
1e-12.  Determinism: moments bitwise equal run to run."""
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


def disordered(shape=(13, 11), nvac=37, onsite=True, open_x=False, seed=5):
    """13x11 cells = 572 sites minus 37 vacancies = 535 sites: 3 tiles of 256 with a ragged tail."""
    full = W.honeycomb(shape[0], shape[1], periodic_x=not open_x, periodic_y=True)
    lat = W.remove_sites(full, W.vacancy_mask(full.n, nvac, seed)) if nvac else full
    if onsite:
        lat.onsite = W.anderson(lat.n, 2.7, seed + 1)
    return lat


def scale_for(lat, e0=0.0):
    return (3 * 2.7 + (1.35 if lat.onsite is not None else 0.0) + abs(e0)) * 1.05


def rand_vectors(n, R, seed):
    rng = np.random.default_rng(seed)
    v = rng.normal(size=(n, R)) + 1j * rng.normal(size=(n, R))
    return v / np.linalg.norm(v, axis=0)


# --------------------------------------------------------------------------------- moments
@pytest.mark.parametrize("R", [1, 2, 4, 8])
@pytest.mark.parametrize("onsite", [False, True])
def test_dos_moments(B, kgo, R, onsite):
    lat = disordered(onsite=onsite)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, R, 3)
    M = 96
    mu = host(B.dos_moments(h, dev(phi), M))
    assert mu.shape == (R, M)
    for r in range(R):
        want = kgo.dos_moments(olat, 0.0, s, phi[:, r], M)
        assert relerr(mu[r], want) <= TOL
        assert abs(mu[r, 0] - 1.0) < 1e-13


@pytest.mark.parametrize("e0", [0.0, 0.35])
def test_moments_distinct_left_right(B, kgo, e0):
    lat = disordered()
    s = scale_for(lat, e0)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, e0, s)
    R, M = 2, 64
    L, Rv = rand_vectors(lat.n, R, 1), rand_vectors(lat.n, R, 2)
    mu = host(B.moments(h, dev(L), dev(Rv), M))
    for r in range(R):
        want = kgo.moments(olat, e0, s, L[:, r], Rv[:, r], M)
        assert relerr(mu[r], want) <= TOL


def test_moments_bitwise_reproducible_and_graph_equals_plain(B):
    import torch
    lat = disordered()
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, scale_for(lat))
    phi = dev(W.random_phase_vectors(lat.n, 4, 9))
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        a = B.dos_moments(h, phi, 200)          # side stream: CUDA-graph path
        b = B.dos_moments(h, phi, 200)
    st.synchronize()
    h.set_option(B.KG_OPT_USE_GRAPHS, 0)
    c = B.dos_moments(h, phi, 200)              # plain launches
    torch.cuda.synchronize()
    assert host(a).tobytes() == host(b).tobytes() == host(c).tobytes()


def test_generic_width_ring(B, kgo):
    """kmax = 2: the runtime-width kernel; 1-D ring closed form Tr[T_n]/N on unit vectors."""
    n = 700
    olat = ring(kgo, n)
    lat = W.Lattice(n, 2, olat.nn, olat.nl, olat.hop, None, olat.x, olat.y, olat.period_x, 0.0)
    s = 2 * 2.7 * 1.05
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = rand_vectors(n, 2, 4)
    mu = host(B.dos_moments(h, dev(phi), 50))
    for r in range(2):
        assert relerr(mu[r], kgo.dos_moments(olat, 0.0, s, phi[:, r], 50)) <= TOL
    v = host(B.apply_velocity(h, dev(phi)))
    for r in range(2):
        assert relerr(v[:, r], kgo.apply_velocity(olat, olat.x, olat.period_x, phi[:, r])) <= 1e-13


# --------------------------------------------------------------------------------- evolve / velocity
@pytest.mark.parametrize("R", [1, 4, 16])
@pytest.mark.parametrize("dt", [0.9, -2.3])
def test_evolve(B, kgo, R, dt):
    lat = disordered()
    e0 = 0.2
    s = scale_for(lat, e0)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, e0, s)
    phi = rand_vectors(lat.n, R, 6)
    out = host(B.evolve(h, dev(phi), dt))
    for r in range(0, R, max(1, R // 4)):
        want = kgo.evolve(olat, e0, s, phi[:, r], dt)
        assert relerr(out[:, r], want) <= 1e-12
    assert np.allclose(np.linalg.norm(out, axis=0), 1.0, atol=1e-12)      # |U phi| = |phi|
    back = host(B.evolve(h, dev(out), -dt))
    assert np.max(np.abs(back - phi)) < 1e-12                              # U(-dt)U(dt) phi = phi


@pytest.mark.parametrize("open_x", [False, True])
def test_apply_velocity(B, kgo, open_x):
    lat = disordered(open_x=open_x)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = rand_vectors(lat.n, 8, 7)
    out = host(B.apply_velocity(h, dev(phi)))
    for r in range(8):
        want = kgo.apply_velocity(olat, olat.x, olat.period_x, phi[:, r])
        assert relerr(out[:, r], want) <= 1e-13
    # transport along y instead (config 3 passes the armchair coordinate)
    h2 = B.from_lattice(lat, lat.y, lat.period_y, 0.0, s)
    out = host(B.apply_velocity(h2, dev(phi[:, :1].copy())))
    assert relerr(out[:, 0], kgo.apply_velocity(olat, olat.y, olat.period_y, phi[:, 0])) <= 1e-13


@pytest.mark.parametrize("R", [1, 2])
def test_evolve_x(B, kgo, R):
    """(psi, psix) <- (U psi, U psix + [X,U] psi) against the oracle's literal Alg. 6 + Alg. 7."""
    lat = disordered()
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    psi0, psix0 = rand_vectors(lat.n, R, 8), rand_vectors(lat.n, R, 9)
    dt = 1.1
    psi, psix = dev(psi0), dev(psix0)
    B.evolve_x(h, psi, psix, dt)
    psi, psix = host(psi), host(psix)
    for r in range(R):
        want_psi = kgo.evolve(olat, 0.0, s, psi0[:, r], dt)
        want_x = kgo.evolve(olat, 0.0, s, psix0[:, r], dt) + \
            kgo.comm_evolve(olat, olat.x, olat.period_x, 0.0, s, psi0[:, r], dt)
        assert relerr(psi[:, r], want_psi) <= 1e-12
        assert relerr(psix[:, r], want_x) <= 1e-12


# --------------------------------------------------------------------------------- VAC / MSD
@pytest.mark.parametrize("R,onsite", [(1, True), (2, False), (8, True)])
def test_vac(B, kgo, R, onsite):
    lat = disordered(onsite=onsite)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, R, 11)
    M, nt, dt = 48, 3, 0.6
    mu = host(B.vac(h, dev(phi), M, nt, dt))
    assert mu.shape == (R, nt + 1, M)
    for r in range(0, R, max(1, R // 2)):
        want = kgo.vac(olat, olat.x, olat.period_x, 0.0, s, phi[:, r], M, nt, dt)
        assert relerr(mu[r], want) <= TOL


@pytest.mark.parametrize("R,onsite,open_x", [(1, True, False), (4, False, True), (8, True, False)])
def test_msd(B, kgo, R, onsite, open_x):
    lat = disordered(onsite=onsite, open_x=open_x)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, R, 12)
    M, nt, dt = 48, 3, 0.6
    mu = host(B.msd(h, dev(phi), M, nt, dt))
    assert np.all(mu[:, 0, :] == 0)                                   # row 0 exactly 0
    for r in range(0, R, max(1, R // 2)):
        want = kgo.msd(olat, olat.x, olat.period_x, 0.0, s, phi[:, r], M, nt, dt)
        assert relerr(mu[r], want) <= TOL


def test_config1_full(B, kgo):
    """BASELINE config 1 in full: 4096 sites, M = 256 DOS moments, VAC and MSD over 16 steps."""
    c = W.make_config(1)
    lat = c.lattice
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, c.xcoord, c.period, c.e0, c.scale)
    phi = W.random_phase_vectors(lat.n, 1, c.seed)
    d = host(B.dos_moments(h, dev(phi), c.M))[0]
    assert relerr(d, kgo.dos_moments(olat, c.e0, c.scale, phi[:, 0], c.M)) <= TOL
    v = host(B.vac(h, dev(phi), c.M, c.n_steps, c.dt_fs))[0]
    assert relerr(v, kgo.vac(olat, c.xcoord, c.period, c.e0, c.scale, phi[:, 0], c.M, c.n_steps, c.dt_fs)) <= TOL
    m = host(B.msd(h, dev(phi), c.M, c.n_steps, c.dt_fs))[0]
    assert relerr(m, kgo.msd(olat, c.xcoord, c.period, c.e0, c.scale, phi[:, 0], c.M, c.n_steps, c.dt_fs)) <= TOL


# --------------------------------------------------------------------------------- boundary
def test_host_pointer_arguments(B, kgo):
    """The C ABI accepts host arrays: results identical to the device-pointer path."""
    import torch
    lat = disordered()
    s = scale_for(lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, 2, 13)
    mu_d = host(B.dos_moments(h, dev(phi), 40))
    mu_h = B.dos_moments(h, phi, 40)                     # numpy in, numpy out
    torch.cuda.synchronize()
    assert isinstance(mu_h, np.ndarray) and mu_h.tobytes() == mu_d.tobytes()
    pinned = torch.from_numpy(phi).pin_memory()
    out = torch.empty_like(pinned).pin_memory()
    B.evolve(h, pinned, 0.7, out=out)
    torch.cuda.synchronize()
    assert np.array_equal(out.numpy(), host(B.evolve(h, dev(phi), 0.7)))
    v_h = B.vac(h, phi, 16, 1, 0.5)
    torch.cuda.synchronize()
    assert v_h.tobytes() == host(B.vac(h, dev(phi), 16, 1, 0.5)).tobytes()


def test_csr_constructor_matches_list(B):
    lat = disordered()
    s = scale_for(lat)
    nl = lat.nl.reshape(3, lat.n); hop = lat.hop.reshape(3, lat.n)
    rowptr = np.zeros(lat.n + 1, np.int64); rowptr[1:] = np.cumsum(lat.nn)
    col = np.concatenate([nl[:lat.nn[i], i] for i in range(lat.n)]).astype(np.int32)
    val = np.concatenate([hop[:lat.nn[i], i] for i in range(lat.n)])
    h1 = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h2 = B.create_hamiltonian_csr(lat.n, rowptr, col, val, lat.onsite, lat.x, lat.period_x, 0.0, s)
    phi = dev(W.random_phase_vectors(lat.n, 1, 14))
    assert host(B.dos_moments(h1, phi, 30)).tobytes() == host(B.dos_moments(h2, phi, 30)).tobytes()
    # device-resident construction arrays work too
    h3 = B.create_hamiltonian(lat.n, 3, dev(lat.nn), dev(lat.nl), dev(lat.hop), dev(lat.onsite),
                              dev(lat.x), lat.period_x, 0.0, s)
    assert host(B.dos_moments(h3, phi, 30)).tobytes() == host(B.dos_moments(h1, phi, 30)).tobytes()


def test_error_codes(B):
    lat = disordered()
    s = scale_for(lat)
    with pytest.raises(B.KgError) as e:                              # spectrum outside [-1, 1]
        B.from_lattice(lat, lat.x, lat.period_x, 0.0, 5.0)
    assert e.value.code == B.KG_ESPECTRUM
    bad = W.Lattice(lat.n, 3, lat.nn, lat.nl.copy(), lat.hop, lat.onsite, lat.x, lat.y, lat.period_x, lat.period_y)
    bad.nl[5] = lat.n + 3
    with pytest.raises(B.KgError) as e:
        B.from_lattice(bad, bad.x, bad.period_x, 0.0, s)
    assert e.value.code == B.KG_EINVAL
    asym = W.Lattice(lat.n, 3, lat.nn, lat.nl, lat.hop.copy(), lat.onsite, lat.x, lat.y, lat.period_x, lat.period_y)
    asym.hop[7] *= 1.5
    with pytest.raises(B.KgError) as e:
        B.from_lattice(asym, asym.x, asym.period_x, 0.0, s * 2)
    assert e.value.code == B.KG_EINVAL and "symmetric" in str(e.value)
    nan = W.Lattice(lat.n, 3, lat.nn, lat.nl, lat.hop, lat.onsite.copy(), lat.x, lat.y, lat.period_x, lat.period_y)
    nan.onsite[3] = np.nan
    with pytest.raises(B.KgError) as e:
        B.from_lattice(nan, nan.x, nan.period_x, 0.0, s)
    assert e.value.code == B.KG_EINVAL
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = dev(W.random_phase_vectors(lat.n, 3, 1))
    with pytest.raises(B.KgError) as e:
        B.dos_moments(h, phi, 8)                                     # R = 3 unsupported
    assert e.value.code == B.KG_EUNSUPPORTED
    phi = dev(W.random_phase_vectors(lat.n, 1, 1))
    with pytest.raises(B.KgError):
        B.dos_moments(h, phi, 1)                                     # M < 2
    with pytest.raises(B.KgError):
        B.evolve(h, phi, 0.0)                                        # dt = 0
    with pytest.raises(B.KgError):
        B.evolve(h, phi, 1.0, out=phi)                               # aliasing


def test_tiny_and_isolated_sites(B, kgo):
    """n = 4 (one cell) and a lattice where vacancies leave isolated (0-neighbour) sites."""
    lat = W.honeycomb(1, 1)
    olat = to_oracle_lattice(kgo, lat)
    s = 3 * 2.7 * 1.05
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = rand_vectors(4, 1, 3)
    assert relerr(host(B.dos_moments(h, dev(phi), 20))[0], kgo.dos_moments(olat, 0.0, s, phi[:, 0], 20)) <= TOL
    full = W.honeycomb(4, 4)
    vac = np.zeros(full.n, np.uint8)
    nl = full.nl.reshape(3, full.n)
    vac[nl[:, 10]] = 1                                                # isolate site 10
    lat = W.remove_sites(full, vac)
    assert lat.nn.min() == 0
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = rand_vectors(lat.n, 1, 5)
    assert relerr(host(B.msd(h, dev(phi), 16, 2, 0.5))[0],
                  kgo.msd(olat, olat.x, olat.period_x, 0.0, s, phi[:, 0], 16, 2, 0.5)) <= TOL


# --------------------------------------------------------------------------------- reconstruction
@pytest.mark.parametrize("jackson", [True, False])
def test_kpm_reconstruct(B, kgo, jackson):
    """eqs 29-31 + Jackson kernel (eq 35) on the device against the oracle: config 1's DOS on its
    1001-point grid (M = 256), MSD rows (several rows at once), host and device pointers."""
    cfg = W.make_config(1)
    lat = cfg.lattice
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    phi = dev(W.random_phase_vectors(lat.n, 1, cfg.seed))
    en = W.energy_grid(cfg.n_energies)
    mu = B.dos_moments(h, phi, cfg.M)
    rho = host(B.kpm_reconstruct(mu, cfg.e0, cfg.scale, dev(en), jackson))
    want = kgo.kpm_reconstruct(host(mu)[0], cfg.e0, cfg.scale, en, jackson)
    assert rho.shape == (1, cfg.n_energies)
    assert relerr(rho[0], want) <= TOL
    if jackson:
        assert np.all(rho > 0)
        assert abs(np.sum(0.5 * (rho[0, 1:] + rho[0, :-1]) * np.diff(en)) - 1.0) < 2e-2   # int rho dE = 1
    msd = host(B.msd(h, phi, 64, 3, cfg.dt_fs))                   # [1][4][64]
    f = B.kpm_reconstruct(msd, cfg.e0, cfg.scale, en, jackson)     # numpy in -> numpy out
    assert f.shape == (1, 4, cfg.n_energies)
    for k in range(4):
        assert relerr(f[0, k], kgo.kpm_reconstruct(msd[0, k], cfg.e0, cfg.scale, en, jackson)) <= TOL
    with pytest.raises(B.KgError) as e:
        B.kpm_reconstruct(mu, cfg.e0, cfg.scale, np.array([0.0, cfg.scale]), jackson)
    assert e.value.code == B.KG_EINVAL


def test_transport_config2_like(B, kgo):
    """The whole post-processing chain of config 2 on a scaled-down twin (50x50 cells, 0.5 %
    vacancies): moments -> rho~, rho~C_vv, rho~DX2 on a 501-point grid -> sigma_GK, sigma_E1,
    sigma_E2, L, G, every table against the oracle's own chain; device and host pointers."""
    cfg = W.make_config(2, shrink=5)
    lat = cfg.lattice
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    phi = W.random_phase_vectors(lat.n, 1, cfg.seed)
    M, nt = 128, 6
    en = W.energy_grid(501)
    d_en = dev(en)
    rho = B.kpm_reconstruct(B.dos_moments(h, dev(phi), M), cfg.e0, cfg.scale, d_en)[0]
    fvac = B.kpm_reconstruct(B.vac(h, dev(phi), M, nt, cfg.dt_fs), cfg.e0, cfg.scale, d_en)[0]
    fmsd = B.kpm_reconstruct(B.msd(h, dev(phi), M, nt, cfg.dt_fs), cfg.e0, cfg.scale, d_en)[0]
    dens = 8.0 / (3 * np.sqrt(3) * 0.142 ** 2)             # 2N/Omega of graphene, nm^-2
    got = B.transport(rho, fvac, fmsd, cfg.dt_fs, dens, 2.0)
    v = phi[:, 0].copy()
    orho = kgo.kpm_reconstruct(kgo.dos_moments(olat, cfg.e0, cfg.scale, v, M), cfg.e0, cfg.scale, en)
    ovac = kgo.vac(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, M, nt, cfg.dt_fs)
    omsd = kgo.msd(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, M, nt, cfg.dt_fs)
    ofvac = np.stack([kgo.kpm_reconstruct(ovac[k], cfg.e0, cfg.scale, en) for k in range(nt + 1)])
    ofmsd = np.stack([kgo.kpm_reconstruct(omsd[k], cfg.e0, cfg.scale, en) for k in range(nt + 1)])
    want = kgo.transport(orho, ofvac, ofmsd, cfg.dt_fs, dens, 2.0)
    for key in ("sigma_gk", "sigma_e1", "sigma_e2", "length_nm", "conductance"):
        assert relerr(host(got[key]), want[key]) <= 1e-9, key
    # host pointers, subset of outputs
    hg = B.transport(None, None, host(fmsd), cfg.dt_fs, dens)
    assert hg["sigma_gk"] is None
    assert relerr(hg["sigma_e2"], want["sigma_e2"]) <= 1e-9


# --------------------------------------------------------------------------------- Fourier-transform method
@pytest.mark.parametrize("R", [1, 4])
def test_fourier_moments_and_ftm_reconstruct(B, kgo, R):
    """Alg. 4 (F_n = <phi_L|U(n dtau)|phi_R>, n = -Nm..Nm) and eqs 22-24 + Hanning window on the
    device against the oracle; distinct and identical left/right vectors; host pointers."""
    lat = disordered()
    e0 = 0.15
    s = scale_for(lat, e0)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, e0, s)
    Nm, dtau = 12, np.pi * W.HBAR / s                       # dtau = pi hbar / s
    L, Rv = rand_vectors(lat.n, R, 21), rand_vectors(lat.n, R, 22)
    F = host(B.fourier_moments(h, dev(L), dev(Rv), Nm, dtau))
    assert F.shape == (R, 2 * Nm + 1)
    for r in range(R):
        assert relerr(F[r], kgo.fourier_moments(olat, e0, s, L[:, r], Rv[:, r], Nm, dtau)) <= TOL
    d = dev(Rv)
    Fd = B.fourier_moments(h, d, d, Nm, dtau)               # DOS moments, eq 25
    Fh = B.fourier_moments(h, Rv, Rv, Nm, dtau)             # host in -> host out
    assert host(Fd).tobytes() == Fh.tobytes()
    assert np.max(np.abs(Fh[:, Nm] - 1.0)) < 1e-13
    assert np.max(np.abs(Fh[:, ::-1] - np.conj(Fh))) < 1e-12
    en = np.linspace(-9.0, 9.0, 301)
    for window in (True, False):
        f = host(B.ftm_reconstruct(Fd, dtau, dev(en), window))
        for r in range(R):
            assert relerr(f[r], kgo.ftm_reconstruct(Fh[r], dtau, en, window)) <= TOL
    f_host = B.ftm_reconstruct(Fh, dtau, en)
    assert relerr(f_host, host(B.ftm_reconstruct(Fd, dtau, dev(en)))) <= 1e-13


def test_run_config_driver(B):
    """The end-to-end driver (moments -> reconstruction -> transport) on config 1 in full."""
    from paper_1307_0288_b200 import run_config
    s = run_config.main(["--config", "1"])
    assert abs(s["mu0"] - 1.0) < 1e-12
    assert abs(s["dos_integral"] - 1.0) < 5e-3
    assert abs(s["sigma_e2_over_e1_last"] - 0.5) < 0.05        # pristine sheet: ballistic
    assert s["kernel_launches"] > 0
