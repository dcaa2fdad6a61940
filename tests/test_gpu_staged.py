"""GPU parity of the TMA-staged moment kernel (csrc/kg_staged.cuh) against the CPU oracle.

The staged kernel is the default for the recursion+dot steps (kmax = 3, contiguous vectors);
these cases pin down what is specific to it: the hopping dictionary (one value, a few values,
too many values -> fp64 hoppings staged), the ring of stages wrapping several times per CTA,
the alternating sweep direction, ragged last tile, every R, and bitwise agreement of repeated
runs.  Tolerance as in test_gpu_parity.py (BASELINE.json: <= 1e-10 max-norm relative)."""
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


def sheet(ncx, ncy, nvac, onsite, seed=11):
    full = W.honeycomb(ncx, ncy)
    lat = W.remove_sites(full, W.vacancy_mask(full.n, nvac, seed)) if nvac else full
    if onsite:
        lat.onsite = W.anderson(lat.n, 2.7, seed + 1)
    return lat


def set_hoppings(lat, kind):
    """Symmetric per-bond hoppings: a function of the unordered pair (i, NL_ik)."""
    n = lat.n
    nl = lat.nl.reshape(3, n).astype(np.int64)
    i = np.arange(n)[None, :]
    lo, hi = np.minimum(i, nl), np.maximum(i, nl)
    if kind == "three":
        vals = np.array([-2.7, -2.5, -3.0])
        hop = vals[(lo + hi) % 3]
    else:   # "many": a different value on (almost) every bond
        hop = -2.7 * (1.0 + 0.1 * np.sin(12.9898 * lo + 78.233 * hi))
    used = np.arange(3)[:, None] < lat.nn[None, :]
    lat.hop = np.where(used, hop, 0.0).reshape(-1)
    return lat


def scale_for(lat):
    return (3 * 3.0 + (1.35 if lat.onsite is not None else 0.0)) * 1.05


@pytest.mark.parametrize("R", [1, 2, 4, 8])
@pytest.mark.parametrize("kind", ["uniform", "three", "many"])
@pytest.mark.parametrize("onsite", [False, True])
def test_staged_moments_hopping_kinds(B, kgo, R, kind, onsite):
    lat = sheet(17, 13, 41, onsite)        # 884 - 41 = 843 sites: ragged last tile for every R
    if kind != "uniform":
        lat = set_hoppings(lat, kind)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, R, 3)
    rng = np.random.default_rng(R)
    L = rng.normal(size=(lat.n, R)) + 1j * rng.normal(size=(lat.n, R))
    M = 80
    h.set_option(B.KG_OPT_ONE_LAUNCH, 0)   # one launch per step here (the single-launch loop: tests/test_gpu_small.py)
    launches0 = h.launch_count
    mu = host(B.moments(h, dev(L), dev(phi), M))
    for r in range(R):
        want = kgo.moments(olat, 0.0, s, L[:, r], phi[:, r], M)
        assert relerr(mu[r], want) <= TOL
    # the staged kernel and the one-thread-per-element kernel compute the same steps
    h.set_option(B.KG_OPT_STAGED, 0)
    mu_plain = host(B.moments(h, dev(L), dev(phi), M))
    assert relerr(mu, mu_plain) <= 1e-12
    assert h.launch_count - launches0 == 2 * M       # (M-1 steps + 1 reduction) twice


@pytest.mark.parametrize("alternate", [0, 1])
@pytest.mark.parametrize("dict_on", [0, 1])
def test_staged_ring_wraps_many_tiles_per_cta(B, kgo, alternate, dict_on):
    """62 500 sites x R = 8 = 977 tiles of 512 elements on <= 296 CTAs: every CTA runs several
    tiles and the 2-3 stage ring wraps; vectors 0 and 7 against the oracle."""
    lat = sheet(125, 125, 0, True)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_ALTERNATE, alternate)
    if not dict_on:
        h.set_option(B.KG_OPT_DICT, 0)
    R, M = 8, 24
    phi = W.random_phase_vectors(lat.n, R, 5)
    mu = host(B.dos_moments(h, dev(phi), M))
    for r in (0, 7):
        assert relerr(mu[r], kgo.dos_moments(olat, 0.0, s, phi[:, r], M)) <= TOL
    again = host(B.dos_moments(h, dev(phi), M))
    assert mu.tobytes() == again.tobytes()           # bitwise reproducible


@pytest.mark.parametrize("stages,ctas", [(2, 1), (2, 3), (4, 1), (6, 1)])
def test_staged_ring_shapes(B, kgo, stages, ctas):
    lat = sheet(60, 50, 100, True)                    # 11 900 sites
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_STAGES, stages)
    h.set_option(B.KG_OPT_STAGED_CTAS, ctas)
    phi = W.random_phase_vectors(lat.n, 1, 6)
    mu = host(B.dos_moments(h, dev(phi), 40))
    assert relerr(mu[0], kgo.dos_moments(olat, 0.0, s, phi[:, 0], 40)) <= TOL


def test_staged_vac_msd(B, kgo):
    """Drivers on top of the staged kernel (VAC's first two steps read a strided phi_R and fall
    back to the plain kernel; MSD is staged from step 2 on)."""
    lat = sheet(20, 16, 30, True)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    R, M, nt, dt = 2, 48, 2, 0.7
    phi = W.random_phase_vectors(lat.n, R, 8)
    vac = host(B.vac(h, dev(phi), M, nt, dt))
    msd = host(B.msd(h, dev(phi), M, nt, dt))
    for r in range(R):
        assert relerr(vac[r], kgo.vac(olat, olat.x, olat.period_x, 0.0, s, phi[:, r], M, nt, dt)) <= TOL
        assert relerr(msd[r], kgo.msd(olat, olat.x, olat.period_x, 0.0, s, phi[:, r], M, nt, dt)) <= TOL


@pytest.mark.parametrize("R", [1, 8, 16])
@pytest.mark.parametrize("dict_on", [0, 1])
def test_staged_evolve_many_tiles(B, kgo, R, dict_on):
    """Alg. 6 on the staged kernel (MODE_EVO): 62 500 sites, every CTA runs several tiles;
    against the oracle (vector 0) and against the one-thread-per-element kernel (all vectors)."""
    lat = sheet(125, 125, 0, True)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    if not dict_on:
        h.set_option(B.KG_OPT_DICT, 0)
    phi = W.random_phase_vectors(lat.n, R, 5)
    dt = -1.7
    out = host(B.evolve(h, dev(phi), dt))
    assert relerr(out[:, 0], kgo.evolve(olat, 0.0, s, phi[:, 0].copy(), dt)) <= 1e-12
    assert np.allclose(np.linalg.norm(out, axis=0), 1.0, atol=1e-12)
    h.set_option(B.KG_OPT_STAGED, 0)
    plain = host(B.evolve(h, dev(phi), dt))
    assert relerr(out, plain) <= 1e-13


@pytest.mark.parametrize("R", [1, 4, 8])
@pytest.mark.parametrize("kind", ["uniform", "many"])
def test_staged_evolve_x_many_tiles(B, kgo, R, kind):
    """Eq 44 / Alg. 7 on the staged pair kernel (MODE_PAIR), two consecutive steps so that the
    second one starts from a non-zero psix; vacancies + on-site disorder; vector R-1 vs oracle."""
    lat = sheet(110, 90, 300, True)          # 39 300 sites
    if kind != "uniform":
        lat = set_hoppings(lat, kind)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, R, 7)
    dt = 1.3
    psi, psix = dev(phi), dev(np.zeros_like(phi))
    for _ in range(2):
        B.evolve_x(h, psi, psix, dt)
    want_psi, want_x = phi[:, R - 1].copy(), np.zeros(lat.n, complex)
    for _ in range(2):                       # eq 44 with the oracle's literal Alg. 6 + Alg. 7
        want_x = kgo.evolve(olat, 0.0, s, want_x, dt) + \
            kgo.comm_evolve(olat, olat.x, olat.period_x, 0.0, s, want_psi, dt)
        want_psi = kgo.evolve(olat, 0.0, s, want_psi, dt)
    assert relerr(host(psi)[:, R - 1], want_psi) <= 1e-12
    assert relerr(host(psix)[:, R - 1], want_x) <= 1e-12
    h.set_option(B.KG_OPT_STAGED, 0)
    p2, x2 = dev(phi), dev(np.zeros_like(phi))
    for _ in range(2):
        B.evolve_x(h, p2, x2, dt)
    assert relerr(host(psix), host(x2)) <= 1e-13


@pytest.mark.parametrize("M", [2, 3, 4, 63, 64])
@pytest.mark.parametrize("R", [1, 4])
@pytest.mark.parametrize("staged", [0, 1])
def test_doubling_moments(B, kgo, M, R, staged):
    """phi_L = phi_R: two moments per Chebyshev step from 2 T_a T_b = T_{a+b} + T_{|a-b|}
    (mu_{2n+1} = 2<T_n|T_{n+1}> - mu_1, mu_{2n+2} = 2<T_{n+1}|T_{n+1}> - mu_0) against the
    oracle's literal Alg. 5, for odd / even / minimal M, and against the literal GPU path."""
    lat = sheet(30, 26, 77, True)          # 3043 sites
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_STAGED, staged)
    h.set_option(B.KG_OPT_ONE_LAUNCH, 0)   # count the per-step launches (single-launch loop: tests/test_gpu_small.py)
    rng = np.random.default_rng(M)
    phi = rng.normal(size=(lat.n, R)) + 1j * rng.normal(size=(lat.n, R))     # not normalised
    d = dev(phi)
    l0 = h.launch_count
    mu = host(B.dos_moments(h, d, M))
    assert h.launch_count - l0 == M // 2 + 1                # M/2 sweeps + the reduction
    for r in range(R):
        assert relerr(mu[r], kgo.dos_moments(olat, 0.0, s, phi[:, r].copy(), M)) <= TOL
    h.set_option(B.KG_OPT_DOUBLING, 0)
    l0 = h.launch_count
    lit = host(B.dos_moments(h, d, M))
    assert h.launch_count - l0 == M                         # literal Alg. 5: M-1 sweeps + reduction
    assert relerr(mu, lit) <= 1e-13


@pytest.mark.parametrize("R", [1, 2, 8])
@pytest.mark.parametrize("staged", [0, 1])
@pytest.mark.parametrize("M", [2, 3, 33, 48])
def test_vac_cross_doubling(B, kgo, R, staged, M):
    """VAC with phi_L != phi_R: [V psi | chi] advanced as one 2R-wide batch and
    mu_{2m+1} = 2<T_m L|T_{m+1} R> - mu_1, mu_{2m+2} = 2<T_{m+1} L|T_{m+1} R> - mu_0 (MODE_MOMX)
    against the oracle's literal Alg. 2 + Alg. 5, and against the literal GPU path."""
    lat = sheet(40, 34, 90, True)           # 5350 sites: several tiles for every width
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    h.set_option(B.KG_OPT_STAGED, staged)
    phi = W.random_phase_vectors(lat.n, R, 12)
    nt, dt = 2, 0.8
    mu = host(B.vac(h, dev(phi), M, nt, dt))
    for r in sorted({0, R - 1}):
        want = kgo.vac(olat, olat.x, olat.period_x, 0.0, s, phi[:, r].copy(), M, nt, dt)
        assert relerr(mu[r], want) <= TOL
    h.set_option(B.KG_OPT_DOUBLING, 0)
    lit = host(B.vac(h, dev(phi), M, nt, dt))
    assert relerr(mu, lit) <= 1e-12


@pytest.mark.parametrize("R", [1, 8])
def test_guard_bands_and_inputs_untouched(B, R):
    """compute-sanitizer is closed on this pool, so out-of-bounds writes are looked for directly:
    every caller-owned array sits between canary bands, sizes leave a ragged last tile, and after
    each call the bands and the read-only inputs must be bit-identical to what they were."""
    import torch
    lat = sheet(33, 29, 61, True)                      # 3767 sites: ragged for both tile sizes
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, scale_for(lat))
    n, G = lat.n, 4096
    canary = complex(1.2345e300, -6.789e299)

    def guarded(shape_rows, cols):
        buf = torch.full((G + shape_rows * cols + G,), canary, dtype=torch.complex128, device="cuda")
        return buf, buf[G:G + shape_rows * cols].view(shape_rows, cols)

    def bands_ok(buf, rows, cols):
        return bool((buf[:G] == canary).all()) and bool((buf[G + rows * cols:] == canary).all())

    phi_np = W.random_phase_vectors(n, R, 2)
    pbuf, phi = guarded(n, R)
    phi.copy_(torch.from_numpy(phi_np))
    keep = phi.clone()
    M, nt = 37, 1
    obuf, out = guarded(n, R)
    B.evolve(h, phi, 0.8, out=out)
    xbuf, psix = guarded(n, R)
    psix.zero_()
    qbuf, psi = guarded(n, R)
    psi.copy_(phi)
    B.evolve_x(h, psi, psix, 0.8)
    vbuf, vout = guarded(n, R)
    B.apply_velocity(h, phi, out=vout)
    mbuf, mu = guarded(R, M)
    B.dos_moments(h, phi, M, mu=mu)
    cbuf, muv = guarded(R * (nt + 1), M)
    B.vac(h, phi, M, nt, 0.8, mu=muv.view(R, nt + 1, M))
    dbuf, mud = guarded(R * (nt + 1), M)
    B.msd(h, phi, M, nt, 0.8, mu=mud.view(R, nt + 1, M))
    fbuf, F = guarded(R, 7)
    B.fourier_moments(h, phi, phi, 3, 0.3, F=F)
    torch.cuda.synchronize()
    assert torch.equal(phi, keep)                                     # inputs never modified
    for buf, rows, cols in ((pbuf, n, R), (obuf, n, R), (xbuf, n, R), (qbuf, n, R), (vbuf, n, R),
                            (mbuf, R, M), (cbuf, R * (nt + 1), M), (dbuf, R * (nt + 1), M), (fbuf, R, 7)):
        assert bands_ok(buf, rows, cols)
    for t in (out, psi, psix, vout, mu, muv, mud, F):                  # and every output was written
        assert not bool((t == canary).any()) and bool(torch.isfinite(t.real).all())


def grid_lattice(shape, t=-1.0, a=0.3, seed=4, onsite_w=0.0):
    """Simple hyper-cubic tight-binding lattice (chain / square / cubic), periodic in every
    direction: kmax = 2 * dim neighbours per site in the paper's k-major list; x = first axis."""
    dims = tuple(shape)
    n = int(np.prod(dims))
    coords = np.stack(np.unravel_index(np.arange(n), dims), axis=0)
    nbrs = []
    for ax in range(len(dims)):
        for step in (+1, -1):
            c = coords.copy()
            c[ax] = (c[ax] + step) % dims[ax]
            nbrs.append(np.ravel_multi_index(tuple(c), dims))
    kmax = len(nbrs)
    nl = np.concatenate(nbrs).astype(np.int32)
    hop = np.full(kmax * n, t)
    ons = None
    if onsite_w:
        ons = onsite_w * (np.random.default_rng(seed).random(n) - 0.5)
    lat = W.Lattice(n, kmax, np.full(n, kmax, np.int32), nl, hop, ons, coords[0] * a,
                    np.zeros(n), dims[0] * a, 0.0)
    return lat


@pytest.mark.parametrize("shape", [(5000,), (90, 70), (22, 18, 16)])
@pytest.mark.parametrize("R", [1, 4])
def test_staged_other_row_widths(B, kgo, shape, R):
    """The staged kernels for K = 2, 4, 6 (chain, square, cubic Anderson models): moments with
    distinct and identical vectors, VAC, MSD, evolve against the oracle, and against the
    one-thread-per-element kernels."""
    lat = grid_lattice(shape, onsite_w=1.0)
    s = (lat.kmax * 1.0 + 0.5) * 1.05
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, R, 9)
    rng = np.random.default_rng(3)
    L = rng.normal(size=(lat.n, R)) + 1j * rng.normal(size=(lat.n, R))
    M, nt, dt = 30, 1, 0.9
    got = {"mom": host(B.moments(h, dev(L), dev(phi), M)), "dos": host(B.dos_moments(h, dev(phi), M)),
           "vac": host(B.vac(h, dev(phi), M, nt, dt)), "msd": host(B.msd(h, dev(phi), M, nt, dt)),
           "evo": host(B.evolve(h, dev(phi), dt))}
    r = R - 1
    v = phi[:, r].copy()
    assert relerr(got["mom"][r], kgo.moments(olat, 0.0, s, L[:, r].copy(), v, M)) <= TOL
    assert relerr(got["dos"][r], kgo.dos_moments(olat, 0.0, s, v, M)) <= TOL
    assert relerr(got["vac"][r], kgo.vac(olat, olat.x, olat.period_x, 0.0, s, v, M, nt, dt)) <= TOL
    assert relerr(got["msd"][r], kgo.msd(olat, olat.x, olat.period_x, 0.0, s, v, M, nt, dt)) <= TOL
    assert relerr(got["evo"][:, r], kgo.evolve(olat, 0.0, s, v, dt)) <= 1e-12
    l0 = h.launch_count
    h.set_option(B.KG_OPT_STAGED, 0)
    assert relerr(host(B.vac(h, dev(phi), M, nt, dt)), got["vac"]) <= 1e-12
    assert relerr(host(B.msd(h, dev(phi), M, nt, dt)), got["msd"]) <= 1e-12
    assert h.launch_count > l0


@pytest.mark.parametrize("R", [1, 8])
def test_vac_msd_bitwise_reproducible(B, R):
    """No atomics anywhere on the path: repeated kg_vac / kg_msd calls (cross-doubling shuffles,
    per-CTA partials, fixed-order final sum) give identical bits."""
    lat = sheet(70, 60, 200, True)          # 16 600 sites
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, scale_for(lat))
    phi = dev(W.random_phase_vectors(lat.n, R, 4))
    a = host(B.vac(h, phi, 50, 2, 0.8)); b = host(B.vac(h, phi, 50, 2, 0.8))
    c = host(B.msd(h, phi, 50, 2, 0.8)); d = host(B.msd(h, phi, 50, 2, 0.8))
    assert a.tobytes() == b.tobytes() and c.tobytes() == d.tobytes()


@pytest.mark.parametrize("R", [1, 2, 16])
@pytest.mark.parametrize("dt", [2.1, -0.6, 0.004])
def test_clenshaw_evolve(B, kgo, R, dt):
    """U(dt) phi by Clenshaw's backward recurrence (default) against the oracle's literal Alg. 6 and
    against the library's forward recursion + accumulation; E0 != 0 (global phase), both time
    directions, and a tiny dt whose series has fewer than 4 terms (falls back to Alg. 6)."""
    lat = sheet(60, 50, 100, True)                    # 11 900 sites
    e0 = 0.25
    s = scale_for(lat) + 0.3
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, e0, s)
    phi = W.random_phase_vectors(lat.n, R, 13)
    l0 = h.launch_count
    out = host(B.evolve(h, dev(phi), dt))
    n_p, _ = B.bessel_terms(s * abs(dt) / W.HBAR)
    assert h.launch_count - l0 == n_p - 1             # one sweep per term beyond the first
    assert relerr(out[:, R - 1], kgo.evolve(olat, e0, s, phi[:, R - 1].copy(), dt)) <= 1e-12
    h.set_option(B.KG_OPT_CLENSHAW, 0)
    fwd = host(B.evolve(h, dev(phi), dt))
    assert relerr(out, fwd) <= 1e-13
    back = host(B.evolve(h, dev(out), -dt))
    assert np.max(np.abs(back - phi)) < 1e-12         # U(-dt) U(dt) = 1


@pytest.mark.parametrize("R", [1, 8])
def test_clenshaw_pair(B, kgo, R):
    """Eq 44 by the Clenshaw form of the (b, e) pair recursion (default) against the oracle's literal
    Alg. 6 + Alg. 7 over two steps (non-zero psix on the second) and against the forward pair
    recursion; then MSD moments through it."""
    lat = sheet(60, 50, 100, True)
    s = scale_for(lat)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    phi = W.random_phase_vectors(lat.n, R, 17)
    dt = 1.9
    psi, psix = dev(phi), dev(np.zeros_like(phi))
    for _ in range(2):
        B.evolve_x(h, psi, psix, dt)
    r = R - 1
    wp, wx = phi[:, r].copy(), np.zeros(lat.n, complex)
    for _ in range(2):
        wx = kgo.evolve(olat, 0.0, s, wx, dt) + kgo.comm_evolve(olat, olat.x, olat.period_x, 0.0, s, wp, dt)
        wp = kgo.evolve(olat, 0.0, s, wp, dt)
    assert relerr(host(psi)[:, r], wp) <= 1e-12 and relerr(host(psix)[:, r], wx) <= 1e-12
    msd = host(B.msd(h, dev(phi), 24, 2, dt))
    h.set_option(B.KG_OPT_CLENSHAW, 0)
    p2, x2 = dev(phi), dev(np.zeros_like(phi))
    for _ in range(2):
        B.evolve_x(h, p2, x2, dt)
    assert relerr(host(psix), host(x2)) <= 1e-13 and relerr(host(psi), host(p2)) <= 1e-13
    assert relerr(msd, host(B.msd(h, dev(phi), 24, 2, dt))) <= 1e-12
    assert relerr(msd[r], kgo.msd(olat, olat.x, olat.period_x, 0.0, s, phi[:, r].copy(), 24, 2, dt)) <= TOL
