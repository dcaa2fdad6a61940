"""Pins of the CPU oracle (oracle/kgo.c) against things OTHER than itself: values the paper
prints (tests/golden/paper_values.txt), closed forms, invariants, textbook results and dense
exact diagonalisation (numpy.linalg) on lattices of <= 512 sites.  Chosen so that a plausible
mistake in any oracle function (dropped term, wrong sign or index, transposed / unconjugated
operand, wrong factor of 2, hbar or s) fails at least one test.  CPU only."""
import numpy as np
import pytest
import scipy.special

from helpers import HBAR, cheb_T, dense_h, golden, rand_state, relerr, ring

T = -2.7
A = 0.142
S_GRAPHENE = 3 * 2.7 * 1.05


def small_disordered(kgo, open_x=False):
    """6x5 cells (120 sites) with 8 vacancies and Anderson disorder: no symmetry left."""
    full = kgo.honeycomb(6, 5, periodic_x=not open_x, periodic_y=True)
    vac = kgo.vacancy_mask(full.n, 8, 11)
    lat = kgo.remove_sites(full, vac)
    lat.onsite = kgo.anderson(lat.n, 2.7, 5)
    return lat


def eig(lat):
    H = dense_h(lat)
    assert np.allclose(H, H.T)
    E, Vec = np.linalg.eigh(H)
    return H, E, Vec


def dense_U(E, Vec, dt):
    """exp(-i H dt / hbar) from the eigen-decomposition."""
    return (Vec * np.exp(-1j * E * dt / HBAR)) @ Vec.conj().T


def dense_Tn(E, Vec, n, e0, s):
    return (Vec * cheb_T(n, (E - e0) / s)) @ Vec.T


# ------------------------------------------------------------------ H apply / moments (O2, O3)
def test_apply_h_matches_dense(kgo):
    lat = small_disordered(kgo)
    H = dense_h(lat)
    phi = rand_state(lat.n, 0)
    e0, s = 0.3, 11.0
    want = (H @ phi - e0 * phi) / s
    assert relerr(kgo.apply_h(lat, e0, s, phi), want) < 1e-14


def test_mu0_is_one_and_mu1_is_expectation(kgo):
    lat = small_disordered(kgo)
    H = dense_h(lat)
    phi = rand_state(lat.n, 1)
    mu = kgo.dos_moments(lat, 0.0, 10.0, phi, 4)
    assert abs(mu[0] - 1.0) < 1e-14                       # normalised trace: mu_0 = 1
    assert abs(mu[1] - np.vdot(phi, H @ phi) / 10.0) < 1e-14
    assert np.max(np.abs(mu.imag)) < 1e-15                # <phi|T_n(H)|phi> is real


def test_full_trace_closed_forms_pristine(kgo):
    """Tr[T_2(H~)]/N = 2 z t^2/s^2 - 1 (z = 3); odd full-trace moments vanish on the bipartite
    lattice with no on-site terms (BASELINE north_star; reading g20: full trace)."""
    lat = kgo.honeycomb(4, 4)
    n, M = lat.n, 8
    tr = np.zeros(M, complex)
    for j in range(n):
        e = np.zeros(n, complex); e[j] = 1.0
        tr += kgo.dos_moments(lat, 0.0, S_GRAPHENE, e, M)
    tr /= n
    assert abs(tr[0] - 1.0) < 1e-15
    assert abs(tr[2] - (2 * 3 * T**2 / S_GRAPHENE**2 - 1)) < 1e-14
    assert abs(tr[2] - (-0.395313681028)) < 1e-11
    assert np.max(np.abs(tr[1::2])) < 1e-15
    # one-sublattice vector: odd moments exactly zero per vector
    phi = rand_state(n, 3); phi[1::2] = 0; phi /= np.linalg.norm(phi)
    mu = kgo.dos_moments(lat, 0.0, S_GRAPHENE, phi, M)
    assert np.max(np.abs(mu[1::2])) < 1e-16


def test_ring_trace_closed_form(kgo):
    """1-D ring, s = 2|t|: eigenvalues -cos(2 pi j/N) => Tr[T_n]/N = (-1)^n [N | n]."""
    n, M = 12, 30
    lat = ring(kgo, n)
    tr = np.zeros(M, complex)
    for j in range(n):
        e = np.zeros(n, complex); e[j] = 1.0
        tr += kgo.dos_moments(lat, 0.0, 2 * 2.7, e, M)
    tr /= n
    want = np.array([(-1.0) ** m if m % n == 0 else 0.0 for m in range(M)])
    assert np.max(np.abs(tr - want)) < 1e-13


def test_moments_vs_dense_diagonalisation(kgo):
    """mu_n = sum_j conj(<j|phi_L>) <j|phi_R> T_n((E_j-E0)/s) — pins the recursion, the
    scaling/shift, and the conjugation of the LEFT vector."""
    lat = small_disordered(kgo)
    _, E, Vec = eig(lat)
    e0, s = 0.2, (3 * 2.7 + 1.35 + 0.2) * 1.05
    assert np.max(np.abs(E - e0)) < s
    phiL, phiR = rand_state(lat.n, 4), rand_state(lat.n, 5)
    cL, cR = Vec.T @ phiL, Vec.T @ phiR
    M = 200
    want = np.array([np.sum(np.conj(cL) * cR * cheb_T(m, (E - e0) / s)) for m in range(M)])
    got = kgo.moments(lat, e0, s, phiL, phiR, M)
    assert relerr(got, want) < 1e-12
    got_dos = kgo.dos_moments(lat, e0, s, phiR, M)
    want_dos = np.array([np.sum(np.abs(cR) ** 2 * cheb_T(m, (E - e0) / s)) for m in range(M)])
    assert relerr(got_dos, want_dos) < 1e-12


# ------------------------------------------------------------------ Bessel (R4)
def test_bessel_truncation_matches_paper(kgo):
    val, tol = golden("np_at_pi")                          # "about 20" at argument pi, 1e-15
    eps = golden("bessel_accuracy")[0]
    np_pi = kgo.bessel_np(np.pi, eps)
    assert abs(np_pi - val) <= tol and np_pi == 21
    # the terms kept really are all those >= eps, scanning from above (reading g6)
    for x in (0.3, np.pi, 6.3, 14.7, 25.2, 80.0):
        n_p = kgo.bessel_np(x, eps)
        jv = scipy.special.jv(np.arange(n_p + 40), x)
        assert abs(jv[n_p - 1]) >= eps and np.all(np.abs(jv[n_p:]) < eps)
    assert abs(20 / np.pi - golden("kpm_vs_ftm_cost")[0]) < golden("kpm_vs_ftm_cost")[1]


def test_bessel_values(kgo):
    for x in (0.3, np.pi, 6.3, 14.7, 25.2):
        n_p = kgo.bessel_np(x)
        j = kgo.bessel_j(x, n_p)
        assert abs(j[0] ** 2 + 2 * np.sum(j[1:] ** 2) - 1.0) < 2e-15      # sum rule
        assert np.max(np.abs(j - scipy.special.jv(np.arange(n_p), x))) < 2e-15


# ------------------------------------------------------------------ evolution (O4)
@pytest.mark.parametrize("e0", [0.0, 0.4])
def test_evolve_vs_dense_expm(kgo, e0):
    lat = small_disordered(kgo)
    _, E, Vec = eig(lat)
    s = (3 * 2.7 + 1.35 + 0.4) * 1.05
    phi = rand_state(lat.n, 6)
    for dt in (0.25, -0.25, 1.7, -1.7):
        want = dense_U(E, Vec, dt) @ phi
        got = kgo.evolve(lat, e0, s, phi, dt)
        assert relerr(got, want) < 1e-12


def test_evolve_unitarity_and_reversibility(kgo):
    lat = small_disordered(kgo)
    s = (3 * 2.7 + 1.35) * 1.05
    phi = rand_state(lat.n, 7)
    dt = 4 * HBAR / 2.7
    psi = kgo.evolve(lat, 0.0, s, phi, dt)
    assert abs(np.linalg.norm(psi) - 1.0) < 1e-12                 # |U phi| = |phi| to 1e-12
    back = kgo.evolve(lat, 0.0, s, psi, -dt)
    assert np.max(np.abs(back - phi)) < 1e-12                     # U(-dt) U(dt) phi = phi
    assert np.max(np.abs(psi - phi)) > 0.1                        # and it did something


def test_infinite_chain_amplitude(kgo):
    """|<j|U(t)|0>| = |J_j(2|t| t/hbar)| on a chain long enough that wrap-around is negligible."""
    n = 400
    lat = ring(kgo, n)
    e = np.zeros(n, complex); e[0] = 1.0
    tt = 3.0
    psi = kgo.evolve(lat, 0.0, 2 * 2.7 * 1.05, e, tt)
    j = np.minimum(np.arange(n), n - np.arange(n))
    want = np.abs(scipy.special.jv(j, 2 * 2.7 * tt / HBAR))
    assert np.max(np.abs(np.abs(psi) - want)) < 1e-13


# ------------------------------------------------------------------ velocity (O2, a5)
def test_velocity_open_boundary_dense_commutator(kgo):
    """V = (i/hbar)[H, X] as dense matrices when X is single-valued (open along x)."""
    lat = small_disordered(kgo, open_x=True)
    H = dense_h(lat)
    X = np.diag(lat.x)
    V = (1j / HBAR) * (H @ X - X @ H)
    phi = rand_state(lat.n, 8)
    got = kgo.apply_velocity(lat, lat.x, 0.0, phi)
    assert relerr(got, V @ phi) < 1e-14
    # [X, H~]
    s = 9.7
    got = kgo.apply_xh(lat, lat.x, 0.0, s, phi)
    assert relerr(got, (X @ H - H @ X) @ phi / s) < 1e-14


def test_velocity_hermitian_and_trace(kgo):
    """<a|Vb> = <Va|b>; pristine Tr[V^2]/N = (3/2)(t a/hbar)^2 for either axis."""
    lat = kgo.honeycomb(4, 4)
    a, b = rand_state(lat.n, 9), rand_state(lat.n, 10)
    for xc, per in ((lat.x, lat.period_x), (lat.y, lat.period_y)):
        lhs = np.vdot(a, kgo.apply_velocity(lat, xc, per, b))
        rhs = np.vdot(kgo.apply_velocity(lat, xc, per, a), b)
        assert abs(lhs - rhs) < 1e-14
        tr = 0.0
        for j in range(lat.n):
            e = np.zeros(lat.n, complex); e[j] = 1.0
            tr += np.linalg.norm(kgo.apply_velocity(lat, xc, per, e)) ** 2
        assert abs(tr / lat.n - 1.5 * (T * A / HBAR) ** 2) < 1e-13
        assert abs(tr / lat.n - 0.508937) < 1e-6


def test_velocity_group_velocity_on_ring(kgo):
    """Plane wave on a periodic ring: V|k> = (1/hbar) dE/dk |k>, E = 2t cos(ka) — pins the sign
    and the minimum-image convention across the periodic boundary (reading g2)."""
    n = 16
    lat = ring(kgo, n)
    for jk in (1, 3, 5, 11):
        k = 2 * np.pi * jk / (n * A)
        pw = np.exp(1j * k * lat.x) / np.sqrt(n)
        vg = -2 * T * A * np.sin(k * A) / HBAR
        got = kgo.apply_velocity(lat, lat.x, lat.period_x, pw)
        assert np.max(np.abs(got - vg * pw)) < 1e-14


# ------------------------------------------------------------------ commutator evolution (O5)
@pytest.mark.parametrize("e0", [0.0, -0.3])
def test_comm_evolve_open_boundary_dense(kgo, e0):
    """[X, U(dt)] = X U - U X with the dense U (open along x)."""
    lat = small_disordered(kgo, open_x=True)
    _, E, Vec = eig(lat)
    s = (3 * 2.7 + 1.35 + 0.3) * 1.05
    X = np.diag(lat.x)
    phi = rand_state(lat.n, 12)
    for dt in (0.3, 2.1):
        U = dense_U(E, Vec, dt)
        want = (X @ U - U @ X) @ phi
        got = kgo.comm_evolve(lat, lat.x, 0.0, e0, s, phi, dt)
        assert relerr(got, want) < 1e-12


def test_comm_evolve_periodic_eigenbasis(kgo):
    """Under PBC: <a|[X,U(t)]|b> = <a|[X,H]|b> (e^{-iE_b t} - e^{-iE_a t})/(E_b - E_a) in the
    eigenbasis (degenerate pairs -> -(it/hbar) e^{-iE_a t/hbar}), with [X,H] the bond operator."""
    lat = small_disordered(kgo, open_x=False)
    H, E, Vec = eig(lat)
    n = lat.n
    # bond operator [X,H]_{im} = (x_i - x_m)_minimg H_im built from the dense H and coordinates
    dx = lat.x[:, None] - lat.x[None, :]
    dx -= lat.period_x * np.round(dx / lat.period_x)
    XH = dx * (H - np.diag(np.diag(H)))
    XHe = Vec.T @ XH @ Vec
    dt = 1.3
    ph = np.exp(-1j * E * dt / HBAR)
    dE = E[None, :] - E[:, None]                         # E_b - E_a, index [a, b]
    with np.errstate(divide="ignore", invalid="ignore"):
        F = (ph[None, :] - ph[:, None]) / dE
    deg = np.abs(dE) < 1e-9
    F[deg] = (-1j * dt / HBAR) * np.broadcast_to(ph[:, None], (n, n))[deg]
    XU = Vec @ (XHe * F) @ Vec.T
    phi = rand_state(n, 13)
    s = (3 * 2.7 + 1.35) * 1.05
    got = kgo.comm_evolve(lat, lat.x, lat.period_x, 0.0, s, phi, dt)
    assert relerr(got, XU @ phi) < 1e-11


def test_comm_evolve_plane_wave_ring(kgo):
    """Ring: [X,U(t)]|k> = (t/hbar) E'(k) e^{-iE_k t/hbar}|k>."""
    n = 20
    lat = ring(kgo, n)
    tt = 0.9
    for jk in (2, 7):
        k = 2 * np.pi * jk / (n * A)
        pw = np.exp(1j * k * lat.x) / np.sqrt(n)
        Ek = 2 * T * np.cos(k * A)
        dEk = -2 * T * A * np.sin(k * A)
        want = (tt / HBAR) * dEk * np.exp(-1j * Ek * tt / HBAR) * pw
        got = kgo.comm_evolve(lat, lat.x, lat.period_x, 0.0, 2 * 2.7 * 1.05, pw, tt)
        assert np.max(np.abs(got - want)) < 1e-13


# ------------------------------------------------------------------ VAC / MSD drivers (O7, O8)
def test_vac_vs_dense(kgo):
    """mu^VAC_n(t_k) = <V U^dag(t_k) phi | T_n(H~) | U^dag(t_k) V phi>  (eq 33)."""
    lat = small_disordered(kgo, open_x=True)
    H, E, Vec = eig(lat)
    s = (3 * 2.7 + 1.35) * 1.05
    X = np.diag(lat.x)
    V = (1j / HBAR) * (H @ X - X @ H)
    phi = rand_state(lat.n, 14)
    M, nt, dt = 24, 3, 0.7
    got = kgo.vac(lat, lat.x, 0.0, 0.0, s, phi, M, nt, dt)
    assert got.shape == (nt + 1, M)
    want = np.empty_like(got)
    for k in range(nt + 1):
        Ud = dense_U(E, Vec, -k * dt)
        L = V @ (Ud @ phi)
        R = Ud @ (V @ phi)
        for m in range(M):
            want[k, m] = np.vdot(L, dense_Tn(E, Vec, m, 0.0, s) @ R)
    assert relerr(got, want) < 1e-12
    # row 0 equals moments(V phi, V phi)
    vphi = kgo.apply_velocity(lat, lat.x, 0.0, phi)
    assert relerr(got[0], kgo.moments(lat, 0.0, s, vphi, vphi, M)) < 1e-15


def test_msd_vs_dense(kgo):
    """mu^MSD_n(t_k) = <psix_k|T_n(H~)|psix_k>, psix_k = [X, U(t_k)] phi = (X U^k - U^k X) phi
    (eq 34; eq 44 composition)."""
    lat = small_disordered(kgo, open_x=True)
    _, E, Vec = eig(lat)
    s = (3 * 2.7 + 1.35) * 1.05
    X = np.diag(lat.x)
    phi = rand_state(lat.n, 15)
    M, nt, dt = 24, 3, 0.7
    got = kgo.msd(lat, lat.x, 0.0, 0.0, s, phi, M, nt, dt)
    want = np.empty_like(got)
    for k in range(nt + 1):
        U = dense_U(E, Vec, k * dt)
        px = (X @ U - U @ X) @ phi
        for m in range(M):
            want[k, m] = np.vdot(px, dense_Tn(E, Vec, m, 0.0, s) @ px)
    assert np.all(got[0] == 0)                                        # row 0 is exactly 0
    assert relerr(got, want) < 1e-12
    assert np.max(np.abs(got.imag)) < 1e-12 * np.max(np.abs(got))


def test_vac_msd_ragged_schedule_vs_dense(kgo):
    """The branch of the VAC / MSD drivers that every stored output under tests/golden/ goes through
    (tests/golden/make_goldens.py): kgo_vac_sched / kgo_msd_sched with a NON-constant number of moments per
    time step — rows shorter than the row stride, and a row with no moments at all, where the states are
    only advanced.  Pinned (a) directly on the dense formulas, eq 33 and eq 34 + eq 44 composition,
    row by row at the scheduled lengths — so a wrong row stride, a row written to the wrong place or an
    evolution dropped on the skipped row fails here without reference to any other oracle routine; (b) on
    the constant-schedule drivers: a Chebyshev moment does not depend on how many are asked for, so every
    scheduled row is bit for bit the head of the full row; (c) entries behind a row's length stay 0."""
    lat = small_disordered(kgo, open_x=True)
    H, E, Vec = eig(lat)
    s = (3 * 2.7 + 1.35) * 1.05
    X = np.diag(lat.x)
    V = (1j / HBAR) * (H @ X - X @ H)
    phi = rand_state(lat.n, 21)
    dt = 0.7
    Mk = np.array([24, 5, 0, 7, 24], np.int32)
    nt, ld = len(Mk) - 1, int(Mk.max())
    Tn = [dense_Tn(E, Vec, m, 0.0, s) for m in range(ld)]
    got_v = kgo.vac_sched(lat, lat.x, 0.0, 0.0, s, phi, Mk, dt)
    got_m = kgo.msd_sched(lat, lat.x, 0.0, 0.0, s, phi, Mk, dt)
    assert got_v.shape == (nt + 1, ld) and got_m.shape == (nt + 1, ld)
    full_v = kgo.vac(lat, lat.x, 0.0, 0.0, s, phi, ld, nt, dt)
    full_m = kgo.msd(lat, lat.x, 0.0, 0.0, s, phi, ld, nt, dt)
    for k in range(nt + 1):
        Ud = dense_U(E, Vec, -k * dt)
        L, R = V @ (Ud @ phi), Ud @ (V @ phi)
        U = dense_U(E, Vec, k * dt)
        px = (X @ U - U @ X) @ phi
        want_v = np.array([np.vdot(L, Tn[m] @ R) for m in range(Mk[k])])
        want_m = np.array([np.vdot(px, Tn[m] @ px) for m in range(Mk[k])])
        if Mk[k]:
            assert relerr(got_v[k, :Mk[k]], want_v) < 1e-12, k                       # (a)
            if k:
                assert relerr(got_m[k, :Mk[k]], want_m) < 1e-12, k
        assert got_v[k, :Mk[k]].tobytes() == full_v[k, :Mk[k]].tobytes(), k          # (b)
        assert got_m[k, :Mk[k]].tobytes() == full_m[k, :Mk[k]].tobytes(), k
        assert np.all(got_v[k, Mk[k]:] == 0) and np.all(got_m[k, Mk[k]:] == 0)       # (c)
    assert np.all(got_m[0] == 0)
    # a schedule that skips the FIRST row and keeps one moment on the last (row stride 1)
    one = kgo.vac_sched(lat, lat.x, 0.0, 0.0, s, phi, np.array([0, 0, 1], np.int32), dt)
    assert one.shape == (3, 1) and one[0, 0] == 0 and one[1, 0] == 0
    Ud = dense_U(E, Vec, -2 * dt)
    assert abs(one[2, 0] - np.vdot(V @ (Ud @ phi), Ud @ (V @ phi))) < 1e-12 * abs(one[2, 0])


def test_ring_vac_constant_msd_quadratic(kgo):
    """1-D ring: [V,H] = 0 => mu^VAC_n(t) independent of t and mu^MSD_n(t) = t^2 <V phi|T_n|V phi>
    per vector, exactly."""
    n = 64
    lat = ring(kgo, n)
    s = 2 * 2.7 * 1.05
    phi = rand_state(n, 16)
    M, nt, dt = 16, 4, 0.5
    v = kgo.vac(lat, lat.x, lat.period_x, 0.0, s, phi, M, nt, dt)
    m = kgo.msd(lat, lat.x, lat.period_x, 0.0, s, phi, M, nt, dt)
    vphi = kgo.apply_velocity(lat, lat.x, lat.period_x, phi)
    base = kgo.moments(lat, 0.0, s, vphi, vphi, M)
    for k in range(nt + 1):
        assert relerr(v[k], base) < 1e-12
        assert np.max(np.abs(m[k] - (k * dt) ** 2 * base)) < 1e-12 * max(1.0, (k * dt) ** 2) * np.max(np.abs(base))


def test_msd_small_time_limit(kgo):
    """mu^MSD_0(t) = |psix|^2 -> <phi|V^2|phi> t^2 as t -> 0."""
    lat = kgo.honeycomb(4, 4)
    phi = rand_state(lat.n, 17)
    dt = 1e-3
    m = kgo.msd(lat, lat.x, lat.period_x, 0.0, S_GRAPHENE, phi, 2, 1, dt)
    v2 = np.linalg.norm(kgo.apply_velocity(lat, lat.x, lat.period_x, phi)) ** 2
    assert abs(m[1, 0].real / dt**2 - v2) < 1e-4 * v2


# ------------------------------------------------------------------ reconstruction (O9)
def test_reconstruct_single_moments(kgo):
    """mu = delta_{n0} -> 1/(pi s sqrt(1-E~^2)); mu = delta_{n1} -> 2 g_1 E~ /(pi s sqrt(1-E~^2)):
    pins the prefactor, the (2 - delta_n0) factor and T_n; g_0 = 1."""
    M, s, e0 = 16, 8.5, 0.1
    en = np.linspace(-7, 7, 29)
    et = (en - e0) / s
    g = kgo.jackson(M)
    assert abs(g[0] - 1.0) < 1e-15
    mu = np.zeros(M, complex); mu[0] = 1
    assert relerr(kgo.kpm_reconstruct(mu, e0, s, en), 1 / (np.pi * s * np.sqrt(1 - et**2))) < 1e-14
    mu = np.zeros(M, complex); mu[1] = 1
    assert relerr(kgo.kpm_reconstruct(mu, e0, s, en), 2 * g[1] * et / (np.pi * s * np.sqrt(1 - et**2))) < 1e-14
    mu = np.zeros(M, complex); mu[5] = 1j                       # only Re mu enters (reading g12)
    assert np.max(np.abs(kgo.kpm_reconstruct(mu, e0, s, en))) == 0.0


def test_jackson_kernel_positive_normalised_narrow(kgo):
    """Jackson-damped delta: positive everywhere, integrates to 1, width ~ pi s/M; the undamped
    (Dirichlet) kernel is not positive — a wrong alpha or a dropped term breaks positivity."""
    M, s = 64, 1.0
    y = 0.3
    mu = cheb_T(np.arange(M), y).astype(complex)
    # Chebyshev-Gauss nodes: integral f dE = (pi/K) sum sqrt(1-x_k^2) f(x_k)
    K = 4096
    xk = np.cos(np.pi * (np.arange(K) + 0.5) / K)
    f = kgo.kpm_reconstruct(mu, 0.0, s, xk)
    w = np.pi / K * np.sqrt(1 - xk**2)
    assert f.min() > -1e-12
    assert abs(np.sum(w * f) - 1.0) < 1e-12
    mean = np.sum(w * f * xk)
    sig = np.sqrt(np.sum(w * f * (xk - mean) ** 2))
    assert 0.8 < sig / (np.pi / M * np.sqrt(1 - y**2)) < 1.2
    f_raw = kgo.kpm_reconstruct(mu, 0.0, s, xk, use_jackson=False)
    assert f_raw.min() < -0.1
    g = kgo.jackson(M)
    assert np.all(np.diff(g) < 0) and 0 < g[-1] < 0.01


def graphene_dos_closed_form(E, t=2.7):
    """Hobson-Nierenberg closed form, per site (integrates to 1): rho(E) =
    (1/pi^2)(|E|/t^2) K(Z1/Z0)/sqrt(Z0), Z0=(1+e)^2-(e^2-1)^2/4, Z1=4e for e=|E/t|<=1, swapped for
    1<=e<=3; K = complete elliptic integral with PARAMETER m (scipy convention)."""
    e = np.abs(E) / t
    z0 = (1 + e) ** 2 - (e**2 - 1) ** 2 / 4
    z1 = 4 * e
    lo = e <= 1
    Z0 = np.where(lo, z0, z1)
    Z1 = np.where(lo, z1, z0)
    out = (1 / np.pi**2) * (np.abs(E) / t**2) * scipy.special.ellipk(Z1 / Z0) / np.sqrt(Z0)
    return np.where(e < 3, out, 0.0)


def test_pristine_graphene_dos_closed_form(kgo):
    """DOS from oracle moments of random-phase vectors on a 48x48-cell sheet against the
    closed form, away from the van Hove points |E| = |t| and from E = 0 / band edges, within the
    Jackson width pi s/M and the stochastic error ~ 1/sqrt(N)."""
    lat = kgo.honeycomb(48, 48)
    n = lat.n
    M, nvec = 96, 6
    mu = np.zeros(M, complex)
    for r in range(nvec):                                       # average of 6 random-phase vectors
        u = kgo.phase_uniforms(n, 0, r)
        phi = np.exp(2j * np.pi * u) / np.sqrt(n)
        mu_r = kgo.dos_moments(lat, 0.0, S_GRAPHENE, phi, M)
        assert abs(mu_r[0] - 1) < 1e-13
        assert np.max(np.abs(mu_r[1::2])) < 6 / np.sqrt(n)      # statistical, reading g20
        mu += mu_r / nvec
    en = np.concatenate([np.linspace(-7.0, -3.6, 12), np.linspace(-1.9, -0.9, 8),
                         np.linspace(0.9, 1.9, 8), np.linspace(3.6, 7.0, 12)])
    rho = kgo.kpm_reconstruct(mu, 0.0, S_GRAPHENE, en)
    ref = graphene_dos_closed_form(en)
    # closed form integrates to 1 (checks the fixture itself)
    g = np.linspace(-8.1, 8.1, 200001)
    assert abs(np.trapezoid(graphene_dos_closed_form(g), g) - 1.0) < 2e-3
    assert np.max(np.abs(rho - ref) / ref) < 0.12
    assert abs(np.mean((rho - ref) / ref)) < 0.03
    # integral of the reconstructed DOS is mu_0 = 1
    K = 2048
    xk = np.cos(np.pi * (np.arange(K) + 0.5) / K)
    f = kgo.kpm_reconstruct(mu, 0.0, S_GRAPHENE, xk * S_GRAPHENE)
    assert abs(np.sum(np.pi / K * np.sqrt(1 - xk**2) * f) * S_GRAPHENE - 1.0) < 1e-12


# ------------------------------------------------------------------ transport post-processing (O10)
def _chain_closed_forms(en, t=2.7, a=0.142):
    """Infinite 1-D chain, per site and spin: rho~ = 1/(pi sqrt(4t^2 - E^2)); E = 2t cos(ka),
    v = (2ta/hbar) sin(ka) => v^2(E) = (a/hbar)^2 (4t^2 - E^2).  Textbook results."""
    root = np.sqrt(4 * t * t - en ** 2)
    return 1.0 / (np.pi * root), (a / HBAR) ** 2 * root ** 2


def test_transport_ballistic_closed_forms(kgo):
    """Ballistic inputs rho~ v^2 (VAC) and rho~ v^2 t^2 (MSD) of the 1-D chain: sigma_GK = sigma_E1
    (P:532), sigma_E2 = sigma_E1 / 2, L = 2 v t (eq 50), and the Landauer value: one open
    channel, G = 2e^2/h = 2 in units of e^2/h, at every energy in the band and every t > 0 (eq 51,
    52).  A wrong prefactor, a dropped 1/2, a first-order end-point derivative or a wrong
    trapezoid weight breaks one of these."""
    a, nt, dt = 0.142, 7, 0.37
    en = np.linspace(-5.0, 5.0, 41)
    rho, v2 = _chain_closed_forms(en, a=a)
    tk = dt * np.arange(nt + 1)[:, None]
    fvac = np.broadcast_to(rho * v2, (nt + 1, en.size)).copy()
    fmsd = rho * v2 * tk ** 2
    width = 1.0                                   # strip of width 1 nm: Omega = W N a, dens = 2N/Omega
    out = kgo.transport(rho, fvac, fmsd, dt, 2.0 / (a * width), width)
    assert relerr(out["sigma_e1"], out["sigma_gk"]) < 1e-13
    assert relerr(out["sigma_e2"][1:], 0.5 * out["sigma_e1"][1:]) < 1e-13
    assert np.all(out["sigma_e2"][0] == 0)
    assert relerr(out["length_nm"], 2 * np.sqrt(v2) * tk) < 1e-13
    assert np.max(np.abs(out["conductance"][1:] - 2.0)) < 1e-12
    assert np.all(out["conductance"][0] == 0)
    # absolute value of sigma: 2 pi hbar dens rho~ v^2 t
    assert relerr(out["sigma_gk"], 2 * np.pi * HBAR * (2.0 / a) * rho * v2 * tk) < 1e-13


def test_transport_diffusive_and_quadrature(kgo):
    """Diffusive MSD 2 D t: sigma_E1 = sigma_E2 = 2 pi hbar dens rho D, independent of t; and the
    Green-Kubo integral of an exponentially decaying VAC within the trapezoid error bound."""
    nt, dt, dens, D, tau = 40, 0.05, 38.2, 0.6, 0.9
    rho = np.array([0.01, 0.05, 0.11])
    tk = dt * np.arange(nt + 1)[:, None]
    out = kgo.transport(rho, None, rho * 2 * D * tk, dt, dens)
    want = 2 * np.pi * HBAR * dens * rho * D
    assert out["sigma_gk"] is None
    assert relerr(out["sigma_e1"], np.broadcast_to(want, (nt + 1, 3))) < 1e-12
    assert relerr(out["sigma_e2"][1:], np.broadcast_to(want, (nt, 3))) < 1e-12
    fvac = rho * (D / tau) * np.exp(-tk / tau)
    gk = kgo.transport(rho, fvac, None, dt, dens)["sigma_gk"]
    exact = 2 * np.pi * HBAR * dens * rho * D * (1 - np.exp(-tk / tau))
    bound = 2 * np.pi * HBAR * dens * rho * (D / tau ** 3) * dt ** 2 / 12 * tk      # |f''| t dt^2 / 12
    assert np.all(np.abs(gk - exact) <= bound + 1e-15)
    assert np.max(np.abs(gk - exact)) > 0                                            # really a quadrature


def test_transport_end_to_end_ring_conductance(kgo):
    """The whole Einstein chain of the oracle on a pristine ring (Alg. 3 -> eq 31 -> eqs 9, 50, 51):
    one ballistic channel, G = 1 in units of 2e^2/h inside the band (P:515-524 plateaus)."""
    n, t, a = 3000, 2.7, 0.142
    lat = ring(kgo, n, -t, a)
    s = 2 * t * 1.05
    # a state on one site: on the translation-invariant ring <0|A delta(E-H) A|0> = Tr[...]/N
    # exactly, so there is no stochastic error, only the Jackson broadening pi s/M = 0.11 eV
    phi = np.zeros(n, complex); phi[0] = 1.0
    M, nt, dt = 160, 6, 2 * HBAR / t
    en = np.linspace(-1.5 * t, 1.5 * t, 31)
    rho = kgo.kpm_reconstruct(kgo.dos_moments(lat, 0.0, s, phi, M), 0.0, s, en)
    mu = kgo.msd(lat, lat.x, lat.period_x, 0.0, s, phi, M, nt, dt)
    fmsd = np.stack([kgo.kpm_reconstruct(mu[k], 0.0, s, en) for k in range(nt + 1)])
    out = kgo.transport(rho, None, fmsd, dt, 2.0 / a, 1.0)
    g = out["conductance"][1:] / 2.0                      # in 2e^2/h
    print("ring conductance / (2e^2/h): mean %.6f, max dev %.2e" % (np.mean(g), np.max(np.abs(g - 1.0))))
    assert abs(np.mean(g) - 1.0) < 5e-4
    assert np.max(np.abs(g - 1.0)) < 1e-3


# ------------------------------------------------------------------ Fourier-transform method (O11, O12)
@pytest.mark.parametrize("e0", [0.0, 0.3])
def test_fourier_moments_vs_dense(kgo, e0):
    """Alg. 4: F_n = sum_j conj(<j|phi_L>) <j|phi_R> exp(-i E_j n dtau/hbar), n = -Nm..Nm, from the
    dense eigen-decomposition: pins the direction of time for +n / -n, the storage order, the
    conjugated LEFT vector and the repeated application of U(dtau)."""
    lat = small_disordered(kgo)
    _, E, Vec = eig(lat)
    s = (3 * 2.7 + 1.35 + abs(e0)) * 1.05
    phiL, phiR = rand_state(lat.n, 14), rand_state(lat.n, 15)
    cL, cR = Vec.T @ phiL, Vec.T @ phiR
    Nm, dtau = 9, 0.21
    nn_ = np.arange(-Nm, Nm + 1)
    want = np.array([np.sum(np.conj(cL) * cR * np.exp(-1j * E * m * dtau / HBAR)) for m in nn_])
    got = kgo.fourier_moments(lat, e0, s, phiL, phiR, Nm, dtau)
    assert relerr(got, want) < 1e-12
    same = kgo.fourier_moments(lat, e0, s, phiR, phiR, Nm, dtau)
    assert np.max(np.abs(same[::-1] - np.conj(same))) < 1e-13          # F_{-n} = conj(F_n) if L = R
    assert abs(same[Nm] - 1.0) < 1e-14


def test_ftm_reconstruct_closed_forms(kgo):
    """eqs 22-24 + Hanning window eq 28 on a single level E_a (F_n = exp(-i E_a n dtau/hbar)):
    without window the Dirichlet kernel dtau/(2 pi hbar) sin((2Nm+1)x/2)/sin(x/2),
    x = (E-E_a) dtau/hbar; with the window the peak value dtau (Nm+1)/(2 pi hbar) (sum of w_n);
    and the integral over one period 2 pi hbar/dtau is w_0 F_0 = 1 in both cases."""
    Nm, dtau, Ea = 12, 0.35, 0.8
    nn_ = np.arange(-Nm, Nm + 1)
    F = np.exp(-1j * Ea * nn_ * dtau / HBAR)
    period = 2 * np.pi * HBAR / dtau
    en = Ea + np.linspace(-0.5, 0.5, 400, endpoint=False) * period + 1e-3
    x = (en - Ea) * dtau / HBAR
    plain = kgo.ftm_reconstruct(F, dtau, en, use_window=False)
    assert relerr(plain, dtau / (2 * np.pi * HBAR) * np.sin((2 * Nm + 1) * x / 2) / np.sin(x / 2)) < 1e-12
    win = kgo.ftm_reconstruct(F, dtau, en, use_window=True)
    peak = kgo.ftm_reconstruct(F, dtau, np.array([Ea]), use_window=True)[0]
    assert abs(peak - dtau * (Nm + 1) / (2 * np.pi * HBAR)) < 1e-13
    assert abs(np.min(win) / peak + 10 ** (-31.5 / 20)) < 1e-3          # Hann window: highest side lobe -31.5 dB (textbook)
    assert np.min(plain) < -0.15 * np.max(plain)                        # Dirichlet: first side lobe -21 %
    for f in (plain, win):                                              # uniform grid over one period:
        assert abs(np.sum(f) * period / en.size - 1.0) < 1e-12          # exact for trig polynomials


def test_ftm_and_kpm_dos_agree(kgo):
    """The paper's own validation (Fig. 2): DOS of a disordered sheet by the FTM and by the
    KPM from the same random vector, at a matched, coarse resolution; and both against the exact
    levels broadened by the FTM window (dense diagonalisation)."""
    full = kgo.honeycomb(8, 8)
    lat = kgo.remove_sites(full, kgo.vacancy_mask(full.n, 6, 2))
    s = S_GRAPHENE
    _, E, Vec = eig(lat)
    phi = rand_state(lat.n, 21)
    dtau = np.pi * HBAR / s                                             # Delta tau = pi hbar / (Delta E / 2)
    Nm = 40
    en = np.linspace(-7.5, 7.5, 151)
    F = kgo.fourier_moments(lat, 0.0, s, phi, phi, Nm, dtau)
    ftm = kgo.ftm_reconstruct(F, dtau, en)
    # exact: sum_j |<j|phi>|^2 K(E - E_j), K = the windowed kernel of a single level
    c2 = np.abs(Vec.T @ phi) ** 2
    nn_ = np.arange(-Nm, Nm + 1)
    w = 0.5 * (1 + np.cos(np.pi * nn_ / (Nm + 1)))
    K = lambda d: dtau / (2 * np.pi * HBAR) * np.sum(w * np.cos(np.outer(d, nn_) * dtau / HBAR), axis=1)
    exact = np.array([np.sum(c2 * K(e - E)) for e in en])
    assert relerr(ftm, exact) < 1e-11
    # KPM (Jackson, energy-dependent width) and FTM (Hanning, uniform width) broaden differently, so
    # they are compared where broadening drops out: the integrated DOS N(E) = int^E rho dE'
    fine = np.linspace(-8.4, 8.4, 841)
    de = fine[1] - fine[0]
    n_ftm = np.cumsum(kgo.ftm_reconstruct(F, dtau, fine)) * de
    n_kpm = np.cumsum(kgo.kpm_reconstruct(kgo.dos_moments(lat, 0.0, s, phi, 3 * Nm), 0.0, s, fine)) * de
    assert abs(n_ftm[-1] - 1.0) < 1e-3 and abs(n_kpm[-1] - 1.0) < 1e-3
    assert np.max(np.abs(n_kpm - n_ftm)) < 0.01


def test_open_boundary_length_saturates_at_sample_length(kgo):
    """Fig. 3: with a non-periodic boundary along the transport direction the length
    L(E,t) = 2 sqrt(DeltaX^2) (eq 50) is confined by the sample — "the maximum diffusion length ...
    being the length of the sample" — while with periodic boundaries it keeps growing ballistically.
    Pristine sheet 24 x 6 cells, L_x = 24 sqrt(3) a = 5.90 nm, site-localised start in the middle
    so that no stochastic error enters."""
    ncx, ncy = 24, 6
    Lx = ncx * np.sqrt(3.0) * A
    s, M, nt, dt = S_GRAPHENE, 48, 14, 4 * HBAR / 2.7
    en = np.linspace(-2.0, 2.0, 9)
    en = en[np.abs(en) > 0.4]
    lengths = {}
    for periodic in (False, True):
        lat = kgo.honeycomb(ncx, ncy, periodic_x=periodic, periodic_y=True)
        assert abs((lat.period_x if periodic else Lx) - Lx) < 1e-12
        phi = np.zeros(lat.n, complex)
        phi[4 * (3 * ncx + ncx // 2)] = 1.0
        rho = kgo.kpm_reconstruct(kgo.dos_moments(lat, 0.0, s, phi, M), 0.0, s, en)
        mu = kgo.msd(lat, lat.x, lat.period_x if periodic else 0.0, 0.0, s, phi, M, nt, dt)
        fmsd = np.stack([kgo.kpm_reconstruct(mu[k], 0.0, s, en) for k in range(nt + 1)])
        lengths[periodic] = kgo.transport(rho, None, fmsd, dt, 1.0)["length_nm"]
    open_, pbc = lengths[False], lengths[True]
    # early times: identical (the wave has not reached the edges yet)
    assert np.max(np.abs(open_[1] - pbc[1])) < 1e-6 * np.max(pbc[1])
    # late times: confined vs ballistic
    assert np.max(open_) < 1.05 * Lx
    assert np.max(open_[-4:]) > 0.6 * Lx
    assert np.min(pbc[-1]) > 1.5 * Lx
    assert np.all(np.diff(pbc.mean(axis=1)) > 0)


# ------------------------------------------------------------------ zigzag ribbon (Fig. 4)
def zgnr_bands(chains, nk=256):
    """Bloch bands of a zigzag ribbon of `chains` zigzag chains from its textbook tight-binding strip
    Hamiltonian (independent of any generator): 2*chains sites per unit cell; inside a chain the two
    sublattice sites couple with t (1 + e^{-ik}), neighbouring chains couple with t through one bond."""
    ks = np.linspace(-np.pi, np.pi, nk, endpoint=False)
    n = 2 * chains
    out = np.empty((nk, n))
    for q, k in enumerate(ks):
        h = np.zeros((n, n), complex)
        for c in range(chains):
            h[2 * c, 2 * c + 1] = T * (1 + np.exp(-1j * k))
            if c + 1 < chains:
                h[2 * c + 1, 2 * c + 2] = T
        h = h + h.conj().T
        out[q] = np.linalg.eigvalsh(h)
    return ks, out


def test_zgnr_flat_edge_band(kgo):
    """ZGNR of 16 chains x 16 cells = 512 sites: the zero-energy edge band.  Textbook (Fujita et al.;
    the flat band the paper's Fig. 4 b shows as the DOS peak at E = 0): edge states exist for
    2 pi/3 < |k| <= pi, one per edge and k.  With 16 k-points that is 5 k-points x 2 edges = 10 states
    within 0.1 eV of zero.  Checked (i) on the dense spectrum of the generated lattice, (ii) against the
    strip Hamiltonian's bands, (iii) as the weight of the E = 0 peak in the oracle's KPM DOS."""
    ncx, chains = 16, 16
    lat = kgo.zgnr(ncx, chains)
    assert lat.n == 512
    _, E, _ = eig(lat)
    k_edge = [j for j in range(-ncx // 2, ncx // 2) if abs(2 * np.pi * j / ncx) > 2 * np.pi / 3]
    want = 2 * len(k_edge)
    assert want == 10
    assert np.sum(np.abs(E) < 0.1) == want
    # the same levels from the strip Hamiltonian at the ribbon's allowed k
    ks, bands = zgnr_bands(chains, nk=ncx)
    assert np.max(np.abs(np.sort(bands.ravel()) - E)) < 1e-10
    # oracle: full trace of T_n over unit vectors -> rho(E); weight of the peak at E = 0
    M, s = 1200, S_GRAPHENE
    mu = np.zeros(M)
    for i in range(0, lat.n, 1):
        if i % (2 * chains) >= 2 * chains:      # (all sites; translation symmetry is not assumed)
            continue
        phi = np.zeros(lat.n, complex); phi[i] = 1.0
        mu += kgo.dos_moments(lat, 0.0, s, phi, M).real
    mu /= lat.n
    assert relerr(mu, np.array([np.mean(cheb_T(m, E / s)) for m in range(M)])) < 1e-11
    en = np.linspace(-0.1, 0.1, 401)
    rho = kgo.kpm_reconstruct(mu.astype(complex), 0.0, s, en)
    weight = np.trapezoid(rho, en)
    # Jackson width pi s / M = 0.022 eV: the ten levels (|E| <= 0.037 eV) sit well inside the window
    assert abs(weight * lat.n - want) < 0.5


def test_zgnr_first_plateau_conductance(kgo):
    """Ballistic conductance of the pristine ZGNR on its first plateau (Fig. 4 a): one open
    channel for 0 < |E| < E_1, so G -> 1 x 2e^2/h "within a short correlation time" (once the t^2 term of
    DeltaX^2 dominates the bounded inter-band oscillations), from the oracle's Einstein chain kgo_msd ->
    kgo_kpm_reconstruct -> kgo_transport.  The trace is exact: the ribbon is translation invariant along
    x, so the average over the 32 sites of one unit cell of site-localised states IS Tr[...]/N."""
    chains, ncx = 16, 320
    lat = kgo.zgnr(ncx, chains)
    _, bands = zgnr_bands(chains, nk=400)
    # bottom of the second conduction subband: between the edge band and it there is a single band
    pos = np.sort(bands, axis=1)[:, chains:]                  # conduction bands, ascending per k
    e1 = pos[:, 1].min()
    assert 0.5 < e1 < 1.2
    en = np.array([0.5 * e1, 0.7 * e1])
    en = np.concatenate([-en[::-1], en])
    s, M, nt, dt = S_GRAPHENE, 500, 12, 8 * HBAR / 2.7
    cell = [i for i in range(lat.n) if lat.x[i] < lat.x.min() + 0.2]       # the two x-columns of one unit cell
    assert len(cell) == 2 * chains
    rho = np.zeros(len(en)); fmsd = np.zeros((nt + 1, len(en)))
    for i in cell:
        phi = np.zeros(lat.n, complex); phi[i] = 1.0
        rho += kgo.kpm_reconstruct(kgo.dos_moments(lat, 0.0, s, phi, M), 0.0, s, en)
        mu = kgo.msd(lat, lat.x, lat.period_x, 0.0, s, phi, M, nt, dt)
        fmsd += np.stack([kgo.kpm_reconstruct(mu[k], 0.0, s, en) for k in range(nt + 1)])
    rho /= len(cell); fmsd /= len(cell)
    out = kgo.transport(rho, None, fmsd, dt, 2.0 * lat.n / lat.period_x, 1.0)
    g = out["conductance"] / 2.0                               # in 2e^2/h
    assert 2 * np.sqrt(np.max(fmsd[-1] / rho)) < 0.45 * lat.period_x       # the wave packet has not wrapped around
    print("ZGNR first plateau G/(2e^2/h) at t_k, k = 6, 9, 12:", np.round(g[[6, 9, 12]], 4))
    assert np.max(np.abs(g[6:] - 1.0)) < 0.05


# ------------------------------------------------------------------ local density of states
def test_ldos_vacancy_zero_mode(kgo):
    """Local DOS from unit vectors on 8 x 8 cells with ONE vacancy (255 sites).  Textbook: on a
    bipartite lattice with N_B = N_A + 1 there is exactly one zero-energy state and it lives on the
    majority sublattice.  The oracle's moments for |i> equal sum_j |<j|i>|^2 T_n(E_j/s) from the dense
    spectrum, and the weight of its KPM local DOS around E = 0 is the zero mode's |<0|i>|^2: large on a
    neighbour of the vacancy, exactly zero on the minority sublattice."""
    full = kgo.honeycomb(8, 8)
    vac = np.zeros(full.n, np.uint8); vac[4 * (3 * 8 + 3) + 0] = 1            # one A-type site (basis b0)
    lat = kgo.remove_sites(full, vac)
    _, E, Vec = eig(lat)
    assert np.sum(np.abs(E) < 1e-9) == 1
    zero = Vec[:, np.argmin(np.abs(E))]
    gap = np.sort(np.abs(E))[1]
    assert gap > 0.3                                                          # the finite sheet's other levels are far away
    s, M = S_GRAPHENE, 600                                                    # Jackson width pi s / M = 0.045 eV << gap
    nbr = int(np.argmax(np.abs(zero)))                                        # strongest site: next to the vacancy
    assert lat.nn[nbr] == 2
    # a site of the minority sublattice: bipartite => the zero mode vanishes there
    minority = [i for i in range(lat.n) if abs(zero[i]) < 1e-12]
    assert len(minority) == 127
    en = np.linspace(-0.25, 0.25, 501)
    for site, w in ((nbr, zero[nbr] ** 2), (minority[5], 0.0)):
        phi = np.zeros(lat.n, complex); phi[site] = 1.0
        mu = kgo.dos_moments(lat, 0.0, s, phi, M)
        want = np.array([np.sum(Vec[site] ** 2 * cheb_T(m, E / s)) for m in range(M)])
        assert relerr(mu, want) < 1e-12
        weight = np.trapezoid(kgo.kpm_reconstruct(mu, 0.0, s, en), en)
        assert abs(weight - w) < 2e-3
    assert zero[nbr] ** 2 > 0.1


# ------------------------------------------------------------------ next-nearest-neighbour model
def test_nnn_graphene_bands(kgo):
    """Denser Hamiltonian (row width 9): the dense spectrum of the generated next-nearest-neighbour torus
    equals the textbook bands E(k) = t' f(k) +- |t| sqrt(3 + f(k)), f = 2 [cos k.a1 + cos k.a2 + cos k.(a2-a1)]
    (Wallace 1947; Castro Neto et al. RMP 2009 eq 6) on the allowed k, and the oracle's full-trace moments with
    E0 = 3 t' != 0 (the Dirac-point energy) equal the moments of that spectrum."""
    ncx, ncy, t, t2 = 6, 4, -2.7, -0.27
    lat = kgo.honeycomb_nnn(ncx, ncy, t_eV=t, t2_eV=t2)
    _, E, _ = eig(lat)
    h = np.sqrt(3) * A / 2
    a1, a2 = np.array([2 * h, 0.0]), np.array([h, 1.5 * A])
    vals = []
    for p in range(ncx):
        for q in range(ncy):
            for bz in range(2):
                k = np.array([2 * np.pi * p / (ncx * 2 * h), 2 * np.pi * q / (ncy * 3 * A) + bz * 2 * np.pi / (3 * A)])
                f = 2 * (np.cos(k @ a1) + np.cos(k @ a2) + np.cos(k @ (a2 - a1)))
                root = abs(t) * np.sqrt(max(3 + f, 0.0))
                vals += [t2 * f + root, t2 * f - root]
    assert np.max(np.abs(np.sort(vals) - E)) < 1e-12
    e0 = -3 * t2                                                  # Dirac point of this sign convention
    s = (abs(e0) + 3 * abs(t) + 6 * abs(t2)) * 1.05
    M = 40
    mu = np.zeros(M)
    for i in range(lat.n):
        phi = np.zeros(lat.n, complex); phi[i] = 1.0
        mu += kgo.dos_moments(lat, e0, s, phi, M).real
    assert relerr(mu / lat.n, np.array([np.mean(cheb_T(m, (E - e0) / s)) for m in range(M)])) < 1e-12
