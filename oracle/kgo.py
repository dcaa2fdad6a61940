"""ctypes binding of the CPU oracle (oracle/kgo.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, by ``__graft_entry__.smoke()`` and by the
``cpu_baseline`` / ``--impl reference`` legs of ``bench.py``.  The product package
``paper_1307_0288_b200`` never imports this module, and this module never imports it.

Only argument marshalling lives here; all arithmetic is in kgo.c, which follows
PAPER.md (Alg. 5-8, eqs 29-46) step by step.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kgo.c")
_LIB = os.path.join(_HERE, "libkgo.so")

HBAR = 0.6582119569  # eV fs, same literal as KGO_HBAR in kgo.c


def build(force: bool = False) -> str:
    """Compile kgo.c -> libkgo.so with gcc (-O2, no fast-math, no OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=gnu99", "-fPIC", "-shared", "-ffp-contract=off",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.kgo_mix64.restype = C.c_uint64
        _lib.kgo_mix64.argtypes = [C.c_uint64] * 3
        _lib.kgo_uniform.restype = C.c_double
        _lib.kgo_uniform.argtypes = [C.c_uint64] * 3
        _lib.kgo_bessel_np.restype = C.c_int
        _lib.kgo_bessel_np.argtypes = [C.c_double, C.c_double]
        _lib.kgo_compact.restype = C.c_int64
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _c128(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


class Lattice:
    """Plain container: the paper's neighbour-list Hamiltonian (D1-D3, eq 13-14)."""

    def __init__(self, n, kmax, nn, nl, hop, onsite, x, y, period_x, period_y):
        self.n, self.kmax = int(n), int(kmax)
        self.nn, self.nl, self.hop = _i32(nn), _i32(nl), _f64(hop)
        self.onsite = _f64(onsite)
        self.x, self.y = _f64(x), _f64(y)
        self.period_x, self.period_y = float(period_x), float(period_y)


# ----------------------------------------------------------------------------- generators
def mix64(seed, stream, index):
    return int(lib().kgo_mix64(C.c_uint64(seed), C.c_uint64(stream), C.c_uint64(index)))


def uniform(seed, stream, index):
    return float(lib().kgo_uniform(C.c_uint64(seed), C.c_uint64(stream), C.c_uint64(index)))


def honeycomb(ncx, ncy, periodic_x=True, periodic_y=True, a_nm=0.142, t_eV=-2.7):
    n = 4 * ncx * ncy
    x = np.empty(n); y = np.empty(n)
    nn = np.empty(n, np.int32); nl = np.empty(3 * n, np.int32)
    lib().kgo_honeycomb(C.c_int64(ncx), C.c_int64(ncy), C.c_int(int(periodic_x)),
                        C.c_int(int(periodic_y)), C.c_double(a_nm), _p(x), _p(y), _p(nn), _p(nl))
    hop = hop_from_nn(nn, t_eV)
    h = np.sqrt(3.0) * a_nm / 2.0
    px = 2 * ncx * h if periodic_x else 0.0
    py = 6 * ncy * (a_nm / 2.0) if periodic_y else 0.0
    return Lattice(n, 3, nn, nl, hop, None, x, y, px, py)


def honeycomb_nnn(ncx, ncy, periodic_x=True, periodic_y=True, a_nm=0.142, t_eV=-2.7, t2_eV=-0.27):
    """Honeycomb sheet with nearest (t) and next-nearest (t2) neighbour hopping, row width 9."""
    n = 4 * ncx * ncy
    x = np.empty(n); y = np.empty(n)
    nn = np.empty(n, np.int32); nl = np.empty(9 * n, np.int32); hop = np.empty(9 * n)
    lib().kgo_honeycomb_nnn(C.c_int64(ncx), C.c_int64(ncy), C.c_int(int(periodic_x)), C.c_int(int(periodic_y)),
                            C.c_double(a_nm), C.c_double(t_eV), C.c_double(t2_eV), _p(x), _p(y), _p(nn), _p(nl), _p(hop))
    h = np.sqrt(3.0) * a_nm / 2.0
    px = 2 * ncx * h if periodic_x else 0.0
    py = 6 * ncy * (a_nm / 2.0) if periodic_y else 0.0
    return Lattice(n, 9, nn, nl, hop, None, x, y, px, py)


def hop_from_nn(nn, t_eV):
    """hop[k*n+i] = t for k < nn[i], 0 for unused slots (ELL padding)."""
    n = nn.shape[0]
    k = np.arange(3, dtype=np.int32)[:, None]
    return np.where(k < nn[None, :], float(t_eV), 0.0).reshape(3 * n)


def vacancy_mask(n_full, n_vac, seed):
    vac = np.zeros(n_full, np.uint8)
    rc = lib().kgo_vacancy_mask(C.c_int64(n_full), C.c_int64(n_vac), C.c_uint64(seed), _p(vac))
    assert rc == 0
    return vac


def remove_sites(lat: Lattice, vacant, t_eV=-2.7):
    n_out = int(lat.n - int(np.count_nonzero(vacant)))
    x = np.empty(n_out); y = np.empty(n_out)
    nn = np.empty(n_out, np.int32); nl = np.empty(3 * n_out, np.int32)
    vacant = np.ascontiguousarray(vacant, np.uint8)
    got = lib().kgo_compact(C.c_int64(lat.n), _p(vacant), _p(lat.x), _p(lat.y), _p(lat.nn),
                            _p(lat.nl), C.c_int64(n_out), _p(x), _p(y), _p(nn), _p(nl))
    assert got == n_out
    return Lattice(n_out, 3, nn, nl, hop_from_nn(nn, t_eV), None, x, y, lat.period_x, lat.period_y)


def zgnr(ncx, n_chains, a_nm=0.142, t_eV=-2.7):
    """Zigzag ribbon of n_chains zigzag chains (even), ncx cells (2 ncx dimer lines) long, periodic
    along x: kgo_honeycomb (open along y) + kgo_zgnr_mask + kgo_compact."""
    sheet = honeycomb(ncx, n_chains // 2 + 1, periodic_x=True, periodic_y=False, a_nm=a_nm, t_eV=t_eV)
    vac = np.zeros(sheet.n, np.uint8)
    rc = lib().kgo_zgnr_mask(C.c_int64(ncx), C.c_int64(n_chains), _p(vac))
    assert rc == 0
    return remove_sites(sheet, vac, t_eV)


def anderson(n, w_eV, seed):
    eps = np.empty(n)
    lib().kgo_anderson(C.c_int64(n), C.c_double(w_eV), C.c_uint64(seed), _p(eps))
    return eps


def phase_uniforms(n, seed, r):
    u = np.empty(n)
    lib().kgo_phase_uniforms(C.c_int64(n), C.c_uint64(seed), C.c_int(r), _p(u))
    return u


# ----------------------------------------------------------------------------- operators
def _lat_args(lat):
    return (C.c_int64(lat.n), C.c_int(lat.kmax), _p(lat.nn), _p(lat.nl), _p(lat.hop))


def apply_h(lat, e0, s, phi):
    phi = _c128(phi); out = np.empty_like(phi)
    lib().kgo_apply_h(*_lat_args(lat), _p(lat.onsite), C.c_double(e0), C.c_double(s), _p(phi), _p(out))
    return out


def apply_xh(lat, xcoord, period, s, phi):
    phi = _c128(phi); out = np.empty_like(phi); xc = _f64(xcoord)
    lib().kgo_apply_xh(*_lat_args(lat), _p(xc), C.c_double(period), C.c_double(s), _p(phi), _p(out))
    return out


def apply_velocity(lat, xcoord, period, phi):
    phi = _c128(phi); out = np.empty_like(phi); xc = _f64(xcoord)
    lib().kgo_apply_v(*_lat_args(lat), _p(xc), C.c_double(period), _p(phi), _p(out))
    return out


def moments(lat, e0, s, phiL, phiR, M):
    phiL = _c128(phiL); phiR = _c128(phiR); mu = np.empty(M, np.complex128)
    rc = lib().kgo_moments(*_lat_args(lat), _p(lat.onsite), C.c_double(e0), C.c_double(s),
                           _p(phiL), _p(phiR), C.c_int(M), _p(mu))
    assert rc == 0
    return mu


def dos_moments(lat, e0, s, phi, M):
    phi = _c128(phi); mu = np.empty(M, np.complex128)
    rc = lib().kgo_dos_moments(*_lat_args(lat), _p(lat.onsite), C.c_double(e0), C.c_double(s),
                               _p(phi), C.c_int(M), _p(mu))
    assert rc == 0
    return mu


def bessel_np(x, eps=1e-15):
    return int(lib().kgo_bessel_np(C.c_double(x), C.c_double(eps)))


def bessel_j(x, np_):
    j = np.empty(np_)
    lib().kgo_bessel_j(C.c_double(x), C.c_int(np_), _p(j))
    return j


def evolve(lat, e0, s, phi, dt_fs, eps=1e-15):
    phi = _c128(phi); out = np.empty_like(phi)
    rc = lib().kgo_evolve(*_lat_args(lat), _p(lat.onsite), C.c_double(e0), C.c_double(s), _p(phi),
                          C.c_double(dt_fs), C.c_double(eps), _p(out))
    assert rc == 0
    return out


def comm_evolve(lat, xcoord, period, e0, s, phi, dt_fs, eps=1e-15):
    phi = _c128(phi); out = np.empty_like(phi); xc = _f64(xcoord)
    rc = lib().kgo_comm_evolve(*_lat_args(lat), _p(lat.onsite), _p(xc), C.c_double(period),
                               C.c_double(e0), C.c_double(s), _p(phi), C.c_double(dt_fs),
                               C.c_double(eps), _p(out))
    assert rc == 0
    return out


def vac(lat, xcoord, period, e0, s, phi, M, n_steps, dt_fs, eps=1e-15):
    phi = _c128(phi); xc = _f64(xcoord); mu = np.empty((n_steps + 1, M), np.complex128)
    rc = lib().kgo_vac(*_lat_args(lat), _p(lat.onsite), _p(xc), C.c_double(period), C.c_double(e0),
                       C.c_double(s), _p(phi), C.c_int(M), C.c_int(n_steps), C.c_double(dt_fs),
                       C.c_double(eps), _p(mu))
    assert rc == 0
    return mu


def msd(lat, xcoord, period, e0, s, phi, M, n_steps, dt_fs, eps=1e-15):
    phi = _c128(phi); xc = _f64(xcoord); mu = np.empty((n_steps + 1, M), np.complex128)
    rc = lib().kgo_msd(*_lat_args(lat), _p(lat.onsite), _p(xc), C.c_double(period), C.c_double(e0),
                       C.c_double(s), _p(phi), C.c_int(M), C.c_int(n_steps), C.c_double(dt_fs),
                       C.c_double(eps), _p(mu))
    assert rc == 0
    return mu


def _sched(fn, lat, xcoord, period, e0, s, phi, Mk, dt_fs, eps):
    phi = _c128(phi); xc = _f64(xcoord)
    Mk = np.ascontiguousarray(Mk, dtype=np.int32)
    n_steps, ld = Mk.shape[0] - 1, int(Mk.max())
    mu = np.zeros((n_steps + 1, ld), np.complex128)
    rc = fn(*_lat_args(lat), _p(lat.onsite), _p(xc), C.c_double(period), C.c_double(e0),
            C.c_double(s), _p(phi), C.c_int(n_steps), _p(Mk), C.c_int(ld), C.c_double(dt_fs),
            C.c_double(eps), _p(mu))
    assert rc == 0
    return mu


def vac_sched(lat, xcoord, period, e0, s, phi, Mk, dt_fs, eps=1e-15):
    """kgo_vac with Mk[k] moments at time step k (0 = none); returns [len(Mk)][max Mk], unused
    entries 0."""
    return _sched(lib().kgo_vac_sched, lat, xcoord, period, e0, s, phi, Mk, dt_fs, eps)


def msd_sched(lat, xcoord, period, e0, s, phi, Mk, dt_fs, eps=1e-15):
    return _sched(lib().kgo_msd_sched, lat, xcoord, period, e0, s, phi, Mk, dt_fs, eps)


def jackson(M):
    g = np.empty(M)
    lib().kgo_jackson(C.c_int(M), _p(g))
    return g


def kpm_reconstruct(mu, e0, s, energies, use_jackson=True):
    mu = _c128(mu); en = _f64(energies); f = np.empty(en.shape[0])
    lib().kgo_kpm_reconstruct(C.c_int(mu.shape[0]), _p(mu), C.c_int(int(use_jackson)),
                              C.c_double(e0), C.c_double(s), C.c_int(en.shape[0]), _p(en), _p(f))
    return f


def transport(rho, fvac, fmsd, dt_fs, dens_per_nm2, width_nm=1.0):
    """O10: dict of sigma_gk, sigma_e1, sigma_e2, length_nm, conductance ([nt+1][ne] each, in e^2/h
    resp. nm) from rho [ne], fvac / fmsd [nt+1][ne] (either may be None)."""
    rho = _f64(rho)
    ref = fvac if fvac is not None else fmsd
    nt, ne = ref.shape[0] - 1, ref.shape[1]
    fv = None if fvac is None else _f64(fvac)
    fm = None if fmsd is None else _f64(fmsd)
    out = {}
    for name, need in (("sigma_gk", fv), ("sigma_e1", fm), ("sigma_e2", fm), ("length_nm", fm), ("conductance", fm)):
        out[name] = None if need is None else np.empty((nt + 1, ne))
    lib().kgo_transport(C.c_int(nt), C.c_int(ne), C.c_double(dt_fs), C.c_double(dens_per_nm2),
                        C.c_double(width_nm), _p(rho), _p(fv), _p(fm), _p(out["sigma_gk"]),
                        _p(out["sigma_e1"]), _p(out["sigma_e2"]), _p(out["length_nm"]), _p(out["conductance"]))
    return out


def fourier_moments(lat, e0, s, phiL, phiR, Nm, dtau_fs, eps=1e-15):
    """O11 (Alg. 4): F[n + Nm] = <phiL|U(n dtau)|phiR>, n = -Nm..Nm."""
    phiL = _c128(phiL); phiR = _c128(phiR); F = np.empty(2 * Nm + 1, np.complex128)
    rc = lib().kgo_fourier_moments(*_lat_args(lat), _p(lat.onsite), C.c_double(e0), C.c_double(s),
                                   _p(phiL), _p(phiR), C.c_int(Nm), C.c_double(dtau_fs),
                                   C.c_double(eps), _p(F))
    assert rc == 0
    return F


def ftm_reconstruct(F, dtau_fs, energies, use_window=True):
    """O12 (eqs 22-24, 28): f(E) from Fourier moments F[n + Nm]."""
    F = _c128(F); en = _f64(energies); f = np.empty(en.shape[0])
    Nm = (F.shape[0] - 1) // 2
    lib().kgo_ftm_reconstruct(C.c_int(Nm), _p(F), C.c_int(int(use_window)), C.c_double(dtau_fs),
                              C.c_int(en.shape[0]), _p(en), _p(f))
    return f
