"""Thin Python binding of libkg (include/kg.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of ``csrc/``; torch is used for device
memory and streams.  The names mirror the C ABI: ``create_hamiltonian``, ``dos_moments``,
``moments``, ``evolve``, ``apply_velocity``, ``evolve_x``, ``vac``, ``msd``.  Tensors may live
on the GPU or on the host (the C ABI accepts either kind of pointer).  There is no CPU
fallback: if ``libkg.so`` is missing the import raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libkg.so")

if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} not found: build it with `python -m paper_1307_0288_b200.build` "
        "(or __graft_entry__.build()); there is no CPU fallback for the kg_* calls")

_lib = C.CDLL(LIB_PATH)

KG_OK, KG_EINVAL, KG_ENOMEM, KG_ECUDA, KG_ESPECTRUM, KG_EUNSUPPORTED = range(6)
KG_OPT_USE_GRAPHS, KG_OPT_BLOCKS_PER_SM, KG_OPT_THREADS = 1, 2, 3
KG_OPT_STAGED, KG_OPT_STAGES, KG_OPT_STAGED_CTAS, KG_OPT_ALTERNATE, KG_OPT_DICT, KG_OPT_DOUBLING = 4, 5, 6, 7, 8, 9
KG_OPT_CLENSHAW = 10
KG_OPT_PDL = 11
KG_OPT_REORDER = 12
KG_OPT_TWO_STEP = 13
KG_OPT_CHECK_INPUT = 14
KG_OPT_ONE_LAUNCH = 15

_vp, _i64, _i32, _dbl, _int = C.c_void_p, C.c_int64, C.c_int32, C.c_double, C.c_int
_lib.kg_last_error.restype = C.c_char_p
_lib.kg_last_error.argtypes = []
_lib.kg_create_hamiltonian.argtypes = [C.POINTER(_vp), _i64, _i32, _vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _dbl, _vp]
_lib.kg_create_hamiltonian_csr.argtypes = [C.POINTER(_vp), _i64, _vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _dbl, _vp]
_lib.kg_destroy_hamiltonian.argtypes = [_vp]
_lib.kg_workspace_bytes.restype = C.c_size_t
_lib.kg_workspace_bytes.argtypes = [_vp]
_lib.kg_num_sites.restype = _i64
_lib.kg_num_sites.argtypes = [_vp]
_lib.kg_launch_count.restype = _i64
_lib.kg_launch_count.argtypes = [_vp]
_lib.kg_moments.argtypes = [_vp, _vp, _vp, _int, _int, _vp, _vp]
_lib.kg_dos_moments.argtypes = [_vp, _vp, _int, _int, _vp, _vp]
_lib.kg_evolve.argtypes = [_vp, _vp, _vp, _int, _dbl, _dbl, _vp]
_lib.kg_apply_velocity.argtypes = [_vp, _vp, _vp, _int, _vp]
_lib.kg_evolve_x.argtypes = [_vp, _vp, _vp, _int, _dbl, _dbl, _vp]
_lib.kg_vac.argtypes = [_vp, _vp, _int, _int, _int, _dbl, _dbl, _vp, _vp]
_lib.kg_msd.argtypes = [_vp, _vp, _int, _int, _int, _dbl, _dbl, _vp, _vp]
_lib.kg_bessel_terms.argtypes = [_dbl, _dbl, C.POINTER(_int), _vp, _int]
_lib.kg_set_option.argtypes = [_vp, _int, _i64]
_lib.kg_set_default_option.argtypes = [_int, _i64]
_lib.kg_transport.argtypes = [_int, _int, _dbl, _dbl, _dbl] + [_vp] * 9
_lib.kg_fourier_moments.argtypes = [_vp, _vp, _vp, _int, _int, _dbl, _dbl, _vp, _vp]
_lib.kg_ftm_reconstruct.argtypes = [_vp, _i64, _int, _int, _dbl, _vp, _int, _vp, _vp]
_lib.kg_kpm_reconstruct.argtypes = [_vp, _i64, _int, _int, _dbl, _dbl, _vp, _int, _vp, _vp]
_lib.kg_kpm_reconstruct_noalloc.argtypes = [_vp, _i64, _int, _int, _dbl, _dbl, _vp, _int, _vp, _vp]
KG_KPM_NOALLOC_MAX_M = 16384


class KgError(RuntimeError):
    def __init__(self, code):
        self.code = code
        super().__init__(f"libkg error {code}: {_lib.kg_last_error().decode()}")


def _check(rc):
    if rc != KG_OK:
        raise KgError(rc)


def _ptr(t):
    """Address of a torch tensor / numpy array (host or device), None -> NULL."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.flags.c_contiguous
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _stream(stream=None):
    if stream is None:
        stream = torch.cuda.current_stream()
    return stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream)


def _vec(t, n):
    """Accept [n] or [n, R] complex128; return (tensor, R)."""
    assert t.dtype in (torch.complex128, np.complex128), "vectors must be complex128"
    if t.ndim == 1:
        return t, 1
    assert t.ndim == 2 and t.shape[0] == n
    return t, int(t.shape[1])


def _empty_like_mu(ref, shape):
    if isinstance(ref, np.ndarray):
        return np.empty(shape, np.complex128)
    return torch.empty(shape, dtype=torch.complex128, device=ref.device)


class Hamiltonian:
    """Owner of a ``kg_hamiltonian*``."""

    def __init__(self, handle, n):
        self._h = _vp(handle)
        self.n = n

    def close(self):
        if self._h:
            _lib.kg_destroy_hamiltonian(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def workspace_bytes(self):
        return int(_lib.kg_workspace_bytes(self._h))

    @property
    def launch_count(self):
        return int(_lib.kg_launch_count(self._h))

    def set_option(self, option, value):
        _check(_lib.kg_set_option(self._h, option, value))


def set_default_option(option, value):
    """kg_set_default_option: create-time options (KG_OPT_REORDER) for handles created afterwards."""
    _check(_lib.kg_set_default_option(option, value))


def create_hamiltonian(n, kmax, nn, nl, hop_eV, onsite_eV, x_nm, period_x_nm, e0_eV, scale_eV,
                       stream=None) -> Hamiltonian:
    """kg_create_hamiltonian: arrays are int32 / float64 numpy arrays or torch tensors (host or
    device), in the paper's k-major neighbour-list layout."""
    out = _vp()
    _check(_lib.kg_create_hamiltonian(C.byref(out), n, kmax, _ptr(nn), _ptr(nl), _ptr(hop_eV),
                                      _ptr(onsite_eV), _ptr(x_nm), period_x_nm, e0_eV, scale_eV,
                                      _stream(stream)))
    return Hamiltonian(out.value, n)


def create_hamiltonian_csr(n, rowptr, col, hop_eV, onsite_eV, x_nm, period_x_nm, e0_eV, scale_eV,
                           stream=None) -> Hamiltonian:
    out = _vp()
    _check(_lib.kg_create_hamiltonian_csr(C.byref(out), n, _ptr(rowptr), _ptr(col), _ptr(hop_eV),
                                          _ptr(onsite_eV), _ptr(x_nm), period_x_nm, e0_eV,
                                          scale_eV, _stream(stream)))
    return Hamiltonian(out.value, n)


def from_lattice(lat, xcoord, period, e0, scale, stream=None) -> Hamiltonian:
    """Convenience: workloads.Lattice (numpy, host) -> Hamiltonian."""
    return create_hamiltonian(lat.n, lat.kmax, np.ascontiguousarray(lat.nn, np.int32),
                              np.ascontiguousarray(lat.nl, np.int32),
                              np.ascontiguousarray(lat.hop, np.float64),
                              None if lat.onsite is None else np.ascontiguousarray(lat.onsite, np.float64),
                              np.ascontiguousarray(xcoord, np.float64), float(period), float(e0),
                              float(scale), stream)


def moments(h: Hamiltonian, phiL, phiR, M, mu=None, stream=None):
    phiR, R = _vec(phiR, h.n)
    phiL, RL = _vec(phiL, h.n)
    assert R == RL
    if mu is None:
        mu = _empty_like_mu(phiR, (R, M))
    _check(_lib.kg_moments(h._h, _ptr(phiL), _ptr(phiR), R, M, _ptr(mu), _stream(stream)))
    return mu


def dos_moments(h: Hamiltonian, phi, M, mu=None, stream=None):
    phi, R = _vec(phi, h.n)
    if mu is None:
        mu = _empty_like_mu(phi, (R, M))
    _check(_lib.kg_dos_moments(h._h, _ptr(phi), R, M, _ptr(mu), _stream(stream)))
    return mu


def evolve(h: Hamiltonian, phi, dt_fs, bessel_eps=1e-15, out=None, stream=None):
    phi, R = _vec(phi, h.n)
    if out is None:
        out = np.empty_like(phi) if isinstance(phi, np.ndarray) else torch.empty_like(phi)
    _check(_lib.kg_evolve(h._h, _ptr(phi), _ptr(out), R, dt_fs, bessel_eps, _stream(stream)))
    return out


def apply_velocity(h: Hamiltonian, phi, out=None, stream=None):
    phi, R = _vec(phi, h.n)
    if out is None:
        out = np.empty_like(phi) if isinstance(phi, np.ndarray) else torch.empty_like(phi)
    _check(_lib.kg_apply_velocity(h._h, _ptr(phi), _ptr(out), R, _stream(stream)))
    return out


def evolve_x(h: Hamiltonian, psi, psix, dt_fs, bessel_eps=1e-15, stream=None):
    """In place: (psi, psix) <- (U psi, U psix + [X,U] psi)."""
    psi, R = _vec(psi, h.n)
    psix, Rx = _vec(psix, h.n)
    assert R == Rx
    _check(_lib.kg_evolve_x(h._h, _ptr(psi), _ptr(psix), R, dt_fs, bessel_eps, _stream(stream)))
    return psi, psix


def vac(h: Hamiltonian, phi, M, n_steps, dt_fs, bessel_eps=1e-15, mu=None, stream=None):
    phi, R = _vec(phi, h.n)
    if mu is None:
        mu = _empty_like_mu(phi, (R, n_steps + 1, M))
    _check(_lib.kg_vac(h._h, _ptr(phi), R, M, n_steps, dt_fs, bessel_eps, _ptr(mu), _stream(stream)))
    return mu


def msd(h: Hamiltonian, phi, M, n_steps, dt_fs, bessel_eps=1e-15, mu=None, stream=None):
    phi, R = _vec(phi, h.n)
    if mu is None:
        mu = _empty_like_mu(phi, (R, n_steps + 1, M))
    _check(_lib.kg_msd(h._h, _ptr(phi), R, M, n_steps, dt_fs, bessel_eps, _ptr(mu), _stream(stream)))
    return mu


def bessel_terms(x, bessel_eps=1e-15):
    """(N_p, J_0..J_{N_p-1}) as the library computes them (host arithmetic, no GPU needed)."""
    n_p = _int()
    _check(_lib.kg_bessel_terms(x, bessel_eps, C.byref(n_p), None, 0))
    j = np.empty(n_p.value)
    _check(_lib.kg_bessel_terms(x, bessel_eps, C.byref(n_p), j.ctypes.data, n_p.value))
    return n_p.value, j


def kpm_reconstruct(mu, e0_eV, scale_eV, energies_eV, jackson=True, stream=None):
    """kg_kpm_reconstruct: mu [..., M] complex128 (torch or numpy, host or device) ->
    f [..., n_energies] float64 of the same kind (eqs 29-31, 35)."""
    M = int(mu.shape[-1])
    lead = tuple(mu.shape[:-1])
    rows = int(np.prod(lead)) if lead else 1
    ne = int(energies_eV.shape[0])
    if isinstance(mu, np.ndarray):
        f = np.empty(lead + (ne,), np.float64)
    else:
        f = torch.empty(lead + (ne,), dtype=torch.float64, device=mu.device)
    _check(_lib.kg_kpm_reconstruct(_ptr(mu), rows, M, int(bool(jackson)), float(e0_eV), float(scale_eV),
                                   _ptr(energies_eV), ne, _ptr(f), _stream(stream)))
    return f


def kpm_reconstruct_noalloc(mu, e0_eV, scale_eV, energies_eV, f, jackson=True, stream=None):
    """kg_kpm_reconstruct_noalloc: the reconstruction of ``kpm_reconstruct`` for callers that cannot
    allocate GPU memory (all of it already belongs to their own arena, or an allocation would stall
    a latency-bound loop).  Nothing is allocated here either: ``mu`` [..., M], ``energies_eV`` and the
    output ``f`` [..., n_energies] are CUDA tensors the caller made beforehand, M must not exceed
    ``KG_KPM_NOALLOC_MAX_M``, and the weights go to one fixed array per GPU inside libkg — so calls
    that could overlap on the GPU (different streams) must be ordered by the caller.  Returns ``f``."""
    M = int(mu.shape[-1])
    lead = tuple(mu.shape[:-1])
    rows = int(np.prod(lead)) if lead else 1
    ne = int(energies_eV.shape[0])
    assert tuple(f.shape) == lead + (ne,) and f.dtype in (torch.float64, np.float64)
    _check(_lib.kg_kpm_reconstruct_noalloc(_ptr(mu), rows, M, int(bool(jackson)), float(e0_eV), float(scale_eV),
                                           _ptr(energies_eV), ne, _ptr(f), _stream(stream)))
    return f


def transport(rho, fvac, fmsd, dt_fs, dens_per_nm2, width_nm=1.0, stream=None):
    """kg_transport: dict of sigma_gk (needs fvac), sigma_e1, sigma_e2, length_nm, conductance
    (need fmsd) as [n_steps+1][n_energies] arrays of the same kind as the inputs (eqs 6-11, 50-51)."""
    ref = fvac if fvac is not None else fmsd
    nt, ne = int(ref.shape[0]) - 1, int(ref.shape[1])

    def new():
        if isinstance(ref, np.ndarray):
            return np.empty((nt + 1, ne), np.float64)
        return torch.empty((nt + 1, ne), dtype=torch.float64, device=ref.device)
    out = {"sigma_gk": new() if fvac is not None else None}
    for k in ("sigma_e1", "sigma_e2"):
        out[k] = new() if fmsd is not None else None
    for k in ("length_nm", "conductance"):                 # eq 50-51 need rho~ as well
        out[k] = new() if fmsd is not None and rho is not None else None
    _check(_lib.kg_transport(nt, ne, float(dt_fs), float(dens_per_nm2), float(width_nm), _ptr(rho), _ptr(fvac),
                             _ptr(fmsd), _ptr(out["sigma_gk"]), _ptr(out["sigma_e1"]), _ptr(out["sigma_e2"]),
                             _ptr(out["length_nm"]), _ptr(out["conductance"]), _stream(stream)))
    return out


def fourier_moments(h: Hamiltonian, phiL, phiR, Nm, dtau_fs, bessel_eps=1e-15, F=None, stream=None):
    """kg_fourier_moments (Alg. 4): F[r, n + Nm] = <phiL_r|U(n dtau)|phiR_r>, n = -Nm..Nm."""
    phiR, R = _vec(phiR, h.n)
    phiL, RL = _vec(phiL, h.n)
    assert R == RL
    if F is None:
        F = _empty_like_mu(phiR, (R, 2 * Nm + 1))
    _check(_lib.kg_fourier_moments(h._h, _ptr(phiL), _ptr(phiR), R, Nm, dtau_fs, bessel_eps, _ptr(F), _stream(stream)))
    return F


def ftm_reconstruct(F, dtau_fs, energies_eV, window=True, stream=None):
    """kg_ftm_reconstruct: F [..., 2Nm+1] -> f [..., n_energies] (eqs 22-24, 28)."""
    Nm = (int(F.shape[-1]) - 1) // 2
    lead = tuple(F.shape[:-1])
    rows = int(np.prod(lead)) if lead else 1
    ne = int(energies_eV.shape[0])
    if isinstance(F, np.ndarray):
        f = np.empty(lead + (ne,), np.float64)
    else:
        f = torch.empty(lead + (ne,), dtype=torch.float64, device=F.device)
    _check(_lib.kg_ftm_reconstruct(_ptr(F), rows, Nm, int(bool(window)), float(dtau_fs), _ptr(energies_eV), ne,
                                   _ptr(f), _stream(stream)))
    return f
