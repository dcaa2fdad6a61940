"""Seeded synthetic inputs: graphene lattices, disorder, random-phase vectors, the five
BASELINE.json configs.

This module holds NONE of the method's arithmetic (no H application, no recursion, no
Bessel/Jackson): it only builds the inputs of ``kg_create_hamiltonian`` and the random
vectors, following the paper's lattice conventions (N_x dimer lines along
zigzag, N_y zigzag chains along armchair, a = 0.142 nm, L_x = sqrt(3) N_x a / 2,
L_y = 3 N_y a / 2), its hopping (eq 13: -gamma_0, gamma_0 = 2.7 eV) and its vacancy
model.  The recipe (counter PRNG, site numbering, neighbour order, vacancy
selection) is stated in DESIGN.md "Input recipe"; the test oracle implements the same recipe
independently in C and tests/test_generators.py compares the two bit for bit.

numpy, vectorised (a 16 M-site sheet takes a few seconds).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

A_NM = 0.142          # bond length
T_EV = -2.7           # hopping matrix element -gamma_0, eq 13
HBAR = 0.6582119569   # eV fs

_M1 = np.uint64(0x9E3779B97F4A7C15)
_M2 = np.uint64(0xD1B54A32D192ED03)
_F1 = np.uint64(0xBF58476D1CE4E5B9)
_F2 = np.uint64(0x94D049BB133111EB)


def mix64(seed: int, stream: int, index) -> np.ndarray:
    """Counter-based 64-bit hash (SplitMix64 finaliser over a (seed, stream, index) counter)."""
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64((((seed + 1) * 0x9E3779B97F4A7C15) & 0xFFFFFFFFFFFFFFFF)
                      ^ (((stream + 1) * 0xD1B54A32D192ED03) & 0xFFFFFFFFFFFFFFFF))
        z = z + idx * _M1
        z = z ^ (z >> np.uint64(30))
        z = z * _F1
        z = z ^ (z >> np.uint64(27))
        z = z * _F2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform(seed: int, stream: int, index) -> np.ndarray:
    """u = (bits >> 11) * 2**-53 in [0, 1)."""
    return (mix64(seed, stream, index) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


@dataclass
class Lattice:
    """Neighbour-list Hamiltonian in the paper's layout: k-major ELL."""
    n: int
    kmax: int
    nn: np.ndarray          # int32 [n]
    nl: np.ndarray          # int32 [kmax*n], nl[k*n+i]; unused slots hold i
    hop: np.ndarray         # float64 [kmax*n] eV; unused slots 0
    onsite: np.ndarray | None   # float64 [n] eV or None
    x: np.ndarray           # float64 [n] nm (zigzag coordinate)
    y: np.ndarray           # float64 [n] nm (armchair coordinate)
    period_x: float         # nm, 0 = open
    period_y: float
    meta: dict = field(default_factory=dict)


def honeycomb(ncx: int, ncy: int, periodic_x=True, periodic_y=True, a_nm=A_NM, t_eV=T_EV) -> Lattice:
    """ncx x ncy rectangular 4-atom cells (paper N_x = 2 ncx, N_y = 2 ncy)."""
    n = 4 * ncx * ncy
    site = np.arange(n, dtype=np.int64)
    b = site & 3
    cell = site >> 2
    cx = cell % ncx
    cy = cell // ncx
    h = np.sqrt(3.0) * a_nm / 2.0
    q = a_nm / 2.0
    hx = np.where(b >= 2, 1, 0)
    hy = np.array([0, 2, 3, 5], dtype=np.int64)[b]
    x = (2 * cx + hx).astype(np.float64) * h
    y = (6 * cy + hy).astype(np.float64) * q

    # neighbour k of basis b: (dcx, dcy, basis'), in recipe order
    dcx = np.array([[0, 0, -1], [0, 0, -1], [0, 0, 1], [0, 0, 1]], dtype=np.int64)
    dcy = np.array([[0, -1, -1], [0, 0, 0], [0, 0, 0], [0, 1, 1]], dtype=np.int64)
    nb = np.array([[1, 3, 3], [0, 2, 2], [3, 1, 1], [2, 0, 0]], dtype=np.int64)

    cand = np.empty((3, n), dtype=np.int64)
    valid = np.ones((3, n), dtype=bool)
    for k in range(3):
        mx = cx + dcx[b, k]
        my = cy + dcy[b, k]
        okx = (mx >= 0) & (mx < ncx)
        oky = (my >= 0) & (my < ncy)
        if periodic_x:
            mx = np.mod(mx, ncx)
        else:
            valid[k] &= okx
        if periodic_y:
            my = np.mod(my, ncy)
        else:
            valid[k] &= oky
        cand[k] = 4 * (my * ncx + np.clip(mx, 0, ncx - 1)) + nb[b, k]
    nn, nl = _pack_neighbours(cand, valid, n)
    hop = _hop_from_nn(nn, t_eV)
    return Lattice(n, 3, nn, nl, hop, None, x, y,
                   2 * ncx * h if periodic_x else 0.0,
                   6 * ncy * q if periodic_y else 0.0,
                   {"ncx": ncx, "ncy": ncy})


def _pack_neighbours(cand, valid, n, values=None):
    """Shift valid neighbours down to slots 0..nn-1 keeping their order; pad with self (and 0 in the
    optional per-slot values, which are packed the same way)."""
    kmax = cand.shape[0]
    nn = valid.sum(axis=0).astype(np.int32)
    slot = np.cumsum(valid, axis=0) - 1            # target slot of each valid candidate
    nl = np.tile(np.arange(n, dtype=np.int64), (kmax, 1))
    vals = None if values is None else np.zeros((kmax, n))
    for k in range(kmax):
        sel = valid[k]
        nl[slot[k, sel], np.nonzero(sel)[0]] = cand[k, sel]
        if values is not None:
            vals[slot[k, sel], np.nonzero(sel)[0]] = values[k]
    if values is None:
        return nn, nl.astype(np.int32).reshape(kmax * n)
    return nn, nl.astype(np.int32).reshape(kmax * n), vals.reshape(kmax * n)


T2_EV = -0.27         # next-nearest-neighbour hopping t' = 0.1 |t| (graphene: 0.02-0.2 |t| in the literature)


def honeycomb_nnn(ncx: int, ncy: int, periodic_x=True, periodic_y=True, a_nm=A_NM, t_eV=T_EV, t2_eV=T2_EV) -> Lattice:
    """Honeycomb sheet with next-nearest-neighbour hopping (a "more complicated tight-binding
    model" with a denser Hamiltonian): row width 9 — the three nearest neighbours of `honeycomb` in the
    same order (hopping t), then the six second neighbours at distance sqrt(3) a (hopping t2) in the
    order (+2,0) (-2,0) (+1,+3) (-1,+3) (+1,-3) (-1,-3) of displacements in units (h, a/2)."""
    n = 4 * ncx * ncy
    site = np.arange(n, dtype=np.int64)
    b = site & 3
    cell = site >> 2
    cx = cell % ncx
    cy = cell // ncx
    h = np.sqrt(3.0) * a_nm / 2.0
    q = a_nm / 2.0
    x = (2 * cx + np.where(b >= 2, 1, 0)).astype(np.float64) * h
    y = (6 * cy + np.array([0, 2, 3, 5], dtype=np.int64)[b]).astype(np.float64) * q
    # (dcx, dcy, basis') per basis b and neighbour k: three nearest, six second neighbours
    tab = np.array([
        [(0, 0, 1), (0, -1, 3), (-1, -1, 3), (1, 0, 0), (-1, 0, 0), (0, 0, 2), (-1, 0, 2), (0, -1, 2), (-1, -1, 2)],
        [(0, 0, 0), (0, 0, 2), (-1, 0, 2), (1, 0, 1), (-1, 0, 1), (0, 0, 3), (-1, 0, 3), (0, -1, 3), (-1, -1, 3)],
        [(0, 0, 3), (0, 0, 1), (1, 0, 1), (1, 0, 2), (-1, 0, 2), (1, 1, 0), (0, 1, 0), (1, 0, 0), (0, 0, 0)],
        [(0, 0, 2), (0, 1, 0), (1, 1, 0), (1, 0, 3), (-1, 0, 3), (1, 1, 1), (0, 1, 1), (1, 0, 1), (0, 0, 1)],
    ], dtype=np.int64)
    cand = np.empty((9, n), dtype=np.int64)
    valid = np.ones((9, n), dtype=bool)
    for k in range(9):
        mx = cx + tab[b, k, 0]
        my = cy + tab[b, k, 1]
        okx = (mx >= 0) & (mx < ncx)
        oky = (my >= 0) & (my < ncy)
        if periodic_x:
            mx = np.mod(mx, ncx)
        else:
            valid[k] &= okx
        if periodic_y:
            my = np.mod(my, ncy)
        else:
            valid[k] &= oky
        cand[k] = 4 * (np.clip(my, 0, ncy - 1) * ncx + np.clip(mx, 0, ncx - 1)) + tab[b, k, 2]
    nn, nl, hop = _pack_neighbours(cand, valid, n, values=[t_eV] * 3 + [t2_eV] * 6)
    return Lattice(n, 9, nn, nl, hop, None, x, y,
                   2 * ncx * h if periodic_x else 0.0, 6 * ncy * q if periodic_y else 0.0,
                   {"ncx": ncx, "ncy": ncy, "t2_eV": t2_eV})


def _hop_from_nn(nn, t_eV):
    k = np.arange(3, dtype=np.int32)[:, None]
    return np.where(k < nn[None, :], float(t_eV), 0.0).reshape(-1)


def vacancy_mask(n_full: int, n_vac: int, seed: int) -> np.ndarray:
    """The n_vac sites with the smallest (key, index), key_j = mix64(seed, 0, j)."""
    keys = mix64(seed, 0, np.arange(n_full, dtype=np.uint64))
    order = np.argsort(keys, kind="stable")       # stable: ties resolved by index
    vac = np.zeros(n_full, dtype=np.uint8)
    vac[order[:n_vac]] = 1
    return vac


def n_vacancies(concentration: float, n_full: int) -> int:
    return int(np.floor(concentration * n_full + 0.5))


def remove_sites(lat: Lattice, vacant: np.ndarray, t_eV=T_EV) -> Lattice:
    """Delete-and-compact (reading g15): survivors keep their order, lists are re-indexed."""
    keep = vacant == 0
    n = lat.n
    newidx = np.cumsum(keep, dtype=np.int64) - 1
    n_out = int(keep.sum())
    old = np.nonzero(keep)[0]
    nl_old = lat.nl.reshape(3, n)[:, old].astype(np.int64)           # [3][n_out] old indices
    k = np.arange(3)[:, None]
    valid = (k < lat.nn[old][None, :]) & keep[nl_old]
    cand = newidx[nl_old]
    nn, nl = _pack_neighbours(cand, valid, n_out)
    return Lattice(n_out, 3, nn, nl, _hop_from_nn(nn, t_eV), None, lat.x[old].copy(),
                   lat.y[old].copy(), lat.period_x, lat.period_y, dict(lat.meta))


def zgnr(ncx: int, n_chains: int, a_nm=A_NM, t_eV=T_EV) -> Lattice:
    """Zigzag graphene nanoribbon (the paper's ballistic test system, Fig. 4: "65536 x 16"):
    n_chains zigzag chains (even; the paper's N_y), ncx cells = 2 ncx dimer lines (N_x) long, periodic
    along x (zigzag direction = transport axis).  Cut from a sheet of ncx x (n_chains/2 + 1) cells open
    along y by removing the bottom cell row's b0 sites and the top row's b1, b2, b3 sites: the cut runs
    through the vertical bonds, so both edges are zigzag and every edge site keeps two neighbours
    (the open sheet itself has "bearded" edges: sites hanging on one bond)."""
    assert n_chains >= 2 and n_chains % 2 == 0
    ncy = n_chains // 2 + 1
    sheet = honeycomb(ncx, ncy, periodic_x=True, periodic_y=False, a_nm=a_nm, t_eV=t_eV)
    site = np.arange(sheet.n, dtype=np.int64)
    b, cy = site & 3, (site >> 2) // ncx
    vacant = (((cy == 0) & (b == 0)) | ((cy == ncy - 1) & (b != 0))).astype(np.uint8)
    lat = remove_sites(sheet, vacant, t_eV)
    lat.meta.update({"n_chains": n_chains, "width_nm": (1.5 * n_chains - 1.0) * a_nm})
    return lat


def anderson(n: int, w_eV: float, seed: int) -> np.ndarray:
    """eps_j = W (u(seed, 1, j) - 1/2)."""
    return w_eV * (uniform(seed, 1, np.arange(n, dtype=np.uint64)) - 0.5)


def random_phase_vectors(n: int, R: int, seed: int) -> np.ndarray:
    """[n][R] complex128, phi_r[j] = exp(2 pi i u(seed, 16+r, j)) / sqrt(n), unit norm (g1)."""
    out = np.empty((n, R), dtype=np.complex128)
    idx = np.arange(n, dtype=np.uint64)
    inv = 1.0 / np.sqrt(float(n))
    for r in range(R):
        ang = 2.0 * np.pi * uniform(seed, 16 + r, idx)
        out[:, r] = (np.cos(ang) + 1j * np.sin(ang)) * inv
    return out


# ----------------------------------------------------------------------------- configs
@dataclass
class Config:
    name: str
    lattice: Lattice
    xcoord: np.ndarray      # transport coordinate handed to kg_create_hamiltonian
    period: float           # its period (0 = open)
    scale: float            # s = Delta E of BASELINE.json (half-width), eV
    e0: float
    R: int
    M: int
    n_steps: int
    dt_fs: float
    seed: int
    n_energies: int


def _dt(mult):  # Delta t = mult * hbar/|t|
    return mult * HBAR / abs(T_EV)


def make_config(idx: int, shrink: int = 1) -> Config:
    """BASELINE.json configs[idx-1], idx in 1..5.  ``shrink`` divides the linear cell counts
    (tests use it for scaled-down twins of the large sheets; bench uses shrink=1)."""
    t = abs(T_EV)
    if idx == 1:
        lat = honeycomb(32 // shrink, 32 // shrink)
        return Config("c1_pristine_32x32", lat, lat.x, lat.period_x, 3 * t * 1.05, 0.0,
                      1, 256, 16, _dt(1), 0, 1001)
    if idx == 2:
        full = honeycomb(250 // shrink, 250 // shrink)
        vac = vacancy_mask(full.n, n_vacancies(0.005, full.n), 1)
        lat = remove_sites(full, vac)
        return Config("c2_vacancies_250x250", lat, lat.x, lat.period_x, 3 * t * 1.05, 0.0,
                      4, 1000, 200, _dt(2), 1, 501)
    if idx == 3:
        # AGNR: 30 dimer lines wide (15 cells, open along x), periodic along y (armchair axis,
        # the transport direction): pass y as the transport coordinate (reading g16).
        lat = honeycomb(15, 20000 // shrink, periodic_x=False, periodic_y=True)
        return Config("c3_agnr_30x20000", lat, lat.y, lat.period_y, 3 * t * 1.05, 0.0,
                      1, 2000, 400, _dt(1), 0, 1001)
    if idx == 4:
        lat = honeycomb(1000 // shrink, 1000 // shrink)
        lat.onsite = anderson(lat.n, t, 2)
        return Config("c4_anderson_1000x1000", lat, lat.x, lat.period_x, (3 * t + t / 2) * 1.05,
                      0.0, 1, 3000, 100, _dt(4), 2, 1001)
    if idx == 5:
        full = honeycomb(2000 // shrink, 2000 // shrink)
        vac = vacancy_mask(full.n, n_vacancies(0.001, full.n), 3)
        lat = remove_sites(full, vac)
        return Config("c5_batched_2000x2000", lat, lat.x, lat.period_x, 3 * t * 1.05, 0.0,
                      8, 3000, 50, _dt(8), 3, 1001)
    if idx == 6:
        # the paper's own ballistic system (Fig. 4): ZGNR with N_x = 65536 dimer lines
        # (32768 cells) and N_y = 16 zigzag chains = 1 048 576 sites; Einstein MSD, transport along x
        lat = zgnr(32768 // shrink, 16)
        return Config("zgnr_65536x16", lat, lat.x, lat.period_x, 3 * t * 1.05, 0.0,
                      1, 2000, 400, _dt(1), 0, 1001)
    raise ValueError("config index must be 1..6 (6 = the paper's ZGNR 65536 x 16)")


def energy_grid(n_energies: int) -> np.ndarray:
    """E_j = -3|t| + 6|t| j/(n-1) (reading g13)."""
    t = abs(T_EV)
    return -3 * t + 6 * t * np.arange(n_energies) / (n_energies - 1)
