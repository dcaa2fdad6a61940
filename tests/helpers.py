"""Test-only helpers: dense matrices built directly from the neighbour-list arrays, golden
fixture reader, lattice conversion between the package's and the oracle's containers.
None of this is used by the product or by the oracle."""
import os

import numpy as np

HBAR = 0.6582119569
GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def golden(name):
    """Read `name value tol # citation` lines from tests/golden/paper_values.txt."""
    with open(os.path.join(GOLDEN, "paper_values.txt")) as f:
        for line in f:
            line = line.split("#")[0].split()
            if len(line) >= 3 and line[0] == name:
                return float(line[1]), float(line[2])
    raise KeyError(name)


def dense_h(lat):
    """H[i, m] from (nn, nl, hop, onsite): H_{i,NL_ik} = hop_ik, H_ii = onsite_i (eV)."""
    n = lat.n
    H = np.zeros((n, n))
    nl = lat.nl.reshape(lat.kmax, n)
    hop = lat.hop.reshape(lat.kmax, n)
    for k in range(lat.kmax):
        for i in range(n):
            if k < lat.nn[i]:
                H[i, nl[k, i]] += hop[k, i]
    if lat.onsite is not None:
        H += np.diag(lat.onsite)
    return H


def to_oracle_lattice(kgo, lat):
    """package workloads.Lattice -> oracle Lattice (same arrays, oracle's own container)."""
    return kgo.Lattice(lat.n, lat.kmax, lat.nn, lat.nl, lat.hop, lat.onsite, lat.x, lat.y,
                       lat.period_x, lat.period_y)


def ring(kgo, n, t=-2.7, a=0.142, periodic=True):
    """1-D chain of n sites as a neighbour list (kmax = 2)."""
    i = np.arange(n)
    if periodic:
        nn = np.full(n, 2, np.int32)
        nl = np.concatenate([(i + 1) % n, (i - 1) % n]).astype(np.int32)
        hop = np.full(2 * n, t)
        period = n * a
    else:
        nn = np.full(n, 2, np.int32); nn[0] = 1; nn[-1] = 1
        first = np.where(i + 1 < n, i + 1, i - 1)
        second = np.where((i + 1 < n) & (i - 1 >= 0), i - 1, i)
        nl = np.concatenate([first, second]).astype(np.int32)
        hop = np.concatenate([np.full(n, t), np.where(nn == 2, t, 0.0)])
        period = 0.0
    x = i * a
    return kgo.Lattice(n, 2, nn, nl, hop, None, x, np.zeros(n), period, 0.0)


def rand_state(n, seed):
    rng = np.random.default_rng(seed)
    v = rng.normal(size=n) + 1j * rng.normal(size=n)
    return v / np.linalg.norm(v)


def cheb_T(n, x):
    return np.cos(n * np.arccos(np.clip(x, -1.0, 1.0)))


def relerr(a, b):
    """max-norm error normalised by the largest magnitude of the reference (BASELINE north_star)."""
    a = np.asarray(a); b = np.asarray(b)
    d = np.max(np.abs(a - b))
    m = np.max(np.abs(b))
    return d / m if m > 0 else d
