"""Lattice / disorder / PRNG generators: the package's numpy implementation
(paper_1307_0288_b200.workloads) against the oracle's independent C implementation
(oracle/kgo.c), bit for bit, plus the properties the paper's conventions fix."""
import numpy as np
import pytest

from paper_1307_0288_b200 import workloads as W
from helpers import golden


def _same_lattice(a, b):
    assert a.n == b.n
    assert np.array_equal(a.nn, b.nn)
    assert np.array_equal(a.nl, b.nl)
    assert np.array_equal(a.hop, b.hop)
    assert a.x.tobytes() == b.x.tobytes()          # bit-exact coordinates
    assert a.y.tobytes() == b.y.tobytes()
    assert a.period_x == b.period_x and a.period_y == b.period_y


def test_prng_bit_exact(kgo):
    idx = np.array([0, 1, 2, 17, 2**31 + 5, 2**40 + 3], dtype=np.uint64)
    for seed in (0, 1, 2, 3, 12345):
        for stream in (0, 1, 16, 23):
            got = W.mix64(seed, stream, idx)
            for j, i in enumerate(idx):
                assert int(got[j]) == kgo.mix64(seed, stream, int(i))
    u = W.uniform(3, 16, np.arange(1000, dtype=np.uint64))
    assert np.array_equal(u, kgo.phase_uniforms(1000, 3, 0))
    assert u.min() >= 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 0.05


@pytest.mark.parametrize("ncx,ncy,px,py", [(4, 4, True, True), (7, 5, True, True),
                                           (5, 9, False, True), (6, 4, True, False),
                                           (3, 3, False, False), (1, 1, True, True)])
def test_honeycomb_bit_exact(kgo, ncx, ncy, px, py):
    _same_lattice(W.honeycomb(ncx, ncy, px, py), kgo.honeycomb(ncx, ncy, px, py))


def test_vacancies_and_compaction_bit_exact(kgo):
    full_p = W.honeycomb(20, 15)
    full_o = kgo.honeycomb(20, 15)
    nv = W.n_vacancies(0.05, full_p.n)
    assert nv == 60
    vp = W.vacancy_mask(full_p.n, nv, 7)
    vo = kgo.vacancy_mask(full_o.n, nv, 7)
    assert np.array_equal(vp, vo) and int(vp.sum()) == nv
    _same_lattice(W.remove_sites(full_p, vp), kgo.remove_sites(full_o, vo))


def test_anderson_bit_exact(kgo):
    assert np.array_equal(W.anderson(5000, 2.7, 2), kgo.anderson(5000, 2.7, 2))
    e = W.anderson(200000, 2.7, 2)
    assert e.min() >= -1.35 and e.max() < 1.35 and abs(e.mean()) < 0.01
    assert abs(e.var() - 2.7**2 / 12) < 0.01


def test_config_counts():
    # BASELINE.json: config 2 removes 0.5 % of 250 000 sites; config 5 0.1 % of 16 M
    assert W.n_vacancies(0.005, 250000) == 1250
    assert W.n_vacancies(0.001, 16000000) == 16000


def test_honeycomb_properties():
    a = golden("bond_length_nm")[0]
    lat = W.honeycomb(6, 5)
    n = lat.n
    nl = lat.nl.reshape(3, n)
    assert np.all(lat.nn == 3)                                   # torus: every site has 3 neighbours
    i = np.arange(n)
    for k in range(3):
        m = nl[k]
        dx = lat.x[m] - lat.x
        dy = lat.y[m] - lat.y
        dx -= lat.period_x * np.round(dx / lat.period_x)
        dy -= lat.period_y * np.round(dy / lat.period_y)
        assert np.allclose(np.hypot(dx, dy), a, rtol=0, atol=1e-15)   # every bond has length a
        assert np.all((m & 1) != (i & 1))                        # bipartite: A <-> B only
        back = nl[:, m]                                          # adjacency symmetric
        assert np.all((back == i[None, :]).sum(axis=0) == 1)
    # three distinct neighbours
    assert np.all((nl[0] != nl[1]) & (nl[1] != nl[2]) & (nl[0] != nl[2]))


def test_lengths_match_paper():
    # L_x = sqrt(3) N_x a / 2 with N_x = 2 ncx dimer lines; paper prints 126 / 252 / 12 nm
    for name, ncx in (("Lx_nm_Nx1024", 512), ("Lx_nm_Nx2048", 1024)):
        val, tol = golden(name)
        lat = W.honeycomb(ncx, 1)
        assert abs(lat.period_x - val) < tol
    val, tol = golden("W_nm_Nx95")
    assert abs(np.sqrt(3) * 95 * 0.142 / 2 - val) < tol
    # L_y = 3 N_y a / 2, N_y = 2 ncy
    lat = W.honeycomb(2, 7)
    assert abs(lat.period_y - 3 * 14 * 0.142 / 2) < 1e-12


def test_ribbon_edges():
    # AGNR of config 3 (open along x): edge columns lose one neighbour, interior keeps 3
    lat = W.honeycomb(5, 8, periodic_x=False, periodic_y=True)
    assert set(np.unique(lat.nn)) == {2, 3}
    edge = (lat.x == lat.x.min()) | (lat.x == lat.x.max())
    assert np.all(lat.nn[edge] == 2) and np.all(lat.nn[~edge] == 3)
    nl = lat.nl.reshape(3, lat.n)
    pad = np.arange(3)[:, None] >= lat.nn[None, :]
    assert np.all(nl[pad] == np.broadcast_to(np.arange(lat.n), (3, lat.n))[pad])
    assert np.all(lat.hop.reshape(3, lat.n)[pad] == 0.0)


def test_vacancy_lattice_consistency():
    full = W.honeycomb(12, 12)
    vac = W.vacancy_mask(full.n, 30, 1)
    lat = W.remove_sites(full, vac)
    assert lat.n == full.n - 30
    nl = lat.nl.reshape(3, lat.n)
    i = np.arange(lat.n)
    deg = np.zeros(lat.n, int)
    for k in range(3):
        sel = k < lat.nn
        m = nl[k, sel]
        # surviving bonds still have length a and are symmetric
        dx = lat.x[m] - lat.x[sel]; dy = lat.y[m] - lat.y[sel]
        dx -= lat.period_x * np.round(dx / lat.period_x)
        dy -= lat.period_y * np.round(dy / lat.period_y)
        assert np.allclose(np.hypot(dx, dy), 0.142, atol=1e-15, rtol=0)
        np.add.at(deg, m, 1)
    assert np.array_equal(deg, lat.nn)                # in-degree == out-degree
    # 3 * removed bonds minus bonds between two vacancies
    assert lat.nn.sum() <= 3 * lat.n - 3 * 30 + 2 * 30


def test_random_phase_vectors():
    phi = W.random_phase_vectors(4096, 3, 0)
    assert phi.shape == (4096, 3)
    assert np.allclose(np.abs(phi) * 64.0, 1.0, atol=1e-14)
    assert np.allclose(np.linalg.norm(phi, axis=0), 1.0, atol=1e-14)   # unit norm (reading g1)
    assert abs(np.vdot(phi[:, 0], phi[:, 1])) < 0.1


def test_make_config_small():
    c = W.make_config(1)
    assert c.lattice.n == 4096 and c.M == 256 and c.n_steps == 16 and c.R == 1
    assert abs(c.scale - 8.505) < 1e-12
    assert abs(c.dt_fs - 0.6582119569 / 2.7) < 1e-15
    c3 = W.make_config(3, shrink=100)
    assert c3.lattice.n == 15 * 200 * 4 and c3.period == c3.lattice.period_y
    c4 = W.make_config(4, shrink=50)
    assert abs(c4.scale - 9.9225) < 1e-12 and c4.lattice.onsite is not None


@pytest.mark.parametrize("ncx,chains", [(7, 4), (16, 16), (5, 2)])
def test_zgnr_bit_exact_and_zigzag_edges(kgo, ncx, chains):
    """Zigzag ribbon (the paper's Fig. 4 system, "65536 x 16"): the two independent generators
    agree bit for bit; N = N_x N_y sites (N_x = 2 ncx dimer lines, N_y chains); both edges are
    zigzag — no site hangs on one bond (the open sheet's bearded edge), the 2 ncx sites of the outermost
    y rows have exactly two neighbours, every other site three; bipartite; the cut runs through the
    vertical bonds (width (3 N_y / 2 - 1) a)."""
    a, b = kgo.zgnr(ncx, chains), W.zgnr(ncx, chains)
    assert a.n == b.n == 2 * ncx * chains
    for f in ("nn", "nl", "hop", "x", "y"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    assert a.period_x == b.period_x and b.period_y == 0.0
    assert set(np.unique(b.nn)) <= {2, 3} and b.nn.min() >= 2
    edge = (b.y == b.y.min()) | (b.y == b.y.max())
    assert edge.sum() == 2 * ncx and np.all(b.nn[edge] == 2) and np.all(b.nn[~edge] == 3)
    assert abs((b.y.max() - b.y.min()) - (1.5 * chains - 1.0) * 0.142) < 1e-12
    nl = b.nl.reshape(3, b.n)
    i = np.broadcast_to(np.arange(b.n), (3, b.n))
    valid = np.arange(3)[:, None] < b.nn[None, :]
    dx = b.x[nl] - b.x[i]
    dx -= b.period_x * np.round(dx / b.period_x)
    bond = np.hypot(dx, b.y[nl] - b.y[i])[valid]
    assert np.max(np.abs(bond - 0.142)) < 1e-12                              # every bond has length a
    # symmetric adjacency
    pairs = set(zip(i[valid].tolist(), nl[valid].tolist()))
    assert all((m, n) in pairs for n, m in pairs)


def test_zgnr_config_counts():
    cfg = W.make_config(6, shrink=64)
    assert cfg.lattice.n == 1_048_576 // 64 and cfg.R == 1 and cfg.M == 2000
    assert abs(cfg.period - 65536 // 64 * np.sqrt(3.0) * 0.142 / 2) < 1e-9      # L_x = sqrt(3) N_x a / 2


@pytest.mark.parametrize("args", [(5, 4, True, True), (6, 3, False, True), (3, 5, True, False), (4, 4, False, False)])
def test_honeycomb_nnn_bit_exact(kgo, args):
    """Next-nearest-neighbour sheet (row width 9, two hopping values): the two generators agree bit for
    bit; on the torus every site has 3 first neighbours at distance a and 6 second neighbours at sqrt(3) a
    on its own sublattice; the adjacency is symmetric with equal hoppings both ways."""
    a, b = kgo.honeycomb_nnn(*args), W.honeycomb_nnn(*args)
    for f in ("nn", "nl", "hop", "x", "y"):
        assert np.array_equal(getattr(a, f), getattr(b, f)), f
    assert b.kmax == 9
    nl, hop = b.nl.reshape(9, b.n), b.hop.reshape(9, b.n)
    i = np.broadcast_to(np.arange(b.n), (9, b.n))
    valid = np.arange(9)[:, None] < b.nn[None, :]
    dx, dy = b.x[nl] - b.x[i], b.y[nl] - b.y[i]
    if b.period_x > 0:
        dx -= b.period_x * np.round(dx / b.period_x)
    if b.period_y > 0:
        dy -= b.period_y * np.round(dy / b.period_y)
    dist = np.hypot(dx, dy)
    first, second = valid & (hop == -2.7), valid & (hop == -0.27)
    assert np.all(first | second == valid)
    assert np.max(np.abs(dist[first] - 0.142)) < 1e-12 and np.max(np.abs(dist[second] - np.sqrt(3) * 0.142)) < 1e-12
    sub = (np.arange(b.n) & 1)                                   # b0, b2 on one sublattice, b1, b3 on the other
    assert np.all(sub[nl][first] != sub[i][first]) and np.all(sub[nl][second] == sub[i][second])
    if args[2] and args[3]:
        assert np.all(b.nn == 9) and np.all(first.sum(axis=0) == 3) and np.all(second.sum(axis=0) == 6)
    pairs = {(int(p), int(m)): float(v) for p, m, v in zip(i[valid], nl[valid], hop[valid])}
    assert all(pairs.get((m, p)) == v for (p, m), v in pairs.items())
