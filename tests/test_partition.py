"""Host logic of the site re-ordering done at create (csrc/kg_partition.h), on the CPU: the order is a
permutation, aligned power-of-two ranges are compact patches (few bonds leave them), and the grouped form
keeps every site's caller index modulo 8 (what makes the shared-memory gathers of a staged tile bank-conflict
free).  The header is plain C++: it is compiled here with g++ into a small command-line tool."""
import os
import subprocess

import numpy as np
import pytest

from paper_1307_0288_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def cli(tmp_path_factory):
    exe = str(tmp_path_factory.mktemp("partition") / "partition_cli")
    subprocess.run(["g++", "-O2", "-std=c++17", "-o", exe, os.path.join(HERE, "native", "partition_cli.cpp")], check=True)
    return exe


def run(cli, lat, leaf, group, tmp_path):
    fin, fout = str(tmp_path / "in.bin"), str(tmp_path / "out.bin")
    with open(fin, "wb") as f:
        f.write(np.ascontiguousarray(lat.nn, dtype=np.int32).tobytes())
        f.write(np.ascontiguousarray(lat.nl, dtype=np.int32).tobytes())
    subprocess.run([cli, str(lat.n), str(lat.kmax), str(leaf), str(group), fin, fout], check=True)
    return np.fromfile(fout, dtype=np.int32)


def leaving_fraction(lat, perm, block):
    """fraction of bonds whose two ends lie in different aligned blocks of `block` internal sites"""
    iperm = np.empty(lat.n, dtype=np.int64)
    iperm[perm] = np.arange(lat.n)
    nl = lat.nl.reshape(lat.kmax, lat.n).astype(np.int64)
    valid = np.arange(lat.kmax)[:, None] < lat.nn[None, :]
    a = (iperm[None, :] // block).repeat(lat.kmax, axis=0)
    b = iperm[nl] // block
    return float(np.mean((a != b)[valid]))


@pytest.mark.parametrize("group", [1, 8])
def test_partition_is_a_compact_permutation(cli, tmp_path, group):
    lat = W.honeycomb(200, 40)                     # 32 000 sites, row-major cells: a 512-site range is part of one cell row
    perm = run(cli, lat, 64, group, tmp_path)
    assert np.array_equal(np.sort(perm), np.arange(lat.n))
    before = leaving_fraction(lat, np.arange(lat.n), 512)
    after = leaving_fraction(lat, perm, 512)
    assert before > 0.30                           # caller order: every third bond leaves its 512-site strip
    assert after < 0.12                            # compact patch of 512 sites: perimeter / area
    assert leaving_fraction(lat, perm, 1024) < after      # larger aligned ranges are compact too
    if group == 8:
        assert np.array_equal(perm % 8, np.arange(lat.n) % 8)      # caller index modulo 8 is kept


def test_partition_grouped_ragged_and_disconnected(cli, tmp_path):
    """n not a multiple of 8 (the trailing partial octet stays last), vacancies (irregular degrees) and two
    disconnected components."""
    full = W.honeycomb(40, 36, periodic_x=False, periodic_y=False)
    lat = W.remove_sites(full, W.vacancy_mask(full.n, 35, 7))       # 5725 sites = 715 octets + 5
    assert lat.n % 8 == 5
    perm = run(cli, lat, 64, 8, tmp_path)
    assert np.array_equal(np.sort(perm), np.arange(lat.n))
    assert np.array_equal(perm[: lat.n // 8 * 8] % 8, np.arange(lat.n // 8 * 8) % 8)
    assert np.array_equal(perm[lat.n // 8 * 8:], np.arange(lat.n // 8 * 8, lat.n))
    assert leaving_fraction(lat, perm, 512) < 0.15
    # two copies of a ribbon side by side, no bonds between them
    a = W.honeycomb(8, 64, periodic_x=False, periodic_y=True)
    nl2 = np.concatenate([a.nl.reshape(3, a.n), a.nl.reshape(3, a.n) + a.n], axis=1).reshape(-1)
    two = W.Lattice(2 * a.n, 3, np.concatenate([a.nn, a.nn]), nl2.astype(np.int32), np.concatenate([a.hop.reshape(3, a.n)] * 2, axis=1).reshape(-1),
                    None, np.concatenate([a.x, a.x]), np.concatenate([a.y, a.y]), 0.0, a.period_y)
    perm = run(cli, two, 64, 8, tmp_path)
    assert np.array_equal(np.sort(perm), np.arange(two.n))
