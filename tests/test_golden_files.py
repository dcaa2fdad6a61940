"""The stored oracle outputs (tests/golden/c*_*.npz, written by tests/golden/make_goldens.py from
oracle/ only): every piece the GPU comparison needs is there, says where it came from, and is
consistent with what the mathematics fixes — the M'-prefix stored at the first / last time step is bit
for bit the head of the full row stored for that step (moments do not depend on how many are asked
for), mu_0 = 1 for the unit-norm vector, |mu_m| <= 1, the DOS moments are real, MSD starts from 0 and
its zeroth moment ||psix_k||^2 grows."""
import ast
import hashlib
import os

import numpy as np
import pytest

from helpers import GOLDEN

PIECES = {2: ("dos", "vac", "msd"), 3: ("dos", "msd"), 4: ("dos", "vac", "msd"), 5: ("dos", "msd"), 6: ("dos", "msd")}
VECTORS = {2: (0, 2, 3), 3: (0,), 4: (0,), 5: (0, 3, 4, 7), 6: (0,)}
SHAPES = {2: (248750, 1000, 200, 64), 3: (1200000, 2000, 400, 64), 4: (4000000, 3000, 100, 64),
          5: (15984000, 3000, 50, 16), 6: (1048576, 2000, 400, 64)}


def load(name):
    d = np.load(os.path.join(GOLDEN, name + ".npz"))
    return d, ast.literal_eval(str(d["meta"]))


def _arith_sha256_today():
    """sha256 of oracle/kgo.c from its first operator function to the end: everything the stored numbers are
    computed by (the generators above it are pinned bit for bit by tests/test_generators.py)."""
    src = open(os.path.join(os.path.dirname(GOLDEN), os.pardir, "oracle", "kgo.c"), "rb").read()
    return hashlib.sha256(src[src.index(b"static double kgo_bond_dx"):]).hexdigest()


def _recorded_versions():
    """tests/golden/oracle_versions.txt: file sha256 -> arithmetic sha256 of the kgo.c versions that wrote files
    before the files recorded the arithmetic hash themselves (make_goldens.py --record-versions)."""
    table = {}
    with open(os.path.join(GOLDEN, "oracle_versions.txt")) as f:
        for line in f:
            w = line.split("#")[0].split()
            if len(w) >= 2:
                table[w[0]] = w[1]
    return table


def test_stored_outputs_were_written_by_todays_oracle_arithmetic():
    """Every stored file was written by a kgo.c whose operators, recursions, series and drivers are byte for
    byte today's: if the oracle's arithmetic is changed after a file was written this fails until the file is
    regenerated, so the GPU is never compared with numbers the current oracle would not produce."""
    today, table = _arith_sha256_today(), _recorded_versions()
    files = sorted(f for f in os.listdir(GOLDEN) if f.endswith(".npz"))
    assert len(files) >= 24
    for name in files:
        meta = ast.literal_eval(str(np.load(os.path.join(GOLDEN, name))["meta"]))
        wrote = meta.get("oracle_arith_sha256") or table.get(meta["oracle_kgo_c_sha256"])
        assert wrote is not None, f"{name}: kgo.c version {meta['oracle_kgo_c_sha256'][:12]} is not in oracle_versions.txt"
        assert wrote == today, f"{name} was written by a different oracle arithmetic: regenerate it (make_goldens.py --piece {name[:-4]})"


@pytest.mark.parametrize("idx", [2, 3, 4, 5, 6])
def test_stored_oracle_outputs(idx):
    n, M, nt, Mp = SHAPES[idx]
    for r in VECTORS[idx]:
        for job in PIECES[idx]:
            d, meta = load(f"c{idx}_{job}_v{r}")
            assert meta["written_by"] == "tests/golden/make_goldens.py" and meta["shrink"] == 1
            assert (meta["n"], meta["M"], meta["nt"], meta["Mp"], meta["vector"]) == (n, M, nt, Mp, r)
            assert len(meta["oracle_kgo_c_sha256"]) == 64 and len(meta["phi_sha256"]) == 64 and len(meta["git_commit"]) >= 7
            if job == "dos":
                mu = d["mu"]
                assert mu.shape == (M,) and abs(mu[0] - 1.0) < 1e-12
                assert np.max(np.abs(mu)) <= 1.0 + 1e-12 and np.max(np.abs(mu.imag)) < 1e-12
                continue
            prefix, full, full_k = d["prefix"], d["full"], d["full_k"]
            assert prefix.shape == (nt + 1, Mp) and full.shape == (len(full_k), M)
            assert list(full_k) == ([0, nt] if job == "vac" else [nt])
            for row, k in zip(full, full_k):
                assert row[:Mp].tobytes() == prefix[k].tobytes()
            assert np.all(np.isfinite(prefix.view(float))) and np.all(np.isfinite(full.view(float)))
            if job == "msd":
                assert np.all(prefix[0] == 0)                                  # eq 44 starts from psix_0 = 0
                norm2 = prefix[:, 0].real                                       # mu_0(t_k) = ||psix_k||^2
                assert np.all(norm2[1:] > 0) and np.all(np.abs(prefix[:, 0].imag) < 1e-12 * norm2.max())
                assert np.all(np.abs(prefix[1:]) <= norm2[1:, None] * (1 + 1e-12))    # |<x|T_m|x>| <= ||x||^2
            else:
                assert np.all(np.abs(prefix[:, 0]) > 0)
