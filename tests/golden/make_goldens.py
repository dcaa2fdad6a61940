#!/usr/bin/env python
"""Writes the stored oracle outputs (tests/golden/c*_*.npz) for BASELINE.json configs 2-5 and the paper's ZGNR (config 6 of workloads.make_config).

    python tests/golden/make_goldens.py --all --jobs 6         # every piece, 6 oracle processes
    python tests/golden/make_goldens.py --piece c4_msd_v0      # one piece in this process

Calls ONLY `oracle/` (the plain C oracle and its own lattice / vacancy / Anderson / random-number
generators — bit-identical to the product's numpy generators by tests/test_generators.py) and numpy.
Nothing here imports, reads or runs the CUDA path, and no stored value comes from it.

What is stored follows SURVEY.md 8(d) "Parity protocol": the single-threaded oracle cannot finish the
full jobs of configs 3-5 in reasonable time, but Chebyshev moments do not depend on how many are asked
for (only the Jackson damping does), so the oracle runs ALL time steps of each config and tabulates

  * a prefix of M' moments at EVERY time step t_k, k = 0..N_t      (`prefix`  [N_t+1][M'])
  * all M moments at the first and the last time step               (`full`    [len(full_k)][M])
  * all M DOS moments                                               (`mu`      [M])

per random vector.  tests/test_gpu_goldens.py runs the FULL GPU jobs and compares every stored entry.

config | lattice                                   | vectors | M    | N_t | M'
   2   | 250x250 cells, 0.5 % vacancies (seed 1)   | 0, 2, 3 | 1000 | 200 | 64
   3   | AGNR 15 x 20000 cells                     | 0       | 2000 | 400 | 64
   4   | 1000x1000 cells, Anderson W=|t| (seed 2)  | 0       | 3000 | 100 | 64
   5   | 2000x2000 cells, 0.1 % vacancies (seed 3) | 0,3,4,7 | 3000 |  50 | 16
   6   | ZGNR 65536 x 16 (the paper's Fig. 4)      | 0       | 2000 | 400 | 64

(Config 5's vectors 3 and 4 sit in the two middle column-pair planes of the GPU's wide-batch path, one in
each column position; 0 and 7 in the outer planes.)

Every file records the sha256 of oracle/kgo.c, the git commit of the tree that wrote it, the config
parameters and the sha256 of the random vector's bytes.  Files written from round 3 on also record
`oracle_arith_sha256`, the sha256 of kgo.c from `kgo_bond_dx` to the end of the file — everything the
stored numbers are computed by (operators, recursions, Bessel series, drivers), without the lattice /
random-number generators above it, which tests/test_generators.py pins bit for bit on their own.  For the
files written before that, `--record-versions` recomputes the same hash from the recorded git commit and
writes tests/golden/oracle_versions.txt (`file sha256, arithmetic sha256, commit` per kgo.c version that
wrote a stored file).  tests/test_golden_files.py compares these with today's kgo.c: a change to the
oracle's arithmetic after a file was written fails there until the file is regenerated.
Host time on 8 cores: about 2.5 h.
"""
from __future__ import annotations

import argparse
import hashlib
import os
import subprocess
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

T = 2.7                     # |t| = gamma_0, eV (eq 13)
HBAR = 0.6582119569         # eV fs

# name: (vectors, M, N_t, dt in units of hbar/|t|, M', wants)
CONFIGS = {
    2: dict(vectors=(0, 2, 3), M=1000, nt=200, dt_mult=2, Mp=64, seed=1, wants=("dos", "vac", "msd")),
    3: dict(vectors=(0,), M=2000, nt=400, dt_mult=1, Mp=64, seed=0, wants=("dos", "msd")),
    4: dict(vectors=(0,), M=3000, nt=100, dt_mult=4, Mp=64, seed=2, wants=("dos", "vac", "msd")),
    5: dict(vectors=(0, 3, 4, 7), M=3000, nt=50, dt_mult=8, Mp=16, seed=3, wants=("dos", "msd")),
    6: dict(vectors=(0,), M=2000, nt=400, dt_mult=1, Mp=64, seed=0, wants=("dos", "msd")),
}


def lattice(idx, shrink=1):
    """BASELINE.json configs[idx-1] from the oracle's own generators (DESIGN.md section 3 recipe).
    Returns (lattice, transport coordinate, its period, scale s)."""
    from oracle import kgo
    s = 3 * T * 1.05
    if idx == 2:
        full = kgo.honeycomb(250 // shrink, 250 // shrink)
        nv = int(np.floor(0.005 * full.n + 0.5))
        lat = kgo.remove_sites(full, kgo.vacancy_mask(full.n, nv, 1))
        return lat, lat.x, lat.period_x, s
    if idx == 3:
        lat = kgo.honeycomb(15, 20000 // shrink, periodic_x=False, periodic_y=True)
        return lat, lat.y, lat.period_y, s
    if idx == 4:
        lat = kgo.honeycomb(1000 // shrink, 1000 // shrink)
        lat.onsite = kgo.anderson(lat.n, T, 2)
        return lat, lat.x, lat.period_x, (3 * T + T / 2) * 1.05
    if idx == 5:
        full = kgo.honeycomb(2000 // shrink, 2000 // shrink)
        nv = int(np.floor(0.001 * full.n + 0.5))
        lat = kgo.remove_sites(full, kgo.vacancy_mask(full.n, nv, 3))
        return lat, lat.x, lat.period_x, s
    if idx == 6:
        lat = kgo.zgnr(32768 // shrink, 16)
        return lat, lat.x, lat.period_x, s
    raise ValueError(idx)


def random_phase(n, seed, r):
    """phi_j = exp(2 pi i u_j)/sqrt(n), u_j = u(seed, 16 + r, j) from the oracle's generator (g1, g19)."""
    from oracle import kgo
    ang = 2.0 * np.pi * kgo.phase_uniforms(n, seed, r)
    return (np.cos(ang) + 1j * np.sin(ang)) * (1.0 / np.sqrt(float(n)))


def pieces(shrink=1):
    out = []
    for idx, c in CONFIGS.items():
        for r in c["vectors"]:
            for job in c["wants"]:
                out.append(f"c{idx}_{job}_v{r}")
    return out


def cost(piece):
    """Rough oracle cost (H-type sweeps x sites) used to start the longest pieces first."""
    idx, job = int(piece[1]), piece.split("_")[1]
    c = CONFIGS[idx]
    n = {2: 0.25e6, 3: 1.2e6, 4: 4e6, 5: 16e6, 6: 1.05e6}[idx]
    n_p = {2: 28, 3: 21, 4: 42, 5: 57, 6: 21}[idx]
    if job == "dos":
        return n * c["M"]
    per_step = (5 if job == "msd" else 2) * n_p + c["Mp"]
    return n * (c["nt"] * per_step + 2 * c["M"])


ARITH_START = b"static double kgo_bond_dx"      # first function of kgo.c after the generators


def arith_sha256(src: bytes) -> str:
    """sha256 of kgo.c from its first operator function to the end (see the module docstring)."""
    return hashlib.sha256(src[src.index(ARITH_START):]).hexdigest()


def provenance():
    with open(os.path.join(ROOT, "oracle", "kgo.c"), "rb") as f:
        src = f.read()
    osha = hashlib.sha256(src).hexdigest()
    try:
        commit = subprocess.run(["git", "-C", ROOT, "rev-parse", "HEAD"], capture_output=True, text=True,
                                check=True).stdout.strip()
    except Exception:
        commit = "unknown"
    return osha, arith_sha256(src), commit


def record_versions(outdir):
    """tests/golden/oracle_versions.txt: for every (kgo.c sha256, git commit) recorded in a stored file,
    the arithmetic hash of kgo.c AS IT WAS at that commit (read with `git show`)."""
    import ast
    seen = {}
    for name in sorted(os.listdir(outdir)):
        if name.endswith(".npz"):
            meta = ast.literal_eval(str(np.load(os.path.join(outdir, name))["meta"]))
            seen[meta["oracle_kgo_c_sha256"]] = meta["git_commit"]
    lines = ["# kgo.c versions that wrote the stored oracle outputs: file sha256, sha256 from kgo_bond_dx to the end, commit",
             "# written by tests/golden/make_goldens.py --record-versions (git show <commit>:oracle/kgo.c)"]
    for osha, commit in sorted(seen.items(), key=lambda kv: kv[1]):
        src = subprocess.run(["git", "-C", ROOT, "show", f"{commit}:oracle/kgo.c"], capture_output=True, check=True).stdout
        if hashlib.sha256(src).hexdigest() != osha:      # written from a tree with uncommitted changes to kgo.c
            with open(os.path.join(ROOT, "oracle", "kgo.c"), "rb") as f:
                src = f.read()
            assert hashlib.sha256(src).hexdigest() == osha, f"kgo.c with sha256 {osha} is neither at {commit} nor in the tree"
        lines.append(f"{osha} {arith_sha256(src)} {commit}")
    with open(os.path.join(outdir, "oracle_versions.txt"), "w") as f:
        f.write("\n".join(lines) + "\n")
    print("\n".join(lines))


def run_piece(piece, outdir, shrink=1, nt_override=None):
    from oracle import kgo
    kgo.build()
    cname, job, vname = piece.split("_")
    idx, r = int(cname[1:]), int(vname[1:])
    c = CONFIGS[idx]
    t0 = time.time()
    lat, xc, period, s = lattice(idx, shrink)
    phi = random_phase(lat.n, c["seed"], r)
    M, Mp = c["M"], c["Mp"]
    nt = c["nt"] if nt_override is None else nt_override
    dt = c["dt_mult"] * HBAR / T
    osha, asha, commit = provenance()
    meta = dict(config=idx, vector=r, n=lat.n, M=M, Mp=Mp, nt=nt, dt_fs=dt, scale=s, e0=0.0, seed=c["seed"],
                shrink=shrink, phi_sha256=hashlib.sha256(phi.tobytes()).hexdigest(), oracle_kgo_c_sha256=osha, oracle_arith_sha256=asha,
                git_commit=commit, written_by="tests/golden/make_goldens.py")
    arrays = {}
    if job == "dos":
        arrays["mu"] = kgo.dos_moments(lat, 0.0, s, phi, M)
    else:
        # all time steps with the M' prefix; full rows at both ends (MSD row 0 is exactly 0: eq 44
        # starts from psix_0 = 0, so only the last row is stored in full for it)
        Mk = np.full(nt + 1, Mp, np.int32)
        full_k = [0, nt] if job == "vac" else [nt]
        for k in full_k:
            Mk[k] = M
        fn = kgo.vac_sched if job == "vac" else kgo.msd_sched
        tab = fn(lat, xc, period, 0.0, s, phi, Mk, dt)
        arrays["prefix"] = np.ascontiguousarray(tab[:, :Mp])
        arrays["full_k"] = np.asarray(full_k, np.int32)
        arrays["full"] = np.ascontiguousarray(tab[full_k, :M])
    meta["oracle_seconds"] = round(time.time() - t0, 1)
    os.makedirs(outdir, exist_ok=True)
    path = os.path.join(outdir, piece + ".npz")
    np.savez_compressed(path, meta=np.array(repr(meta)), **arrays)
    print(f"{piece}: {meta['oracle_seconds']} s -> {path}", flush=True)


def main():
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--piece", help="e.g. c4_msd_v0")
    ap.add_argument("--all", action="store_true")
    ap.add_argument("--jobs", type=int, default=4, help="oracle processes run side by side with --all")
    ap.add_argument("--out", default=HERE)
    ap.add_argument("--shrink", type=int, default=1, help="debug: divide the linear size of the lattices")
    ap.add_argument("--time-steps", type=int, default=None, help="debug: override N_t")
    ap.add_argument("--skip-existing", action="store_true")
    ap.add_argument("--record-versions", action="store_true", help="write oracle_versions.txt from the stored files and git")
    args = ap.parse_args()
    if args.record_versions:
        record_versions(args.out)
        return
    if args.piece:
        run_piece(args.piece, args.out, args.shrink, args.time_steps)
        return
    if not args.all:
        ap.error("give --piece NAME or --all")
    from oracle import kgo
    kgo.build()
    todo = sorted(pieces(), key=cost, reverse=True)
    if args.skip_existing:
        todo = [p for p in todo if not os.path.exists(os.path.join(args.out, p + ".npz"))]
    running = []
    while todo or running:
        while todo and len(running) < args.jobs:
            p = todo.pop(0)
            cmd = [sys.executable, os.path.abspath(__file__), "--piece", p, "--out", args.out,
                   "--shrink", str(args.shrink)]
            if args.time_steps is not None:
                cmd += ["--time-steps", str(args.time_steps)]
            running.append((p, subprocess.Popen(cmd)))
        time.sleep(2)
        for p, proc in list(running):
            if proc.poll() is not None:
                running.remove((p, proc))
                if proc.returncode != 0:
                    raise SystemExit(f"piece {p} failed with exit code {proc.returncode}")


if __name__ == "__main__":
    main()
