"""N > 1 path on CPU: two processes over gloo exercise the replica plumbing that bench.py uses
under torchrun (rank bookkeeping, vector ownership, max / mean over ranks) and the
site-update accounting.  No GPU, no kg_* compute calls."""
import os
import socket
import sys

import numpy as np
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1307_0288_b200 import replicas
    from paper_1307_0288_b200 import workloads as W
    ctx = replicas.init_from_env("gloo")
    assert (ctx.rank, ctx.world) == (rank, world)
    R = 2
    own = replicas.vector_streams(rank, R)
    # a rank's vectors are the global vector set's columns rank*R .. rank*R+R-1
    allv = W.random_phase_vectors(64, world * R, 7)
    mine = W.random_phase_vectors(64, own.stop, 7)[:, own.start:own.stop]
    assert mine.tobytes() == np.ascontiguousarray(allv[:, own.start:own.stop]).tobytes()
    ctx.barrier()
    tmax = ctx.max_over_ranks(10.0 + rank)
    tsum = ctx.sum_over_ranks(1.5)
    mu = torch.tensor([1.0 + rank, 2.0j * (rank + 1)], dtype=torch.complex128)
    avg = ctx.mean_over_ranks(mu)
    torch.save({"tmax": tmax, "tsum": tsum, "avg": avg, "own": list(own)},
               os.path.join(out_dir, f"r{rank}.pt"))
    ctx.finalize()


def test_two_rank_replicas_gloo(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    res = [torch.load(os.path.join(tmp_path, f"r{r}.pt")) for r in range(world)]
    for r in res:
        assert r["tmax"] == 11.0                      # slowest rank
        assert r["tsum"] == 3.0
        assert torch.allclose(r["avg"], torch.tensor([1.5, 3.0j], dtype=torch.complex128))
    assert res[0]["own"] == [0, 1] and res[1]["own"] == [2, 3]


def test_single_process_context_needs_no_process_group():
    sys.path.insert(0, ROOT)
    from paper_1307_0288_b200 import replicas
    for k in ("RANK", "WORLD_SIZE", "LOCAL_RANK"):
        os.environ.pop(k, None)
    ctx = replicas.init_from_env("gloo")
    assert ctx.world == 1 and ctx.max_over_ranks(3.0) == 3.0
    mu = torch.tensor([1 + 2j], dtype=torch.complex128)
    assert torch.equal(ctx.mean_over_ranks(mu), mu)


def test_site_update_accounting_matches_survey_table():
    """H-applications per vector for DOS / VAC~MSD on the five configs
    (C1 255 / 4 975, C2 999 / 211 599, C3 1 999 / 817 599, C4 2 999 / 311 099, C5 2 999 / 158 549).
    bench.site_updates counts the launches the library actually makes; VAC adds the velocity
    applications (1 + one per time row), which the survey's round figure leaves out, and MSD skips
    the M - 1 applications of row k = 0, whose moments are exactly 0 (psix_0 = 0) and are written
    without being computed."""
    sys.path.insert(0, ROOT)
    import bench
    table = {1: (256, 16, 21, 255, 4975), 2: (1000, 200, 28, 999, 211599), 3: (2000, 400, 21, 1999, 817599),
             4: (3000, 100, 42, 2999, 311099), 5: (3000, 50, 57, 2999, 158549)}
    for _, (M, nt, n_p, dos, corr) in table.items():
        u = bench.site_updates(1, 1, M, nt, n_p)
        assert u["dos"] == dos
        assert u["msd"] == corr - (M - 1)
        assert u["vac"] == corr + 1 + (nt + 1)
