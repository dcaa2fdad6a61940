"""Full-size parity of BASELINE.json configs 2-5 against STORED oracle outputs, and long time loops
against the LIVE oracle.

Stored outputs: tests/golden/c<config>_<dos|vac|msd>_v<vector>.npz, written by
tests/golden/make_goldens.py from `oracle/` only (SURVEY.md 8(d) "Parity protocol"): per random
vector an M'-moment prefix at EVERY time step of the config, all M moments at the first / last time
step, and all M DOS moments.  The tests below run the FULL GPU jobs — every time step, every moment,
every vector of the batch, in the launch configuration bench.py times — and compare every stored
entry at 1e-10 (max-norm relative, BASELINE.json), row by row (each time step normalised by its own
largest magnitude, which is stricter than one norm for the whole table: MSD grows like t^2).

The live-oracle tests cover what the stored files cannot: every vector of a batch, R in {4, 8}, the
CUDA-graph / programmatic-dependent-launch / plain-launch variants, and the one-thread-per-element
kernels, each over tens to hundreds of consecutive time steps (ping-pong state buffers, alternating
sweep direction, Clenshaw recurrences, cached graph replay)."""
import ast
import os

import numpy as np
import pytest

from helpers import GOLDEN, relerr, to_oracle_lattice
from paper_1307_0288_b200 import workloads as W

pytestmark = pytest.mark.gpu
TOL = 1e-10


@pytest.fixture(scope="module")
def B():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_1307_0288_b200 import binding
    return binding


def dev(x):
    import torch
    return torch.from_numpy(np.ascontiguousarray(x)).cuda()


def host(t):
    return t.cpu().numpy()


def load_piece(name):
    path = os.path.join(GOLDEN, name + ".npz")
    assert os.path.exists(path), f"{path} missing: run tests/golden/make_goldens.py --piece {name}"
    d = np.load(path)
    return d, ast.literal_eval(str(d["meta"]))


def rowwise_err(got, want):
    """max over rows of (max |got - want| / max |want|); all-zero rows must match exactly."""
    worst = 0.0
    for g, w in zip(got, want):
        m = np.max(np.abs(w))
        d = np.max(np.abs(g - w))
        worst = max(worst, d / m if m > 0 else (0.0 if d == 0 else np.inf))
    return worst


# config 5 runs its 8 vectors as four column-pair planes: 0 / 7 are in the outer planes, 3 / 4 in the two middle
# ones, and both column positions of a plane are covered
VECTORS = {2: (0, 2, 3), 3: (0,), 4: (0,), 5: (0, 3, 4, 7), 6: (0,)}
WANTS = {2: ("vac", "msd"), 3: ("msd",), 4: ("vac", "msd"), 5: ("msd",), 6: ("msd",)}


@pytest.mark.parametrize("idx", [2, 3, 4, 5, 6])
def test_full_job_against_stored_oracle_outputs(B, idx):
    """The whole config — kg_dos_moments(M), kg_vac / kg_msd over ALL N_t time steps with ALL M
    moments, all R vectors in one batch — compared on every stored oracle entry.  idx 6 is the paper's
    own ballistic system, the zigzag ribbon 65536 x 16 of Fig. 4 (workloads.make_config(6))."""
    import torch
    cfg = W.make_config(idx)
    lat = cfg.lattice
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    phi = W.random_phase_vectors(lat.n, cfg.R, cfg.seed)
    dphi = dev(phi)
    stream = torch.cuda.Stream()                 # a capturable stream, as run_config uses
    with torch.cuda.stream(stream):
        dos = B.dos_moments(h, dphi, cfg.M)
        out = {job: (B.vac if job == "vac" else B.msd)(h, dphi, cfg.M, cfg.n_steps, cfg.dt_fs) for job in WANTS[idx]}
    stream.synchronize()
    dos = host(dos)
    out = {k: host(v) for k, v in out.items()}
    compared = 0
    for r in VECTORS[idx]:
        d, meta = load_piece(f"c{idx}_dos_v{r}")
        assert meta["n"] == lat.n and meta["M"] == cfg.M and meta["shrink"] == 1
        assert relerr(dos[r], d["mu"]) <= TOL
        compared += d["mu"].size
        for job in WANTS[idx]:
            d, meta = load_piece(f"c{idx}_{job}_v{r}")
            assert meta["n"] == lat.n and meta["nt"] == cfg.n_steps and meta["M"] == cfg.M
            assert abs(meta["dt_fs"] - cfg.dt_fs) < 1e-15 and abs(meta["scale"] - cfg.scale) < 1e-12
            got = out[job][r]
            assert got.shape == (cfg.n_steps + 1, cfg.M)
            Mp = meta["Mp"]
            assert d["prefix"].shape == (cfg.n_steps + 1, Mp)
            assert rowwise_err(got[:, :Mp], d["prefix"]) <= TOL, (job, r)
            assert rowwise_err(got[d["full_k"]], d["full"]) <= TOL, (job, r, "full rows")
            compared += d["prefix"].size + d["full"].size
            if job == "msd":
                assert np.all(got[0] == 0)                                      # eq 44 starts from psix_0 = 0
    print(f"config {idx}: {compared} stored oracle entries compared")


def _twin(idx, shrink):
    cfg = W.make_config(idx, shrink=shrink)
    return cfg, cfg.lattice


def test_config2_twin_all_200_steps_live_oracle(B, kgo):
    """Config 2 scaled down (50 x 50 cells, 0.5 % vacancies, R = 4) over ALL 200 time steps of the
    config, M' = 32 moments at every step, all four vectors, VAC and MSD, against the live oracle."""
    cfg, lat = _twin(2, 5)
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    phi = W.random_phase_vectors(lat.n, cfg.R, cfg.seed)
    Mp, nt = 32, cfg.n_steps
    assert nt == 200 and cfg.R == 4
    vac = host(B.vac(h, dev(phi), Mp, nt, cfg.dt_fs))
    msd = host(B.msd(h, dev(phi), Mp, nt, cfg.dt_fs))
    for r in range(cfg.R):
        v = phi[:, r].copy()
        assert rowwise_err(vac[r], kgo.vac(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, Mp, nt, cfg.dt_fs)) <= TOL
        assert rowwise_err(msd[r], kgo.msd(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, Mp, nt, cfg.dt_fs)) <= TOL


@pytest.fixture(scope="module")
def batched_case(kgo):
    """64 x 64 cells with vacancies and Anderson disorder, R = 8, 24 time steps, M' = 48: oracle
    tables for every vector, computed once and compared with each launch variant."""
    full = W.honeycomb(64, 64)
    lat = W.remove_sites(full, W.vacancy_mask(full.n, 80, 11))
    lat.onsite = W.anderson(lat.n, 2.7, 12)
    s = (3 * 2.7 + 1.35) * 1.05
    olat = to_oracle_lattice(kgo, lat)
    R, Mp, nt, dt = 8, 48, 24, 2 * W.HBAR / 2.7
    phi = W.random_phase_vectors(lat.n, R, 13)
    want_vac = np.stack([kgo.vac(olat, lat.x, lat.period_x, 0.0, s, phi[:, r].copy(), Mp, nt, dt) for r in range(R)])
    want_msd = np.stack([kgo.msd(olat, lat.x, lat.period_x, 0.0, s, phi[:, r].copy(), Mp, nt, dt) for r in range(R)])
    return lat, s, phi, Mp, nt, dt, want_vac, want_msd


@pytest.mark.parametrize("variant", ["default-side-stream", "graphs-off-pdl-off", "graphs-on-pdl-on", "one-thread-kernels",
                                     "literal-alg5-alg6"])
@pytest.mark.parametrize("R", [4, 8])
def test_batched_time_loops_launch_variants(B, batched_case, variant, R):
    import torch
    lat, s, phi, Mp, nt, dt, want_vac, want_msd = batched_case
    h = B.from_lattice(lat, lat.x, lat.period_x, 0.0, s)
    if variant == "graphs-off-pdl-off":
        h.set_option(B.KG_OPT_USE_GRAPHS, 0); h.set_option(B.KG_OPT_PDL, 0)
    elif variant == "graphs-on-pdl-on":
        h.set_option(B.KG_OPT_USE_GRAPHS, 1); h.set_option(B.KG_OPT_PDL, 1)
    elif variant == "one-thread-kernels":
        h.set_option(B.KG_OPT_STAGED, 0)
    elif variant == "literal-alg5-alg6":
        h.set_option(B.KG_OPT_DOUBLING, 0); h.set_option(B.KG_OPT_CLENSHAW, 0)
    dphi = dev(phi[:, :R])
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        vac = B.vac(h, dphi, Mp, nt, dt)
        msd = B.msd(h, dphi, Mp, nt, dt)
    stream.synchronize()
    vac, msd = host(vac), host(msd)
    for r in range(R):
        assert rowwise_err(vac[r], want_vac[r]) <= TOL, (variant, r)
        assert rowwise_err(msd[r], want_msd[r]) <= TOL, (variant, r)


def test_config4_twin_beyond_graph_and_pdl_thresholds(B, kgo):
    """Config 4 scaled down to 333 x 333 cells (443 556 sites: above the programmatic-dependent-launch
    threshold 2^18, with tiles spread over all CTAs) over 20 time steps, M' = 32 at every step and
    M = 600 at the last one, VAC and MSD against the live oracle."""
    cfg, lat = _twin(4, 3)
    assert lat.n > 1 << 18
    olat = to_oracle_lattice(kgo, lat)
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)
    phi = W.random_phase_vectors(lat.n, 1, cfg.seed)
    Mp, Mfull, nt = 32, 600, 20
    Mk = np.full(nt + 1, Mp); Mk[nt] = Mfull
    vac = host(B.vac(h, dev(phi), Mfull, nt, cfg.dt_fs))[0]
    msd = host(B.msd(h, dev(phi), Mfull, nt, cfg.dt_fs))[0]
    v = phi[:, 0].copy()
    want_vac = kgo.vac_sched(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, Mk, cfg.dt_fs)
    want_msd = kgo.msd_sched(olat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale, v, Mk, cfg.dt_fs)
    assert rowwise_err(vac[:, :Mp], want_vac[:, :Mp]) <= TOL
    assert rowwise_err(msd[:, :Mp], want_msd[:, :Mp]) <= TOL
    assert relerr(vac[nt], want_vac[nt]) <= TOL and relerr(msd[nt], want_msd[nt]) <= TOL
