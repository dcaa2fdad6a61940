#!/usr/bin/env python
"""bench.py — throughput of the Chebyshev hot path (arXiv 1307.0288) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl b200|reference]

One STEP = one pass of the whole hot path on the
BASELINE.json roofline configuration (config 4: 1000x1000 cells = 4,000,000 sites, Anderson
disorder W = |t|, 1 random-phase vector, M = 3000 moments, dt = 4 hbar/|t| => N_p = 42):

    kg_dos_moments(M)  +  kg_vac(M, n_steps = T)  +  kg_msd(M, n_steps = T)        (T = 1)

i.e. DOS moments, then the first T of the config's 100 correlation-time steps of the
Green-Kubo (VAC) and Einstein (MSD) loops.  Every time step of those loops does identical
work (2 evolutions + M-1 fused recursion+dot kernels), so the RATE (Gsite-updates/s) does not
depend on T; T = 1 keeps the default run within minutes.  `--time-steps 100` runs the full job.

Metric: Gsite-updates/s.  One site-update = one output element of H~ phi in one Chebyshev
step for one vector; a pair-commutator launch (a2+a6) counts as two.

N > 1 (torchrun): replicas only — the path does not shard (BASELINE.json: "no sharding, no
inter-GPU collectives").  Each rank runs the same step on its own random vector (the paper
averages 10-100 independent vectors, eq 21); the only exchange is the final average of
the [M] moment arrays (a few KB).  Weak scaling.

The JSON line carries `roofline` (dominant kernel, measured live with CUDA events on the
launching stream) and `cpu_baseline` (the oracle, as it stands, timed on the host cores on a
bounded sample of the same workload).  `--impl reference` times the oracle only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gsite-updates/s (H~.phi per Chebyshev step, fp64 complex)"
UNIT = "Gsite-updates/s"

# algorithmic bytes per site-update of the dominant kernel (fused recursion + moment dot,
# general ELL, K = 3): 48 (T_m, T_{m-1}, T_{m+1}) + 16 (phi_L) + (12 idx + 24 hop + 8 onsite)/R
# -- SURVEY.md 8(d), DESIGN.md "Roofline".
def mom_bytes_per_update(R: int, kmax: int = 3, phi_l_stream: bool = True) -> float:
    return 48.0 + (16.0 if phi_l_stream else 0.0) + (kmax * 12.0 + 8.0) / R


def must_move_bytes_per_update(R: int, kmax: int = 3, onsite: bool = True, dictionary: bool = True) -> float:
    """What the LAUNCHED doubling sweep has to move through HBM with no cache reuse between launches:
    T_m and T_{m-1} read, T_{m+1} written (48 B per element) + the matrix row shared by the R columns:
    4 B packed index per neighbour (the fp64 hopping rides in the index word when the hopping
    dictionary applies, else + 8 B) + 8 B on-site energy when the model has a diagonal."""
    return 48.0 + (kmax * (4.0 if dictionary else 12.0) + (8.0 if onsite else 0.0)) / R


def site_updates(n: int, R: int, M: int, nt: int, n_p: int, doubling: bool = False) -> dict:
    """H~-applications one step really performs.  The oracle runs the literal
    Alg. 5 (M-1 applications per moment set); the CUDA path gets two moments per sweep from the
    product identity: M/2 applications per set when phi_L = phi_R (DOS, MSD),
    2 * (M/2) for VAC rows k >= 1, whose sweep advances both phi_L and phi_R (row k = 0 has phi_L = phi_R and
    costs M/2); it is credited only with those."""
    per_set = M // 2 if doubling else M - 1
    dos = per_set
    # VAC: V phi once; per time point V psi_k + one moment set — at t = 0 phi_L = phi_R = V phi, so the
    # doubling path runs it on one column (no velocity application either: chi_0 is copied), later rows
    # advance both chains
    if doubling:
        vac = 1 + per_set + nt * (1 + 2 * per_set) + nt * 2 * (n_p - 1)
    else:
        vac = 1 + (nt + 1) * (1 + (M - 1)) + nt * 2 * (n_p - 1)
    # MSD row k = 0 is exactly 0 (psix_0 = 0) and is written, not computed: nt moment sets
    msd = nt * per_set + nt * 2 * (n_p - 1)
    per_vec = {"dos": dos, "vac": vac, "msd": msd}
    return {k: v * n * R for k, v in per_vec.items()}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def ncu_traffic(key: str):
    """dram bytes per launch of the dominant kernel from the committed ncu --set full summary."""
    p = os.path.join(ROOT, "profiles", "traffic.txt")
    if not os.path.exists(p):
        return None
    with open(p) as f:
        for line in f:
            parts = line.split("#")[0].split()
            if len(parts) >= 2 and parts[0] == key:
                return float(parts[1])
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc = index, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100", "-i", str(self.index)], stdout=subprocess.PIPE,
                stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "samples": len(sm),
                "reasons": sorted(reasons)}


# --------------------------------------------------------------------------------------
# oracle legs (cpu_baseline, --impl reference): the only places bench.py executes oracle/
# --------------------------------------------------------------------------------------
# SURVEY 8(d) "CPU baseline": K consecutive steps of recursion + dot (Alg. 5: kgo_apply_h, the
# axpy of l.6 and the long-double inner product of l.7) on the config's own lattice, one vector,
# single-threaded oracle as it stands.  The same sample in both legs; site-updates = the H~
# applications the oracle really executes (kgo_moments with M moments calls kgo_apply_h M - 1 times).
ORACLE_SAMPLE_M = 101


def oracle_step(cfg, olat, phi, m_sample=ORACLE_SAMPLE_M):
    from oracle import kgo
    kgo.moments(olat, cfg.e0, cfg.scale, phi, phi, m_sample)


def oracle_units(cfg, m_sample=ORACLE_SAMPLE_M):
    return (m_sample - 1) * cfg.lattice.n


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.lower().startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def oracle_inputs(cfg):
    from oracle import kgo
    from paper_1307_0288_b200 import workloads as W
    kgo.build()
    lat = cfg.lattice
    olat = kgo.Lattice(lat.n, lat.kmax, lat.nn, lat.nl, lat.hop, lat.onsite, lat.x, lat.y,
                       lat.period_x, lat.period_y)
    phi = W.random_phase_vectors(lat.n, 1, cfg.seed)[:, 0].copy()
    return olat, phi


def sample_text(cfg, m_sample=ORACLE_SAMPLE_M):
    return (f"{m_sample - 1} consecutive steps of recursion + dot (kgo_moments, literal Alg. 5: kgo_apply_h + axpy + "
            f"long-double inner product per step) on the {cfg.name} lattice ({cfg.lattice.n} sites), 1 vector, "
            f"1 thread of '{cpu_model()}' ({os.cpu_count()} logical cores on the host); site-updates = H~ applications "
            "the oracle executes")


def cpu_baseline_block(value, seconds, cfg):
    return {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "seconds": seconds,
            "cpu_model": cpu_model(), "host_cores_available": os.cpu_count(),
            "build": "gcc -O2 -ffp-contract=off, no OpenMP (oracle/kgo.py)", "sample": sample_text(cfg)}


def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    olat, phi = oracle_inputs(cfg)
    units = oracle_units(cfg)
    for _ in range(args.warmup):
        oracle_step(cfg, olat, phi)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_step(cfg, olat, phi)
    dt = time.perf_counter() - t0
    val = units * args.steps / dt / 1e9
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "c128 (fp64 complex)",
            "data": "synthetic", "config": workload_config(cfg, args, 1),
            "cpu_baseline": cpu_baseline_block(val, dt / args.steps, cfg),
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(cfg, args, n_ranks):
    return {"workload": f"BASELINE.json configs[{args.config - 1}] ({cfg.name}): {cfg.lattice.n} sites, "
                        f"R={cfg.R} vector(s) per GPU, M={cfg.M}, dt={cfg.dt_fs:.6g} fs; step = kg_dos_moments + "
                        f"kg_vac + kg_msd with {args.time_steps} of the config's {cfg.n_steps} time steps",
            "sites": cfg.lattice.n, "R": cfg.R, "M": cfg.M, "time_steps": args.time_steps,
            "parallelism": f"replicas x{n_ranks} (independent random vectors, no data-path collective)",
            "l2": f"inputs larger than L2: one moment sweep moves >= {80 * cfg.lattice.n * cfg.R / 1e6:.0f} MB vs 126 MB L2; no flush "
                  "(consecutive Chebyshev sweeps are the workload)"}


# --------------------------------------------------------------------------------------
# B200 arm
# --------------------------------------------------------------------------------------
def run_b200(args, cfg):
    import numpy as np
    import torch
    from paper_1307_0288_b200 import binding as B
    from paper_1307_0288_b200 import replicas
    from paper_1307_0288_b200 import workloads as W

    ctx = replicas.init_from_env("nccl")
    rank, world, local = ctx.rank, ctx.world, ctx.local_rank
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local)
    lat = cfg.lattice
    n, R, M, nt = lat.n, cfg.R, cfg.M, args.time_steps
    torch.cuda.synchronize()
    t_create = time.perf_counter()
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)      # synchronises (validation result)
    t_create = time.perf_counter() - t_create
    n_p, _ = B.bessel_terms(cfg.scale * cfg.dt_fs / W.HBAR)
    units = site_updates(n, R, M, nt, n_p, doubling=True)
    units_literal = sum(site_updates(n, R, M, nt, n_p).values())
    units_step = sum(units.values())

    # each rank its own random vectors (streams 16 + rank*R + r of the config's seed)
    own = replicas.vector_streams(rank, R)
    phi_np = W.random_phase_vectors(n, own.stop, cfg.seed)[:, own.start:own.stop].copy()
    phi_dev = torch.from_numpy(phi_np).cuda()
    mu_dos = torch.empty((R, M), dtype=torch.complex128, device="cuda")
    mu_vac = torch.empty((R, nt + 1, M), dtype=torch.complex128, device="cuda")
    mu_msd = torch.empty((R, nt + 1, M), dtype=torch.complex128, device="cuda")
    # end-to-end leg: pinned HOST buffers through the same C-ABI calls
    phi_host = torch.from_numpy(phi_np).pin_memory()
    mu_dos_h = torch.empty((R, M), dtype=torch.complex128).pin_memory()
    mu_vac_h = torch.empty((R, nt + 1, M), dtype=torch.complex128).pin_memory()
    mu_msd_h = torch.empty((R, nt + 1, M), dtype=torch.complex128).pin_memory()
    h2d = 3 * phi_host.numel() * 16
    d2h = (mu_dos_h.numel() + mu_vac_h.numel() + mu_msd_h.numel()) * 16

    def step_dev():
        B.dos_moments(h, phi_dev, M, mu=mu_dos)
        B.vac(h, phi_dev, M, nt, cfg.dt_fs, mu=mu_vac)
        B.msd(h, phi_dev, M, nt, cfg.dt_fs, mu=mu_msd)

    def step_host():
        B.dos_moments(h, phi_host, M, mu=mu_dos_h)
        B.vac(h, phi_host, M, nt, cfg.dt_fs, mu=mu_vac_h)
        B.msd(h, phi_host, M, nt, cfg.dt_fs, mu=mu_msd_h)

    stream = torch.cuda.current_stream()

    def timed(fn, k):
        """K steps bracketed by barrier + synchronize; device time by CUDA events on the launching
        stream; max over ranks."""
        torch.cuda.synchronize(); ctx.barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = h.launch_count
        e0.record(stream)
        for _ in range(k):
            fn()
        e1.record(stream)
        torch.cuda.synchronize(); ctx.barrier()
        return ctx.max_over_ranks(e0.elapsed_time(e1)), h.launch_count - l0

    # the first moments call of a handle also builds the two-step kernel's tile plans on the host (once per handle)
    t_first = None
    if args.warmup > 0:
        t_first = time.perf_counter()
        step_dev(); torch.cuda.synchronize()
        t_first = time.perf_counter() - t_first
    for _ in range(args.warmup - 1):
        step_dev()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ms, launches = timed(step_dev, args.steps)
    clocks = sampler.stop() if rank == 0 else None
    for _ in range(max(1, min(args.warmup, 1))):
        step_host()
    ms_e2e, _ = timed(step_host, args.steps)

    # trace average over the replicas' random vectors (eq 21): the only exchange
    mu_avg = ctx.mean_over_ranks(mu_dos.mean(dim=0))
    mu0 = complex(mu_avg[0].item())

    # The two moment kernels of the step, each timed as a DIFFERENCE OF TWO SERIES LENGTHS of the same call, so
    # that everything that does not scale with M cancels exactly — first step, final reduction, velocity, column
    # copies (including the re-layout copies of the column-pair planes on wider batches), the evolution — and
    # only pass launches remain, counted by the library's launch counter over the same two calls:
    #   one-column form (DOS, MSD rows, VAC row 0; MODE_MOM2 on R columns):  kg_dos_moments(M) - kg_dos_moments(M1)
    #   cross form (VAC rows k >= 1; MODE_MOMX on the batch [V psi_k | chi_k], 2R columns):
    #       [kg_vac(n_steps = 2, M) - kg_vac(1, M)] - [kg_vac(2, M1) - kg_vac(1, M1)]
    # All live CUDA events on the launching stream.  On the roofline config the passes are the TWO-STEP kernel
    # kg_tb2_kernel (T_m+1 and T_m+2 per pass, tile + two halo rings in shared memory); d(launches) against
    # d(Chebyshev steps) says which kernel ran.
    reps = 3
    C = 2 * R
    M1 = max(8, (M // 2) & ~3)

    def timed_calls(fn):
        fn(); torch.cuda.synchronize()
        l0 = h.launch_count
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(reps):
            fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e3 / reps, (h.launch_count - l0) // reps

    def vac_step(m):
        """time and launches of ONE more time step of kg_vac at series length m"""
        mu_v = [torch.empty((R, k + 1, m), dtype=torch.complex128, device="cuda") for k in (1, 2)]
        us1, l1 = timed_calls(lambda: B.vac(h, phi_dev, m, 1, cfg.dt_fs, mu=mu_v[0]))
        us2, l2 = timed_calls(lambda: B.vac(h, phi_dev, m, 2, cfg.dt_fs, mu=mu_v[1]))
        return us2 - us1, l2 - l1

    def dos_call(m):
        mu = torch.empty((R, m), dtype=torch.complex128, device="cuda")
        return timed_calls(lambda: B.dos_moments(h, phi_dev, m, mu=mu))

    dsteps = M // 2 - M1 // 2                            # Chebyshev steps between the two series lengths (doubling)
    (us_a, l_a), (us_b, l_b) = vac_step(M), vac_step(M1)
    momx_t = (us_a - us_b, l_a - l_b)
    (us_a, l_a), (us_b, l_b) = dos_call(M), dos_call(M1)
    mom2_t = (us_a - us_b, l_a - l_b)
    peak, peak_src = peaks()
    ons = lat.onsite is not None

    def kernel_block(mode, cols, d_us, d_launches):
        """roofline entry of one moment kernel: `d_launches` more launches performed `dsteps` more Chebyshev
        steps on `cols` columns in `d_us` more microseconds"""
        one_launch = d_launches <= 0                     # the whole loop is one cluster launch: no per-pass launches to count
        nl = 1 if one_launch else d_launches
        spl = dsteps / nl                                # Chebyshev steps per launch
        us = d_us / nl
        two = (not one_launch) and spl > 1.5
        if one_launch:
            kname = "kg_small_kernel (launch-bound size: all Chebyshev steps after the first in ONE cluster launch, vectors in distributed shared memory)"
        elif two:
            kname = (f"kg_tb2_kernel<C={min(cols, 2)}, K={lat.kmax}, {mode}, NSTEP=2> (two Chebyshev steps per pass: tile + two halo rings in "
                     "shared memory, TMA-staged streams, four inner products per pass"
                     + (f"; the {cols} columns as {cols // 2} column-pair planes side by side in one launch)" if cols > 2 else ")"))
        else:
            kname = (f"kg_staged_kernel<R={cols}, {mode}> (fused T_m+1 = 2H~T_m - T_m-1 + two inner products; TMA-staged streams, "
                     "hopping dictionary, alternating sweep)")
        if two:
            # must-move bytes of a two-step pass, per site: T_m, T_m-1 read and T_m+1, T_m+2 written (64 B per
            # column), 8 B of tile-local matrix row (4 x uint16) per plane of <= 2 columns, 8 B on-site energy per
            # plane; halo re-reads not counted
            planes = max(1, cols // 2)
            bl = (64.0 * cols + planes * (8.0 + (8.0 if ons else 0.0))) * n
            bdef = ("must-move bytes of the launched two-step pass: (64 C + 8 + 8) B per site and column-pair plane (T_m, T_m-1 read, "
                    "T_m+1, T_m+2 written for C columns; tile-local matrix row; on-site energy), no halo, no cache reuse between launches")
            tkey = f"{cfg.name}_tb2_{'momx' if mode == 'MODE_MOMX' else 'mom2'}_C{cols}"
        else:
            bl = must_move_bytes_per_update(cols, lat.kmax, ons) * n * cols * (spl if one_launch else 1.0)
            bdef = ("must-move bytes of the launched one-step sweep: (48 + (4 K + 8)/C) B per site-update (T_m, T_m-1 read, T_m+1 "
                    "written, packed index + on-site row shared by the C columns)"
                    + (" times the steps of the one launch (which keeps them in shared memory: not an HBM figure)" if one_launch else ""))
            tkey = f"{cfg.name}_{'momx' if mode == 'MODE_MOMX' else 'mom2'}_R{cols}"
        upd = n * cols * spl
        b8d = mom_bytes_per_update(cols, lat.kmax, phi_l_stream=False) * upd
        ach = bl / (us * 1e-6) / 1e9
        blk = {"bound": "hbm", "kernel": kname, "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
               "peak_source": peak_src, "frac_of_nominal_8TBs": ach / 8000.0, "bytes_per_launch": bl, "bytes_definition": bdef,
               "chebyshev_steps_per_launch": spl,
               "timed_as": f"difference of the same call at M = {M} and M = {M1}: {d_launches} launches, {dsteps} Chebyshev steps, {d_us:.1f} us",
               "survey_8d_general_ell": {"bytes_per_launch": b8d, "achieved": b8d / (us * 1e-6) / 1e9, "frac": b8d / (us * 1e-6) / 1e9 / peak,
                                         "note": "SURVEY 8(d) doubling row, 48 + (12 K + 8)/C B per site-update of a one-step sweep "
                                                 "with fp64 hoppings streamed, times the site-updates one launch performs; the launched "
                                                 "kernel moves far fewer bytes (two steps per pass, hopping dictionary), so this "
                                                 "fraction exceeds 1 - the roofline fraction is `frac`, on the bytes really required"},
               "us_per_launch": us, "gsu_per_s": upd / (us * 1e-6) / 1e9, "traffic": ncu_traffic(tkey)}
        if 48.0 * n * cols <= 126e6:
            blk["l2_resident"] = (f"T_m, T_m-1 and T_m+1 of the {cols} columns are {48.0 * n * cols / 1e6:.0f} MB and stay in the 126 MB L2 "
                                  "from launch to launch: this launch is not HBM-bound and `frac` is not a roofline fraction")
        elif blk["frac"] > 1.0:
            blk["warning"] = "frac > 1 against must-move bytes: the timed launches are not the kernel named here"
        return blk

    momx = kernel_block("MODE_MOMX", C, *momx_t)
    mom2 = kernel_block("MODE_MOM2", R, *mom2_t)
    # which of the two dominates: passes of a moment set of M moments x time per pass (the first step and the
    # reduction of every set are left out of the shares)
    sets_us = {"momx": (M // 2 - 1) / momx["chebyshev_steps_per_launch"] * momx["us_per_launch"],
               "mom2": (M // 2 - 1) / mom2["chebyshev_steps_per_launch"] * mom2["us_per_launch"]}
    t_momx = nt * sets_us["momx"]                                        # VAC rows k = 1 .. nt
    t_mom2 = (2 + nt) * sets_us["mom2"]                                  # DOS, VAC row 0, MSD rows 1 .. nt
    step_us = ms / args.steps * 1e3
    momx["share_of_step"] = t_momx / step_us
    mom2["share_of_step"] = t_mom2 / step_us
    roofline, other = (mom2, momx) if t_mom2 >= t_momx else (momx, mom2)
    roofline["second_kernel"] = other
    # the bench step runs T = --time-steps of the config's N_t time steps, which over-weights the one-column form
    # (DOS and VAC row 0 are once per job): the same two measured kernels weighted by the pass counts of the FULL
    # job, DOS + kg_vac(N_t) + kg_msd(N_t)
    jt_momx, jt_mom2 = cfg.n_steps * sets_us["momx"], (2 + cfg.n_steps) * sets_us["mom2"]
    roofline["job_weighted"] = {
        "n_steps": cfg.n_steps, "frac": (jt_momx * momx["frac"] + jt_mom2 * mom2["frac"]) / (jt_momx + jt_mom2),
        "moment_time_share": {"MODE_MOMX": jt_momx / (jt_momx + jt_mom2), "MODE_MOM2": jt_mom2 / (jt_momx + jt_mom2)},
        "note": "time-weighted mean of the two kernels' roofline fractions over the moment passes of the config's full job "
                "(= their must-move bytes / their time / peak); evolutions not included"}

    if rank != 0:
        ctx.finalize()
        return
    value = units_step * world * args.steps / (ms * 1e-3) / 1e9
    e2e = units_step * world * args.steps / (ms_e2e * 1e-3) / 1e9
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "c128 (fp64 complex)", "data": "synthetic",
            "config": workload_config(cfg, args, world),
            "site_updates_per_step_per_gpu": units,
            "literal_alg5_equivalent": {"site_updates_per_step_per_gpu": units_literal,
                                        "value": units_literal * world * args.steps / (ms * 1e-3) / 1e9,
                                        "note": "what the same outputs cost with M-1 sweeps per moment set (Alg. 5 as "
                                                "written); value above counts only the sweeps really launched"}, "n_p": n_p, "mu0_trace_average": [mu0.real, mu0.imag],
            "clocks": clocks,
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                    "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": int(launches),
            "setup": {"create_s": t_create, "first_step_s": t_first, "steady_step_s": ms / args.steps * 1e-3,
                      "note": "once per handle, outside the timed region: kg_create_hamiltonian from host arrays (H2D copy, site "
                              "re-ordering on the host, validation + scaling + dictionary on the device); the first step also builds "
                              "the tile plans of the two-step kernel and sizes the workspace"},
            "roofline": roofline}
    if world == 1 and not args.no_cpu_baseline:
        olat, phi1 = oracle_inputs(cfg)
        oracle_step(cfg, olat, phi1, 3)                      # touch the pages once
        t0 = time.perf_counter()
        oracle_step(cfg, olat, phi1)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = cpu_baseline_block(oracle_units(cfg) / dt / 1e9, dt, cfg)
    print(json.dumps(line), flush=True)
    ctx.finalize()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json config index 1..5 (default 4, the roofline config)")
    ap.add_argument("--time-steps", type=int, default=1, help="correlation-time steps of kg_vac / kg_msd per bench step")
    ap.add_argument("--shrink", type=int, default=1, help="divide the lattice's linear size (debug only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        print("note: warmup < 3 violates the timing rules; use only for debugging", file=sys.stderr)
    from paper_1307_0288_b200 import workloads as W
    cfg = W.make_config(args.config, shrink=args.shrink)
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_b200(args, cfg)


if __name__ == "__main__":
    main()
