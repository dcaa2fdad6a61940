"""Run one BASELINE.json configuration in full through the C-ABI library and post-process it.

    python -m paper_1307_0288_b200.run_config --config 4 [--out DIR] [--time-steps N]

For the chosen config (1..5, `workloads.make_config`) this computes what BASELINE.json lists as its
outputs — DOS moments, VAC and/or MSD moments over all its correlation-time steps — then, still
on the device, the KPM reconstructions on the config's energy grid (eqs 29-31, 35), the running
conductivities sigma_GK / sigma_E1 / sigma_E2 in e^2/h (eqs 6, 9, 11) and, for the ribbon, the
ballistic conductance (eqs 50-51).  It prints one JSON line with timings (`setup_s` = synthetic lattice and vectors generated with numpy on the
host + `create_s`, the kg_create_hamiltonian call alone) and a few physical
sanity numbers (integral of the DOS, Einstein vs Green-Kubo agreement, conductance near the band
centre) and, with --out, saves the arrays as a compressed .npz.

Only argument marshalling and bookkeeping happen here; every number comes from the CUDA kernels
behind include/kg.h.  Needs a GPU.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

# which correlation functions each config asks for (BASELINE.json "configs")
WANTS = {1: ("dos", "vac", "msd"), 2: ("dos", "vac", "msd"), 3: ("dos", "msd"),
         4: ("dos", "vac", "msd"), 5: ("dos", "msd"), 6: ("dos", "msd")}
A_NM = 0.142
GRAPHENE_DENS = 8.0 / (3.0 * np.sqrt(3.0) * A_NM ** 2)      # 2N/Omega of a honeycomb sheet, nm^-2


def main(argv=None):
    ap = argparse.ArgumentParser(description=__doc__.split("\n\n")[0])
    ap.add_argument("--config", type=int, required=True, choices=[1, 2, 3, 4, 5, 6],
                    help="BASELINE.json config 1..5, or 6 = the paper's ZGNR 65536 x 16 (Fig. 4)")
    ap.add_argument("--time-steps", type=int, default=None, help="override the config's number of time steps")
    ap.add_argument("--moments", type=int, default=None, help="override the config's M")
    ap.add_argument("--out", default=None, help="directory for <config name>.npz")
    ap.add_argument("--no-warmup", action="store_true", help="skip the untimed warm-up calls (one moment set per call, "
                    "one post-processing pass: module loading, workspace and plan allocation)")
    args = ap.parse_args(argv)

    import torch
    from . import binding as B
    from . import workloads as W

    assert torch.cuda.is_available(), "run_config needs a CUDA device (there is no CPU fallback)"
    t0 = time.perf_counter()
    cfg = W.make_config(args.config)
    lat = cfg.lattice
    n, R = lat.n, cfg.R
    M = args.moments or cfg.M
    nt = cfg.n_steps if args.time_steps is None else args.time_steps
    torch.cuda.synchronize()
    t_create = time.perf_counter()
    h = B.from_lattice(lat, cfg.xcoord, cfg.period, cfg.e0, cfg.scale)        # synchronises (validation result)
    t_create = time.perf_counter() - t_create
    phi = torch.from_numpy(W.random_phase_vectors(n, R, cfg.seed)).cuda()
    energies = torch.from_numpy(W.energy_grid(cfg.n_energies)).cuda()
    t_setup = time.perf_counter() - t0
    # a side stream: the library replays launch-bound moment loops as CUDA graphs, which the
    # legacy default stream cannot capture
    prev_stream = torch.cuda.current_stream()
    stream = torch.cuda.Stream()
    torch.cuda.set_stream(stream)

    def timed(fn):
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = h.launch_count
        e0.record(stream)
        out = fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return out, e0.elapsed_time(e1) * 1e-3, h.launch_count - l0

    wants = WANTS[args.config]
    res, timing = {}, {}
    if not args.no_warmup:
        # untimed: loads the kernels, sizes the workspace for M moments, builds the tile plan
        w_dos = B.dos_moments(h, phi, M)
        w_vac = B.vac(h, phi, M, 0, cfg.dt_fs) if "vac" in wants else None
        w_msd = B.msd(h, phi, M, 1 if nt >= 1 else 0, cfg.dt_fs) if "msd" in wants else None
        B.kpm_reconstruct(w_dos, cfg.e0, cfg.scale, energies)
        for w in (w_vac, w_msd):
            if w is not None and nt >= 1:
                f = B.kpm_reconstruct(w, cfg.e0, cfg.scale, energies).mean(dim=0).contiguous()
        del w_dos, w_vac, w_msd
        torch.cuda.synchronize()
    mu_dos, timing["dos_s"], timing["dos_launches"] = timed(lambda: B.dos_moments(h, phi, M))
    res["mu_dos"] = mu_dos
    if "vac" in wants:
        res["mu_vac"], timing["vac_s"], timing["vac_launches"] = timed(lambda: B.vac(h, phi, M, nt, cfg.dt_fs))
    if "msd" in wants:
        res["mu_msd"], timing["msd_s"], timing["msd_launches"] = timed(lambda: B.msd(h, phi, M, nt, cfg.dt_fs))

    # post-processing on the device; the stochastic trace is the mean over the R random vectors
    def post():
        out = {"rho": B.kpm_reconstruct(mu_dos, cfg.e0, cfg.scale, energies).mean(dim=0)}
        fvac = fmsd = None
        if "mu_vac" in res:
            fvac = B.kpm_reconstruct(res["mu_vac"], cfg.e0, cfg.scale, energies).mean(dim=0).contiguous()
        if "mu_msd" in res:
            fmsd = B.kpm_reconstruct(res["mu_msd"], cfg.e0, cfg.scale, energies).mean(dim=0).contiguous()
        if nt >= 1 and (fvac is not None or fmsd is not None):
            if args.config in (3, 6):
                # ribbon of N sites and length L_s: dens * W = 2N/L_s, so with width_nm = 1 the
                # conductance (W/L) sigma_E1 needs dens = 2N/(L_s * 1 nm)
                dens, width = 2.0 * n / cfg.period, 1.0
            else:
                dens, width = GRAPHENE_DENS, 1.0
            out.update(B.transport(out["rho"].contiguous(), fvac, fmsd, cfg.dt_fs, dens, width))
        out["f_vac"], out["f_msd"] = fvac, fmsd
        return out

    pp, timing["post_s"], _ = timed(post)
    torch.cuda.set_stream(prev_stream)
    host = {k: v.cpu().numpy() for k, v in {**res, **pp}.items() if v is not None}
    en = energies.cpu().numpy()

    summary = {"config": cfg.name, "sites": n, "R": R, "M": M, "time_steps": nt, "dt_fs": cfg.dt_fs,
               "setup_s": round(t_setup, 3), "create_s": round(t_create, 3), **{k: (round(v, 4) if isinstance(v, float) else v) for k, v in timing.items()},
               "workspace_GB": round(h.workspace_bytes / 1e9, 3)}
    sweeps = timing["dos_launches"] + timing.get("vac_launches", 0) + timing.get("msd_launches", 0)
    summary["kernel_launches"] = int(sweeps)
    summary["mu0"] = float(np.mean(host["mu_dos"][:, 0].real))
    summary["dos_integral"] = float(np.trapezoid(host["rho"], en))
    inner = np.abs(en) < 2.0
    if "sigma_gk" in host and "sigma_e1" in host and nt >= 4:
        k = nt - 1                                   # central difference available
        gk, e1 = host["sigma_gk"][k][inner], host["sigma_e1"][k][inner]
        summary["sigma_e1_vs_gk_rel_l2"] = float(np.linalg.norm(e1 - gk) / np.linalg.norm(gk))
        summary["sigma_gk_mean_e2_per_h"] = float(np.mean(gk))
    if "sigma_e1" in host and nt >= 2:
        summary["sigma_e1_last_mean_e2_per_h"] = float(np.mean(host["sigma_e1"][nt - 1][inner]))
        summary["sigma_e2_over_e1_last"] = float(np.mean(host["sigma_e2"][nt - 1][inner]) /
                                                 np.mean(host["sigma_e1"][nt - 1][inner]))
        summary["length_nm_last_mean"] = float(np.mean(host["length_nm"][nt][inner]))
    if args.config in (3, 6) and "conductance" in host and nt >= 2:
        g = host["conductance"][nt - 1] / 2.0        # in 2e^2/h
        summary["G_2e2h_at_|E|<0.5eV_mean"] = float(np.mean(g[np.abs(en) < 0.5]))
        summary["G_2e2h_at_1.0-1.2eV_mean"] = float(np.mean(g[(np.abs(en) > 1.0) & (np.abs(en) < 1.2)]))
    if args.out:
        os.makedirs(args.out, exist_ok=True)
        path = os.path.join(args.out, cfg.name + ".npz")
        np.savez_compressed(path, energies=en, **host)
        summary["saved"] = path
    print(json.dumps(summary), flush=True)
    return summary


if __name__ == "__main__":
    sys.exit(0 if main() else 1)
