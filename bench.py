#!/usr/bin/env python
"""bench.py -- LJ-liquid time steps per second on one B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config lj_64k] [--impl reference]

A "step" is one MD time step: the whole hot path (half kick + drift + buffer
check, list rebuild when the buffer is exceeded, LJ force/energy/virial, half
kick; Hilbert sort every `sort_period` steps).  The K timed steps are consecutive
steps of one trajectory that has first been advanced `--equil` + W steps from the
seeded lattice start, so the fluid has melted.

Prints ONE JSON line (rank 0).  Multi-GPU: replicas only (DESIGN.md section
"Multi-GPU"): every rank runs an independent system with its own seed, no
collective on the data path; torch.distributed (NCCL) is used for the barrier
and the max-over-ranks time only.

--impl reference times the ORACLE (oracle/orc.c, fp64, OpenMP over i) on the
host cores for a bounded number of the same steps.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1308_5587_b200 import workloads as wl  # noqa: E402

METRIC = "lj_liquid_timesteps_per_s"
UNIT = "timesteps/s"
# FP32 peak for the "alu" roofline (DESIGN.md section "Rooflines"): 148 SMs x 128 FP32
# lanes x 2 flop/FMA x 1.965 GHz (clocks.max.sm, B200_PROFILING.md table).
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
PAPER_TITAN_STEPS_PER_S = 1270.0   # PAPER.md:143, GK110, same N=64000 workload shape (context)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured"
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append([x.strip() for x in ln.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm = [float(r[0]) for r in self.rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({names[k] for r in self.rows if len(r) >= 7 for k in range(4) if r[3 + k].lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


def cpu_oracle_steps_per_s(w, state, nsteps):
    """The oracle as it stands, timed on this box's host cores."""
    from oracle import orc
    p = orc.Params.of(w)
    orc.lib()
    t0 = time.perf_counter()
    out = orc.run_nve(state.pos, state.vel, state.image, state.type, state.L, p, w.r_buff, w.dt, nsteps)
    dt = time.perf_counter() - t0
    return nsteps / dt, dt, orc.num_threads(), out["builds"]


def run_reference(args, w):
    """--impl reference: the oracle on the host cores, bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    state = wl.make_state(w)
    # bounded: the oracle does ~2.5e7 pair evaluations per second per core
    per_step = w.N * 70 / 2.0e7 / max(1, os.cpu_count() or 1) * 4
    cap = max(2, int(40.0 / max(per_step, 1e-6)))
    K = max(1, min(args.steps, cap))
    W = max(0, min(args.warmup, max(1, cap // 10)))
    from oracle import orc
    p = orc.Params.of(w)
    warm = orc.run_nve(state.pos, state.vel, state.image, state.type, state.L, p, w.r_buff, w.dt, W)
    t0 = time.perf_counter()
    orc.run_nve(warm["pos"], warm["vel"], warm["image"], state.type, state.L, p, w.r_buff, w.dt, K,
                forces=(warm["F"], warm["U"], warm["W"]))
    el = time.perf_counter() - t0
    v = K / el
    sample = f"{K} consecutive steps of {w.name} (N={w.N}) after {W} warm-up steps from the seeded lattice start, list rebuilds included"
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": K, "warmup": W,
            "ms_per_step": 1e3 * el / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": config_of(w, args, {}),
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def max_over_ranks(x, dist, device):
    """Replicas only: the one quantity the ranks exchange is a time, reduced with MAX."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, steps, ms_max):
    """Independent systems, one per rank: steps of all ranks over the slowest rank's time."""
    return world * steps / (ms_max * 1e-3)


def config_of(w, args, extra):
    c = {"workload": w.name, "N": w.N, "rho": w.rho, "T": w.T, "r_cut": w.r_cut_max, "r_buff": w.r_buff, "dt": w.dt,
         "ntypes": w.ntypes, "shift": "energy" if w.shift else "none", "sort_period": w.sort_period,
         "equil_steps": args.equil, "parallelism": "replicas" if args.gpus > 1 else "single"}
    c.update(extra)
    return c


# Algorithmic work of the step kernel.  Per LISTED pair the kernel must do
# 3 sub, 3 mul/fma (r^2), 1 compare = 7 ALU ops / 9 flops; per pair inside r_cut in addition 1 rcp, 2 mul (r^-6),
# 3 (f/r), 3 (energy), 3 mul + 3 add (force), 6 fma (virial) = 24 ALU ops / 33 flops (an FMA counts 2 flops, 1 op).
OPS_LISTED, FLOPS_LISTED, OPS_INCUT, FLOPS_INCUT = 7, 9, 24, 33


def force_work(g, w):
    """Algorithmic bytes, flops and ALU ops of one launch of the force kernel."""
    pairs = int(g.get_nlist_sizes()[-1])
    N = w.N
    # 16-bit list entries + position in, force + virial out, + velocity and position in and out when the step is fused in
    bytes_ = 2 * pairs + N * (16 + 16 + 32) + N * (16 + 16 + 16 + 16)
    frac_in = (w.r_cut_max / w.r_max) ** 3 if w.ntypes == 1 else 0.55
    flops = FLOPS_LISTED * pairs + FLOPS_INCUT * frac_in * pairs
    ops = OPS_LISTED * pairs + OPS_INCUT * frac_in * pairs
    return pairs, bytes_, flops, ops


def ncu_traffic(kernel):
    """dram__bytes_read + dram__bytes_write per launch from the committed ncu capture (profiles/), or None."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f).get(kernel)
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10000)
    ap.add_argument("--warmup", type=int, default=1000)
    ap.add_argument("--equil", type=int, default=2000, help="untimed steps before the warm-up (melting the lattice)")
    ap.add_argument("--config", default="lj_64k", choices=list(wl.CONFIGS))
    ap.add_argument("--impl", default="hb", choices=["hb", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-also", action="store_true", help="skip the short N=1M measurement")
    ap.add_argument("--tune", default="", help="comma list name=value of hb tunables")
    args = ap.parse_args()
    w = wl.CONFIGS[args.config]
    if args.impl == "reference":
        run_reference(args, w)
        return

    import torch
    from paper_1308_5587_b200 import hb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    if args.warmup < 3:
        args.warmup = 3
    hbm_peak, peak_kind = measured_peaks()
    tun = dict(kv.split("=") for kv in args.tune.split(",") if kv)

    def make_system(wk, seed):
        st = wl.make_state(wk, seed=seed)
        g = hb.System.from_workload(wk)
        for k, v in tun.items():
            g.set_tunable(k, int(v))
        g.set_state(st.pos, st.type, st.vel, st.image)
        g.build_nlist(0.0, wk.r_buff)
        g.compute_lj(wk.shift)
        return g, st

    def timed_run(g, wk, K):
        """K steps between CUDA events on the stream the library launches on."""
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0 = g.stats()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        e0.record()
        g.run_nve(wk.dt, K, wk.sort_period)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        ms = max_over_ranks(ms, dist, "cuda")
        s1 = g.stats()
        return ms, {k: s1[k] - s0[k] for k in ("rebuilds", "sorts", "kernel_launches", "graph_launches", "overflow_retries")}

    g, st0 = make_system(w, seed=w.seed + rank)
    g.run_nve(w.dt, args.equil, w.sort_period)
    g.run_nve(w.dt, args.warmup, w.sort_period)
    sampler = ClockSampler(local)
    sampler.start()
    ms, delta = timed_run(g, w, args.steps)
    clocks = sampler.stop()
    value = whole_job_value(world, args.steps, ms)
    th = g.thermo()
    stats = g.stats()

    # ---- per-kernel rooflines, measured live with CUDA events on the launching stream ----
    # (hb_time_stage: the launches of one stage captured into one graph, CUDA events around the graph launch)
    pairs, fbytes, fflops, fops = force_work(g, w)
    t_step = g.time_stage("lj_nve", 200)                    # the kernel a step of hb_run_nve is: force + kicks + drift
    t_force = g.time_stage("lj_force", 200)                 # the same kernel without the integration
    t_step_cold = g.time_stage("lj_nve", 20, 512 << 20)     # L2 flushed before every launch
    t_nlist = g.time_stage("nlist", 50)
    t_cells = g.time_stage("cells", 50)
    t_rebuild = g.time_stage("rebuild", 50)
    t_nve = g.time_stage("nve", 200)
    rate = delta["rebuilds"] / args.steps
    share_step_kernel = t_step * args.steps / ms
    roof_alu = {"bound": "alu", "achieved": fflops / (t_step * 1e-3) / 1e12, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                "kernel": "lj_tile_kernel", "ms": t_step, "traffic": ncu_traffic("lj_tile_kernel"),
                "peak_source": "nominal fp32: 148 SM x 128 lanes x 2 flop x 1.965 GHz (DESIGN.md); no measured fp32 peak exists",
                "alu_ops_frac": fops / (t_step * 1e-3) / (FP32_PEAK_TFLOPS * 1e12 / 2),
                "alu_ops_note": "algorithmic ALU instructions (an FMA is one) per second over 148 x 128 x 1.965 GHz issue slots"}
    roof_alu["frac"] = roof_alu["achieved"] / roof_alu["peak"]
    roof_hbm = {"bound": "hbm", "achieved": fbytes / (t_step_cold * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s",
                "kernel": "lj_tile_kernel", "ms": t_step_cold, "traffic": ncu_traffic("lj_tile_kernel"),
                "peak_source": f"MEASURED_PEAKS.json hbm_gbs ({peak_kind}); L2 flushed before every launch"}
    roof_hbm["frac"] = roof_hbm["achieved"] / roof_hbm["peak"]
    nl_bytes = 2 * pairs + w.N * (16 + 4 + 64)              # positions in, 16-bit entries + count out, reorder copy-back
    nl_tests = 27.0 * w.N * w.N / stats["cells_per_axis"] ** 3
    kernels = {
        "lj_step": {"ms_warm_l2": t_step, "ms_cold_l2": t_step_cold, "ms_force_only": t_force, "pairs": pairs,
                    "algorithmic_bytes": fbytes, "algorithmic_flops": fflops, "algorithmic_alu_ops": fops,
                    "share_of_step": share_step_kernel},
        "nlist": {"ms": t_nlist, "algorithmic_bytes": nl_bytes, "gbs": nl_bytes / (t_nlist * 1e-3) / 1e9,
                  "frac_hbm": nl_bytes / (t_nlist * 1e-3) / 1e9 / hbm_peak, "distance_tests": nl_tests,
                  "alu_ops_frac": 8 * nl_tests / (t_nlist * 1e-3) / (FP32_PEAK_TFLOPS * 1e12 / 2)},
        "cells": {"ms": t_cells, "algorithmic_bytes": 36 * w.N + 100 * w.N},
        "rebuild": {"ms": t_rebuild, "per_step": rate, "ms_per_step": rate * t_rebuild},
        "nve_standalone": {"ms": t_nve, "algorithmic_bytes": 108 * w.N, "gbs": 108 * w.N / (t_nve * 1e-3) / 1e9},
        "step_model": {"ms": t_step + rate * t_rebuild, "launch_gaps_ms": ms / args.steps - (t_step + rate * t_rebuild)},
    }

    # ---- end to end through the C ABI with HOST buffers ----
    s_now = g.get_state()
    pos_h, vel_h, typ_h, img_h = (np.ascontiguousarray(s_now[k]) for k in ("pos", "vel", "type", "image"))
    Ke = max(1, min(args.steps, 2000))
    g.set_state(pos_h, typ_h, vel_h, img_h)
    g.run_nve(w.dt, 50, w.sort_period)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    g.set_state(pos_h, typ_h, vel_h, img_h)                      # H2D inside the timed region
    g.run_nve(w.dt, Ke, w.sort_period)
    g.get_state_into(pos=pos_h, type=typ_h, vel=vel_h, image=img_h)  # D2H inside the timed region
    th_e = g.thermo()
    el = time.perf_counter() - t0
    el = max_over_ranks(el, dist, "cuda")
    e2e = {"value": world * Ke / el, "unit": UNIT, "steps_per_call": Ke, "h2d_bytes_per_step": w.N * 40 / Ke,
           "d2h_bytes_per_step": (w.N * 40 + 96) / Ke, "h2d_bytes_per_call": w.N * 40, "d2h_bytes_per_call": w.N * 40 + 96,
           "note": "hb_set_state(host) + hb_run_nve + hb_get_state(host) + hb_thermo, wall clock"}
    g.close()

    also = {}
    if not args.no_also and world == 1 and args.config == "lj_64k":
        w2 = wl.CONFIGS["lj_1m"]
        g2, _ = make_system(w2, seed=w2.seed)
        g2.run_nve(w2.dt, 600, w2.sort_period)
        ms2, d2 = timed_run(g2, w2, 1000)
        p2, b2, f2, o2 = force_work(g2, w2)
        tf2 = g2.time_stage("lj_nve", 30)
        tn2 = g2.time_stage("nlist", 10)
        also = {"lj_1m": {"timesteps_per_s": 1000 / (ms2 * 1e-3), "particle_steps_per_s": 1000 * w2.N / (ms2 * 1e-3),
                          "ms_per_step": ms2 / 1000, "rebuilds": d2["rebuilds"], "lj_step_ms": tf2,
                          "lj_step_hbm_gbs": b2 / (tf2 * 1e-3) / 1e9, "lj_step_hbm_frac": b2 / (tf2 * 1e-3) / 1e9 / hbm_peak,
                          "lj_step_alu_frac": f2 / (tf2 * 1e-3) / 1e12 / FP32_PEAK_TFLOPS,
                          "nlist_ms": tn2, "mean_nbrs": p2 / w2.N, "inputs": "larger than L2 (126 MB list + tables)"}}
        g2.close()
        # opt-in variant, NOT the headline: inner steps of a chunk compute forces only (tunable thermo_every = 0);
        # same trajectory bit for bit, energies and virials valid whenever hb_run_nve returns
        tun["thermo_every"] = "0"
        g3, _ = make_system(w, seed=w.seed + rank)
        del tun["thermo_every"]
        g3.run_nve(w.dt, args.equil + args.warmup, w.sort_period)
        ms3, d3 = timed_run(g3, w, min(args.steps, 4000))
        also["lj_64k_thermo_every_0"] = {"timesteps_per_s": min(args.steps, 4000) / (ms3 * 1e-3),
                                         "note": "U_i and W_i only in the last step of each 100-step chunk; opt-in, not the headline"}
        g3.close()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # about 15 s of CPU work: the oracle takes ~1.5e-7 s per particle per step on the 16 cores of these boxes
        n_cpu = max(2, min(2000, int(15.0 / (w.N * 1.5e-7 * 16 / max(1, os.cpu_count() or 1)))))
        v, secs, cores, builds = cpu_oracle_steps_per_s(w, st0, n_cpu)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {n_cpu} steps of {w.name} (N={w.N}) from the seeded lattice start incl. the initial list build "
                         f"and {builds} builds, {secs:.1f} s"}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": config_of(w, args, {
                "l2": ("working set (list + particle data) is smaller than the 126 MB L2: the K timed steps are consecutive steps "
                       "of one trajectory, each consuming the previous step's output; no flush between steps"
                       if w.N < 400_000 else "inputs larger than L2"),
                "row_pitch": stats["row_pitch"], "cells_per_axis": stats["cells_per_axis"], "mean_nbrs": pairs / w.N,
                "tunables": {k: g_tun for k, g_tun in tun.items()}}),
            "particle_steps_per_s": value * w.N,
            "context_paper": {"gtx_titan_gk110_steps_per_s": PAPER_TITAN_STEPS_PER_S, "ratio": value / world / PAPER_TITAN_STEPS_PER_S,
                              "note": "PAPER.md:143, other hardware and an equilibrated start: context, not vs_baseline"},
            "run": {**delta, "E_per_particle": (th["K"] + th["U"]) / w.N, "T": 2 * th["K"] / (3 * w.N),
                    "max_nbrs": stats["max_nbrs"]},
            "roofline": roof_alu,
            "roofline_other": roof_hbm,
            "kernels": kernels,
            "cpu_baseline": cpu,
            "e2e": e2e,
            "gpu_launches": delta["kernel_launches"],
            "clocks": clocks,
            "also": also,
        }
        print(json.dumps(line))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
