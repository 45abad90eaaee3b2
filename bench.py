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
# Nominal FP32 peak, for context beside the measured one (DESIGN.md section "Rooflines"): 148 SMs x 128 FP32
# lanes x 2 flop/FMA x 1.965 GHz (clocks.max.sm, B200_PROFILING.md table).  The roofline fractions below use
# the peaks hb_measure_peak measures in this very run (FFMA chains, L2 reads, shared-memory loads).
FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12
ISSUE_SLOTS_PER_S = 148 * 128 * 1.965e9        # thread-instructions per second at one warp instruction per scheduler per cycle
SMEM_NOMINAL_GBS = 148 * 128 * 1.965e9 / 1e9   # 128 B per cycle per SM
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


def cpu_oracle_steps_per_s(w, state, nsteps, threads=None):
    """The oracle as it stands, timed on this box's host cores (threads = None: all of them)."""
    import ctypes
    from oracle import orc
    p = orc.Params.of(w)
    orc.lib()
    all_threads = orc.num_threads()
    gomp = ctypes.CDLL("libgomp.so.1")
    if threads is not None:
        gomp.omp_set_num_threads(int(threads))
    try:
        used = orc.num_threads()
        t0 = time.perf_counter()
        out = orc.run_nve(state.pos, state.vel, state.image, state.type, state.L, p, w.r_buff, w.dt, nsteps)
        dt = time.perf_counter() - t0
    finally:
        gomp.omp_set_num_threads(all_threads)
    return nsteps / dt, dt, used, out["builds"]


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
# An inner step of hb_run_nve needs the forces only (tunable thermo_every = 0, the default: U_i and W_i of a step
# nobody can read are not computed): per pair inside r_cut 1 rcp, 2 mul (r^-6), 1 fma + 2 mul (f/r), 3 fma (force)
# = 9 ALU ops / 13 flops.
OPS_LISTED, FLOPS_LISTED, OPS_INCUT, FLOPS_INCUT = 7, 9, 24, 33
OPS_INCUT_F, FLOPS_INCUT_F = 9, 13


def force_work(g, w, thermo):
    """Algorithmic bytes, flops and ALU ops of one launch of the step kernel (thermo: with U_i and W_i)."""
    pairs = int(g.get_nlist_sizes()[-1])
    N = w.N
    # 16-bit list entries + position in, force (+ virial) out, + velocity and position in and out (the step is fused in)
    bytes_ = 2 * pairs + N * (16 + 16 + (32 if thermo else 0)) + N * (16 + 16 + 16 + 16)
    frac_in = (w.r_cut_max / w.r_max) ** 3 if w.ntypes == 1 else 0.55
    flops = FLOPS_LISTED * pairs + (FLOPS_INCUT if thermo else FLOPS_INCUT_F) * frac_in * pairs
    ops = OPS_LISTED * pairs + (OPS_INCUT if thermo else OPS_INCUT_F) * frac_in * pairs
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
    ap.add_argument("--n", type=int, default=0, help="run the config's fluid at another particle number (scaling studies)")
    args = ap.parse_args()
    w = wl.CONFIGS[args.config]
    if args.n > 0:
        w = wl.scaled(w, args.n)
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
    # The headline is the path north_star names -- force, ENERGY and VIRIAL in every step, the paper's kernel
    # -- so the tunable thermo_every is 1 here unless --tune says otherwise.  The library's default
    # (0: U_i and W_i in the last step of every chunk only, same trajectory bit for bit) is the named optimisation
    # reported beside it as "value_thermo_every_0" and also.lj_64k_thermo_every_0.
    tun.setdefault("thermo_every", "1")

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
    g.run_nve(w.dt, args.steps, w.sort_period)       # rehearsal of the timed call itself: same chunking, untimed
    builds0 = g.stats()["graph_builds"]
    sampler = ClockSampler(local)
    sampler.start()
    if args.steps >= 2000:
        # two halves, so that a drift of the rate during the run would show
        h1 = args.steps // 2
        ms_a, delta_a = timed_run(g, w, h1)
        ms_b, delta_b = timed_run(g, w, args.steps - h1)
        ms = ms_a + ms_b
        delta = {k: delta_a[k] + delta_b[k] for k in delta_a}
        halves = {"first_half_steps_per_s": whole_job_value(world, h1, ms_a),
                  "second_half_steps_per_s": whole_job_value(world, args.steps - h1, ms_b)}
    else:
        ms, delta = timed_run(g, w, args.steps)
        halves = {}
    clocks = sampler.stop()
    graph_builds_timed = g.stats()["graph_builds"] - builds0
    value = whole_job_value(world, args.steps, ms)
    th = g.thermo()
    stats = g.stats()
    thermo_every = g.get_tunable("thermo_every")
    g_chunk = g.get_tunable("graph_steps")

    # ---- measured peaks (kernels of this library, this run) ----
    peak_fp32 = g.measure_peak("fp32_tflops")
    peak_l2 = g.measure_peak("l2_gbs")
    peak_smem = g.measure_peak("smem_gbs")

    # ---- per-kernel rooflines, measured live with CUDA events on the launching stream ----
    # (hb_time_stage: the launches of one stage captured into one graph, CUDA events around the graph launch)
    pairs, fbytes, fflops, fops = force_work(g, w, thermo=bool(thermo_every))
    _, tbytes, tflops, tops = force_work(g, w, thermo=True)
    _, _, fflops0, fops0 = force_work(g, w, thermo=False)
    t_step = g.time_stage("lj_nve", 200)                    # the kernel an inner step of hb_run_nve is: force + kicks + drift
    t_force = g.time_stage("lj_force", 200)                 # force + energy + virial, no integration (hb_compute_lj)
    t_step_cold = g.time_stage("lj_nve", 20, 512 << 20)     # L2 flushed before every launch
    t_nlist = g.time_stage("nlist", 50)
    t_cells = g.time_stage("cells", 50)
    t_rebuild = g.time_stage("rebuild", 50)
    t_nve = g.time_stage("nve", 200)
    rate = delta["rebuilds"] / args.steps
    share_step_kernel = t_step * args.steps / ms
    sec = t_step * 1e-3
    roof_alu = {"bound": "alu", "achieved": fflops / sec / 1e12, "peak": peak_fp32, "unit": "TFLOP/s",
                "kernel": "lj_tile_kernel (inner step of hb_run_nve: " + ("force, energy, virial" if thermo_every else "forces only") +
                          ", both half kicks, drift, r_buff/2 check)",
                "ms": t_step, "traffic": ncu_traffic("lj_tile_kernel"),
                "peak_source": "measured in this run: hb_measure_peak fp32_tflops (8 FFMA chains per thread, all SMs); "
                               f"nominal 148 x 128 x 2 x 1.965 GHz = {FP32_NOMINAL_TFLOPS:.1f}",
                "alu_ops_frac": fops / sec / ISSUE_SLOTS_PER_S,
                "alu_ops_note": "algorithmic ALU instructions (an FMA is one) per second over 148 x 128 x 1.965 GHz issue slots",
                "gather_gbs": 16 * pairs / sec / 1e9, "gather_peak_gbs": peak_smem,
                "gather_frac": 16 * pairs / sec / 1e9 / peak_smem,
                "gather_frac_nominal": 16 * pairs / sec / 1e9 / SMEM_NOMINAL_GBS,
                "gather_peak_bytes_per_clk_sm": peak_smem * 1e9 / (148 * 1.965e9),
                "gather_note": "16 B of shared memory read per listed pair (the neighbor's staged position) over the measured "
                               "conflict-free shared-memory load bandwidth (LDS.128, four independent address streams per thread; "
                               "gather_peak_bytes_per_clk_sm = that peak per SM per cycle at 1.965 GHz, 128 B = one wavefront) and, "
                               f"as gather_frac_nominal, over the nominal 128 B/clk/SM = {SMEM_NOMINAL_GBS:.0f} GB/s"}
    roof_alu["frac"] = roof_alu["achieved"] / roof_alu["peak"]
    l2_resident = w.N < 400_000
    mem_peak = peak_l2 if l2_resident else hbm_peak
    t_mem = t_step if l2_resident else t_step_cold
    roof_mem = {"bound": "l2" if l2_resident else "hbm", "achieved": fbytes / (t_mem * 1e-3) / 1e9, "peak": mem_peak, "unit": "GB/s",
                "kernel": "lj_tile_kernel", "ms": t_mem, "traffic": ncu_traffic("lj_tile_kernel"),
                "peak_source": ("measured in this run: hb_measure_peak l2_gbs (32 MB buffer re-read from L2)" if l2_resident else
                                f"MEASURED_PEAKS.json hbm_gbs ({peak_kind}); L2 flushed before every launch")}
    roof_mem["frac"] = roof_mem["achieved"] / roof_mem["peak"]
    nl_bytes = 2 * pairs + w.N * (16 + 4 + 64)              # positions in, 16-bit entries + count out, reorder copy-back
    nl_tests = 27.0 * w.N * w.N / stats["cells_per_axis"] ** 3
    kernels = {
        "lj_step": {"ms_warm_l2": t_step, "ms_cold_l2": t_step_cold, "pairs": pairs,
                    "algorithmic_bytes": fbytes, "algorithmic_flops": fflops, "algorithmic_alu_ops": fops,
                    "share_of_step": share_step_kernel},
        "lj_force_energy_virial": {"ms": t_force, "algorithmic_flops": tflops, "algorithmic_alu_ops": tops,
                                   "tflops": tflops / (t_force * 1e-3) / 1e12, "frac_fp32": tflops / (t_force * 1e-3) / 1e12 / peak_fp32,
                                   "alu_ops_frac": tops / (t_force * 1e-3) / ISSUE_SLOTS_PER_S,
                                   "note": "hb_compute_lj's kernel (the paper's: U_i and W_i with the force, PAPER.md:95), no integration"},
        "nlist": {"ms": t_nlist, "algorithmic_bytes": nl_bytes, "gbs": nl_bytes / (t_nlist * 1e-3) / 1e9,
                  "frac_mem": nl_bytes / (t_nlist * 1e-3) / 1e9 / mem_peak, "distance_tests": nl_tests,
                  "tflops": 9 * nl_tests / (t_nlist * 1e-3) / 1e12, "frac_fp32": 9 * nl_tests / (t_nlist * 1e-3) / 1e12 / peak_fp32,
                  "alu_ops_frac": 8 * nl_tests / (t_nlist * 1e-3) / ISSUE_SLOTS_PER_S,
                  "note": "27 N^2/m^3 distance tests of 8 ALU instructions / 9 flops each (3 sub, 3 mul-add, compare, record)"},
        "cells": {"ms": t_cells, "algorithmic_bytes": 36 * w.N + 100 * w.N},
        "rebuild": {"ms": t_rebuild, "per_step": rate, "ms_per_step": rate * t_rebuild},
        "nve_standalone": {"ms": t_nve, "algorithmic_bytes": 108 * w.N, "gbs": 108 * w.N / (t_nve * 1e-3) / 1e9},
        "step_model": {"ms": t_step + rate * t_rebuild, "launch_gaps_ms": ms / args.steps - (t_step + rate * t_rebuild)},
        "peaks_measured": {"fp32_tflops": peak_fp32, "l2_gbs": peak_l2, "smem_gbs": peak_smem, "hbm_gbs": hbm_peak,
                           "hbm_source": peak_kind},
    }

    # ---- end to end through the C ABI with HOST buffers ----
    s_now = g.get_state()
    def pinned(a):      # page-locked host buffers (the copies in and out of the timed call are DMA transfers)
        t = torch.empty(a.shape, dtype={np.dtype(np.float32): torch.float32, np.dtype(np.int32): torch.int32}[a.dtype]).pin_memory()
        v = t.numpy()
        v[...] = a
        return v, t
    (pos_h, _p0), (vel_h, _p1), (typ_h, _p2), (img_h, _p3) = (pinned(np.ascontiguousarray(s_now[k])) for k in ("pos", "vel", "type", "image"))
    Ke = max(1, min(args.steps, 2000))
    g.set_state(pos_h, typ_h, vel_h, img_h)
    g.run_nve(w.dt, Ke, w.sort_period)                           # rehearsal: the timed call below repeats it
    builds_e = g.stats()["graph_builds"]
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
           "graph_builds_in_timed_region": g.stats()["graph_builds"] - builds_e,
           "note": "hb_set_state(pinned host buffers) + hb_run_nve + hb_get_state(pinned host buffers) + hb_thermo, wall clock"}
    g.close()

    also = {}
    if not args.no_also and world == 1 and args.config == "lj_64k":
        w2 = wl.CONFIGS["lj_1m"]
        g2, _ = make_system(w2, seed=w2.seed)
        g2.run_nve(w2.dt, 600, w2.sort_period)
        ms2, d2 = timed_run(g2, w2, 1000)
        p2, b2, f2, o2 = force_work(g2, w2, thermo=bool(g2.get_tunable("thermo_every")))
        tf2 = g2.time_stage("lj_nve", 30)
        tf2c = g2.time_stage("lj_nve", 10, 512 << 20)
        tn2 = g2.time_stage("nlist", 10)
        tr2 = g2.time_stage("rebuild", 10)
        m2 = g2.stats()["cells_per_axis"]
        also = {"lj_1m": {"timesteps_per_s": 1000 / (ms2 * 1e-3), "particle_steps_per_s": 1000 * w2.N / (ms2 * 1e-3),
                          "ms_per_step": ms2 / 1000, "rebuilds": d2["rebuilds"], "lj_step_ms": tf2, "lj_step_ms_cold_l2": tf2c,
                          "lj_step_hbm_gbs": b2 / (tf2c * 1e-3) / 1e9, "lj_step_hbm_frac": b2 / (tf2c * 1e-3) / 1e9 / hbm_peak,
                          "lj_step_fp32_frac": f2 / (tf2 * 1e-3) / 1e12 / peak_fp32,
                          "lj_step_alu_ops_frac": o2 / (tf2 * 1e-3) / ISSUE_SLOTS_PER_S,
                          "lj_step_gather_frac": 16 * p2 / (tf2 * 1e-3) / 1e9 / peak_smem,
                          "lj_step_gather_frac_nominal": 16 * p2 / (tf2 * 1e-3) / 1e9 / SMEM_NOMINAL_GBS,
                          "nlist_ms": tn2, "rebuild_ms": tr2,
                          "nlist_alu_ops_frac": 8 * 27.0 * w2.N * w2.N / m2 ** 3 / (tn2 * 1e-3) / ISSUE_SLOTS_PER_S,
                          "nlist_hbm_frac": (2 * p2 + w2.N * 84) / (tn2 * 1e-3) / 1e9 / hbm_peak,
                          "mean_nbrs": p2 / w2.N, "inputs": "larger than L2 (126 MB list + tables)"}}
        g2.close()
        # the named optimisation: tunable thermo_every = 0 (the library's default) computes U_i and W_i in the last step
        # of every chunk only; same trajectory bit for bit as the headline, which computes them in every step
        headline_te = tun["thermo_every"]
        tun["thermo_every"] = "0"
        g3, _ = make_system(w, seed=w.seed + rank)
        tun["thermo_every"] = headline_te
        g3.run_nve(w.dt, args.equil + args.warmup, w.sort_period)
        n3 = min(args.steps, 4000)
        g3.run_nve(w.dt, n3, w.sort_period)
        ms3, d3 = timed_run(g3, w, n3)
        t3 = g3.time_stage("lj_nve", 200)
        also["lj_64k_thermo_every_0"] = {"timesteps_per_s": n3 / (ms3 * 1e-3), "lj_step_ms": t3,
                                         "lj_step_fp32_frac": fflops0 / (t3 * 1e-3) / 1e12 / peak_fp32,
                                         "lj_step_alu_ops_frac": fops0 / (t3 * 1e-3) / ISSUE_SLOTS_PER_S,
                                         "note": "inner steps of a chunk compute forces only; U_i and W_i in the last step of "
                                                 "every chunk (valid whenever hb_run_nve returns); not the headline"}
        g3.close()

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # about 15 s of CPU work: the oracle takes ~1.5e-7 s per particle per step on the 16 cores of these boxes
        ncores = max(1, os.cpu_count() or 1)
        n_cpu = max(2, min(2000, int(10.0 / (w.N * 1.5e-7 * 16 / ncores))))
        v, secs, cores, builds = cpu_oracle_steps_per_s(w, st0, n_cpu)
        n_one = max(2, min(n_cpu, int(5.0 / (w.N * 1.5e-7 * 16))))
        v1, secs1, cores1, _ = cpu_oracle_steps_per_s(w, st0, n_one, threads=1)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {n_cpu} steps of {w.name} (N={w.N}) from the seeded lattice start incl. the initial list build "
                         f"and {builds} builds, {secs:.1f} s",
               "one_thread": {"value": v1, "cores": cores1, "sample": f"first {n_one} steps, {secs1:.1f} s"}}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            # `config` holds the workload keys only, the same in both arms (--impl reference prints the same dict);
            # what this arm chose at run time is in `run_config`
            "config": config_of(w, args, {}),
            "run_config": {
                "l2": ("working set (list + particle data) is smaller than the 126 MB L2: the K timed steps are consecutive steps "
                       "of one trajectory, each consuming the previous step's output; no flush between steps"
                       if w.N < 400_000 else "inputs larger than L2"),
                "row_pitch": stats["row_pitch"], "cells_per_axis": stats["cells_per_axis"], "mean_nbrs": pairs / w.N,
                "chunk_steps": g_chunk, "thermo_every": thermo_every,
                "tunables": {k: g_tun for k, g_tun in tun.items()}},
            "value_thermo_every_0": also.get("lj_64k_thermo_every_0", {}).get("timesteps_per_s"),
            "particle_steps_per_s": value * w.N, **halves,
            "graph_builds_in_timed_region": graph_builds_timed,
            "context_paper": {"gtx_titan_gk110_steps_per_s": PAPER_TITAN_STEPS_PER_S, "ratio": value / world / PAPER_TITAN_STEPS_PER_S,
                              "note": "PAPER.md:143, other hardware and an equilibrated start: context, not vs_baseline"},
            "run": {**delta, "E_per_particle": (th["K"] + th["U"]) / w.N, "T": 2 * th["K"] / (3 * w.N),
                    "max_nbrs": stats["max_nbrs"]},
            "roofline": roof_alu,
            "roofline_other": roof_mem,
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
