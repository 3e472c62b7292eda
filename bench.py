#!/usr/bin/env python
"""bench.py -- throughput of the LCS hot path on B200 (BASELINE.json metric: seed-RK4-steps/s and seeds/s to FTLE).

A "step" is one pass of the whole hot path over one batch of synthetic input: with the velocity field resident,
lcs_advect (RK4 flow map of the whole seed grid) followed by lcs_cg_ftle (gradient, Cauchy-Green tensor, FTLE).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

N = 1: the workload is BASELINE.json config 3 (3D ABC flow, 128^3 periodic grid, 256^3 seeds, 500 RK4 steps, fp32),
the 3D Cartesian configuration north_star's roofline target is stated for; --config picks another one.
N > 1 (torchrun, one rank per GPU): the path shards with NO data-path collective -- rank r computes an independent
FTLE volume (the seed grid released at t0 = 0.5 r: the time series of PAPER.md:37) -- so scaling is "weak"; the only
communication is the barrier and the max-over-ranks of the device time.
--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "seed_rk4_steps_per_s"
UNIT = "seed-steps/s"


# ------------------------------------------------------------------------------------------------
def make_workload(cfg: int, rank: int = 0):
    """Full-size BASELINE.json configs (DESIGN.md input recipe).  Returns (workload, [(t0, tf, h), ...])."""
    from paper_2209_13775_b200 import inputs as I
    if cfg == 1:
        w = I.config1()
        runs = [(w.t0, w.tf, w.h)]
    elif cfg == 2:
        w = I.config2()
        runs = [(w.t0, w.tf, w.h)]
    elif cfg == 3:
        w = I.config3()
        t0 = 0.5 * rank                                   # independent FTLE volume per rank (weak scaling)
        runs = [(t0, t0 + 5.0, w.h)]
    elif cfg == 4:
        w = I.config4()
        runs = [(w.t0, w.tf, w.h)]
    elif cfg == 5:
        w = I.config5()
        runs = [(a, b, w.h) for (a, b) in w.meta["windows"]]
    else:
        raise SystemExit("--config must be 1..5")
    return w, runs


def algorithmic_bytes_per_seed_step(w) -> float:
    """SURVEY.md 8.3 / DESIGN.md: gather bytes the straightforward 4-stage scheme must read per seed-step:
    4 stages x stencil nodes x 2 snapshots x dim components x element size (+ mesh data on simplex meshes)."""
    es = w.vel.dtype.itemsize
    if w.kind == 0:
        return 4.0 * (2 ** w.dim) * 2 * w.dim * es
    mesh = (w.dim + 1) * 4 + (w.dim + 1) * w.dim * 8 * (0.5 if w.compute_dtype == np.float32 else 1.0)
    return 4.0 * ((w.dim + 1) * 2 * w.dim * es + mesh)


class ClockSampler:
    """nvidia-smi clocks + throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
                for k, nm in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("sm_max_mhz", 1965.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, 1965.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------
def cpu_baseline(w, runs, budget_s=15.0):
    """The oracle as it stands, OpenMP over seeds on the host cores, on a bounded sample: a contiguous block of the
    seed grid integrated over the full number of steps and taken to FTLE."""
    from oracle import lcs_oracle
    fo = lcs_oracle.OracleField.from_workload(w)
    t0, tf, h = runs[0]
    N = int(round((tf - t0) / h))
    seeds = w.seeds()
    ng = w.ng
    # probe rate on a small block, then size the sample for ~budget_s
    def block(nb):
        nb = [min(nb, ng[a]) for a in range(w.dim)] + [1] * (3 - w.dim)
        if w.dim == 3:
            s = seeds.reshape(ng[2], ng[1], ng[0], 3)
            lo = [(ng[a] - nb[a]) // 2 for a in range(3)]
            return np.ascontiguousarray(s[lo[2]:lo[2] + nb[2], lo[1]:lo[1] + nb[1], lo[0]:lo[0] + nb[0]].reshape(-1, 3)), nb
        s = seeds.reshape(ng[1], ng[0], 2)
        lo = [(ng[a] - nb[a]) // 2 for a in range(2)]
        return np.ascontiguousarray(s[lo[1]:lo[1] + nb[1], lo[0]:lo[0] + nb[0]].reshape(-1, 2)), nb

    def run(nb):
        s, nbb = block(nb)
        t = time.perf_counter()
        F, fl, es = fo.advect(s.astype(np.float64), t0, tf, h)
        cg, ft, st = lcs_oracle.cg_ftle(w.dim, nbb[:w.dim], w.seed_spacing[:w.dim], (0,) * w.dim, (0.0,) * w.dim, F, fl, tf - t0)
        dt = time.perf_counter() - t
        return float(es.sum()), s.shape[0], dt, nbb

    steps, nseeds, dt, nbb = run(8 if w.dim == 3 else 32)
    rate = steps / max(dt, 1e-9)
    target = rate * budget_s / max(N, 1)
    nb = int(round(target ** (1.0 / w.dim)))
    nb = max(8, min(nb, 96 if w.dim == 3 else 1024))
    steps, nseeds, dt, nbb = run(nb)
    cap = 96 if w.dim == 3 else 1024
    for _ in range(3):                                  # the probe under-estimates the rate of short runs: grow the sample
        if dt >= budget_s / 3 or nb >= min(cap, max(ng[:w.dim])):
            break
        nb = max(nb + 1, min(cap, int(nb * (0.7 * budget_s / max(dt, 1e-3)) ** (1.0 / w.dim))))
        steps, nseeds, dt, nbb = run(nb)
    return {"value": steps / dt, "unit": UNIT, "cores": lcs_oracle.max_threads(), "kind": "oracle",
            "seeds_per_s_to_ftle": nseeds / dt,
            "sample": "centred %s block of the seed grid (%d seeds), %d RK4 steps + CG/FTLE, %.1f s" % ("x".join(map(str, nbb[:w.dim])), nseeds, N, dt)}


def reference_arm(args):
    """--impl reference: the oracle timed on the host cores; each step = a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w, runs = make_workload(args.config)
    vals, times = [], []
    for it in range(args.warmup + args.steps):
        r = cpu_baseline(w, runs, budget_s=4.0)
        if it >= args.warmup:
            vals.append(r)
    total_t = sum(float(v["sample"].split()[-2]) for v in vals)
    value = float(np.mean([v["value"] for v in vals]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * total_t / max(len(vals), 1), "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": {"workload": w.name, "sample": vals[-1]["sample"]},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": vals[-1]["cores"], "kind": "oracle", "sample": vals[-1]["sample"]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def reduce_over_ranks(elapsed_ms, seed_steps, seeds, device, world):
    """Whole-job figures: the time is the MAX over ranks, the work is the SUM (every rank integrates its own FTLE volume;
    there is no data-path collective).  Backend-agnostic (nccl on GPUs, gloo in the CPU test)."""
    if world <= 1:
        return float(elapsed_ms), float(seed_steps), float(seeds)
    import torch
    import torch.distributed as dist
    t = torch.tensor([elapsed_ms], dtype=torch.float64, device=device)
    tot = torch.tensor([seed_steps, seeds], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return float(t.item()), float(tot[0].item()), float(tot[1].item())


# ------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--option", action="append", default=[], help="library option key=value (e.g. integrator=2)")
    args = ap.parse_args()
    if args.impl == "reference":
        return reference_arm(args)

    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2209_13775_b200 import build, lcs
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    lcs.lib()

    w, runs = make_workload(args.config, rank)
    ring = 4 if args.config == 5 else 0
    field = lcs.Field.from_workload(w, max_resident_snapshots=ring, pinned=True)
    if args.config == 5:
        field.set_option("field_sets", 12)               # time series: consecutive volumes share 9 of their 10 windows
    for kv in args.option:
        k, v = kv.split("=")
        field.set_option(k, int(v))
    tdt = torch.float32 if w.compute_dtype == np.float32 else torch.float64
    seeds_h = torch.from_numpy(w.seeds()).pin_memory()
    seeds_d = seeds_h.cuda()
    n = w.n_seeds
    flow = torch.empty_like(seeds_d)
    flag = torch.empty(n, dtype=torch.uint8, device="cuda")
    es = torch.empty(n, dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()

    def one_pass():
        """All rows of the hot path over one batch: flow map(s) -> CG -> FTLE.  Returns seed-steps taken."""
        ftles = []
        if args.config == 5:
            field.set_option("field_sets_clear", 0)      # every pass starts without resident blended fields: reuse only WITHIN a pass
        for (t0, tf, h) in runs:
            field.advect(seeds_d, t0, tf, h, flowmap=flow, exit_flag=flag, exit_step=es)
            cg, ftle, st = lcs.cg_ftle(w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, flow, flag, tf - t0,
                                       want_cg=True, want_status=False)
            ftles.append(ftle)
        return ftles

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        one_pass()
    # seed-steps actually taken in one pass (exits shorten trajectories): sum of exit_step
    torch.cuda.synchronize()
    steps_per_pass = 0.0
    for (t0, tf, h) in runs[-1:]:
        steps_per_pass = float(es.sum(dtype=torch.int64).item()) * len(runs) if len(runs) > 1 else float(es.sum(dtype=torch.int64).item())
    field.set_option("time_windows", 1)
    sampler = ClockSampler(local)
    sampler.start()
    l0 = lcs.kernel_launch_count()
    barrier()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record(stream)
    for _ in range(args.steps):
        one_pass()
    ev1.record(stream)
    barrier()
    elapsed_ms = ev0.elapsed_time(ev1)
    launches = lcs.kernel_launch_count() - l0
    clocks = sampler.stop()
    win_ns = field.info("window_time_ns")
    win_launches = field.info("window_launches")
    field.set_option("time_windows", 0)
    elapsed_ms, steps_all, seeds_all = reduce_over_ranks(elapsed_ms, steps_per_pass, float(n * len(runs)), "cuda", world)
    sec_per_step = elapsed_ms * 1e-3 / args.steps
    value = steps_all / sec_per_step

    # end to end through the C-ABI with HOST buffers (H2D seeds + D2H FTLE inside the timed region)
    e2e = None
    if not args.no_e2e:
        ftle_h = torch.empty(n, dtype=tdt).pin_memory()
        esz = seeds_h.element_size()
        def e2e_pass():
            if args.config == 5:
                field.set_option("field_sets_clear", 0)
            for (t0, tf, h) in runs:
                field.ftle_host(w.ng, w.seed_spacing, w.seed_periodic, w.period, seeds_h.numpy(), t0, tf, h, ftle=ftle_h.numpy())
        e2e_pass()
        barrier()
        t0w = time.perf_counter()
        ev0.record(stream)
        for _ in range(args.steps):
            e2e_pass()
        ev1.record(stream)
        barrier()
        e_ms = max(ev0.elapsed_time(ev1), 0.0)
        e_wall = (time.perf_counter() - t0w) * 1e3
        e_ms = max(e_ms, e_wall)                          # copies on the legacy stream: wall clock bounds the region
        te = torch.tensor([e_ms], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": steps_all / (float(te.item()) * 1e-3 / args.steps), "unit": UNIT,
               "h2d_bytes_per_step": int(n * w.dim * esz * len(runs)), "d2h_bytes_per_step": int(n * esz * len(runs)),
               "seeds_per_s_to_ftle": seeds_all / (float(te.item()) * 1e-3 / args.steps)}

    if rank == 0:
        hbm_gbs, sm_max_mhz, peak_src = measured_peaks()
        kernel_s = win_ns * 1e-9 / max(win_launches, 1)                    # average launch duration of the dominant kernel
        bytes_unit = algorithmic_bytes_per_seed_step(w)
        units_per_launch = steps_per_pass * args.steps / max(win_launches, 1)
        achieved = bytes_unit * units_per_launch / max(kernel_s, 1e-12) / 1e9
        share = (win_ns * 1e-9) / (elapsed_ms * 1e-3) if world == 1 else None
        common = {"traffic": None, "seed_steps_per_launch": units_per_launch, "avg_launch_ms": kernel_s * 1e3,
                  "kernel_share_of_step": share, "algorithmic_bytes_per_seed_step": bytes_unit}
        if w.kind == 0 and w.dim == 3 and w.compute_dtype == np.float32:
            # the 3D fp32 Cartesian integrator gathers from L1 (DRAM < 20% of peak) and is bound by
            # FP32 issue slots + L1 wavefronts.  ALU roofline: SURVEY.md 8.3's 720 flop per seed-step against
            # 148 SMs x 128 FP32 lanes x 2 flop x max SM clock.
            flop_unit = 720.0
            peak_tf = 148 * 128 * 2 * sm_max_mhz * 1e6 / 1e12
            ach_tf = flop_unit * units_per_launch / max(kernel_s, 1e-12) / 1e12
            l1_peak = 148 * 128 * sm_max_mhz * 1e6 / 1e9
            roofline = {"bound": "alu", "kernel": "cart_xpair_kernel", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                        "frac": ach_tf / peak_tf, "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x %.0f MHz (DESIGN.md)" % sm_max_mhz,
                        "algorithmic_flop_per_seed_step": flop_unit,
                        "l1_gather": {"achieved": achieved, "peak": l1_peak, "unit": "GB/s", "frac": achieved / l1_peak,
                                      "note": "768 B per seed-step of the straightforward 4-stage scheme against 148 SMs x 128 B/clk; "
                                              "above 1 because the kernel gathers pre-blended fields and reuses corners in registers"},
                        **common}
        elif w.kind == 1 and w.dim == 3 and w.compute_dtype == np.float32:
            # tets in fp32 (config 4): measured DRAM 1.5% of peak, L2 hit 80-96%, issue slots 58%, L1 wavefronts 63%
            # (profiles/r1_cfg4_simplex.md): not HBM-bound.  ALU roofline with SURVEY.md 8.3's 900 flop per seed-step.
            flop_unit = 900.0
            peak_tf = 148 * 128 * 2 * sm_max_mhz * 1e6 / 1e12
            ach_tf = flop_unit * units_per_launch / max(kernel_s, 1e-12) / 1e12
            roofline = {"bound": "alu", "kernel": "simplex_window_kernel", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                        "frac": ach_tf / peak_tf, "peak_source": "derived: 148 SMs x 128 FP32 lanes x 2 x %.0f MHz (DESIGN.md)" % sm_max_mhz,
                        "algorithmic_flop_per_seed_step": flop_unit,
                        "hbm_gather": {"achieved": achieved, "peak": hbm_gbs, "unit": "GB/s", "frac": achieved / hbm_gbs,
                                       "note": "640 B per seed-step of the straightforward scheme against the measured HBM copy peak; far "
                                               "above 1 because the mesh is served by L1/L2 and the held cell skips most gathers"},
                        **common}
        else:
            roofline = {"bound": "hbm", "kernel": "cart_window_kernel" if w.kind == 0 else "simplex_window_kernel",
                        "achieved": achieved, "peak": hbm_gbs, "unit": "GB/s", "frac": achieved / hbm_gbs, "peak_source": peak_src,
                        "note": "algorithmic gather bytes; small fields are served by L1/L2, so this can exceed the HBM copy peak "
                                "(DESIGN.md section 6)", **common}
        tr = os.path.join(ROOT, "profiles", "traffic_cfg%d.txt" % args.config)
        if os.path.exists(tr):
            roofline["traffic"] = json.load(open(tr)).get("dram_bytes_per_launch")
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": sec_per_step * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32" if w.compute_dtype == np.float32 else "f64", "data": "synthetic",
                "config": {"workload": w.name, "baseline_config": args.config, "seeds": n * len(runs), "rk4_steps": w.n_steps,
                           "seed_steps_per_pass": steps_per_pass, "parallelism": "independent FTLE volumes per rank, no collective",
                           "l2": "inputs larger than L2: seeds + tracer state are %.0f MB per pass" % (n * (w.dim * 2 + 3) * 4 / 1e6)},
                "seeds_per_s_to_ftle": seeds_all / sec_per_step, "roofline": roofline, "clocks": clocks, "gpu_launches": int(launches),
                "e2e": e2e}
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(w, runs)
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
