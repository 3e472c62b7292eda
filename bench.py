#!/usr/bin/env python
"""bench.py -- throughput of the LCS hot path on B200 (BASELINE.json metric: seed-RK4-steps/s and seeds/s to FTLE).

A "step" is one pass of the whole hot path over one batch of synthetic input: with the velocity field resident,
lcs_advect (RK4 flow map of the whole seed grid) followed by lcs_cg_ftle (gradient, Cauchy-Green tensor, FTLE).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--extra-configs 4,5|none] [--impl reference]

N = 1: the workload is BASELINE.json config 3 (3D ABC flow, 128^3 periodic grid, 256^3 seeds, 500 RK4 steps, fp32),
the 3D Cartesian configuration north_star's roofline target is stated for; --config picks another one.  The default
line also carries, under "configs", the same figures for configs 4 and 5 (the other two 3D configs of the >= 50% target).
N > 1 (torchrun, one rank per GPU): the path shards with NO data-path collective -- rank r computes an independent
FTLE volume (the seed grid released at t0 = 0.5 r: the time series of PAPER.md:37) -- so scaling is "weak"; the only
communication is the barrier and the max-over-ranks of the device time.
--impl reference times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.

Roofline: every peak is MEASURED in this run by the library's own micro-kernels (lcs_measure_peak: FP32 / FP64 FMA, L1-hit
256-bit gathers, shared-memory gathers, L2 sequential and random-sector reads, random 32-byte HBM gathers, launch latency);
the HBM streaming peak is the driver's MEASURED_PEAKS.json.  `bound` names the resource that the committed ncu counters
(profiles/roofline_cfgN.json, extracted from the --set full tables beside them) show closest to saturation; `frac` is the
useful work the kernel gets out of that resource (bytes its gathers deliver to registers per seed-step x rate) over the
measured peak; the 720 / 900-flop and 768 / 640-byte model figures of SURVEY.md 8.3 are kept beside it.
"""
from __future__ import annotations

import argparse
import gc
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
L2_BYTES = 126e6


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


_PEAKS = None


def measured_peaks(lcs):
    """Peaks measured in THIS run by the library's micro-kernels, plus the driver's HBM copy figure."""
    global _PEAKS
    if _PEAKS is None:
        p = {k: lcs.measure_peak(k) for k in lcs.PEAK_KINDS}
        path = os.path.join(ROOT, "MEASURED_PEAKS.json")
        if os.path.exists(path):
            d = json.load(open(path))
            p["hbm_copy_driver_gbs"] = float(d["hbm_gbs"])
            p["hbm_source"] = "measured (MEASURED_PEAKS.json)"
        else:
            p["hbm_copy_driver_gbs"] = 6650.0
            p["hbm_source"] = "fallback (B200_PROFILING.md)"
        _PEAKS = p
    return _PEAKS


def profile_constants(cfg: int):
    """Per-kernel constants taken from the committed ncu tables (profiles/roofline_cfgN.json names its source table):
    DRAM bytes per launch, bytes the gathers deliver to registers per seed-step, executed warp instructions per seed-step and
    the pipe utilisations that decide which resource binds."""
    for name in ("roofline_cfg%d.json" % cfg, "traffic_cfg%d.txt" % cfg):
        path = os.path.join(ROOT, "profiles", name)
        if os.path.exists(path):
            return json.load(open(path))
    return {}


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
def roofline_block(lcs, cfg, w, kernel_s, units_per_launch, share, win_launches, win_s_per_pass, options=()):
    """The roofline object of one config (see the module docstring)."""
    pk = measured_peaks(lcs)
    prof = profile_constants(cfg)
    rate = units_per_launch / max(kernel_s, 1e-12)                         # seed-steps per second inside the dominant kernel
    bytes_unit = algorithmic_bytes_per_seed_step(w)
    common = {"traffic": prof.get("dram_bytes_per_launch"), "seed_steps_per_launch": units_per_launch, "avg_launch_ms": kernel_s * 1e3,
              "launches_timed": int(win_launches), "kernel_share_of_step": share, "algorithmic_bytes_per_seed_step": bytes_unit,
              "peak_source": "measured in this run (lcs_measure_peak); HBM copy: " + pk["hbm_source"],
              "peaks": {k: v for k, v in pk.items() if k != "hbm_source"},
              "counters": {k: prof[k] for k in ("l1_data_pipe_pct", "issue_slots_pct", "fma_pipe_pct", "fp64_pipe_pct", "dram_pct", "l1_hit_pct",
                                                "lanes_per_instruction", "executed_inst_per_seed_step", "source") if k in prof}}
    three_d_f32 = w.dim == 3 and w.compute_dtype == np.float32
    if three_d_f32:
        cart = w.kind == 0
        flop_unit = 720.0 if cart else 900.0
        model_alu = {"flop_per_seed_step": flop_unit, "achieved": flop_unit * rate / 1e12, "peak": pk["fp32_fma_tflops"], "unit": "TFLOP/s",
                     "frac": flop_unit * rate / 1e12 / pk["fp32_fma_tflops"],
                     "note": "SURVEY.md 8.3 model flop count of the straightforward scheme (not what the kernel executes) over the measured FFMA peak"}
        model_gather = {"bytes_per_seed_step": bytes_unit, "achieved": bytes_unit * rate / 1e9, "unit": "GB/s",
                        "note": "SURVEY.md 8.3 model gather bytes of the straightforward 4-stage scheme; the kernel loads less (pre-blended "
                                "fields / held cell), so this is a statement about the method, not a utilisation"}
        delivered = prof.get("l1_bytes_to_registers_per_seed_step")
        kern = prof.get("kernel", "cart_xpair_kernel" if cart else "simplex_window_kernel")
        staged = cart and any(o.startswith("tma=") and o != "tma=0" for o in options)
        if staged:                                           # the staged variant has no counter table of its own in roofline_cfgN.json
            kern, delivered = "cart_xpair_tma_kernel", 256.0
        peak_key = "smem_records_swizzled_gbs" if staged else "l1_gather_line_gbs"
        if delivered:
            ach = delivered * rate / 1e9
            busy = prof.get("l1_data_pipe_pct")
            return {"bound": "l1", "kernel": kern, "achieved": ach, "peak": pk[peak_key], "unit": "GB/s", "frac": ach / pk[peak_key],
                    "binding_resource_busy": (max(busy) / 100.0 if busy and not staged else None),
                    "binding_resource_busy_note": "l1tex__data_pipe_lsu_wavefronts, % of peak, from the committed ncu table of this kernel "
                                                  "(SURVEY.md 8.3: the binding roofline is the resource with the highest % of its peak); `frac` "
                                                  "counts only the bytes the gathers usefully deliver",
                    "bytes_to_registers_per_seed_step": delivered,
                    "note": "L1 / shared-memory data pipe (128 B per clock per SM into registers): bytes the kernel's gathers actually deliver to "
                            "registers per seed-step (ncu request counts, profiles/) x rate, over the measured best-case gather rate (%s)" % peak_key,
                    "model_alu": model_alu, "model_gather": model_gather, **common}
        return {"bound": "alu", "kernel": kern, "achieved": model_alu["achieved"], "peak": model_alu["peak"], "unit": "TFLOP/s",
                "frac": model_alu["frac"], "note": "no ncu table for this kernel yet: model flop count over the measured FFMA peak",
                "model_gather": model_gather, **common}
    # configs 1-2 (and other small fp64 cases): under / near one wave of threads, fields resident in L1 / L2: latency-bound.
    # report time-to-solution and microseconds per RK4 step (FP64 pipe share for config 2), no HBM fraction.
    us_per_step = win_s_per_pass * 1e6 / max(w.n_steps, 1)
    flop_unit = 250.0 if w.kind == 0 else 400.0
    return {"bound": "latency", "kernel": "cart_window_kernel" if w.kind == 0 else "simplex_window_kernel",
            "achieved": us_per_step, "peak": pk["launch_us"], "unit": "us per RK4 step (all seeds)", "frac": None,
            "fp64_pipe": {"flop_per_seed_step": flop_unit, "achieved": flop_unit * rate / 1e12, "peak": pk["fp64_fma_tflops"], "unit": "TFLOP/s",
                          "frac": flop_unit * rate / 1e12 / pk["fp64_fma_tflops"]},
            "note": "fewer seeds than (or about) one wave of 148 SMs x 2048 threads and fields that live in L1 / L2: bound by launch and "
                    "dependent-load latency; `peak` is the measured empty-launch latency for scale", **common}


def run_config(args, lcs, cfg, steps, warmup, rank, world, local, with_e2e, with_cpu):
    """Times `steps` passes of the hot path on one config; returns the fields of the JSON line (rank 0) or None."""
    import torch
    import torch.distributed as dist
    w, runs = make_workload(cfg, rank)
    ring = args.cfg5_ring if cfg == 5 else 0          # config 5 streams its snapshots from pinned host memory through a ring of device slots
    field = lcs.Field.from_workload(w, max_resident_snapshots=ring, pinned=True)
    series = cfg == 5 and args.cfg5_mode == "series"     # the 16 volumes advanced together through every window (lcs_advect_series)
    if cfg == 5 and not series:
        field.set_option("field_sets", 12)               # volume by volume: consecutive volumes share 9 of their 10 windows
    for kv in args.option:
        k, v = kv.split("=")
        field.set_option(k, int(v))
    tdt = torch.float32 if w.compute_dtype == np.float32 else torch.float64
    slab = args.shard == "volume" and cfg in (3, 4)      # ONE volume across the ranks: seed slabs along the slowest axis + a halo layer
    seeds_all = w.seeds()
    if slab:
        from paper_2209_13775_b200 import shard
        runs = [make_workload(cfg, 0)[1][0]]             # every rank works on the same volume
        plane = int(w.ng[0]) * (int(w.ng[1]) if w.dim == 3 else 1)
        k0, k1 = shard.slab_range(int(w.ng[w.dim - 1]), rank, world)
        seeds_all = np.ascontiguousarray(seeds_all[k0 * plane:k1 * plane])
    seeds_h = torch.from_numpy(seeds_all).pin_memory()
    seeds_d = seeds_h.cuda()
    n = seeds_h.shape[0]
    flow = torch.empty_like(seeds_d)
    flag = torch.empty(n, dtype=torch.uint8, device="cuda")
    es = torch.empty(n, dtype=torch.int32, device="cuda")
    stream = torch.cuda.current_stream()
    # set-up: everything lcs_advect needs is allocated here, once (the hot calls never allocate)
    if series:
        t_starts = [t0 for (t0, tf, h) in runs]
        T_ser, h_ser = runs[0][1] - runs[0][0], runs[0][2]
        flows = torch.empty((len(runs), n, w.dim), dtype=tdt, device="cuda")
        flags = torch.empty((len(runs), n), dtype=torch.uint8, device="cuda")
        ess = torch.empty((len(runs), n), dtype=torch.int32, device="cuda")
        field.advect_series(seeds_d, t_starts, T_ser, h_ser, flowmaps=flows, exit_flags=flags, exit_steps=ess)      # reserves
    else:
        field.reserve(n, max(int(round((tf - t0) / h)) for (t0, tf, h) in runs))

    def one_pass(count=None):
        """All rows of the hot path over one batch: flow map(s) -> CG -> FTLE."""
        if series:
            field.advect_series(seeds_d, t_starts, T_ser, h_ser, flowmaps=flows, exit_flags=flags, exit_steps=ess, reserve=False)
            for k in range(len(runs)):
                lcs.cg_ftle(w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, flows[k], flags[k], T_ser, want_cg=True, want_status=False)
            if count is not None:
                count.append(float(ess.sum(dtype=torch.int64).item()))
            return
        if cfg == 5:
            field.set_option("field_sets_clear", 0)      # every pass starts without resident blended fields: reuse only WITHIN a pass
        for (t0, tf, h) in runs:
            field.advect(seeds_d, t0, tf, h, flowmap=flow, exit_flag=flag, exit_step=es, reserve=False)
            if slab:
                shard.cg_ftle_slab(lcs, w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, flow, flag, tf - t0, rank, world, want_cg=True)
            else:
                lcs.cg_ftle(w.dim, w.ng, w.seed_spacing, w.seed_periodic, w.period, flow, flag, tf - t0, want_cg=True, want_status=False)
            if count is not None:
                count.append(float(es.sum(dtype=torch.int64).item()))

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # inputs of one pass: tracer records (two buffers when re-bundled) + seeds + outputs + the fields gathered from
    state_bytes = n * (32 * 2 + w.dim * 2 * seeds_h.element_size() + 5) + float(np.asarray(w.vel[0]).nbytes) * 2
    flush = state_bytes < L2_BYTES
    flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if flush else None
    for _ in range(max(warmup - 1, 0)):
        one_pass()
    counts = []
    one_pass(counts)                                     # last warm-up pass: seed-steps actually taken (exits shorten trajectories),
    steps_per_pass = float(sum(counts))                  # summed over EVERY run of the pass
    field.set_option("time_windows", 1)
    sampler = ClockSampler(local)
    sampler.start()
    l0 = lcs.kernel_launch_count()
    barrier()
    if flush:
        # small configs: the whole working set would stay in the 126 MB L2 between passes; write a 256 MB buffer between
        # timed passes (outside the per-pass event brackets)
        elapsed_ms = 0.0
        for _ in range(steps):
            flush_buf.fill_(1)
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            ev0.record(stream)
            one_pass()
            ev1.record(stream)
            torch.cuda.synchronize()
            elapsed_ms += ev0.elapsed_time(ev1)
        barrier()
    else:
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(steps):
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
    sec_per_step = elapsed_ms * 1e-3 / steps
    value = steps_all / sec_per_step

    # end to end through the C-ABI with HOST buffers: H2D of the seeds, D2H of the Cauchy-Green tensor and the FTLE inside the
    # timed region (the same outputs the device-timed pass writes)
    e2e = None
    if with_e2e and not slab:                            # (--shard volume: the host-buffer call has no halo exchange; device-timed only)
        ncg = 3 if w.dim == 2 else 6
        ftle_h = torch.empty(n, dtype=tdt).pin_memory()
        cg_h = torch.empty((n, ncg), dtype=tdt).pin_memory()
        esz = seeds_h.element_size()
        e_steps = steps if cfg == args.config else min(steps, 5)

        if series:
            ftle_h = torch.empty((len(runs), n), dtype=tdt).pin_memory()
            cg_h = torch.empty((len(runs), n, ncg), dtype=tdt).pin_memory()

        def e2e_pass():
            if series:
                field.ftle_series_host(w.ng, w.seed_spacing, w.seed_periodic, w.period, seeds_h.numpy(), t_starts, T_ser, h_ser,
                                       ftle=ftle_h.numpy(), cg=cg_h.numpy())
                return
            if cfg == 5:
                field.set_option("field_sets_clear", 0)
            for (t0, tf, h) in runs:
                field.ftle_host(w.ng, w.seed_spacing, w.seed_periodic, w.period, seeds_h.numpy(), t0, tf, h, ftle=ftle_h.numpy(), cg=cg_h.numpy())
        e2e_pass()
        barrier()
        t0w = time.perf_counter()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record(stream)
        for _ in range(e_steps):
            e2e_pass()
        ev1.record(stream)
        barrier()
        e_ms = max(ev0.elapsed_time(ev1), 0.0)
        e_wall = (time.perf_counter() - t0w) * 1e3
        e_ms = max(e_ms, e_wall)                          # copies on the legacy stream: wall clock bounds the region
        te = torch.tensor([e_ms], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e = {"value": steps_all / (float(te.item()) * 1e-3 / e_steps), "unit": UNIT, "steps": e_steps,
               "h2d_bytes_per_step": int(n * w.dim * esz * len(runs)), "d2h_bytes_per_step": int(n * (1 + ncg) * esz * len(runs)),
               "outputs": "cg + ftle", "seeds_per_s_to_ftle": seeds_all / (float(te.item()) * 1e-3 / e_steps)}
        del ftle_h, cg_h

    line = None
    if rank == 0:
        kernel_s = win_ns * 1e-9 / max(win_launches, 1)                    # average launch duration of the dominant kernel
        units_per_launch = steps_per_pass * steps / max(win_launches, 1)
        share = (win_ns * 1e-9) / (elapsed_ms * 1e-3) if world == 1 else None
        roofline = roofline_block(lcs, cfg, w, kernel_s, units_per_launch, share, win_launches, win_ns * 1e-9 / steps, args.option)
        l2_note = ("flushed: a 256 MB buffer is written between timed passes (working set %.1f MB < L2)" % (state_bytes / 1e6)) if flush else \
                  ("inputs larger than L2: tracer records, seeds, outputs and fields are %.0f MB per pass" % (state_bytes / 1e6))
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
                "ms_per_step": sec_per_step * 1e3, "higher_is_better": True, "scaling": "strong" if slab else "weak", "vs_baseline": None,
                "dtype": "f32" if w.compute_dtype == np.float32 else "f64", "data": "synthetic",
                "config": {"workload": w.name, "baseline_config": cfg, "seeds": n * len(runs), "rk4_steps": w.n_steps,
                           "seed_steps_per_pass": steps_per_pass, "parallelism": ("one volume in %d seed slabs, one halo layer of flow map exchanged before lcs_cg_ftle" % world) if slab else
                                          "independent FTLE volumes per rank, no collective",
                           "options": dict(kv.split("=") for kv in args.option), "l2": l2_note,
                           **({"series": "lcs_advect_series: %d volumes, overlapping ones advanced together" % len(runs)} if series else {}),
                           **({"snapshot_ring_slots": ring, "h2d_snapshot_bytes_total": int(field.info("h2d_bytes"))} if cfg == 5 else {})},
                "seeds_per_s_to_ftle": seeds_all / sec_per_step, "roofline": roofline, "clocks": clocks, "gpu_launches": int(launches),
                "e2e": e2e}
        if with_cpu and world == 1:
            line["cpu_baseline"] = cpu_baseline(w, runs)
    field.close()
    del field, seeds_d, flow, flag, es, flush_buf, seeds_h, w
    gc.collect()
    torch.cuda.empty_cache()
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--extra-configs", default="4,5", help="configs whose figures ride along under `configs` (N = 1, default config only)")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--option", action="append", default=[], help="library option key=value (e.g. integrator=2)")
    ap.add_argument("--shard", default="volumes", choices=["volumes", "volume"],
                    help="N > 1: 'volumes' = an independent FTLE volume per rank (weak scaling, no collective); 'volume' = ONE volume of "
                         "config 3 / 4 split into seed slabs with a halo exchange of the flow map before lcs_cg_ftle (strong scaling)")
    ap.add_argument("--cfg5-ring", type=int, default=4, help="config 5: device slots of the snapshot ring (0 = every snapshot resident, no streaming)")
    ap.add_argument("--cfg5-mode", default="series", choices=["series", "volumes"],
                    help="config 5: lcs_advect_series (overlapping volumes advanced together) or one lcs_advect per volume with resident field sets")
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

    line = run_config(args, lcs, args.config, args.steps, max(args.warmup, 1), rank, world, local, not args.no_e2e, not args.no_cpu_baseline)
    extras = []
    if world == 1 and args.config == 3 and args.extra_configs not in ("", "none") and not args.option:
        extras = [int(c) for c in args.extra_configs.split(",") if int(c) != args.config]
    if extras and line is not None:
        line["configs"] = {}
        for c in extras:
            # the other 3D configs of the >= 50% target, same passes / timing rules, fewer passes so that the default run stays short
            sub = run_config(args, lcs, c, min(args.steps, 10), min(max(args.warmup, 1), 3), rank, world, local, not args.no_e2e, False)
            line["configs"][str(c)] = {k: sub[k] for k in ("value", "unit", "steps", "warmup", "ms_per_step", "dtype", "config", "seeds_per_s_to_ftle",
                                                              "roofline", "clocks", "gpu_launches", "e2e")}
    if rank == 0 and line is not None:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
