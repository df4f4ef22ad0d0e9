#!/usr/bin/env python
"""bench.py -- throughput of the fused SHASTA time step on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]

A "step" is one pass of the whole hot path = one SHASTA time step (three fused sweep kernels, the last of
which also writes the six primitive fields) over the whole grid.  Workload at N=1: BASELINE.json configs[3],
the 256^3 "event-by-event hotspots" state (fp64), built by paper_1206_0919_b200.inputs.hotspots (seeded,
synthetic).  N>1: N independent replicas (one event per GPU, a different seed per rank) -- the path does
not exchange data between GPUs, so scaling is "weak" and the only collectives are the
barrier and the max-over-ranks of the timing.

Prints ONE JSON line (rank 0).  Keys beyond the driver contract:
  roofline      dominant kernel, algorithmic bytes / CUDA-event duration, vs MEASURED_PEAKS.json
  step_roofline the whole step: 288 B per cell-update x value / peak
  cpu_baseline  the oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample
  e2e           same metric through the HOST-buffer entry points of the C ABI (copies inside the timing)
`--impl reference` times the oracle only (see reference_arm()).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "cell-updates/sec (fp64, 3 sweeps+cons2prim) at 256^3; % of HBM roofline"
UNIT = "cell-updates/s"
B_SWEEP = 80.0      # algorithmic bytes per cell of one fused sweep: 5 fields read + 5 written, fp64
B_PRIM = 48.0       # + six primitive fields written by the last sweep of a step
B_STEP = 3 * B_SWEEP + B_PRIM   # 288 B per cell-update
HBM_FALLBACK_GBS = 6650.0       # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# fp64 instructions (DADD/DMUL/DFMA/DSETP + 64-bit MUFU seeds) per UPDATED cell of one plain Gamma-law y/z sweep: 174.1 per
# marched cell (producer 96.1 + consumer 78.0, profiles/r2_sass_mix.md: executed-instruction counts of the ncu capture)
# x 1.0625 marched cells per updated cell (segments of 128 re-march 8 halo cells)
FP64_PER_CELL_SWEEP = 185.0
# fp64 issue rate: 16 lanes per SM sub-partition = 64 results/clk/SM nominal; measured 63.9 with the pipe saturated
# (tests/probes/fp64_issue_probe.cu, run by test_fp64_issue_rate_probe; record in profiles/parity_r2.json)
FP64_RESULTS_PER_CLK_SM = 63.9


def sampler_clock_mhz(sampler):
    """median SM clock seen so far by the NVML sampler (max clock if it has no samples yet)"""
    xs = sorted(s[1] for s in sampler.samples)
    return float(xs[len(xs) // 2]) if xs else float(getattr(sampler, "max_mhz", 1965))


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=120)
    ap.add_argument("--warmup", type=int, default=6)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=256, help="grid extent (256 = the metric's workload)")
    ap.add_argument("--precision", type=int, default=64, choices=[64, 32])
    ap.add_argument("--segment", type=int, default=0, help="tuning: cells marched per work item (0 = auto)")
    ap.add_argument("--workload", default="hotspots", choices=["hotspots", "spherical_riemann", "fireball"],
                    help="hotspots = BASELINE.json configs[3], the metric's workload (default); the others are the parity "
                         "configs 3 (general EOS) and 2, offered for profiling: their lines are not the headline metric")
    ap.add_argument("--batch", type=int, default=1, help="independent events per GPU advanced by one launch (SHASTA_BATCH)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    return ap.parse_args()


def hbm_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and clock-event reasons through NVML while the timed regions run."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown",
               0x4: "sw_power_cap", 0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting",
               0x100: "display_clock_setting", 0x10: "sync_boost"}

    def __init__(self, index, uuid=None):
        super().__init__(daemon=True)
        self.index, self.uuid = index, uuid
        self.samples, self.windows, self.stop_flag, self.err = [], [], False, None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            try:
                h = nv.nvmlDeviceGetHandleByUUID(self.uuid)
            except Exception:
                h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            while not self.stop_flag:
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                self.samples.append((time.perf_counter(), nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM), int(r)))
                time.sleep(0.005)
        except Exception as e:          # NVML missing: report it, do not fake numbers
            self.err = repr(e)

    def summary(self):
        if self.err or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "error": self.err or "no samples"}
        inside = [s for s in self.samples if any(a <= s[0] <= b for a, b in self.windows)] or self.samples
        mhz = sorted(s[1] for s in inside)
        bits = 0
        for s in inside:
            bits |= s[2]
        reasons = [n for b, n in self.REASONS.items() if bits & b]
        return {"sm_mhz": mhz[len(mhz) // 2], "sm_max_mhz": self.max_mhz, "reasons": reasons,
                "samples_under_load": len(inside)}


# ------------------------------------------------------------------------------------------------
# the oracle legs (the only places bench.py executes oracle/)
def oracle_sample(size, crop, seed, c=None):
    """Bounded sample of the workload: the central crop^3 sub-box of the size^3 hotspots state."""
    import numpy as np
    from paper_1206_0919_b200 import inputs
    if c is None:
        c = inputs.hotspots(size, steps=1, seed=seed)
    lo = (size - crop) // 2
    sl = (slice(lo, lo + crop),) * 3
    sub = dict(c)
    for k in ("e", "n", "vx", "vy", "vz"):
        sub[k] = np.ascontiguousarray(c[k][sl])
    sub["nx"] = sub["ny"] = sub["nz"] = crop
    return sub


def oracle_time_steps(sub, nsteps, warmup, threads):
    """Times `nsteps` oracle steps (after `warmup`) on the sample; returns (seconds, cells)."""
    from oracle import shasta_oracle as so
    so.build()
    so.set_threads(threads)
    o = so.Oracle(sub["nx"], sub["ny"], sub["nz"], sub["dx"], sub["lam"], sub["gamma"], sub["boundary"],
                  sub["mass"])
    o.set_state(sub["e"], sub["n"], sub["vx"], sub["vy"], sub["vz"])
    if warmup:
        o.step(warmup)
    t0 = time.perf_counter()
    o.step(nsteps)
    o.get_primitives()
    return time.perf_counter() - t0, sub["nx"] * sub["ny"] * sub["nz"]


def cpu_baseline(size, seed, c=None):
    cores = os.cpu_count() or 1
    crop = min(96, size)
    sub = oracle_sample(size, crop, seed, c)
    nsteps = 6
    dt, cells = oracle_time_steps(sub, nsteps, 0, cores)
    return {"value": cells * nsteps / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"central {crop}^3 sub-box of the {size}^3 hotspots state, {nsteps} steps "
                      f"(all six axis orders), oracle/shasta_oracle.c with {cores} OpenMP threads over pencils",
            "seconds": dt}


def reference_arm(args):
    """--impl reference: the oracle as it stands on the host cores; a step = one time step on a bounded
    sample (central sub-box) of the workload.  Rank 0 only."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cores = os.cpu_count() or 1
    total = args.steps + args.warmup
    crop = 96 if total <= 80 else (64 if total <= 300 else 48)
    crop = min(crop, args.size)
    sub = oracle_sample(args.size, crop, SEED0)
    dt, cells = oracle_time_steps(sub, args.steps, args.warmup, cores)
    value = cells * args.steps / dt
    sample = (f"central {crop}^3 sub-box of the {args.size}^3 hotspots state, one time step per bench step, "
              f"oracle/shasta_oracle.c with {cores} OpenMP threads over pencils")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / max(args.steps, 1),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"hotspots {args.size}^3 (BASELINE.json configs[3]), bounded sample: {sample}"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


SEED0 = 12060919


# ------------------------------------------------------------------------------------------------
def ours(args):
    import torch
    from paper_1206_0919_b200 import inputs
    from paper_1206_0919_b200.shasta import Shasta

    from paper_1206_0919_b200 import replicas
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    rank, world, local = replicas.env()
    torch.cuda.set_device(local)
    replicas.init(use_cuda=True)

    def barrier():
        replicas.barrier(use_cuda=True)

    def max_over_ranks(x):
        return replicas.max_over_ranks(x, use_cuda=True)

    # one independent event per rank (weak scaling, replicas: DESIGN.md 9)
    n = args.size
    import numpy as np
    B = max(1, args.batch)
    if args.workload == "hotspots":
        cs = [inputs.hotspots(n, steps=args.steps, seed=replicas.event_seed(rank) + 1000 * b) for b in range(B)]
    else:
        cs = [getattr(inputs, args.workload)(n, steps=args.steps) for b in range(B)]
    c = cs[0]
    ncell = B * n ** 3              # cells advanced per step on this GPU (all events of the batch)
    names = ("e", "n", "vx", "vy", "vz")
    host_in = [torch.from_numpy(c[k] if B == 1 else np.stack([cb[k] for cb in cs])).pin_memory() for k in names]
    host_out = [torch.empty(host_in[0].shape, dtype=torch.float64).pin_memory() for _ in range(6)]
    dev_in = [t.cuda(non_blocking=True) for t in host_in]
    stream = torch.cuda.current_stream()
    s = Shasta(n, n, n, c["dx"], c["lam"], c["gamma"], c["boundary"], c["mass"], precision=args.precision,
               segment=args.segment, batch=B)
    s.set_state(*dev_in)
    K, W = args.steps, args.warmup
    s.step(W)
    torch.cuda.synchronize()

    try:
        uuid = "GPU-" + str(torch.cuda.get_device_properties(local).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local, uuid)
    sampler.start()

    # ---- region A: K steps through shasta_step (the value)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    l0, w0 = s.launch_count, time.perf_counter()
    ev0.record(stream)
    s.step(K)
    ev1.record(stream)
    barrier()
    sampler.windows.append((w0, time.perf_counter()))
    launches = s.launch_count - l0
    ms_total = max_over_ranks(ev0.elapsed_time(ev1))
    value = replicas.aggregate_rate(ncell, K, ms_total, world)

    # ---- region B: the same K steps sweep by sweep, CUDA events around every kernel launch
    from paper_1206_0919_b200.shasta import BRANCH as table
    # The sweeps are issued exactly as shasta_step issues them: a step whose last sweep runs along x leaves its primitives
    # to the first sweep of the next step (emit_primitives = 2); only when no such sweep follows inside the region does
    # the x sweep write them at once (x kernel + element-wise cons2prim_kernel, timed as one entry).
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(3 * K + 1)]
    kinds = []
    base = s.step_index
    barrier()
    w0 = time.perf_counter()
    evs[0].record(stream)
    deferred = False
    for i in range(K):
        for k in range(3):
            a = table[(3 * (base + i) + k) % len(table)]
            emit, label, nbytes = (1 if k == 2 else 0), "", B_SWEEP
            if deferred:
                deferred, emit, label, nbytes = False, 2, "<emit_in>", B_SWEEP + B_PRIM
            elif k == 2 and a == 0:
                nxt = table[(3 * (base + i + 1)) % len(table)]
                if i + 1 < K and nxt != 0:
                    deferred, emit = True, 0
                else:
                    label, nbytes = "+cons2prim_kernel", 2 * B_SWEEP + B_PRIM - 40.0     # 80 + (40 read + 48 written)
            elif k == 2:
                label, nbytes = "<emit>", B_SWEEP + B_PRIM
            s.sweep(a, emit_primitives=emit)
            evs[3 * i + k + 1].record(stream)
            kinds.append((s.kernel_name(a) + label, nbytes))
    barrier()
    sampler.windows.append((w0, time.perf_counter()))
    per = {}
    for j, (name, nbytes) in enumerate(kinds):
        d = per.setdefault(name, {"ms": 0.0, "launches": 0, "bytes": 0.0})
        d["ms"] += evs[j].elapsed_time(evs[j + 1])
        d["launches"] += 1
        d["bytes"] += ncell * nbytes * (args.precision / 64.0)
    ms_sweeps = sum(d["ms"] for d in per.values())
    dom_name = max(per, key=lambda k: per[k]["ms"])
    dom = per[dom_name]
    peak, peak_src = hbm_peak()
    achieved = dom["bytes"] / (dom["ms"] * 1e-3) / 1e9
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")     # written from the committed ncu --set full capture
    if os.path.exists(tpath):
        try:
            traffic = json.load(open(tpath)).get(dom_name)
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "kernel": dom_name, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": "profiles/traffic.json (committed ncu --set full capture, not measured in this run)",
                "peak_source": peak_src,
                "bytes_per_launch": dom["bytes"] / dom["launches"],
                "avg_launch_ms": dom["ms"] / dom["launches"], "share_of_step": dom["ms"] / ms_sweeps,
                "kernels": {k: {"avg_launch_ms": v["ms"] / v["launches"], "launches": v["launches"],
                                "GB/s": v["bytes"] / (v["ms"] * 1e-3) / 1e9} for k, v in per.items()}}
    # the second roof of this path: fp64 instructions per cell and sweep against the fp64 issue rate at the
    # SM clock sampled in this run
    clk = sampler_clock_mhz(sampler)
    fp64_peak = FP64_RESULTS_PER_CLK_SM * torch.cuda.get_device_properties(local).multi_processor_count * clk * 1e6 / 1e9
    fp64_ach = ncell * FP64_PER_CELL_SWEEP / (dom["ms"] / dom["launches"] * 1e-3) / 1e9
    alu_roofline = {"bound": "alu", "kernel": dom_name, "achieved": fp64_ach, "peak": fp64_peak,
                    "unit": "G fp64 warp-lane results/s", "frac": fp64_ach / fp64_peak,
                    "per_cell_sweep": FP64_PER_CELL_SWEEP, "clock_mhz": clk,
                    "results_per_clk_sm": FP64_RESULTS_PER_CLK_SM,
                    "note": "per-cell count: profiles/r2_sass_mix.md; peak: measured 63.9 results/clk/SM (tests/probes/fp64_issue_probe.cu; nominal 64)"}
    step_gbs = value / world * B_STEP * (args.precision / 64.0) / 1e9
    step_roofline = {"bytes_per_cell_update": B_STEP * (args.precision / 64.0), "achieved": step_gbs,
                     "peak": peak, "unit": "GB/s", "frac": step_gbs / peak,
                     "frac_of_nominal_8TBs": step_gbs / 8000.0}

    # ---- e2e: the HOST-buffer entry points; upload + K steps + download inside the timed region
    e2e = None
    if not args.no_e2e:
        def job(nsteps):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            barrier()
            w = time.perf_counter()
            a.record(stream)
            s.set_state_host(*host_in)
            s.step(nsteps)
            s.get_primitives_host(host_out)
            b.record(stream)
            barrier()
            sampler.windows.append((w, time.perf_counter()))
            return max_over_ranks(a.elapsed_time(b))
        job(1)                                                   # warm the staging buffers
        ms_job = job(K)
        ms_rt = job(1)
        h2d, d2h = 5 * 8 * ncell, 6 * 8 * ncell
        e2e = {"value": world * ncell * K / (ms_job * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": h2d / K, "d2h_bytes_per_step": d2h / K,
               "pattern": f"one job = shasta_set_state_host (pinned, {h2d} B) + shasta_step({K}) + "
                          f"shasta_get_primitives_host (pinned, {d2h} B), all inside the timed region "
                          "(the paper uploads an event once and propagates it, PAPER.md:205)",
               "ms_per_job": ms_job,
               "roundtrip_every_step": {"value": world * ncell / (ms_rt * 1e-3), "unit": UNIT,
                                        "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                                        "ms_per_step": ms_rt}}
    sampler.stop_flag = True
    sampler.join(timeout=2.0)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(n, SEED0, c)

    if rank == 0:
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_total / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64" if args.precision == 64 else "f32", "data": "synthetic",
            "config": {"workload": (f"hotspots {n}^3 (BASELINE.json configs[3]): 50 Gaussian hotspots + "
                                    "vz=tanh(z/4), dx=0.1 fm, lambda=0.4, p=e/3, outflow; one event per GPU")
                                   if args.workload == "hotspots" else f"{args.workload} {n}^3 (a parity config, NOT the metric's workload)",
                       "grid": [n, n, n], "batch": B, "cells_per_gpu": ncell, "parallelism": f"replicas x{world}",
                       "l2": "state (2x5 fields ping-pong + 6 primitives, "
                             f"{16 * ncell * args.precision // 8 / 1e6:.0f} MB) is larger than the 126 MB L2; no flush",
                       "timing": "CUDA events on the launching stream, max over ranks"},
            "roofline": roofline, "alu_roofline": alu_roofline, "step_roofline": step_roofline, "cpu_baseline": cpu, "e2e": e2e,
            "gpu_launches": launches, "ms_step_sum_of_kernels": ms_sweeps / K, "clocks": sampler.summary(),
        }))
    replicas.finalize()


def main():
    args = parse_args()
    if args.impl == "reference":
        reference_arm(args)
    else:
        ours(args)


if __name__ == "__main__":
    main()
