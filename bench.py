#!/usr/bin/env python
"""bench.py -- marker RK4 pushes/sec (incl. field gather) of the TRIMEG hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5|cfg2|cfg3] [--impl reference]

One bench "step" = one pass of the whole hot path (DESIGN.md §1 rows a1-a6) over the
workload's marker batch: compact lost markers, then [cell sort -> fused RK4 push of
`sort_every` steps] repeated until the workload's nsteps RK4 steps are done, the field
frozen.  value = marker-RK4-steps of all ranks / max-over-ranks device time.

Default workload (N = 1): BASELINE.json configs[4] ("cfg5": 96x384 mesh, 16 toroidal modes,
2^24 markers, dt = 0.01, 50 steps) -- the 2^24-marker config the north_star target is
quoted on (reading G21).  Inputs are seeded synthetic data of that shape, resident in HBM
before the timed region; they are far larger than L2 (872 MB vs 126 MB).

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores, on a
bounded sample of the same workload.
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

import numpy as np

METRIC = "marker RK4 pushes/sec (incl. field gather)"
# dram__bytes_read.sum + dram__bytes_write.sum of one launch of the push kernel, from the committed ncu --set full
# capture (profiles/r01_fused_push_kernel.md): (workload, push kernel, sort_every, markers) -> bytes; null for anything else
PROFILED_DRAM_BYTES_PER_LAUNCH = {("cfg5", 3, 10, 1 << 24): 1.936e9, ("cfg5", 7, 10, 1 << 24): 1.94e9}
PUSH_KERNEL_NAMES = {0: "push_kernel", 1: "push_warp_kernel<2,4,6>", 2: "push_warp_kernel<4,4,16>", 3: "push_fused_kernel<2,384,1>",
                     4: "push_fused_kernel<3,256,1>", 5: "push_fused_kernel<4,256,1>", 6: "push_fused_kernel<2,192,2>", 7: "push_wcache_kernel<2,12,5>", 8: "push_warp_kernel<2,4,6,4>"}
UNIT = "marker-steps/s"


# ------------------------------------------------------------------ algorithmic work
def flops_per_marker_step(n_modes: int) -> int:
    """F_step = 4 (200 + 170 M): canonical count of SURVEY.md §8(d), FMA = 2 flops."""
    return 4 * (200 + 170 * n_modes)


def bytes_per_marker_call(nsteps_fused: int) -> float:
    """Marker stream of one push call: 52 B read + 44 B written per marker, once per call
    (all fused steps keep the state in registers)."""
    return 96.0


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d.get("hbm_gbs", 6650.0)), "measured (MEASURED_PEAKS.json)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------- clock sampling
class ClockSampler(threading.Thread):
    """nvidia-smi-equivalent clock / throttle-reason samples (NVML) during the timed region."""

    def __init__(self, index: int, period: float = 0.1):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.max_mhz = None
        self._halt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._halt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._halt.wait(self.period)

    def stop(self):
        self._halt.set()
        if self.is_alive():
            self.join(timeout=2.0)
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


# ------------------------------------------------------------------------------- oracle timing
def time_oracle(wl, target_seconds: float, steps: int = 1, warmup: int = 0):
    """Time oracle.push (as it stands) on a bounded strided sample of the workload.
    Returns (marker-steps/s, cores, description, seconds per timed step, sample size, rk4 steps)."""
    import oracle
    from paper_2601_14301_b200 import inputs
    o = oracle.from_workload(wl, inputs)
    o.bell_from_dofs(wl.modes, inputs.field_dofs(wl))
    cores = o.max_threads()
    n_pool = 1 << 16
    pool = inputs.markers(wl, n=n_pool)
    probe_n, probe_steps = 2048, 2
    probe = {k: v[:probe_n] for k, v in pool.items()}
    t0 = time.perf_counter()
    o.push(probe, wl.dt, probe_steps)
    rate = probe_n * probe_steps / (time.perf_counter() - t0)
    rk4 = max(1, min(wl.nsteps, 10))
    n_s = int(min(n_pool, max(1024, rate * target_seconds / rk4)))
    sample = {k: v[:n_s] for k, v in pool.items()}
    for _ in range(warmup):
        o.push(sample, wl.dt, rk4)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.push(sample, wl.dt, rk4)
    dt = (time.perf_counter() - t0) / steps
    desc = (f"first {n_s} markers of the seeded {wl.name} draw x {rk4} RK4 steps per step, "
            f"oracle.push with OpenMP over markers ({cores} threads)")
    return n_s * rk4 / dt, cores, desc, dt, n_s, rk4


def run_reference(args, wl):
    from paper_2601_14301_b200 import dist as D
    rank, _, world = D.env_rank()
    if rank != 0:
        return 0
    budget = 150.0 / max(1, args.steps + args.warmup)
    value, cores, desc, sec, n_s, rk4 = time_oracle(wl, min(20.0, budget), steps=args.steps, warmup=args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, extra={"reference_sample_markers": n_s, "reference_rk4_steps_per_step": rk4}),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(wl, extra=None):
    c = {"workload": f"{wl.name} (BASELINE.json configs[{int(wl.name[3:]) - 1}])",
         "mesh": f"{wl.n_r}x{wl.n_theta} rings x sectors, {wl.n_tri} triangles",
         "toroidal_modes": list(wl.modes), "markers_per_gpu": wl.n_markers, "dt": wl.dt,
         "rk4_steps_per_step": wl.nsteps, "l2": "inputs larger than L2 (no flush needed)"}
    if extra:
        c.update(extra)
    return c


# ----------------------------------------------------------------------------------- GPU arm
def run_gpu(args, wl):
    import torch
    from paper_2601_14301_b200 import binding, inputs
    from paper_2601_14301_b200 import dist as D

    rank, local_rank, world = D.init("nccl")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    binding.load()

    n = wl.n_markers
    sort_every = max(1, min(args.sort_every, wl.nsteps))
    ctx = binding.context_for(wl, inputs)
    ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs(wl)).to(dev), kind=0)
    if args.push_kernel >= 0:
        ctx.set_push_kernel(args.push_kernel)
    m_np = inputs.markers(wl, n=n, seed=D.rank_seed(wl.seed, rank))
    d = binding.markers_to_device(m_np, dev)
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    torch.cuda.synchronize()
    fp64_peak = ctx.measure_fp64_peak()
    fp64_peak3 = ctx.measure_fp64_peak_operands(3)     # DFMA stream with three fresh register operands
    hbm_peak, hbm_src = load_peaks()

    push_events = []
    state = {"n_active": n}

    def one_step(record: bool):
        """One pass of the hot path over the batch; returns marker-steps done."""
        units = 0
        done = 0
        n_act = state["n_active"]
        while done < wl.nsteps:
            k = min(sort_every, wl.nsteps - done)
            if done == 0:
                n_act, _ = ctx.compact(d, n=n_act)    # a6: drop lost markers once per step (syncs to return the count);
            ctx.sort(d, n=n_act)                      # a1  (markers lost since sort to the end of the range and are skipped)
            if record:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
            ctx.push(d, wl.dt, k, n=n_act)            # a2-a6, fused
            if record:
                e1.record()
                push_events.append((e0, e1, n_act * k))
            units += n_act * k
            done += k
        state["n_active"] = n_act
        return units

    for _ in range(args.warmup):
        one_step(False)
    torch.cuda.synchronize()
    st0 = ctx.get_stats()
    sampler = ClockSampler(local_rank)
    D.barrier()
    torch.cuda.synchronize()
    sampler.start()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record()
    units = 0
    for _ in range(args.steps):
        units += one_step(True)
    t_end.record()
    torch.cuda.synchronize()
    D.barrier()
    clocks = sampler.stop()
    seconds = t_start.elapsed_time(t_end) * 1e-3
    st1 = ctx.get_stats()
    launches = st1["n_launches"] - st0["n_launches"]
    tile_counters = ctx.get_tile_counters()

    agg = D.aggregate(units, seconds, {"launches": launches}, device=dev)

    # roofline of the dominant kernel (push_kernel), from the live CUDA-event durations
    push_s = sum(a.elapsed_time(b) for a, b, _ in push_events) * 1e-3
    push_units = sum(u for _, _, u in push_events)
    n_push = len(push_events)
    flops = flops_per_marker_step(len(wl.modes)) * push_units
    byts = bytes_per_marker_call(sort_every) * sum(u / max(1, min(sort_every, wl.nsteps)) for _, _, u in push_events)
    t_fp64 = flops / (fp64_peak * 1e12)
    t_hbm = byts / (hbm_peak * 1e9)
    roof = {
        "bound": "alu", "kernel": PUSH_KERNEL_NAMES.get(ctx.get_push_kernel(), "push kernel"),
        "achieved": flops / push_s * 1e-12, "peak": fp64_peak, "unit": "TFLOP/s",
        "frac": (flops / push_s * 1e-12) / fp64_peak,
        "peak_source": "FP64 DFMA throughput measured live by trimeg_measure_fp64_peak (nominal 148 SM x 64 DFMA/clk x 2 x 1.965 GHz = 37.2)",
        "traffic": PROFILED_DRAM_BYTES_PER_LAUNCH.get((wl.name, ctx.get_push_kernel(), sort_every, n)),
        "peak_three_register_operands": fp64_peak3, "frac_of_three_register_operand_peak": (flops / push_s * 1e-12) / fp64_peak3,
        "peak_three_register_operands_note": "DFMA stream whose three source operands all change from one instruction to the "
                                             "next (a Horner step over several markers): the FP64 pipe reads one 64-bit register "
                                             "operand per cycle, so such a stream issues every 3 cycles instead of 2",
        "algorithmic_flops_per_marker_step": flops_per_marker_step(len(wl.modes)),
        "algorithmic_bytes_per_marker_call": bytes_per_marker_call(sort_every),
        "hbm_time_frac_of_fp64_time": t_hbm / t_fp64, "hbm_peak_gbs": hbm_peak, "hbm_peak_source": hbm_src,
        "launches": n_push, "avg_launch_ms": push_s / max(1, n_push) * 1e3,
        "push_share_of_step": push_s / seconds,
        "tile_counters": tile_counters,
    }

    line = None
    if True:
        # ---- e2e: host buffers through the C ABI, copies inside the timed region
        e2e = None
        if not args.no_e2e:
            h = {k: torch.from_numpy(m_np[k]).pin_memory() for k in ("R", "Z", "phi", "vpar", "mu", "w")}
            h["cell"] = torch.full((n,), -1, dtype=torch.int32).pin_memory()
            ctx.push_host(h, wl.dt, wl.nsteps, locate_first=True)          # warm-up (also allocates)
            D.barrier()
            torch.cuda.synchronize()
            k_e2e = max(1, min(args.steps, 3))
            n_in = int((h["cell"] >= 0).sum())                            # markers still inside after the warm-up call
            lost0 = ctx.get_stats()["n_lost"]
            t0 = time.perf_counter()
            e2e_units = 0
            for _ in range(k_e2e):
                ctx.push_host(h, wl.dt, wl.nsteps, locate_first=False)     # returns when the results are in the host buffers
                e2e_units += n_in * wl.nsteps
                lost1 = ctx.get_stats()["n_lost"]                         # markers flagged lost leave the count of the next step
                n_in -= lost1 - lost0
                lost0 = lost1
            torch.cuda.synchronize()
            e2e_s = time.perf_counter() - t0
            ag2 = D.aggregate(e2e_units, e2e_s, {}, device=dev)
            e2e = {"value": ag2["value"], "unit": UNIT, "h2d_bytes_per_step": n * (6 * 8 + 4),
                   "d2h_bytes_per_step": n * (5 * 8 + 4), "steps": k_e2e,
                   "api": "trimeg_push_host (pinned host SoA in: H2D -> locate/sort of the whole batch -> push -> unsort -> D2H)"}

        cpu = None
        if rank == 0 and world == 1 and not args.no_cpu_baseline:
            v, cores, desc, _, _, _ = time_oracle(wl, 15.0)
            cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

        if rank == 0:
            line = {
                "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": agg["seconds"] / args.steps * 1e3, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": workload_config(wl, extra={"sort_every": sort_every, "parallelism": f"marker-shard x{world}",
                                                     "lost_markers": st1["n_lost"]}),
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(agg["launches"]),
                "roofline": roof, "cpu_baseline": cpu,
                "paper_context": "thesis K1 (one RHS eval, EM, B-spline equilibrium): 1.5e8 marker-RHS/s on 1 H100 "
                                 "(PAPER.md:911) ~ 3.8e7 RK4-step equivalents/s; other hardware, not like-for-like",
            }
            print(json.dumps(line), flush=True)
    return 0


def run_gather_sweep(args, wl):
    """BASELINE.json configs[3]: gather-only sweep (dphi, d/dR, d/dZ at the markers, no push) on the 64 x 256 mesh with
    modes {0, 5, 10}, marker counts 2^16 .. 2^max in powers of 4, markers as drawn and sorted by triangle.  One JSON line."""
    import torch
    from paper_2601_14301_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(0)
    binding.load()
    ctx = binding.context_for(wl, inputs)
    ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs(wl)).cuda(), kind=0)
    hbm_peak, _ = load_peaks()
    fp64_peak = ctx.measure_fp64_peak()
    flops = 25 + 170 * len(wl.modes) + 6                       # gather-only work per marker
    rows = []
    for lg in range(16, args.max_log2 + 1, 2):
        n = 1 << lg
        m = inputs.markers(wl, n=n)
        R, Z, phi = (torch.from_numpy(m[k]).cuda() for k in ("R", "Z", "phi"))
        cell = torch.empty(n, dtype=torch.int32, device="cuda")
        ctx.locate(R, Z, cell=cell)
        order = torch.argsort(cell, stable=True)
        out = {k: torch.empty(n, dtype=torch.float64, device="cuda") for k in ("dphi", "dphi_dR", "dphi_dZ")}
        for name, idx in (("as drawn", None), ("sorted by triangle", order)):
            r, z, p = (R, Z, phi) if idx is None else (R[idx].contiguous(), Z[idx].contiguous(), phi[idx].contiguous())
            ts = []
            for rep in range(3 + max(1, args.steps)):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                ctx.gather(r, z, p, want_dphi=False, out=out)
                e1.record()
                torch.cuda.synchronize()
                if rep >= 3:
                    ts.append(e0.elapsed_time(e1) * 1e-3)
            t = sorted(ts)[len(ts) // 2]
            rows.append({"markers": n, "order": name, "gathers_per_s": n / t, "ms": t * 1e3,
                         "algorithmic_GBps": 48.0 * n / t * 1e-9, "algorithmic_TFLOPs": flops * n / t * 1e-12})
        del R, Z, phi, cell, order, out
    line = {"metric": "field gathers/sec (dphi, d/dR, d/dZ; 3 toroidal modes)", "unit": "gathers/s", "n_gpus": 1,
            "config": workload_config(wl), "dtype": "f64", "data": "synthetic", "hbm_peak_gbs": hbm_peak, "fp64_peak_tflops": fp64_peak,
            "algorithmic_bytes_per_gather": 48, "algorithmic_flops_per_gather": flops, "rows": rows}
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--markers", type=int, default=0, help="override markers per GPU (testing)")
    ap.add_argument("--sort-every", type=int, default=10, help="RK4 steps fused per sort + push call")
    ap.add_argument("--push-kernel", type=int, default=-1, help="trimeg_set_push_kernel variant (-1 = library default)")
    ap.add_argument("--max-log2", type=int, default=26, help="cfg4 gather sweep: largest marker count 2^k")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    from paper_2601_14301_b200 import inputs
    import dataclasses
    wl = inputs.WORKLOADS[args.workload]
    if args.markers:
        wl = dataclasses.replace(wl, n_markers=args.markers)
    if args.workload == "cfg4":
        return run_gather_sweep(args, wl)
    if args.impl == "reference":
        return run_reference(args, wl)
    return run_gpu(args, wl)


if __name__ == "__main__":
    sys.exit(main())
