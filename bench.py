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
# captures under profiles/: (workload, push kernel, sort_every, markers) -> bytes; null for anything else
PROFILED_DRAM_BYTES_PER_LAUNCH = {("cfg5", 2, 10, 1 << 24): 1.94e9}
PUSH_KERNEL_NAMES = {0: "push_kernel", 1: "push_lane_kernel<16>", 2: "push_wcache_kernel<2,12,5>"}
UNIT = "marker-steps/s"


# ------------------------------------------------------------------ algorithmic work
def flops_per_marker_step(n_modes: int) -> int:
    """F_step = 4 (200 + 170 M): canonical count of SURVEY.md §8(d), FMA = 2 flops."""
    return 4 * (200 + 170 * n_modes)


def flops_per_marker_step_spline() -> int:
    """Row f3, field on the cubic B-spline toroidal basis: per stage 200 as above, four REAL quintics with both
    derivatives (85 each, half of a complex mode), 28 for the eight spline weights, 32 for the four weighted sums."""
    return 4 * (200 + 4 * 85 + 28 + 32)


def flops_per_gather(n_modes: int) -> int:
    """Gather only (configs[3]): locator 25 + 170 per mode + 6 for the chain rule."""
    return 25 + 170 * n_modes + 6


def bytes_per_marker_call(nsteps_fused: int) -> float:
    """Marker stream of one push call: 52 B read + 44 B written per marker, once per call
    (all fused steps keep the state on chip)."""
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
def _strided(m, n_s):
    n = m["R"].size
    stride = max(1, n // n_s)
    return {k: np.ascontiguousarray(v[::stride][:n_s]) for k, v in m.items()}, stride


def time_oracle(wl, m_np, target_seconds: float, steps: int = 1, warmup: int = 0, one_core_seconds: float = 0.0, n_phi: int = 0,
                eom_variant: int = 0):
    """Time oracle.push (as it stands, never tuned) the way BASELINE.md §4 / SURVEY.md §8(d) plan it: a STRIDED
    subsample of the workload's seeded marker draw, pushed for the workload's full number of RK4 steps, with OpenMP
    over markers on all host cores -- and, if one_core_seconds > 0, once more on one core with a smaller strided
    sample.  The sample is the largest power of two (at most 2^20) that fits `target_seconds`.  Markers are
    independent, so the rate scales linearly to the full batch.  Returns a dict."""
    import oracle
    from paper_2601_14301_b200 import inputs
    o = oracle.from_workload(wl, inputs, eom_variant=eom_variant)
    if n_phi:
        o.bell_spline_from_dofs(inputs.spline_dofs(wl, n_phi))
    else:
        o.bell_from_dofs(wl.modes, inputs.field_dofs(wl))
    cores = o.max_threads()
    nsteps = max(1, wl.nsteps)
    probe, _ = _strided(m_np, 2048)
    t0 = time.perf_counter()
    o.push(probe, wl.dt, 2)
    rate = probe["R"].size * 2 / (time.perf_counter() - t0)
    n_s = 1 << int(max(10, min(20, np.floor(np.log2(max(1.0, rate * target_seconds / nsteps))))))
    n_s = min(n_s, m_np["R"].size)
    sample, stride = _strided(m_np, n_s)
    for _ in range(warmup):
        o.push(sample, wl.dt, nsteps)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.push(sample, wl.dt, nsteps)
    sec = (time.perf_counter() - t0) / steps
    out = {"value": n_s * nsteps / sec, "cores": cores, "nproc": os.cpu_count(), "seconds_per_step": sec, "sample_markers": n_s,
           "rk4_steps": nsteps,
           "sample": (f"every {stride}-th marker of the seeded {wl.name} draw ({n_s} markers) x the full {nsteps} RK4 steps, "
                      f"oracle.push with OpenMP over markers on {cores} threads (nproc {os.cpu_count()}); "
                      "markers are independent: the rate scales linearly to the full batch")}
    if one_core_seconds > 0:
        n_1 = 1 << int(max(8, np.floor(np.log2(max(1.0, out["value"] / cores * one_core_seconds / nsteps)))))
        n_1 = min(n_1, n_s)
        s1, stride1 = _strided(m_np, n_1)
        t0 = time.perf_counter()
        o.push(s1, wl.dt, nsteps, nthreads=1)
        out["value_one_core"] = n_1 * nsteps / (time.perf_counter() - t0)
        out["sample_one_core"] = f"every {stride1}-th marker ({n_1} markers) x {nsteps} RK4 steps on 1 thread"
        o.push(probe, wl.dt, 1, nthreads=cores)           # restore the OpenMP thread count
    return out


def run_reference(args, wl):
    from paper_2601_14301_b200 import dist as D
    from paper_2601_14301_b200 import inputs
    rank, _, world = D.env_rank()
    if rank != 0:
        return 0
    m_np = inputs.markers(wl, n=wl.n_markers)
    budget = 150.0 / max(1, args.steps + args.warmup)
    r = time_oracle(wl, m_np, min(20.0, budget), steps=args.steps, warmup=args.warmup, n_phi=args.n_phi, eom_variant=args.eom_variant)
    line = {
        "impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["seconds_per_step"] * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(wl, extra={"reference_sample_markers": r["sample_markers"], "reference_rk4_steps_per_step": r["rk4_steps"]}),
        "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "nproc": r["nproc"], "kind": "oracle",
                         "sample": r["sample"],
                         "note": "the oracle is the unoptimised correctness checker (plain monomial sums, gcc -O2): a baseline, "
                                 "not a tuned CPU push; the GPU/oracle ratio is not a like-for-like speedup"},
        "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_config(wl, extra=None, n_phi=0, eom_variant=0, unstructured=False, eq_table=0):
    c = {"workload": f"{wl.name} (BASELINE.json configs[{int(wl.name[3:]) - 1}])",
         "mesh": f"{wl.n_r}x{wl.n_theta} rings x sectors, {wl.n_tri} triangles",
         "toroidal_modes": list(wl.modes), "markers_per_gpu": wl.n_markers, "dt": wl.dt,
         "rk4_steps_per_step": wl.nsteps, "l2": "inputs larger than L2 (no flush needed)"}
    if unstructured:
        c["mesh"] = (f"unstructured: the {wl.n_r}x{wl.n_theta} ring x sector vertices jittered, Delaunay, numbering shuffled"
                     + ("" if unstructured == "shuffled" else ", triangles renumbered along a Hilbert curve (trimeg_mesh_locality_order)")
                     + f"; {wl.n_tri} triangles; box-grid locator (row f4)")
    if eq_table:
        c["equilibrium"] = f"cubic-B-spline tables {eq_table}x{eq_table} of psi (the configs' flux function, elongation 1.2) and F(psi) = B0 R0 (1 + 0.1 psi) (row f4)"
    if eom_variant:
        c["eom_variant"] = {1: "1 (b0* normalised by B/B*par, reading G2)", 2: "2 (reduced equations A.19-A.29, row f4)"}[eom_variant]
    if n_phi:
        c["toroidal_basis"] = f"cubic B-splines on {n_phi} planes (row f3), the mode list's perturbation sampled on the planes"
    if extra:
        c.update(extra)
    return c


# ----------------------------------------------------------------------------------- GPU arm
class PushRun:
    """One workload resident on the current device: context, field, the seeded marker batch (a pristine copy and a
    working copy).  A bench step = restore the batch to the workload's initial state (device copy), compact, then
    [cell sort -> fused push of `sort_every` RK4 steps] until the workload's nsteps are done."""

    def __init__(self, wl, sort_every, push_kernel=-1, seed=None, keep_host=True, n_phi=0, eom_variant=0, unstructured=False, eq_table=0):
        import torch
        from paper_2601_14301_b200 import binding, inputs
        self.torch, self.wl = torch, wl
        self.n = wl.n_markers
        self.sort_every = max(1, min(sort_every, wl.nsteps))
        self.n_phi, self.eom_variant, self.umesh = n_phi, eom_variant, None
        if unstructured:                                   # row f4: the same cross-section as an unstructured triangulation, box-grid locator
            Rv, Zv, tri = inputs.unstructured_mesh(wl)
            if unstructured != "shuffled":                 # the caller's one-off renumbering along a Hilbert curve (include/trimeg.h)
                tri = np.ascontiguousarray(tri[binding.mesh_locality_order(Rv, Zv, tri)])
            self.umesh = (Rv, Zv, tri)
            self.ctx = binding.Context.unstructured(*self.umesh, wl.params(eom_variant, 0))
            self.ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs_at(wl, self.umesh[0], self.umesh[1])).cuda(), kind=0)
        else:
            self.ctx = binding.context_for(wl, inputs, eom_variant=eom_variant)
            if n_phi:                                      # row f3: the same perturbation on n_phi B-spline planes
                self.ctx.field_upload_spline(torch.from_numpy(inputs.spline_dofs(wl, n_phi)).cuda(), kind=0)
            else:
                self.ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs(wl)).cuda(), kind=0)
        self.eq_tab = None
        if eq_table:                                       # row f4: the configs' circular flux function, elongated by 1.2, as B-spline tables
            self.eq_tab = inputs.equilibrium_table(wl, eq_table, eq_table, 33, kappa=1.2, f1=0.1)
            self.ctx.equilibrium_upload(self.eq_tab)
        if push_kernel >= 0:
            self.ctx.set_push_kernel(push_kernel)
        m_np = inputs.markers(wl, n=self.n, seed=seed)
        self.d0 = binding.markers_to_device(m_np, "cuda")
        self.ctx.locate(self.d0["R"], self.d0["Z"], cell=self.d0["cell"])
        self.d = {k: torch.empty_like(v) for k, v in self.d0.items()}
        self.m_np = m_np if keep_host else None
        self.push_events = []
        self.n_start = None
        torch.cuda.synchronize()

    def step(self, record):
        wl, ctx, d = self.wl, self.ctx, self.d
        for k, v in self.d0.items():                      # every step starts from the config's initial state
            d[k].copy_(v)
        n_act, _ = ctx.compact(d, n=self.n)               # a6: drop the markers outside the mesh (syncs to return the count)
        self.n_start = n_act
        done = 0
        while done < wl.nsteps:
            k = min(self.sort_every, wl.nsteps - done)
            ctx.sort(d, n=n_act)                          # a1 (markers lost since go to the end of the range and are skipped)
            if record:
                e0, e1 = self.torch.cuda.Event(enable_timing=True), self.torch.cuda.Event(enable_timing=True)
                e0.record()
            ctx.push(d, wl.dt, k, n=n_act)                # a2-a6, fused
            if record:
                e1.record()
                self.push_events.append((e0, e1, n_act * k))
            done += k

    def run(self, steps, warmup, barrier=lambda: None, device_index=0):
        torch = self.torch
        for _ in range(warmup):
            self.step(False)
        torch.cuda.synchronize()
        st0 = self.ctx.get_stats()
        sampler = ClockSampler(device_index)
        barrier()
        torch.cuda.synchronize()
        sampler.start()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        for _ in range(steps):
            self.step(True)
        t1.record()
        torch.cuda.synchronize()
        barrier()
        clocks = sampler.stop()
        st1 = self.ctx.get_stats()
        lost = st1["n_lost"] - st0["n_lost"]
        # unit count: a marker that leaves the mesh during a bench step counts ZERO steps for that step (lower bound)
        units = self.wl.nsteps * (steps * self.n_start - lost)
        return {"units": units, "seconds": t0.elapsed_time(t1) * 1e-3, "clocks": clocks, "launches": st1["n_launches"] - st0["n_launches"],
                "lost_per_step": lost / max(1, steps), "n_start": self.n_start}

    def kernel_name(self):
        k = self.ctx.get_push_kernel()
        if self.n_phi and k == 1:
            return "push_lane_kernel<16> (B-spline plane records)"
        core = not (self.n_phi or self.eom_variant == 2 or self.umesh is not None or getattr(self, "eq_tab", None) is not None)
        if k == 2 and len(self.wl.modes) <= 14 and core:
            return "push_wcache_kernel<2,16,5>"                    # TRIMEG_WCACHE_16_MAX_MODES, core build
        return PUSH_KERNEL_NAMES.get(k, "push kernel")

    def flops_unit(self):
        f = flops_per_marker_step_spline() if self.n_phi else flops_per_marker_step(len(self.wl.modes))
        # reduced equations (row f4): no curl b, no B*_par -- 140 instead of 200 flops per stage outside the gather
        return f - 4 * 60 if self.eom_variant == 2 else f

    def roofline(self, fp64_peak, seconds):
        wl = self.wl
        push_s = sum(a.elapsed_time(b) for a, b, _ in self.push_events) * 1e-3
        push_units = sum(u for _, _, u in self.push_events)
        n_push = len(self.push_events)
        flops = self.flops_unit() * push_units
        return {"bound": "alu", "kernel": self.kernel_name(),
                "achieved": flops / push_s * 1e-12, "peak": fp64_peak, "unit": "TFLOP/s",
                "frac": (flops / push_s * 1e-12) / fp64_peak, "launches": n_push, "avg_launch_ms": push_s / max(1, n_push) * 1e3,
                "push_share_of_step": push_s / seconds, "units_per_launch": push_units / max(1, n_push)}

    def check_against_oracle(self, stride=4096):
        """Push a fresh 1/stride strided sample of the batch for the workload's nsteps in the launch pattern that was
        timed (locate, then [sort -> push sort_every steps] ...) and compare it with the oracle; also: every state
        array of the batch that was timed is finite."""
        import oracle
        torch = self.torch
        from paper_2601_14301_b200 import binding, inputs
        wl = self.wl
        for k in ("R", "Z", "phi", "vpar", "w"):
            assert bool(torch.isfinite(self.d[k][: self.n_start]).all()), f"non-finite {k} after the timed steps"
        sample = {k: np.ascontiguousarray(v[::stride]) for k, v in self.m_np.items()}
        ds = binding.markers_to_device(sample, "cuda")
        self.ctx.locate(ds["R"], ds["Z"], cell=ds["cell"])
        ident = torch.arange(ds["R"].numel(), device="cuda")
        done = 0
        while done < wl.nsteps:
            k = min(self.sort_every, wl.nsteps - done)
            perm = self.ctx.sort(ds, want_perm=True)
            ident = ident[perm]
            self.ctx.push(ds, wl.dt, k)
            done += k
        got = {k: np.empty_like(v.cpu().numpy()) for k, v in ds.items()}
        idx = ident.cpu().numpy()
        for k, v in ds.items():
            got[k][idx] = v.cpu().numpy()
        if self.umesh is not None:
            o = oracle.Oracle.unstructured(*self.umesh, wl.params(self.eom_variant, 0))
            o.bell_from_dofs(wl.modes, inputs.field_dofs_at(wl, self.umesh[0], self.umesh[1]))
        else:
            o = oracle.from_workload(wl, inputs, eom_variant=self.eom_variant)
            if self.n_phi:
                o.bell_spline_from_dofs(inputs.spline_dofs(wl, self.n_phi))
            else:
                o.bell_from_dofs(wl.modes, inputs.field_dofs(wl))
        if self.eq_tab is not None:
            o.set_equilibrium_table(self.eq_tab)
        want = o.push(sample, wl.dt, wl.nsteps)
        assert np.array_equal(got["cell"] < 0, want["cell"] < 0), "lost-marker sets differ"
        worst = 0.0
        for k, scale in (("R", wl.R0), ("Z", wl.a), ("vpar", 1.0), ("w", max(1e-4, float(np.abs(want["w"]).max())))):
            worst = max(worst, float((np.abs(got[k] - want[k]) / np.maximum(np.maximum(np.abs(got[k]), np.abs(want[k])), scale)).max()))
        dphi = np.abs((got["phi"] - want["phi"] + np.pi) % (2 * np.pi) - np.pi).max() / (2 * np.pi)
        worst = max(worst, float(dphi))
        cells_differ = int((got["cell"] != want["cell"]).sum())
        tol = 1e-9 * max(1.0, wl.nsteps / 20.0)
        assert worst < tol, f"bench parity check failed: {worst} >= {tol}"
        # note: the library's own Bell expansion (kind 0) vs the oracle's LU: 1e-11 relative per coefficient
        return {"sample_markers": int(sample["R"].size), "rk4_steps": wl.nsteps, "max_rel_err": worst, "tolerance": tol,
                "cells_differ": cells_differ, "lost_in_sample": int((want["cell"] < 0).sum()), "finite": True}

    def close(self):
        self.ctx.close()
        self.d = self.d0 = None
        self.torch.cuda.empty_cache()


def e2e_run(ctx, wl, m_np, k_e2e, device_value, D=None, dev=None):
    """The metric through trimeg_push_host with pinned host SoA buffers: every call starts from the config's initial state
    (restored untimed), H2D and D2H inside the timed region; one warm-up call (it also allocates)."""
    import torch
    n = m_np["R"].size
    keys = ("R", "Z", "phi", "vpar", "mu", "w")
    h0 = {k: torch.from_numpy(m_np[k]) for k in keys}
    h = {k: torch.empty_like(h0[k]).pin_memory() for k in keys}
    h["cell"] = torch.empty(n, dtype=torch.int32).pin_memory()
    e2e_s, e2e_units = 0.0, 0
    for it in range(1 + k_e2e):
        for k in keys:
            h[k].copy_(h0[k])
        h["cell"].fill_(-1)
        if D is not None:
            D.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ctx.push_host(h, wl.dt, wl.nsteps, locate_first=True)     # returns when the results are in the host buffers
        dt_call = time.perf_counter() - t0
        if it > 0:
            e2e_s += dt_call
            e2e_units += int((h["cell"] >= 0).sum()) * wl.nsteps  # markers lost on the way count zero steps
    if D is not None:
        ag2 = D.aggregate(e2e_units, e2e_s, {}, device=dev)
        value = ag2["value"]
    else:
        value = e2e_units / e2e_s
    del h, h0
    ctx.release_host_buffers()
    return {"value": value, "unit": UNIT, "h2d_bytes_per_step": n * 6 * 8, "d2h_bytes_per_step": n * (5 * 8 + 4), "steps": k_e2e,
            "frac_of_device_value": value / device_value,
            "api": "trimeg_push_host (pinned host SoA in: chunks of the batch go H2D -> locate -> cell sort -> push, re-sort "
                   "every 10 steps -> unsort -> D2H on three streams, copies under the push of other chunks)"}


def gather_rows(ctx, wl, log2s, reps, hbm_peak, fp64_peak):
    """BASELINE.json configs[3]: gather only (dphi, d/dR, d/dZ, no push), markers as drawn and sorted by triangle.
    Markers as drawn: every marker reads the coefficient record of a random triangle; the row's `frac_record_gather` is the
    record bytes per second against the same access pattern without arithmetic (trimeg_measure_gather_peak on a table of
    the field's size)."""
    import torch
    from paper_2601_14301_b200 import inputs
    flops = flops_per_gather(len(wl.modes))
    rec_bytes = 16 * 21 * len(wl.modes)
    gather_peak = ctx.measure_gather_peak(rec_bytes * wl.n_tri, rec_bytes) if rec_bytes else None
    rows = []
    for lg in log2s:
        n = 1 << lg
        pos = inputs.positions(wl, n)
        R, Z, phi = (torch.from_numpy(pos[k]).cuda() for k in ("R", "Z", "phi"))
        del pos
        cell = torch.empty(n, dtype=torch.int32, device="cuda")
        ctx.locate(R, Z, cell=cell)
        out = {k: torch.empty(n, dtype=torch.float64, device="cuda") for k in ("dphi", "dphi_dR", "dphi_dZ")}
        for name in ("as drawn", "sorted by triangle"):
            if name == "sorted by triangle":
                order = torch.argsort(cell, stable=True)
                R, Z, phi, cell = R[order].contiguous(), Z[order].contiguous(), phi[order].contiguous(), cell[order].contiguous()
                del order
            ts = []
            for rep in range(3 + max(1, reps)):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                ctx.gather(R, Z, phi, cell_hint=cell, want_dphi=False, out=out)
                e1.record()
                torch.cuda.synchronize()
                if rep >= 3:
                    ts.append(e0.elapsed_time(e1) * 1e-3)
            t = sorted(ts)[len(ts) // 2]
            rows.append({"markers": n, "order": name, "gathers_per_s": n / t, "ms": t * 1e3,
                         "algorithmic_GBps": 52.0 * n / t * 1e-9, "frac_hbm": 52.0 * n / t * 1e-9 / hbm_peak,
                         "algorithmic_TFLOPs": flops * n / t * 1e-12, "frac_fp64": flops * n / t * 1e-12 / fp64_peak})
            if name == "as drawn" and gather_peak:
                rows[-1].update({"record_GBps": rec_bytes * n / t * 1e-9, "record_gather_peak_GBps": gather_peak,
                                 "frac_record_gather": rec_bytes * n / t * 1e-9 / gather_peak})
        del R, Z, phi, cell, out
        torch.cuda.empty_cache()
    return rows


def run_gpu(args, wl):
    import dataclasses
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
    run = PushRun(wl, args.sort_every, args.push_kernel, seed=D.rank_seed(wl.seed, rank), n_phi=args.n_phi, eom_variant=args.eom_variant,
                  unstructured=args.unstructured, eq_table=args.eq_table)
    ctx = run.ctx
    fp64_peak = ctx.measure_fp64_peak()
    fp64_peak3 = ctx.measure_fp64_peak_operands(3)     # DFMA stream with three fresh register operands
    hbm_peak, hbm_src = load_peaks()

    res = run.run(args.steps, args.warmup, barrier=D.barrier, device_index=local_rank)
    agg = D.aggregate(res["units"], res["seconds"], {"launches": res["launches"]}, device=dev)
    tile_counters = ctx.get_tile_counters()

    roof = run.roofline(fp64_peak, res["seconds"])
    flops_unit = run.flops_unit()
    t_fp64 = flops_unit * roof["units_per_launch"] / (fp64_peak * 1e12)
    t_hbm = bytes_per_marker_call(run.sort_every) * res["n_start"] / (hbm_peak * 1e9)
    roof.update({
        "peak_source": "FP64 DFMA throughput measured live by trimeg_measure_fp64_peak (nominal 148 SM x 64 DFMA/clk x 2 x 1.965 GHz = 37.2)",
        "traffic": PROFILED_DRAM_BYTES_PER_LAUNCH.get((wl.name, ctx.get_push_kernel(), run.sort_every, n)),
        "peak_three_register_operands": fp64_peak3, "frac_of_three_register_operand_peak": roof["achieved"] / fp64_peak3,
        "algorithmic_flops_per_marker_step": flops_unit,
        "algorithmic_bytes_per_marker_call": bytes_per_marker_call(run.sort_every),
        "hbm_time_frac_of_fp64_time": t_hbm / t_fp64, "hbm_peak_gbs": hbm_peak, "hbm_peak_source": hbm_src,
        "schedule_counters": tile_counters,
    })

    # ---- the bench checks what it timed: finiteness of the timed batch, a fresh strided sample against the oracle
    check = None
    if rank == 0 and not args.no_check:
        check = run.check_against_oracle(stride=max(1, n // 4096))

    # ---- e2e: host buffers through the C ABI, copies inside the timed region
    e2e = None
    if not args.no_e2e:
        e2e = e2e_run(ctx, wl, run.m_np, max(1, min(args.steps, 3)), agg["value"], D, dev)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.unstructured and not args.eq_table:
        r = time_oracle(wl, run.m_np, 15.0, one_core_seconds=6.0, n_phi=args.n_phi, eom_variant=args.eom_variant)
        cpu = {"value": r["value"], "unit": UNIT, "cores": r["cores"], "nproc": r["nproc"], "kind": "oracle", "sample": r["sample"],
               "value_one_core": r.get("value_one_core"), "sample_one_core": r.get("sample_one_core"),
               "note": "the oracle is the unoptimised correctness checker (plain monomial sums, gcc -O2): a baseline, not a "
                       "tuned CPU push; the GPU/oracle ratio is not a like-for-like speedup"}
    run.close()

    # ---- the other configs, device-timed the same way (N = 1 only): short runs, same live peaks
    sweep = None
    if rank == 0 and world == 1 and not args.no_sweep and wl.name == "cfg5" and not args.markers and not args.n_modes and not args.n_phi and not args.eom_variant and not args.unstructured and not args.eq_table:
        sweep = {}
        for name in ("cfg2", "cfg3"):
            w2 = inputs.WORKLOADS[name]
            r2 = PushRun(w2, args.sort_every, -1, keep_host=True)
            out = r2.run(2, 3)
            rf = r2.roofline(fp64_peak, out["seconds"])
            chk = None if args.no_check else r2.check_against_oracle(stride=max(1, w2.n_markers // 2048))
            e2 = None if args.no_e2e else e2e_run(r2.ctx, w2, r2.m_np, 1, out["units"] / out["seconds"])
            sweep[name] = {"value": out["units"] / out["seconds"], "unit": UNIT, "steps": 2, "warmup": 3,
                           "ms_per_step": out["seconds"] / 2 * 1e3, "kernel": rf["kernel"], "frac": rf["frac"],
                           "achieved_tflops": rf["achieved"], "avg_launch_ms": rf["avg_launch_ms"],
                           "push_share_of_step": rf["push_share_of_step"], "clocks": out["clocks"],
                           "config": workload_config(w2, extra={"sort_every": r2.sort_every}), "oracle_check": chk, "e2e": e2}
            r2.close()
            del r2
        w4 = inputs.WORKLOADS["cfg4"]
        c4 = binding.context_for(w4, inputs)
        c4.field_upload(w4.modes, torch.from_numpy(inputs.field_dofs(w4)).cuda(), kind=0)
        sampler = ClockSampler(local_rank)
        sampler.start()
        rows = gather_rows(c4, w4, (24, 28), 2, hbm_peak, fp64_peak)
        sweep["cfg4"] = {"metric": "field gathers/sec (dphi, d/dR, d/dZ; 3 toroidal modes)", "unit": "gathers/s",
                         "algorithmic_bytes_per_gather": 52, "algorithmic_flops_per_gather": flops_per_gather(len(w4.modes)),
                         "rows": rows, "clocks": sampler.stop(), "config": workload_config(w4)}
        c4.close()
        # row f3: cfg5's mesh, markers and perturbation with the field on 32 cubic B-spline planes
        r3 = PushRun(inputs.WORKLOADS["cfg5"], args.sort_every, -1, keep_host=True, n_phi=32)
        out = r3.run(2, 3)
        rf = r3.roofline(fp64_peak, out["seconds"])
        chk = None if args.no_check else r3.check_against_oracle(stride=max(1, r3.wl.n_markers // 2048))
        sweep["spline_cfg5"] = {"value": out["units"] / out["seconds"], "unit": UNIT, "steps": 2, "warmup": 3,
                                "ms_per_step": out["seconds"] / 2 * 1e3, "kernel": rf["kernel"], "frac": rf["frac"],
                                "achieved_tflops": rf["achieved"], "avg_launch_ms": rf["avg_launch_ms"],
                                "algorithmic_flops_per_marker_step": r3.flops_unit(),
                                "push_share_of_step": rf["push_share_of_step"], "clocks": out["clocks"],
                                "config": workload_config(r3.wl, n_phi=32, extra={"sort_every": r3.sort_every}), "oracle_check": chk}
        r3.close()
        del r3
        # row f4: cfg5's cross-section as an unstructured triangulation (Hilbert-renumbered), box-grid locator
        r4 = PushRun(inputs.WORKLOADS["cfg5"], args.sort_every, -1, keep_host=True, unstructured="hilbert")
        out = r4.run(2, 3)
        rf = r4.roofline(fp64_peak, out["seconds"])
        chk = None if args.no_check else r4.check_against_oracle(stride=max(1, r4.wl.n_markers // 2048))
        sweep["unstructured_cfg5"] = {"value": out["units"] / out["seconds"], "unit": UNIT, "steps": 2, "warmup": 3,
                                      "ms_per_step": out["seconds"] / 2 * 1e3, "kernel": rf["kernel"], "frac": rf["frac"],
                                      "achieved_tflops": rf["achieved"], "avg_launch_ms": rf["avg_launch_ms"],
                                      "push_share_of_step": rf["push_share_of_step"], "clocks": out["clocks"],
                                      "config": workload_config(r4.wl, unstructured="hilbert", extra={"sort_every": r4.sort_every}),
                                      "oracle_check": chk}
        r4.close()
        del r4
        sweep["em_cfg5"] = em_run(inputs.WORKLOADS["cfg5"], 3, fp64_peak, hbm_peak, with_oracle=not args.no_check)
        sweep["scatter_cfg5"] = scatter_run(inputs.WORKLOADS["cfg5"], 3, fp64_peak, hbm_peak, with_oracle=not args.no_check)

    if rank == 0:
        line = {
            "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": agg["seconds"] / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(wl, n_phi=args.n_phi, eom_variant=args.eom_variant, unstructured=args.unstructured, eq_table=args.eq_table, extra={"sort_every": run.sort_every, "parallelism": f"marker-shard x{world}",
                                                 "lost_markers_per_step": res["lost_per_step"],
                                                 "unit_count": "every bench step restarts from the config's initial state; a marker "
                                                               "that leaves the mesh during a step counts zero steps for it"}),
            "clocks": res["clocks"], "e2e": e2e, "gpu_launches": int(agg["launches"]),
            "roofline": roof, "cpu_baseline": cpu, "oracle_check": check, "config_sweep": sweep,
            "paper_context": "thesis K1 (one RHS eval, EM, B-spline equilibrium): 1.5e8 marker-RHS/s on 1 H100 "
                             "(PAPER.md:911) ~ 3.8e7 RK4-step equivalents/s; other hardware, not like-for-like",
        }
        print(json.dumps(line), flush=True)
    return 0


def flops_per_scatter(n_modes: int) -> int:
    """Particle-to-grid projection (row f1), per marker: locator 25 + 20 for the monomials, per mode 21 complex x real
    multiply-adds (84 flops) + the rotation of the toroidal factor (8)."""
    return 45 + 92 * n_modes


def scatter_run(wl, reps, fp64_peak, hbm_peak, with_oracle=True):
    """trimeg_scatter on the workload's marker batch (order as drawn), device-timed per call with CUDA events."""
    import torch
    from paper_2601_14301_b200 import binding, inputs
    ctx = binding.context_for(wl, inputs)
    ctx.field_upload(wl.modes, torch.from_numpy(inputs.field_dofs(wl)).cuda(), kind=0)
    n = wl.n_markers
    m = inputs.markers(wl, n=n)
    m["w"] = np.random.default_rng([wl.seed, 7]).standard_normal(n)
    d = binding.markers_to_device(m, "cuda")
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    out = torch.empty((len(wl.modes), wl.n_vert, 6), dtype=torch.complex128, device="cuda")
    n_in = int((d["cell"] >= 0).sum())
    fl = flops_per_scatter(len(wl.modes))
    rows = []
    for order in ("as drawn", "cell-sorted"):
        if order == "cell-sorted":
            ctx.sort(d)                                   # the order the push leaves the markers in
        st0 = ctx.get_stats()
        ts = []
        for rep in range(3 + reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.scatter(d, out=out)
            e1.record()
            torch.cuda.synchronize()
            if rep >= 3:
                ts.append(e0.elapsed_time(e1) * 1e-3)
        launches = (ctx.get_stats()["n_launches"] - st0["n_launches"]) // (3 + reps)
        t = sorted(ts)[len(ts) // 2]
        rows.append({"order": order, "value": n_in / t, "unit": "markers/s", "ms_per_call": t * 1e3, "launches_per_call": int(launches),
                     "achieved_tflops": fl * n_in / t * 1e-12, "frac": fl * n_in / t * 1e-12 / fp64_peak})
    best = rows[1]
    res = {"metric": "markers projected per second (trimeg_scatter, row f1)", "value": best["value"], "unit": "markers/s",
           "ms_per_call": best["ms_per_call"], "markers": n, "markers_inside": n_in, "order": best["order"], "rows": rows,
           "roofline": {"bound": "alu", "kernel": "whole call, 6 launches (scatter_moments_kernel dominates)", "achieved": best["achieved_tflops"],
                        "peak": fp64_peak, "unit": "TFLOP/s", "frac": best["frac"],
                        "algorithmic_flops_per_marker": fl, "algorithmic_bytes_per_marker": 36,
                        "hbm_time_frac_of_fp64_time": (36.0 / (hbm_peak * 1e9)) / (fl / (fp64_peak * 1e12))},
           "config": workload_config(wl)}
    if with_oracle:
        import oracle
        o = oracle.from_workload(wl, inputs)
        o.set_modes(wl.modes)
        stride = max(1, n // (1 << 17))
        sl = slice(0, None, stride)
        t0 = time.perf_counter()
        want = o.scatter(m["R"][sl], m["Z"][sl], m["phi"][sl], m["w"][sl])
        dt_o = time.perf_counter() - t0
        ds = binding.markers_to_device({k: np.ascontiguousarray(v[sl]) for k, v in m.items()}, "cuda")
        ctx.locate(ds["R"], ds["Z"], cell=ds["cell"])
        got = ctx.scatter(ds).cpu().numpy()
        err = max(float(np.abs(got[k] - want[k]).max() / np.abs(want[k]).max()) for k in range(len(wl.modes)))
        assert err < 1e-11, f"scatter parity check failed: {err}"
        res["oracle_check"] = {"sample_markers": int(m["R"][sl].size), "max_rel_err_per_mode": err}
        res["cpu_baseline"] = {"value": o.last_scatter_count / dt_o, "unit": "markers/s", "kind": "oracle", "cores": o.max_threads(),
                               "sample": f"every {stride}-th marker ({m['R'][sl].size}), oracle.scatter (one toroidal mode per thread)"}
    ctx.close()
    del d, out
    torch.cuda.empty_cache()
    return res


def flops_per_rhs_em(n_modes: int) -> int:
    """One electromagnetic right-hand side (row f2, the thesis's K1): locator 25, three gathers of 170 per mode + 6, and
    ~330 for equilibrium, b*, the equations and the weight rate (the electrostatic 155 + the dA^s / dA^h terms)."""
    return 25 + 3 * (170 * n_modes + 6) + 330


def em_run(wl, reps, fp64_peak, hbm_peak, with_oracle=True):
    """trimeg_rhs_em (K1) and trimeg_pullback (K2) on the workload's marker batch, as drawn and cell-sorted; the three fields
    are seeded like the workload's own (amplitudes 1e-3, 1e-3, 3e-4)."""
    import torch
    from paper_2601_14301_b200 import binding, inputs
    ctx = binding.context_for(wl, inputs)
    dofs = [inputs.field_dofs(wl, seed=wl.seed + 100 * a, sigma=sg) for a, sg in enumerate((1e-3, 1e-3, 3e-4))]
    ctx.field_upload(wl.modes, torch.from_numpy(dofs[0]).cuda(), kind=0)
    ctx.field_upload_aux(binding.FIELD_AS, torch.from_numpy(dofs[1]).cuda(), kind=0)
    ctx.field_upload_aux(binding.FIELD_AH, torch.from_numpy(dofs[2]).cuda(), kind=0)
    n = wl.n_markers
    m = inputs.markers(wl, n=n)
    d = binding.markers_to_device(m, "cuda")
    ctx.locate(d["R"], d["Z"], cell=d["cell"])
    n_in = int((d["cell"] >= 0).sum())
    fl = flops_per_rhs_em(len(wl.modes))
    rows = []
    for order in ("as drawn", "cell-sorted"):
        if order == "cell-sorted":
            ctx.sort(d)
        for op in ("rhs_em", "pullback"):
            ts = []
            u0, w0 = d["vpar"].clone(), d["w"].clone()
            for rep in range(3 + reps):
                if op == "pullback":
                    d["vpar"].copy_(u0); d["w"].copy_(w0)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                out = ctx.rhs_em(d) if op == "rhs_em" else ctx.pullback(d)
                e1.record()
                torch.cuda.synchronize()
                if rep >= 3:
                    ts.append(e0.elapsed_time(e1) * 1e-3)
            d["vpar"].copy_(u0); d["w"].copy_(w0)
            t = sorted(ts)[len(ts) // 2]
            row = {"op": op, "order": order, "value": n_in / t, "unit": "markers/s", "ms_per_call": t * 1e3}
            if op == "rhs_em":
                row.update({"achieved_tflops": fl * n_in / t * 1e-12, "frac": fl * n_in / t * 1e-12 / fp64_peak})
            else:
                row.update({"algorithmic_GBps": 60.0 * n_in / t * 1e-9, "frac_hbm": 60.0 * n_in / t * 1e-9 / hbm_peak})
            rows.append(row)
    best = [r for r in rows if r["op"] == "rhs_em" and r["order"] == "cell-sorted"][0]
    res = {"metric": "marker right-hand sides per second, electromagnetic model (trimeg_rhs_em, the thesis's K1); pullbacks per second (K2)",
           "value": best["value"], "unit": "marker-RHS/s", "markers": n, "markers_inside": n_in, "rows": rows,
           "roofline": {"bound": "alu", "kernel": "rhs_em_kernel", "achieved": best["achieved_tflops"], "peak": fp64_peak, "unit": "TFLOP/s",
                        "frac": best["frac"], "algorithmic_flops_per_marker": fl, "algorithmic_bytes_per_marker": 92},
           "paper_context": "thesis K1, 32e6 electrons on 1 H100: 0.21 s = 1.5e8 marker-RHS/s; K2 + density + g2p2g 0.10-0.13 s "
                            "(PAPER.md:911-917; EQDSK equilibrium, cubic splines in phi: other hardware, not like-for-like)",
           "config": workload_config(wl)}
    if with_oracle:
        import oracle
        o = oracle.from_workload(wl, inputs)
        coefs = [o.bell_from_dofs(wl.modes, x) for x in dofs]
        o.set_coeffs(wl.modes, coefs[0]); o.set_aux_coeffs(0, coefs[1]); o.set_aux_coeffs(1, coefs[2])
        stride = max(1, n // (1 << 17))
        ms = {k: np.ascontiguousarray(v[::stride]) for k, v in m.items()}
        t0 = time.perf_counter()
        want = o.rhs_em(ms["R"], ms["Z"], ms["phi"], ms["vpar"], ms["mu"], ms["w"])
        dt_o = time.perf_counter() - t0
        ds = binding.markers_to_device(ms, "cuda")
        got = ctx.rhs_em(ds)
        err = max(float(np.abs(got[k].cpu().numpy() - want[k]).max() / np.abs(want[k]).max()) for k in ("dRdt", "dZdt", "dphidt", "dudt", "dwdt"))
        assert err < 1e-10, f"rhs_em parity check failed: {err}"      # library Bell expansion vs the oracle's: 1e-11 per coefficient
        res["oracle_check"] = {"sample_markers": int(ms["R"].size), "max_rel_err": err}
        res["cpu_baseline"] = {"value": ms["R"].size / dt_o, "unit": "marker-RHS/s", "kind": "oracle", "cores": o.max_threads(),
                               "sample": f"every {stride}-th marker ({ms['R'].size}), oracle.rhs_em with OpenMP over markers"}
    ctx.close()
    del d
    torch.cuda.empty_cache()
    return res


def run_em(args, wl):
    import torch
    from paper_2601_14301_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(0)
    binding.load()
    ctx = binding.context_for(wl, inputs)
    fp64_peak = ctx.measure_fp64_peak()
    ctx.close()
    hbm_peak, _ = load_peaks()
    res = em_run(wl, max(3, args.steps), fp64_peak, hbm_peak)
    res.update({"n_gpus": 1, "dtype": "f64", "data": "synthetic", "higher_is_better": True})
    print(json.dumps(res), flush=True)
    return 0


def run_scatter(args, wl):
    import torch
    from paper_2601_14301_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(0)
    binding.load()
    ctx = binding.context_for(wl, inputs)
    fp64_peak = ctx.measure_fp64_peak()
    ctx.close()
    hbm_peak, _ = load_peaks()
    res = scatter_run(wl, max(3, args.steps), fp64_peak, hbm_peak)
    res.update({"n_gpus": 1, "dtype": "f64", "data": "synthetic", "higher_is_better": True})
    print(json.dumps(res), flush=True)
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
    rows = gather_rows(ctx, wl, range(args.min_log2, args.max_log2 + 1, 2), args.steps, hbm_peak, fp64_peak)
    line = {"metric": "field gathers/sec (dphi, d/dR, d/dZ; 3 toroidal modes)", "unit": "gathers/s", "n_gpus": 1,
            "config": workload_config(wl), "dtype": "f64", "data": "synthetic", "hbm_peak_gbs": hbm_peak, "fp64_peak_tflops": fp64_peak,
            "algorithmic_bytes_per_gather": 52, "algorithmic_flops_per_gather": flops_per_gather(len(wl.modes)), "rows": rows}
    print(json.dumps(line), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=4)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--op", default="push", choices=["push", "scatter", "em"],
                    help="scatter: time trimeg_scatter (row f1); em: trimeg_rhs_em and trimeg_pullback (row f2) on the workload's markers")
    ap.add_argument("--workload", default="cfg5", choices=["cfg1", "cfg2", "cfg3", "cfg4", "cfg5"])
    ap.add_argument("--markers", type=int, default=0, help="override markers per GPU (testing)")
    ap.add_argument("--n-modes", type=int, default=0, help="override the toroidal mode list by n = 0, 2, ..., 2 (K - 1) (schedule selection sweeps)")
    ap.add_argument("--n-phi", type=int, default=0, help="row f3: the field on N cubic B-spline toroidal planes instead of the harmonic mode list")
    ap.add_argument("--eom-variant", type=int, default=0, choices=[0, 1, 2], help="trimeg_params.eom_variant (2: the reduced equations A.19-A.29, row f4)")
    ap.add_argument("--unstructured", nargs="?", const="hilbert", default=None, choices=["hilbert", "shuffled"],
                    help="row f4: the workload's cross-section as an unstructured triangulation (jittered Delaunay, shuffled numbering) with "
                         "the box-grid locator; 'hilbert' (default): triangles renumbered by trimeg_mesh_locality_order first, 'shuffled': as generated")
    ap.add_argument("--eq-table", type=int, default=0, help="row f4: equilibrium from N x N cubic-B-spline tables (the configs' flux function elongated by 1.2, F' != 0) instead of the analytic one")
    ap.add_argument("--sort-every", type=int, default=10, help="RK4 steps fused per sort + push call")
    ap.add_argument("--push-kernel", type=int, default=-1, help="trimeg_set_push_kernel variant (-1 = library default)")
    ap.add_argument("--min-log2", type=int, default=16, help="cfg4 gather sweep: smallest marker count 2^k")
    ap.add_argument("--max-log2", type=int, default=28, help="cfg4 gather sweep: largest marker count 2^k")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the short device-timed runs of cfg2, cfg3, cfg4 (config_sweep)")
    ap.add_argument("--no-check", action="store_true", help="skip the oracle check of a strided sample after the timed steps")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 0)
    from paper_2601_14301_b200 import inputs
    import dataclasses
    wl = inputs.WORKLOADS[args.workload]
    if args.markers:
        wl = dataclasses.replace(wl, n_markers=args.markers)
    if args.n_modes:
        wl = dataclasses.replace(wl, modes=tuple(range(0, 2 * args.n_modes, 2)))
    if args.workload == "cfg4":
        return run_gather_sweep(args, wl)
    if args.impl == "reference":
        return run_reference(args, wl)
    if args.op == "scatter":
        return run_scatter(args, wl)
    if args.op == "em":
        return run_em(args, wl)
    return run_gpu(args, wl)


if __name__ == "__main__":
    sys.exit(main())
