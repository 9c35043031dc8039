#!/usr/bin/env python
"""bench.py -- ADI step throughput of the wave2d hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3|cfg2|cfg4_f64|cfg4_f32|cfg5|cfg1]
                    [--impl ours|reference] [--no-cpu-baseline]

A "step" is one ADI time step of the whole hot path (fused RHS + x-sweep solve,
fused RHS + y-sweep solve, level rotation) over the whole grid of the workload.  The default workload is
config 3 of BASELINE.json (fp64 4096^2, the one the north_star's roofline target is quoted on); it fits
one GPU (0.4 GB).  Its three fields (403 MB) exceed the 126 MB L2, and every sweep streams 2 fields in
and 1 out, so successive timed steps cannot reuse L2 contents ("inputs larger than L2").

Prints ONE JSON line (rank 0).  Keys follow the graft bench contract; `roofline` is the dominant kernel
(the slower of the two sweep kernels) timed live with CUDA events on the launching stream through
wave2d_profile_sweeps; `cpu_baseline` is the oracle as it stands on the host cores on a bounded sample;
`e2e` is the same metric through the public API with HOST buffers (H2D of phi and D2H of u inside the
timed region, every iteration).

Multi-GPU: the path does not shard without an exchange: "replicas only".  Under torchrun
every rank runs an independent replica of the workload on its own GPU; value = total point-updates of all
ranks / max-over-ranks device time; no data-path collective.

--impl reference: the reference arm of this tier is the CPU oracle (oracle/), timed as it stands on the
host cores on a bounded sample of the same workload (rank 0 only).
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

METRIC = "ADI step throughput (Gpoint-updates/s) fp64; achieved HBM GB/s vs peak"
UNIT = "Gpoint-updates/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=960)
    ap.add_argument("--warmup", type=int, default=24)
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--scheme", type=int, default=0, choices=[0, 1],
                    help="0: the paper's split scheme (2.11)-(2.12) (default, the north_star path); "
                         "1: factorised unsplit scheme (2.8), 5 field passes per step (SURVEY.md 8f NEXT-2)")
    ap.add_argument("--tau-factor", type=float, default=1.0,
                    help="off-config: multiply the workload's tau (16: alpha = 128, the exact whole-line solvers run)")
    ap.add_argument("--speed-field", action="store_true",
                    help="off-config (SURVEY.md 8f NEXT-4): c(t) cs(x,y) with a smooth seeded positive field cs; the "
                         "variable-coefficient solvers run, 4 field passes per sweep")
    ap.add_argument("--dense-source", action="store_true",
                    help="off-config: replace the workload's source shape by one that is non-zero on the whole grid "
                         "(wave2d_set_source with a full grid: + 1 field read per sweep)")
    ap.add_argument("--sharded", action="store_true",
                    help="off-default (SURVEY.md 8f NEXT-3): ONE simulation over the N ranks -- every rank owns a row block "
                         "with halo rows refreshed from its neighbours after every step (paper_2006_10142_b200/sharded.py); "
                         "strong scaling.  The default for N > 1 stays N independent replicas (north_star: no sharding)")
    ap.add_argument("--solver", type=int, default=0, choices=[0, 1, 2, 3],
                    help="off-default: wave2d_set_option('solver'): 0 auto, 1 exact whole-line, 2 streamed, 3 small-grid cluster")
    ap.add_argument("--opt", action="append", default=[], metavar="NAME=VALUE",
                    help="off-default: any wave2d_set_option tuning option (repeatable), e.g. --opt tail_min=2")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps per end-to-end iteration (default: --steps)")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md clocks line)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.ok = index, [], None, True

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100", "-i",
                 str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.t = threading.Thread(target=self._read, daemon=True)
        self.t.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self, t0=None, t1=None):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.t.join(timeout=2)
        sm, mx, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def load_workload(name: str, steps_needed: int):
    from paper_2006_10142_b200 import workloads as W
    w = W.by_name(name)
    if steps_needed > w.M:   # more timed steps than the config's M: extend the time axis with the same recipe
        w = W.by_name(name, M=steps_needed)
    return w


class NvmlSampler:
    """SM clock + throttle reasons sampled every 5 ms through NVML while the timed region runs."""

    def __init__(self, torch_index: int):
        self.rows, self.stop_flag, self.ok = [], False, False
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            uuid = str(torch.cuda.get_device_properties(torch_index).uuid)
            if not uuid.startswith("GPU-"):
                uuid = "GPU-" + uuid
            try:
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(torch_index)
            self.nv = pynvml
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:   # noqa: BLE001
            self.err = repr(e)

    def start(self):
        if not self.ok:
            return
        self.t = threading.Thread(target=self._loop, daemon=True)
        self.t.start()

    def _loop(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                rs = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
                self.rows.append((time.perf_counter(), float(mhz), int(rs), pw))
            except Exception:
                pass
            time.sleep(0.005)

    def stop(self, t0=None, t1=None):
        if not self.ok:
            return None
        self.stop_flag = True
        self.t.join(timeout=2)
        nv = self.nv
        rows = [r for r in self.rows if (t0 is None or r[0] >= t0) and (t1 is None or r[0] <= t1)] or self.rows
        bits = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
                "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
                "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
                "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        reasons = sorted(n for n, b in bits.items() if any(r[2] & b for r in rows))
        return {"sm_mhz": float(np.median([r[1] for r in rows])) if rows else None, "sm_max_mhz": self.max_mhz,
                "power_w_max": max((r[3] for r in rows), default=None), "samples": len(rows), "reasons": reasons}


def field_bytes(w):
    return w.points * (8 if w.dtype == "f64" else 4)


def time_oracle(w, budget_s: float, min_steps: int = 2):
    """The oracle as it stands on the host cores: first `steps` time steps of workload w (full grid)."""
    from oracle import oracle
    o = oracle.Wave2DOracle(w.N1, w.N2, w.l, w.tau, w.M)
    try:
        o.set_speed(w.c_half)
        if w.s is not None:
            o.set_source(w.s, w.g_half)
        o.set_initial(w.phi, w.psi)
        t0 = time.perf_counter()
        o.run(1)
        t1 = time.perf_counter() - t0
        steps = int(max(min_steps, min(w.M - 1, budget_s / max(t1, 1e-6))))
        t0 = time.perf_counter()
        o.run(steps)
        dt = time.perf_counter() - t0
    finally:
        o.close()
    return {"value": w.points * steps / dt / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": f"{steps} time steps of {w.name} on the full {w.n1}x{w.n2} grid after 1 untimed step "
                      f"({dt:.1f} s, oracle/wave2d_oracle.c: Thomas per line, OpenMP over lines, fp64)",
            "seconds": dt, "steps": steps}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


def run_reference(args):
    """Reference arm of this tier: the CPU oracle, K timed steps after W warm-up steps, rank 0 only."""
    rank, world, _ = dist_env()
    if rank != 0:
        return
    from oracle import oracle
    oracle.build()
    K, Wm = args.steps, args.warmup
    w = load_workload(args.workload, K + Wm + 1)
    # bounded sample: one calibration step on the full grid; if W+K full-grid steps would take more than
    # ~150 s, the sample is the same recipe on a grid with fewer rows (N2 reduced), stated in `sample`.
    o = oracle.Wave2DOracle(w.N1, w.N2, w.l, w.tau, w.M)
    o.set_speed(w.c_half)
    if w.s is not None:
        o.set_source(w.s, w.g_half)
    o.set_initial(w.phi, w.psi)
    t0 = time.perf_counter(); o.run(1); t1 = time.perf_counter() - t0
    o.close()
    N2 = w.N2
    est = t1 * (K + Wm)
    if est > 150.0:
        N2 = max(64, int(w.N2 * 150.0 / est) // 64 * 64)
    rows = N2 - 1
    phi = np.ascontiguousarray(w.phi[:rows])
    s = None if w.s is None else np.ascontiguousarray(w.s[:rows])
    o = oracle.Wave2DOracle(w.N1, N2, w.l * 1.0, w.tau, w.M)
    # keep h2 = l/N2 of the full workload: the strip is [0,l] x [0, l*N2/N2_full]; the oracle takes one l,
    # so the strip uses its own h2 -- only the arithmetic cost per point matters for this timing.
    o.set_speed(w.c_half)
    if s is not None:
        o.set_source(s, w.g_half)
    o.set_initial(phi, None)
    o.run(Wm)
    t0 = time.perf_counter()
    o.run(K)
    dt = time.perf_counter() - t0
    o.close()
    pts = (w.N1 - 1) * rows
    value = pts * K / dt / 1e9
    sample = (f"{K} timed steps (after {Wm}) of {w.name} on " +
              (f"the full {w.n1}x{w.n2} grid" if N2 == w.N2 else
               f"a {w.n1}x{rows} strip of its {w.n1}x{w.n2} grid (full grid would take ~{est:.0f} s)"))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
            "warmup": Wm, "ms_per_step": dt / K * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N1": w.N1, "N2": w.N2, "tau": w.tau, "sample_points": pts},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def traced_sweeps(make_handle, budget_steps, samples=5):
    """Median over `samples` graph replays of 2 steps of: the span of the last x sweep and of the last y sweep (first CTA
    start -> last CTA end, ns, from wave2d_get_trace) and of the gap between the two (y's first start - x's last end;
    negative = the sweeps overlap by programmatic launch / early start).  None where the solver family records no trace."""
    per = max(1, min(2, budget_steps // samples))
    try:
        h = make_handle(trace=1)
    except Exception:
        return None
    try:
        h.run(0)
        h.run(per)                                   # warm
        xs, ys, gaps = [], [], []
        for _ in range(samples):
            h.run(per)
            tx, ty = h.trace(0), h.trace(1)          # synchronises the stream
            x0, x1 = int(tx[:, 0].min()), int(tx[:, 1].max())
            y0, y1 = int(ty[:, 0].min()), int(ty[:, 1].max())
            xs.append(x1 - x0)
            ys.append(y1 - y0)
            gaps.append(y0 - x1)
        return {"ns_x": float(np.median(xs)), "ns_y": float(np.median(ys)), "ns_gap_x_to_y": float(np.median(gaps)),
                "samples": samples, "ctas_x": int(tx.shape[0]), "ctas_y": int(ty.shape[0])}
    except Exception:
        return None
    finally:
        h.close()


def run_ours(args):
    import torch
    from paper_2006_10142_b200.replicas import Ranks

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path is CUDA only, there is no CPU fallback")
    torch.cuda.set_device(local)
    from paper_2006_10142_b200 import build as _build
    if local == 0:
        _build.build()                      # no-op when libwave2d.so is up to date
    else:
        for _ in range(600):                # other ranks wait for rank 0's build (atomic rename)
            if not _build.needs_build():
                break
            time.sleep(0.5)
    ranks = Ranks("nccl", torch.device("cuda", local))

    def barrier():
        ranks.barrier()
        torch.cuda.synchronize()

    max_over_ranks = ranks.max_over_ranks

    from paper_2006_10142_b200 import binding as B
    K, Wm = args.steps, args.warmup
    PROF = 12                                             # per-kernel timing pass (plain launches + events)
    w = load_workload(args.workload, Wm + K + PROF + 2)
    if args.tau_factor != 1.0:
        w.tau *= args.tau_factor
        w.name += f" with tau x {args.tau_factor:g} (off-config)"
    sch = args.scheme
    npdt = np.float64 if w.dtype == "f64" else np.float32
    esz = 8 if w.dtype == "f64" else 4
    fbytes = field_bytes(w)

    # pinned host buffers (the e2e leg copies from / to these every iteration)
    phi_pin = torch.empty((w.n2, w.n1), dtype=torch.float64 if esz == 8 else torch.float32).pin_memory()
    phi_pin.numpy()[...] = w.phi.astype(npdt, copy=False)
    out_pin = torch.empty_like(phi_pin).pin_memory()

    stream = torch.cuda.Stream()
    cs = None
    if args.speed_field:
        yy = np.linspace(0.0, 1.0, w.n2)[:, None]
        xx = np.linspace(0.0, 1.0, w.n1)[None, :]
        cs = 1.0 + 0.4 * np.sin(2 * np.pi * xx) * np.cos(np.pi * yy) + 0.3 * xx - 0.2 * yy
        w.name += " with speed field cs(x,y) (off-config)"
    if args.dense_source:
        yy = np.linspace(0.0, 1.0, w.n2)[:, None]
        xx = np.linspace(0.0, 1.0, w.n1)[None, :]
        w.s = 1.0 + 0.5 * np.sin(3 * np.pi * xx) * np.cos(2 * np.pi * yy)      # non-zero everywhere
        if w.g_half is None:
            w.g_half = np.cos(np.arange(2 * w.M) * 0.01)
        w.name += " with a dense source s(x,y) (off-config)"

    def make_handle(**extra):
        h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
        h.set_stream(stream)
        if sch:
            h.set_option("scheme", sch)      # factorised (2.8): set_initial stands at level 1, every run step is a solve
        if args.solver:
            h.set_option("solver", args.solver)
        for kv in args.opt:
            name, _, val = kv.partition("=")
            h.set_option(name, float(val))
        for name, val in extra.items():
            h.set_option(name, float(val))
        h.set_speed(w.c_half)
        if cs is not None:
            h.set_speed_field(cs.astype(npdt))
        if w.s is not None:
            h.set_source(w.s.astype(npdt, copy=False), w.g_half)
        h.set_initial(phi_pin)
        return h

    h = make_handle()

    sampler = NvmlSampler(local)
    if not sampler.ok:
        sampler = ClockSampler(local)   # nvidia-smi fallback (coarser: 100 ms)
    sampler.start()

    # ---- device-resident timing: W warm-up steps, then exactly K steps between two events on the stream
    h.run(0)                                # plan + graphs (captured, instantiated, uploaded) before anything is timed
    h.run(Wm)
    h.sync()
    l0 = h.info("launches")
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    tw0 = time.perf_counter()
    ev0.record(stream)
    h.run(K)
    ev1.record(stream)
    h.sync()
    barrier()
    tw1 = time.perf_counter()
    ms = max_over_ranks(float(ev0.elapsed_time(ev1)))
    launches = int(h.info("launches") - l0)
    graph_replays, plain_sweeps = int(h.info("graph_launches")), int(h.info("plain_sweeps"))
    clocks = sampler.stop(tw0, tw1) or {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable"]}

    # ---- per-kernel timing of the two sweep kernels, live, CUDA events on the same stream
    ms_x, ms_y = h.profile_sweeps(PROF)
    geom = {k: h.info(k) for k in ("solver_x", "solver_y", "halo_x", "halo_y", "chunks_x", "chunks_y", "grid_x",
                                   "grid_y", "ctas_per_sm_x", "ctas_per_sm_y", "threads_x", "threads_y",
                                   "smem_x", "smem_y", "nbk_x", "nbk_y", "quota_x", "quota_y", "unit_x", "unit_y")}

    # ---- per-sweep spans measured INSIDE graph replays: a second handle with option "trace" records every CTA's start and
    # end (GPU global timer); a sweep's span = first CTA start -> last CTA end of its last launch in a replayed chunk.
    traced = traced_sweeps(make_handle, PROF)

    # ---- end to end through the public API with HOST buffers: H2D(phi) + K steps + D2H(u) per iteration
    Ke = args.e2e_steps or K
    e2e_iters = 3
    h.set_initial(phi_pin); h.run(min(Ke, 12)); h.get(out_pin)          # warm the path once
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_iters):
        h.set_initial(phi_pin)        # pinned host -> device (u^0 and u^{-1/2})
        h.run(Ke)
        h.get(out_pin)                # device -> pinned host, synchronises
    barrier()
    e2e_s = max_over_ranks((time.perf_counter() - t0) / e2e_iters)
    h.close()

    peak, peak_src = measured_peaks()
    pts = w.points
    value = world * pts * K / (ms * 1e-3) / 1e9
    dom = "x" if ms_x >= ms_y else "y"
    # algorithmic bytes per launch: read 2 fields, write 1; scheme 1's y sweep reads 1, writes 1
    bytes_x, bytes_y = 3 * fbytes, (2 if sch else 3) * fbytes
    if args.speed_field:                      # + the speed field in every sweep
        bytes_x, bytes_y = 4 * fbytes, 4 * fbytes
    if args.dense_source:                     # + the source shape in every sweep that adds f (scheme 1: the x sweep only)
        bytes_x += fbytes
        bytes_y += 0 if sch else fbytes
    sweep_bytes = bytes_x if dom == "x" else bytes_y
    passes = (8 if args.speed_field else 5 if sch else 6) + (0 if not args.dense_source else 1 if sch else 2)
    step_s = ms * 1e-3 / K
    # The timed region is K steps = K launches of each sweep kernel back to back (graph replay), timed by the two
    # events above.  The dominant kernel's average launch duration in that region is its share of the step (from
    # the per-launch events of wave2d_profile_sweeps, which add a launch gap per kernel) times the step time.
    share_dom = max(ms_x, ms_y) / (ms_x + ms_y)
    ms_dom = step_s * 1e3 * share_dom
    method = "share"
    if traced is not None:                    # measured span of the kernel inside a replayed graph
        ms_dom = traced["ns_" + dom] * 1e-6
        method = "trace"
    achieved = sweep_bytes / (ms_dom * 1e-3) / 1e9
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": w.dtype, "data": "synthetic",
        "config": {"workload": w.name, "N1": w.N1, "N2": w.N2, "unknowns": [w.n1, w.n2], "tau": w.tau, "M": w.M,
                   "scheme": ("split (2.11)-(2.12), 6 field passes per step" if not sch else
                              "factorised unsplit (2.8), 5 field passes per step (SURVEY.md 8f NEXT-2)"),
                   "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (no collective)",
                   "l2": (f"working set {3 * fbytes / 1e6:.0f} MB (3 fields) "
                          + ("> 126 MB L2: inputs larger than L2, no flush needed" if 3 * fbytes > 126e6 * 1.5
                             else "fits the 126 MB L2: L2-resident, HBM fraction not meaningful")),
                   "geometry": geom},
        "clocks": clocks,
        "gpu_launches": launches,
        "e2e": {"value": world * pts * Ke / e2e_s / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": fbytes / Ke, "d2h_bytes_per_step": fbytes / Ke,
                "steps_per_call": Ke, "seconds_per_call": e2e_s,
                "what": "wave2d_set_initial(pinned host phi) + wave2d_run(steps_per_call) + wave2d_get(pinned host u), "
                        "wall clock incl. both copies; bytes are per call / steps_per_call"},
        "roofline": {"bound": "hbm", "kernel": (f"wave2d_exact_{dom}<{w.dtype}>" if geom["solver_x"] == 1 else
                                                f"wave2d_sweep_panel<{w.dtype}, dir={dom}>" if geom["solver_x"] != 3 else
                                                f"wave2d_line_steps<{w.dtype}> (both half-steps of every step in one "
                                                "launch; each sweep is given half of it)"), "achieved": achieved,
                     "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                     "peak_source": peak_src, "bytes_per_launch": sweep_bytes,
                     "ms_per_launch": ms_dom, "share_of_step": share_dom, "method": method,
                     "how": "method 'trace' (default): the kernel's span inside a replayed graph, first CTA start -> last "
                            "CTA end by the GPU global timer (option trace, wave2d_get_trace), median of 5 replays of a "
                            "second handle with the same configuration; consecutive sweeps overlap by programmatic launch "
                            "and early start, so the spans of a step add up to more than the step time (see 'traced'). "
                            "method 'share' (fallback where a solver family records no trace; also in 'model_share'): step "
                            "time of the K-step timed region x the kernel's share from the per-launch events of "
                            "wave2d_profile_sweeps -- a model, not a measurement. 'isolated' = plain launches with an "
                            "event pair per kernel; ncu (serialised, cold) in profiles/. Every fraction is algorithmic "
                            "bytes / time / the copy rate in MEASURED_PEAKS.json, which is a copy kernel's rate, not a "
                            "hardware ceiling: values near or above 1 mean 'as fast as that copy', the DRAM traffic "
                            "measured by ncu is 0.93-1.00 x the algorithmic bytes (profiles/traffic.csv)",
                     "graph_replays_total": graph_replays, "sweeps_outside_graphs": plain_sweeps,
                     "isolated": {"what": "plain launches, one event pair per kernel (includes a launch gap)",
                                  "ms_x": ms_x, "ms_y": ms_y,
                                  "gbs_x": bytes_x / ms_x / 1e6, "gbs_y": bytes_y / ms_y / 1e6,
                                  "frac_x": bytes_x / ms_x / 1e6 / peak, "frac_y": bytes_y / ms_y / 1e6 / peak},
                     "model_share": {"what": "step time split by the isolated launches' shares (a model)",
                                     "frac_x": bytes_x / (step_s * 1e3 * ms_x / (ms_x + ms_y)) / 1e6 / peak,
                                     "frac_y": bytes_y / (step_s * 1e3 * ms_y / (ms_x + ms_y)) / 1e6 / peak},
                     "traced": None if traced is None else dict(
                         traced, what="span of one launch inside a replayed graph: first CTA start -> last CTA end",
                         overlap_note="ns_gap_x_to_y < 0: the y sweep's first CTA starts before the x sweep's last one ends"),
                     "frac_x": (bytes_x / traced["ns_x"] / peak if traced is not None else
                                bytes_x / (step_s * 1e3 * ms_x / (ms_x + ms_y)) / 1e6 / peak),
                     "frac_y": (bytes_y / traced["ns_y"] / peak if traced is not None else
                                bytes_y / (step_s * 1e3 * ms_y / (ms_x + ms_y)) / 1e6 / peak),
                     "step_passes": passes, "step_frac": passes * fbytes / step_s / 1e9 / peak,
                     "step_frac6": 6 * fbytes / step_s / 1e9 / peak, "step_frac5": 5 * fbytes / step_s / 1e9 / peak},
    }
    traffic_file = os.path.join(ROOT, "profiles", "traffic.csv")
    line["roofline"]["traffic_source"] = "profiles/traffic.csv: dram__bytes_read.sum + dram__bytes_write.sum of one " \
                                         "committed ncu --set full capture of this kernel (not measured by this run)"
    if os.path.exists(traffic_file):
        try:
            key = f"{w.name}:{dom}" + (":scheme1" if sch else "")
            for ln in open(traffic_file).read().splitlines()[1:]:
                k, v = ln.rsplit(",", 1)
                if k == key:
                    line["roofline"]["traffic"] = int(v)
        except Exception:
            pass
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            from oracle import oracle
            oracle.build()
            line["cpu_baseline"] = time_oracle(w, budget_s=15.0)
        print(json.dumps(line), flush=True)
    ranks.close()


def run_sharded(args):
    """One simulation sharded by grid rows over the ranks; a step = run(1) on every block + the halo refresh."""
    import torch
    from paper_2006_10142_b200.replicas import Ranks
    from paper_2006_10142_b200 import build as _build, sharded as S
    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the hot path is CUDA only, there is no CPU fallback")
    torch.cuda.set_device(local)
    if local == 0:
        _build.build()
    else:
        for _ in range(600):
            if not _build.needs_build():
                break
            time.sleep(0.5)
    dev = torch.device("cuda", local)
    ranks = Ranks("nccl", dev)
    K, Wm = args.steps, args.warmup
    w = load_workload(args.workload, Wm + K + 2)
    shards, G = S.make_shards(w.N1, w.N2, w.l, w.tau, w.M, w.dtype, world, w.phi, w.psi, w.c_half, w.s, w.g_half,
                              ranks=[rank])
    sh = shards[0]
    ex = S.DistExchange(sh, rank, world, dev) if world > 1 else None

    def steps(n):
        for _ in range(n):
            sh.step(1)
            if ex is not None:
                ex.refresh()

    sh.engine.run(0)
    steps(Wm)
    sh.engine.sync()
    ranks.barrier(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    steps(K)
    sh.engine.sync()
    ranks.barrier(); torch.cuda.synchronize()
    sec = ranks.max_over_ranks(time.perf_counter() - t0)   # (run(1) + get/set_rows synchronise the stream every step)
    # end to end: this rank's block of phi from pinned host memory, K sharded steps, its owned rows back to pinned host memory
    blk = sh.block
    tdt = torch.float64 if w.dtype == "f64" else torch.float32
    phi_pin = torch.from_numpy(np.ascontiguousarray(blk.local(w.phi))).to(tdt).pin_memory()
    out_pin = torch.empty((blk.b - blk.a, w.n1), dtype=tdt).pin_memory()

    def e2e_once():
        sh.engine.set_initial(phi_pin)
        steps(K)
        sh.engine.get_rows(0, blk.top, blk.b - blk.a, out_pin)      # synchronises

    e2e_once()
    ranks.barrier(); torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(3):
        e2e_once()
    ranks.barrier(); torch.cuda.synchronize()
    e2e_sec = ranks.max_over_ranks((time.perf_counter() - t0) / 3)
    peak, peak_src = measured_peaks()
    esz = 8 if w.dtype == "f64" else 4
    line = {"metric": METRIC, "value": w.points * K / sec / 1e9, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": sec / K * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": w.dtype, "data": "synthetic",
            "config": {"workload": w.name + " sharded by grid rows (off-default, SURVEY.md 8f NEXT-3)", "N1": w.N1, "N2": w.N2,
                       "parallelism": f"{world} row blocks, {G} halo rows refreshed per step and cut (NCCL point-to-point)",
                       "rows_owned": sh.block.b - sh.block.a, "rows_local": sh.block.rows},
            "gpu_launches": int(sh.engine.info("launches")),
            "roofline": {"bound": "hbm", "achieved": 6 * w.points * esz * K / sec / 1e9, "peak": peak * world, "unit": "GB/s",
                         "frac": 6 * w.points * esz * K / sec / 1e9 / (peak * world), "traffic": None, "peak_source": peak_src,
                         "how": "6 field passes of the whole grid / wall time of K steps incl. the halo exchange, against "
                                "N x the measured single-GPU peak"},
            "e2e": {"value": w.points * K / e2e_sec / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": phi_pin.numel() * phi_pin.element_size() / K,
                    "d2h_bytes_per_step": out_pin.numel() * out_pin.element_size() / K, "steps_per_call": K,
                    "what": "per rank: wave2d_set_initial(pinned host block of phi) + K sharded steps (halo refresh included) "
                            "+ wave2d_get_rows(owned rows -> pinned host); wall clock, max over ranks; bytes are this "
                            "rank's per call / K"}}
    line["roofline"]["per_gpu"] = {"achieved": line["roofline"]["achieved"] / world, "peak": peak,
                                   "frac": line["roofline"]["achieved"] / world / peak}
    if rank == 0:
        print(json.dumps(line), flush=True)
    sh.engine.close()
    ranks.close()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.sharded:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
