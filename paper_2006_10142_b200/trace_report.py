"""Per-CTA trace of the two sweep kernels (option "trace", wave2d_get_trace): when every CTA started and ended,
on which SM, and how many pieces of work it ran.

    python -m paper_2006_10142_b200.trace_report [--workload cfg3|cfg2|cfg4_f64|cfg4_f32|cfg5] [--scheme 0|1]

The sweeps are launched one by one here (wave2d_profile_sweeps), so consecutive kernels overlap less than in the
graph replay that bench.py times.  Needs a B200; prints plain text.
"""
from __future__ import annotations

import argparse

import numpy as np

from . import binding as B
from . import workloads as W


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="cfg3")
    ap.add_argument("--scheme", type=int, default=0)
    args = ap.parse_args()
    M = 40
    make = {"cfg3": lambda: W.cfg3(M=M), "cfg2": lambda: W.cfg2(M=M), "cfg4_f64": lambda: W.cfg4(M=M),
            "cfg4_f32": lambda: W.cfg4(M=M, dtype="f32"), "cfg5": lambda: W.cfg5(M=M)}
    w = make[args.workload]()
    npdt = np.float64 if w.dtype == "f64" else np.float32
    h = B.Wave2D(w.N1, w.N2, w.l, w.tau, w.M, w.dtype)
    try:
        h.set_option("trace", 1)
        if args.scheme:
            h.set_option("scheme", args.scheme)
        h.set_speed(w.c_half)
        if w.s is not None:
            h.set_source(w.s.astype(npdt), w.g_half)
        h.set_initial(w.phi.astype(npdt))
        h.run(12)
        h.sync()
        ms_x, ms_y = h.profile_sweeps(6)
        print(f"{args.workload} scheme {args.scheme}: {w.n1} x {w.n2} {w.dtype}; isolated launches "
              f"{1e3 * ms_x:.1f} us (x), {1e3 * ms_y:.1f} us (y)")
        for d, name in ((0, "x sweep"), (1, "y sweep")):
            t = h.trace(d).astype(np.int64)
            t0 = t[:, 0].min()
            dur = (t[:, 1] - t[:, 0]) / 1e3
            end = (t[:, 1] - t0) / 1e3
            print(f"{name}: {len(t)} CTAs on {len(np.unique(t[:, 2]))} SMs, {int(h.info('chunks_x' if d == 0 else 'chunks_y'))} "
                  f"pieces; kernel span {end.max():.1f} us; CTA start spread {(t[:, 0].max() - t0) / 1e3:.1f} us; "
                  f"CTA busy min / median / mean / max {dur.min():.1f} / {np.median(dur):.1f} / {dur.mean():.1f} / "
                  f"{dur.max():.1f} us; CTA end min / mean / max {end.min():.1f} / {end.mean():.1f} / {end.max():.1f} us; "
                  f"pieces per CTA min / max {t[:, 3].min()} / {t[:, 3].max()}")
    finally:
        h.close()


if __name__ == "__main__":
    main()
