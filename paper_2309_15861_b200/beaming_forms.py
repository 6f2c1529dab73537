"""Fluorescence beaming: the weight form against the count form, for variance and speed (section 1.1.1;
SURVEY.md section 8(f)-4; R14 / R28).

    python -m paper_2309_15861_b200.beaming_forms [--segments N] [--seeds K]

Three ways to bring the isotropic fluorescence light of the same segments onto one telescope 10 km away:
  isotropic    every bunch drawn, direction uniform on the sphere (weight 1)
  weight form  R14: every bunch drawn, direction uniform in a fixed 2-degree cone about the line of sight, weight Omega / 4 pi
  count form   R28 (the paper's own): per-segment cone that just holds the telescope, the NUMBER of bunches scaled by
               Omega / 4 pi, weight ~1
All three have the same expected detected light sum(w).  For K seeds the tool prints bunches drawn, hits, the mean of
sum(w) with its relative scatter over the seeds (the Monte-Carlo error of the detected light), the kernel time, and the
figure of merit 1 / (relative variance x time).  Needs a B200: every number comes from the kernels.
"""
from __future__ import annotations

import argparse
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import torch

    import paper_2309_15861_b200 as c8
    import workloads as wl

    ap = argparse.ArgumentParser()
    ap.add_argument("--segments", type=int, default=1_000_000)
    ap.add_argument("--seeds", type=int, default=12)
    ap.add_argument("--yield-scale", type=float, default=250.0,
                    help="fluorescence yield multiplier (configs[2]'s 4 / MeV gives ~1 expected isotropic hit per 10^6 segments)")
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("beaming_forms needs a CUDA device: the photon path has no CPU fallback")
    c8.build()
    cfg = wl.make_config("c3a", n_segments=args.segments)
    seg = cfg["segments"]
    n = len(seg)
    dev = torch.device("cuda:0")
    d_seg = torch.from_numpy(seg.view(np.uint8).reshape(n, 48).copy()).to(dev)
    ctx = c8.Context(cfg["atmosphere"])
    ctx.add_telescopes(cfg["telescopes"])
    stream = torch.cuda.current_stream()
    base = dict(cfg["params"], mode=c8.MODE_TALLY, fl_yield=cfg["params"]["fl_yield"] * args.yield_scale)
    forms = [("isotropic", dict(fl_beam_telescope=-1)),
             ("weight form, 2 deg cone (R14)", dict(fl_beam_telescope=0, fl_beam_halfangle=float(np.radians(2.0)))),
             ("count form, per-segment cone (R28)", dict(fl_beam_telescope=c8.BEAM_ARRAY))]
    print(f"{n} fluorescence segments of configs[2] (yield x {args.yield_scale:g}), telescope of 6 m at 10 km, {args.seeds} seeds\n")
    print("| form | bunches drawn | hits / run | sum w / run | relative scatter of sum w | kernel [ms] | 1 / (variance x time), isotropic = 1 |")
    print("|---|---|---|---|---|---|---|")
    ref = None
    for name, over in forms:
        sw, hits, gen, ms = [], [], 0, []
        for sd in range(args.seeds):
            par = dict(base, seed=1000 + sd, **over)
            ctx.reset_tallies()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctx.propagate_segments(d_seg, par, n=n)
            b.record(stream)
            t, cnt, _ = ctx.read_tallies()
            sw.append(float(t["sum_w"].sum())); hits.append(int(t["hits"].sum())); gen = cnt["generated"]; ms.append(a.elapsed_time(b))
        sw = np.array(sw)
        rel = float(sw.std(ddof=1) / sw.mean()) if sw.mean() > 0 else float("nan")
        t_ms = float(np.min(ms))
        fom = 1.0 / (rel * rel * t_ms) if rel > 0 else float("inf")
        if ref is None:
            ref = fom
        print(f"| {name} | {gen} | {np.mean(hits):.1f} | {sw.mean():.4g} | {rel:.3f} | {t_ms:.3f} | {fom / ref:.3g} |")
    ctx.close()


if __name__ == "__main__":
    main()
