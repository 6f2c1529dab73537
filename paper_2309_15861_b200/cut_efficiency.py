"""Efficiency of the angular particle cut on the synthetic showers -- the stand-in for the paper's Fig. 2
("Efficiency of an angular particle cut for the reduction of atmospheric photons").

    python -m paper_2309_15861_b200.cut_efficiency --workload c2 [--segments N] [--angles 1 2 3 ...]

For every cut angle and both forms of the cut (angle to the experiment centre; smallest angle to a telescope) one
tally-mode pass through the CUDA path gives the fraction of bunches that were not handled (the paper's "reduce the number
of handled particles by up to 90 %") and the fraction of the detected light that the cut loses (its "visible photon
loss"), next to the uncut pass and to the exact culling (C8OPT_FLAG_CULL), which loses nothing by construction.
Prints a markdown table.  Needs a B200: every number comes from the kernels (argument marshalling only here).
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
    ap.add_argument("--workload", default="c2", choices=["c1", "c2", "c4", "c5"])
    ap.add_argument("--segments", type=int, default=None)
    ap.add_argument("--angles", type=float, nargs="*", default=[1, 2, 3, 4, 5, 6, 7, 8, 9, 10])
    ap.add_argument("--repeat", type=int, default=5)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("cut_efficiency needs a CUDA device: the photon path has no CPU fallback")
    c8.build()
    cfg = wl.make_config(args.workload, n_segments=args.segments)
    seg = cfg["segments"]
    n = len(seg)
    dev = torch.device("cuda:0")
    d_seg = torch.from_numpy(seg.view(np.uint8).reshape(n, 48).copy()).to(dev)
    ctx = c8.Context(cfg["atmosphere"])
    ctx.add_telescopes(cfg["telescopes"])
    stream = torch.cuda.current_stream()

    def run(flags, angle_deg=0.0):
        par = dict(cfg["params"], mode=c8.MODE_TALLY, flags=flags, cut_angle=float(np.radians(angle_deg)))
        best = None
        for _ in range(args.repeat):
            ctx.reset_tallies()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            ctx.propagate_segments(d_seg, par, n=n)
            b.record(stream)
            tallies, cnt, _ = ctx.read_tallies()
            ms = a.elapsed_time(b)
            best = ms if best is None else min(best, ms)
        return cnt, float(tallies["sum_w"].sum()), best

    base, w_base, ms_base = run(0)
    cull, w_cull, ms_cull = run(c8.FLAG_CULL)
    # the Cherenkov share of the hits is what the cut can lose; the fluorescence hits (c4) are never cut
    print(f"workload {cfg['name']}: {n} segments, {len(cfg['telescopes'])} telescopes, {base['generated']} bunches, "
          f"{base['hits']} hits, sum of weights {w_base:.6g}; uncut pass {ms_base:.3f} ms\n")
    print("| cut | angle [deg] | bunches not handled | hits lost | detected light lost (sum w) | kernel [ms] | speed-up |")
    print("|---|---|---|---|---|---|---|")
    print(f"| none | - | 0 | 0 | 0 | {ms_base:.3f} | 1.00 |")
    print(f"| exact culling (C8OPT_FLAG_CULL) | - | {cull['culled'] / base['generated']:.4f} | "
          f"{1 - cull['hits'] / base['hits']:.5f} | {1 - w_cull / w_base:.5f} | {ms_cull:.3f} | {ms_base / ms_cull:.2f} |")
    for name, flag in (("experiment centre", c8.FLAG_CUT_CENTRE), ("nearest telescope", c8.FLAG_CUT_TELESCOPES)):
        for ang in args.angles:
            cnt, w, ms = run(flag, ang)
            print(f"| {name} | {ang:g} | {cnt['culled'] / base['generated']:.4f} | {1 - cnt['hits'] / base['hits']:.5f} | "
                  f"{1 - w / w_base:.5f} | {ms:.3f} | {ms_base / ms:.2f} |")
    ctx.close()


if __name__ == "__main__":
    main()
