#!/usr/bin/env python
"""bench.py -- photons generated + propagated per second (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c2] [--impl ours|reference]

A "step" is one pass of the whole hot path (preamble, Philox draw, generation, propagation, sphere
test, tally / record output: every row of SURVEY.md §8(a)) over one batch of synthetic segments.
The default workload is BASELINE.json configs[1] ("c2": 10^6 shower-shaped segments, 5-layer
atmosphere, 4 telescopes, tally mode), the configuration north_star quotes the target on.
Prints ONE JSON line (rank 0).  See DESIGN.md §7 for how each field is measured.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads as wl  # noqa: E402

METRIC = "photons generated+propagated per second"
UNIT = "photons/s"
RECORD_BYTES = 28.0
SEGMENT_BYTES = 48.0

# Algorithmic thread-instructions per photon (DESIGN.md section 7 has the same table, row by row): what the method must do for
# one photon in SASS-level operations, NOT what the kernel executes (ncu's executed count is reported in profiles/).
ALG_PARTS = {
    "philox_block": 42.0,       # Philox4x32-10, S-halves of rounds 1-2 hoisted: 18 IMAD.WIDE + 18 LOP3 + 6
    "uniform": 2.0,             # per uniform: SHF + LOP3 (mantissa stuffing)
    "azimuth": 6.0,             # K0 - u1 L, phi, range scale, 2 MUFU (sin, cos)
    "project": 12.0,            # v_z, 1/v_z (MUFU.RCP), rho, N, plane crossing, sign test
    "pretest_per_tel": 6.0,     # 2 FADD + 2 FFMA/FMUL + FSETP + mask LOP per constant-bank telescope
    "grid_lookup": 15.0,        # cell index, bounds test, 8-byte load, first pre-test (100-telescope array)
    "generic_photon": 34.0,     # fluorescence / generic kinds: emission point, sincospi polynomial, polar angle, direction
    "walk": 14.0,               # index walk, emitter-crossing test, loop
    "reach_vote": 3.0,          # brute-force kernels: OR of the lanes' reach masks over the warp, test, branch
    "queue": 4.0,               # candidate ballot / queue test
    "exact_per_hit": 250.0,     # regenerate + exact test + time + wavelength + weight + commit, per (photon, telescope) hit
    "preamble_per_emitter": 1200.0,   # fp64 preamble of one (segment, process)
    "record_per_hit": 90.0,     # photon output, dense tiles: exact test, arrival time, wavelength, 7-word record staging
    "hist_per_bunch": 92.0,     # ground histogram: v_x, v_y, arrival time, wavelength, radius, bin, 3 shared atomics
}


def alg_instr_per_photon(name: str, photons: float, emitters: float, hits: float, n_tel: int, ground_hist: bool = False,
                         reach_frac: float = 1.0) -> dict:
    """Algorithmic instructions per photon of workload `name`, from ALG_PARTS and the measured counts of the run
    (photons, emitters = (segment, process) pairs with a preamble, hits).  Returns the parts and their sum.
    reach_frac (brute-force kernels, <= 8 telescopes): the share of the photons whose emitter can reach a telescope at
    all (reach mask of the preamble, measured by bench.py with one culling pass); the plane crossing, the pre-tests and
    the candidate dispatch are the method's work for those photons only -- the others are generated and counted."""
    P = ALG_PARTS
    fluor = name in ("c3a", "c3b")
    parts = {}
    if fluor:
        parts["philox"] = P["philox_block"]                     # one block per fluorescence photon
        parts["uniforms"] = 4 * P["uniform"]
        parts["generation"] = P["generic_photon"]
    else:
        parts["philox"] = P["philox_block"] / 2                 # one block per TWO Cherenkov photons (R20)
        parts["uniforms"] = 2 * P["uniform"]
        parts["generation"] = P["azimuth"]
    brute = n_tel <= 8 and not ground_hist and name != "c5g"
    rf = reach_frac if brute else 1.0
    parts["projection"] = P["project"] * rf + (2.0 * (1.0 - rf) if brute else 0.0)      # v_z and its sign test stay (upward count)
    if ground_hist:
        parts["histogram"] = P["hist_per_bunch"]
    elif name == "c5g":
        parts["record"] = P["record_per_hit"] * hits / photons
    else:
        parts["pretests"] = P["grid_lookup"] if n_tel > 8 else P["pretest_per_tel"] * (1 if n_tel <= 1 else 4 if n_tel <= 4 else 8) * rf
        parts["queue"] = P["queue"] * rf
        if brute:
            parts["reach_vote"] = P["reach_vote"] / 2           # once per trip of two photons per lane
        parts["exact_amortised"] = P["exact_per_hit"] * hits / photons
    parts["walk"] = P["walk"]
    parts["preamble_amortised"] = P["preamble_per_emitter"] * emitters / photons
    if name == "c4" and not ground_hist:
        # both processes: the fluorescence share of the photons (~4 %) costs a full block and the generic generation
        parts["fluorescence_share"] = 0.04 * (P["philox_block"] / 2 + 2 * P["uniform"] + P["generic_photon"] - P["azimuth"])
    parts = {k: round(v, 2) for k, v in parts.items()}
    return {"parts": parts, "total": round(sum(parts.values()), 2)}


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), sm_max_mhz=float(p.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed region runs."""

    def __init__(self, index: int, period_s: float = 0.01):
        super().__init__(daemon=True)
        self.index, self.period, self.samples, self.reasons, self.max_mhz = index, period_s, [], set(), None
        self._stop_evt = threading.Event()
        self.paused = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4)}
        while not self._stop_evt.is_set():
            if self.paused:
                time.sleep(self.period)
                continue
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            time.sleep(self.period)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2.0)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


def oracle_baseline(cfg: dict, target_s: float = 15.0) -> dict:
    """Time the fp64 oracle, as it stands, on the host cores on a bounded sample of the workload."""
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    seg = cfg["segments"]
    probe = min(len(seg), 2000)
    t0 = time.perf_counter()
    r = oracle.run(cfg["atmosphere"], cfg["telescopes"], seg[:probe], cfg["params"], want_counts=False, threads=1)
    t1 = time.perf_counter() - t0
    per_seg_core = max(t1 / probe, 1e-9)
    n = int(min(len(seg), max(probe, target_s * cores / per_seg_core)))
    t0 = time.perf_counter()
    r = oracle.run(cfg["atmosphere"], cfg["telescopes"], seg[:n], cfg["params"], want_counts=False, threads=cores)
    dt = time.perf_counter() - t0
    photons = int(r["counters"][1])
    return {"value": photons / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"first {n} of {len(seg)} segments of {cfg['name']} ({photons} photons) in {dt:.2f} s, "
                      f"{cores} threads over contiguous segment ranges"}


def run_reference(args, rank: int):
    """--impl reference: the oracle on host cores (rank 0 only)."""
    if rank != 0:
        return
    cfg = wl.make_config(args.workload, n_segments=args.segments)
    import oracle
    oracle.build()
    cores = os.cpu_count() or 1
    seg = cfg["segments"]
    # each step = a bounded sample of the workload sized for ~2 s on this box
    t0 = time.perf_counter()
    oracle.run(cfg["atmosphere"], cfg["telescopes"], seg[:2000], cfg["params"], want_counts=False, threads=1)
    per_seg_core = (time.perf_counter() - t0) / min(2000, len(seg))
    n = int(min(len(seg), max(2000, 2.0 * cores / per_seg_core)))
    steps = max(1, min(args.steps, 20))
    warm = max(0, min(args.warmup, 2))
    photons = 0
    for _ in range(warm):
        oracle.run(cfg["atmosphere"], cfg["telescopes"], seg[:n], cfg["params"], want_counts=False, threads=cores)
    t0 = time.perf_counter()
    for _ in range(steps):
        r = oracle.run(cfg["atmosphere"], cfg["telescopes"], seg[:n], cfg["params"], want_counts=False, threads=cores)
        photons += int(r["counters"][1])
    dt = time.perf_counter() - t0
    v = photons / dt
    sample = f"each step = first {n} of {len(seg)} segments of {cfg['name']}, {cores} threads"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": 1e3 * dt / steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "segments": len(seg), "sampled_segments_per_step": n},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=["c1", "c2", "c3a", "c3b", "c4", "c5", "c5g"])
    ap.add_argument("--segments", type=int, default=None, help="override the segment count of the workload")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--output-segments", type=int, default=None,
                    help="segment count of the photon-output leg (default: configs[4]'s 10^7)")
    ap.add_argument("--no-output-leg", action="store_true",
                    help="skip the photon-output leg (roofline_output) that the default c2 run adds")
    ap.add_argument("--ground-hist", action="store_true",
                    help="ground-plane radial profile mode (C8OPT_MODE_GROUND_HIST, PAPER.md:85-89) on the workload's "
                         "segments: 1000 bins of 1 m about the shower axis; telescopes are not consulted")
    ap.add_argument("--cull", action="store_true",
                    help="segment culling on (C8OPT_FLAG_CULL): same tallies, `value` then counts culled bunches too")
    ap.add_argument("--cauchy-b", type=float, default=0.0,
                    help="wavelength-dependent refractive index n - 1 = eta (1 + b / lambda^2), b in nm^2 (DESIGN.md R30; "
                         "air: 5670); not the headline configuration, the roofline fraction then does not apply")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist

    import paper_2309_15861_b200 as c8
    from paper_2309_15861_b200.sharding import all_reduce_results, shard_first_id

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the photon path has no CPU fallback")
    from paper_2309_15861_b200.build import build as build_cuda
    build_cuda()      # in-tree nvcc build if libc8opt.so is missing or older than its sources (atomic replace)
    c8.lib()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    # clocks and throttle reasons are sampled over the whole measuring part of the process (warm-up, timed region,
    # end-to-end leg, photon-output leg), every 5 ms
    sampler = ClockSampler(local_rank, period_s=0.005)
    sampler.start()

    # ---- inputs: every rank owns a full-size segment set of its own (weak scaling, independent showers)
    cfg = wl.make_config(args.workload, n_segments=args.segments)
    if world > 1:
        cfg = wl.make_config(args.workload, n_segments=args.segments, seed_offset=rank)
    seg = cfg["segments"]
    n = len(seg)
    first_id = shard_first_id(rank, n)
    tel = np.asarray(cfg["telescopes"], dtype=np.float32)
    n_tel = len(tel)
    par = dict(cfg["params"])
    if args.cull:
        par["flags"] = c8.FLAG_CULL
    if args.cauchy_b > 0.0:
        par["cauchy_b"] = args.cauchy_b
        cfg["params"] = dict(cfg["params"], cauchy_b=args.cauchy_b)       # the oracle leg times the same physics
    if args.ground_hist:
        par["mode"] = c8.MODE_GROUND_HIST
        par["fl_beam_telescope"] = -1
    output_mode = par["mode"] == c8.MODE_OUTPUT
    n_procs = 2 if par["processes"] == 3 else 1
    h_seg = torch.from_numpy(seg.view(np.uint8).reshape(n, 48).copy()).pin_memory()
    d_seg = h_seg.to(dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    stream = torch.cuda.current_stream()
    peaks = load_peaks()

    def time_leg(ctx, par, kw, steps, warmup, hist=False):
        """W untimed + K timed steps of one propagate call over the whole table; device time by CUDA events on the
        launching stream around every step, L2 flushed (untimed) between steps.  Returns (counters, ms per step array,
        launches in the timed region, wall seconds of the timed region)."""
        def step(ev=None):
            flush.fill_(1)
            ctx.reset_tallies()
            if ev is not None:
                ev[0].record(stream)
            ctx.propagate_segments(d_seg, par, n=n, first_segment_id=first_id, **kw)
            if ev is not None:
                ev[1].record(stream)
        for _ in range(warmup):
            step()
        counters = ctx.read_ground_histogram()[2] if hist else ctx.read_tallies()[1]
        events = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        l0 = ctx.launch_count
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        w0 = time.perf_counter()
        for k in range(steps):
            step(events[k])
        torch.cuda.synchronize()
        wall = time.perf_counter() - w0
        if world > 1:
            dist.barrier()
        return counters, np.array([a.elapsed_time(b) for a, b in events]), ctx.launch_count - l0, wall

    def output_buffers(ctx, par, n_tel):
        """Record regions sized by one tally-mode pass (exact record count per telescope + slack)."""
        p0 = dict(par); p0["mode"] = c8.MODE_TALLY
        ctx.reset_tallies()
        ctx.propagate_segments(d_seg, p0, n=n, first_segment_id=first_id)
        t0_, _, _ = ctx.read_tallies()
        caps = (t0_["hits"].astype(np.int64) + 1024)
        offs = np.concatenate([[0], np.cumsum(caps)[:-1]])
        return dict(records=torch.empty((int(caps.sum()), 7), dtype=torch.float32, device=dev),
                    tel_offset=torch.from_numpy(offs).to(dev), tel_capacity=torch.from_numpy(caps).to(dev))

    ctx = c8.Context(cfg["atmosphere"])
    ctx.add_telescopes(tel)
    if args.ground_hist:
        ctx.set_ground_histogram(0.0, 0.0, 1000.0, 1000)
    kw = output_buffers(ctx, par, n_tel) if output_mode else {}

    def read_counters():
        """Synchronise, read the step's result back (D2H) and return the counters."""
        if args.ground_hist:
            return ctx.read_ground_histogram()[2]
        return ctx.read_tallies()[1]

    # ---- timed region: exactly K steps
    counters, step_ms, launches, wall = time_leg(ctx, par, kw, args.steps, args.warmup, hist=args.ground_hist)
    photons_per_step = counters["generated"]
    culled_per_step = counters["culled"]
    hits_per_step = counters["hits"]
    total_ms = float(step_ms.sum())
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
        pc = torch.tensor([photons_per_step], dtype=torch.float64, device=dev)
        dist.all_reduce(pc, op=dist.ReduceOp.SUM)
        photons_all = float(pc.item())
    else:
        photons_all = float(photons_per_step)
    value = photons_all * args.steps / (total_ms * 1e-3)

    # brute-force kernels: the share of the Cherenkov photons whose emitter can reach a telescope at all, from one
    # untimed pass with the exact culling on (it culls exactly the emitters whose reach mask is empty)
    reach_frac = 1.0
    if (n_tel <= 8 and (par["processes"] & 1) and not (args.ground_hist or args.cull or args.cauchy_b > 0.0)
            and args.workload not in ("c5g", "c3a", "c3b") and rank == 0):
        pc = dict(par, mode=c8.MODE_TALLY, flags=c8.FLAG_CULL)
        ctx.reset_tallies()
        ctx.propagate_segments(d_seg, pc, n=n, first_segment_id=first_id)
        cc = ctx.read_tallies()[1]
        reach_frac = 1.0 - cc["culled"] / max(cc["generated"], 1)

    # ---- the job's only exchange: one sum of the per-telescope tallies and counters over the ranks, after
    # the timed region (NCCL all-reduce of a few hundred bytes)
    reduced = None
    if world > 1 and not args.ground_hist:
        tallies, cnt, _ = ctx.read_tallies()
        tallies_all, cnt_all = all_reduce_results(tallies, cnt, device=dev)
        reduced = {"hits_all_ranks": int(tallies_all["hits"].sum()), "generated_all_ranks": int(cnt_all["generated"])}

    # ---- end to end through the C-ABI with HOST buffers: H2D of the segments + kernel + D2H of the tallies
    e2e = None
    if not args.no_e2e:
        # (no NVML queries during this leg: they take the driver's lock, the 28 copies and launches of a call wait for it
        # and the copy engine stands still -- 1.06 ms per call without the sampler, 1.15 - 1.45 ms with it; the clocks of
        # the kernel legs before and after are sampled as before)
        sampler.paused = True
        for _ in range(2):
            ctx.reset_tallies()
            ctx.propagate_segments_host(h_seg, par, n=n, first_segment_id=first_id, **kw)
            read_counters()
        ke = max(3, min(args.steps, 20))
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t0 = time.perf_counter()
        for _ in range(ke):
            ctx.reset_tallies()
            ctx.propagate_segments_host(h_seg, par, n=n, first_segment_id=first_id, **kw)
            read_counters()                             # synchronises + D2H
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        e2e = {"value": photons_all * ke / dt, "unit": UNIT, "h2d_bytes_per_step": int(n * 48),
               "d2h_bytes_per_step": int(1001 * 24 + 8 * 8) if args.ground_hist else int(n_tel * 24 + 8 * 8 + n_tel * 8), "steps": ke,
               "note": "c8opt_propagate_segments_host from pinned host memory (chunked H2D overlapped with the kernels) "
                       "+ c8opt_read_tallies; wall clock"}
        sampler.paused = False

    # ---- photon-output leg (north_star's second roofline): the same segments against one accept-all detector on the
    # observation level, every downward photon written as a 28-byte record ("c5g" at this segment count)
    roofline_output = None
    if args.workload == "c2" and not (args.no_output_leg or args.cull or args.ground_hist or args.cauchy_b > 0.0) and world == 1:
        # "c5g": configs[4]'s segment set (the c2 generator at 10^7 segments) with one accept-all detector
        del kw
        ocfg = wl.make_config("c5g", n_segments=args.output_segments)
        oseg = ocfg["segments"]
        on = len(oseg)
        d_seg = torch.from_numpy(oseg.view(np.uint8).reshape(on, 48).copy()).to(dev)
        n_saved, n = n, on                              # time_leg / output_buffers read n and d_seg
        octx = c8.Context(ocfg["atmosphere"])
        octx.add_telescopes(np.asarray(ocfg["telescopes"], dtype=np.float32))
        opar = dict(ocfg["params"]); opar["mode"] = c8.MODE_OUTPUT
        okw = output_buffers(octx, opar, 1)
        ko = max(3, min(args.steps, 10))
        ocnt, oms, olaunch, _ = time_leg(octx, opar, okw, ko, 3)
        launches += olaunch
        o_s = float(oms.sum()) * 1e-3 / ko
        obytes = RECORD_BYTES * ocnt["records"] + SEGMENT_BYTES * on
        roofline_output = {
            "bound": "hbm", "workload": f"c5g: {on} segments of configs[4] (seed 2), one accept-all detector at h_obs, photon-output mode",
            "achieved": obytes / o_s / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": obytes / o_s / 1e9 / peaks["hbm_gbs"],
            "traffic": None, "traffic_note": "measured per round with ncu --set full: profiles/ncu_c5g_output_r02.md",
            "peak_source": peaks["source"], "algorithmic_bytes_per_launch": obytes,
            "bytes_per_record": RECORD_BYTES, "bytes_per_segment": SEGMENT_BYTES, "records_per_launch": ocnt["records"],
            "kernel": "c8::propagate_kernel<TEL_CONST, coplanar, 1, output>", "kernel_ms": o_s * 1e3, "steps": ko,
            "photons_per_s": ocnt["generated"] / o_s}
        octx.close()
        del okw, d_seg
        n = n_saved

    clocks = sampler.stop()
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (only) kernel
    per_launch_s = total_ms * 1e-3 / args.steps
    alg = alg_instr_per_photon(args.workload, float(photons_per_step - culled_per_step), float(n * n_procs), float(hits_per_step), n_tel,
                               ground_hist=args.ground_hist, reach_frac=reach_frac)
    if args.workload == "c5g":
        bytes_per_launch = RECORD_BYTES * hits_per_step + SEGMENT_BYTES * n
        roofline = {"bound": "hbm", "achieved": bytes_per_launch / per_launch_s / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                    "traffic": None, "peak_source": peaks["source"], "bytes_per_record": RECORD_BYTES, "bytes_per_segment": SEGMENT_BYTES,
                    "algorithmic_bytes_per_launch": bytes_per_launch, "alg_instr_per_photon": alg["total"], "alg_instr_parts": alg["parts"]}
    else:
        peak = 148 * 4 * 32 * peaks["sm_max_mhz"] * 1e6 / 1e12            # thread-instructions / s, issue-slot peak
        # culled bunches cost no photon-loop instructions: the roofline counts the propagated ones only
        roofline = {"bound": "alu", "achieved": alg["total"] * (photons_per_step - culled_per_step) / per_launch_s / 1e12, "peak": peak,
                    "unit": "Tinstr/s", "traffic": None, "peak_source": "148 SM x 4 schedulers x 32 lanes x sm_max_mhz "
                    f"({peaks['source']})", "alg_instr_per_photon": alg["total"], "alg_instr_parts": alg["parts"], "reach_frac": reach_frac,
                    "hbm_achieved_gbs": (SEGMENT_BYTES * n + RECORD_BYTES * (hits_per_step if output_mode else 0)) / per_launch_s / 1e9}
    roofline["traffic_note"] = "not measured in this run; the ncu --set full captures of the round are under profiles/"
    roofline["frac"] = roofline["achieved"] / roofline["peak"]
    roofline["kernel"] = "c8::propagate_kernel"
    roofline["kernel_ms"] = per_launch_s * 1e3

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": cfg["name"], "segments": n, "segments_per_gpu": n, "photons_per_step_per_gpu": photons_per_step,
                   "hits_per_step_per_gpu": hits_per_step, "telescopes": n_tel, "mode": "ground histogram (1000 x 1 m)" if args.ground_hist else "output" if output_mode else "tally",
                   "l2": "flushed between steps (256 MiB fill, untimed)", "timing": "sum of per-step CUDA-event times",
                   "parallelism": f"segments sharded over {world} GPU(s), no data-path collective; one all-reduce of the tallies after the job",
                   "culling": (f"on: {culled_per_step} of the bunches per step are generated but provably miss every telescope "
                               "and skip the photon loop; value counts them (pre-cull equivalent), tallies are identical")
                              if args.cull else "off",
                   "cauchy_b_nm2": args.cauchy_b},
        "roofline": roofline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "wall_s_timed_region": wall, "step_ms_min_med_max": [float(step_ms.min()), float(np.median(step_ms)), float(step_ms.max())],
    }
    if roofline_output is not None:
        out["roofline_output"] = roofline_output
    if reduced is not None:
        out["all_reduce"] = reduced
    if not args.no_cpu_baseline and world == 1:
        out["cpu_baseline"] = oracle_baseline(cfg)
    print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
