"""Helpers of the GPU parity tests: run the CUDA path through the Python binding of the C-ABI,
run the fp64 oracle on the same seeded inputs, and compare by BASELINE.json north_star's
criteria (a)-(d).  Only tests import this module."""
from __future__ import annotations

import os

import numpy as np

import oracle
import workloads as wl

# north_star tolerances
TOL_XY_M = 1e-2          # (c) arrival positions within 1 cm
TOL_DIR_RAD = 1e-5       # (c) directions within 1e-5 rad
TOL_T_NS = 0.1           # (d) arrival times within 0.1 ns
TOL_TALLY_REL = 1e-3     # (b) per-telescope tallied counts within 1e-3 relative
TOL_FLIP_M = 5e-3        # (b) a hit/miss flip is legitimate only if |b_oracle - R| < 5 mm  (R22)
TOL_LAM_REL = 1e-6
TOL_W_REL = 1e-5


def n_threads() -> int:
    return max(1, min(16, os.cpu_count() or 1))


def gpu_run(cfg: dict, mode: int, want_records: bool = True, capacity_per_tel: int | None = None,
            first_id: int = 0, host_segments: bool = False, chunks: int = 1, with_ids: bool = True, region_shift: int = 0):
    """Run cfg through the CUDA path.  Returns dict(counts, tallies, counters, records, tel_count).

    records: structured array sorted by (id, tel) with the 7 record floats, the id and the telescope.
    with_ids=False: no id side buffer is passed (the launch bench.py times); the records then come back in the order
    of the regions, id = 0.  region_shift: every telescope region starts that many records later in the buffer.
    """
    import torch

    import paper_2309_15861_b200 as c8

    seg = cfg["segments"]
    n = len(seg)
    tel = np.asarray(cfg["telescopes"], dtype=np.float32)
    n_tel = len(tel)
    par = dict(cfg["params"])
    par["mode"] = mode
    ctx = c8.Context(cfg["atmosphere"])
    ctx.add_telescopes(tel)
    dev = torch.device("cuda:0")
    d_counts = torch.zeros((n, 2), dtype=torch.int32, device=dev)
    kw = dict(counts=d_counts)
    d_rec = d_ids = None
    if mode == c8.MODE_OUTPUT:
        cap = int(capacity_per_tel if capacity_per_tel is not None else 1 << 20)
        d_rec = torch.zeros((n_tel * cap + region_shift, 7), dtype=torch.float32, device=dev)
        d_ids = torch.zeros(n_tel * cap + region_shift, dtype=torch.int64, device=dev)
        d_off = torch.arange(n_tel, dtype=torch.int64, device=dev) * cap + region_shift
        d_cap = torch.full((n_tel,), cap, dtype=torch.int64, device=dev)
        kw.update(records=d_rec, tel_offset=d_off, tel_capacity=d_cap, ids=d_ids if with_ids else None)
    if host_segments:
        h = torch.from_numpy(seg.view(np.uint8).reshape(n, 48).copy()).pin_memory()
        ctx.propagate_segments_host(h, par, n=n, first_segment_id=first_id, **kw)
    else:
        d_seg = torch.from_numpy(seg.view(np.uint8).reshape(n, 48).copy()).to(dev)
        bounds = [n * i // chunks for i in range(chunks + 1)]
        for lo, hi in zip(bounds[:-1], bounds[1:]):
            kk = dict(kw)
            kk["counts"] = d_counts[lo:]
            ctx.propagate_segments(d_seg[lo:], par, n=hi - lo, first_segment_id=first_id + lo, **kk)
    tallies, counters, tel_count = ctx.read_tallies(allow_overflow=True)
    out = dict(counts=d_counts.cpu().numpy().astype(np.uint32), tallies=tallies, counters=counters,
               tel_count=tel_count, records=None, launches=ctx.launch_count)
    if mode == c8.MODE_OUTPUT and want_records:
        rec_dtype = np.dtype([("x", "<f4"), ("y", "<f4"), ("cx", "<f4"), ("cy", "<f4"), ("t", "<f4"),
                              ("lam", "<f4"), ("w", "<f4"), ("id", "<u8"), ("tel", "<i4")])
        parts = []
        h_rec = d_rec.cpu().numpy()
        h_ids = d_ids.cpu().numpy().view(np.uint64)
        for k in range(n_tel):
            m = int(tel_count[k])
            r = np.zeros(m, dtype=rec_dtype)
            blk = h_rec[region_shift + k * cap: region_shift + k * cap + m]
            for i, name in enumerate(("x", "y", "cx", "cy", "t", "lam", "w")):
                r[name] = blk[:, i]
            r["id"] = h_ids[region_shift + k * cap: region_shift + k * cap + m]
            r["tel"] = k
            parts.append(r)
        rec = np.concatenate(parts) if parts else np.zeros(0, dtype=rec_dtype)
        out["records"] = rec[np.lexsort((rec["tel"], rec["id"]))] if with_ids else rec
        if region_shift:
            assert not h_rec[:region_shift].any(), "records written before the first region"
    ctx.close()
    return out


def oracle_run(cfg: dict, record_capacity: int = 1 << 22, first_id: int = 0):
    res = oracle.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"], cfg["params"], first_id=first_id,
                     want_counts=True, record_capacity=record_capacity, threads=n_threads())
    rec = res["records"]
    if rec is not None:
        res["records"] = rec[np.lexsort((rec["tel"], rec["id"]))]
    return res


def oracle_impact(cfg: dict, rid: int, k: int, first_id: int = 0):
    """Impact parameter b (m) of photon `rid` w.r.t. telescope k, recomputed with the oracle's own pieces."""
    S, tag, j = rid >> 25, (rid >> 24) & 1, rid & 0xFFFFFF
    seg = cfg["segments"][S - first_id]
    tel = np.asarray(cfg["telescopes"], dtype=np.float32).astype(np.float64)
    par = cfg["params"]
    bt = tel[par["fl_beam_telescope"]] if (tag == 1 and par["fl_beam_telescope"] >= 0) else None
    if tag == 1 and par["fl_beam_telescope"] == oracle.BEAM_ARRAY:
        bt = oracle.array_sphere(cfg["telescopes"])
    st, fr = oracle.preamble(cfg["atmosphere"], par, seg, tag, bt)
    assert st == 0 and j < fr.n_b
    ph = oracle.make_photon(fr, par, S, j, tag)
    hit, b2, s_c, s_pl, x, y = oracle.intersect(list(ph.e), list(ph.v), tel[k])
    return hit, float(np.sqrt(max(b2, 0.0))), float(tel[k][3]), float(ph.v[2])


def compare(cfg: dict, g: dict, o: dict, first_id: int = 0, check_records: bool = True, check_upward: bool = True) -> dict:
    """Assert criteria (a)-(d); returns a small report."""
    rep = {}
    # (a) per-segment generated photon counts are bit-exact
    assert np.array_equal(g["counts"], o["counts"]), "criterion (a): per-segment bunch counts differ"
    oc = {name: int(v) for name, v in zip(oracle.COUNTER_NAMES, o["counters"])}
    gc = g["counters"]
    assert gc["segments"] == oc["segments"]
    assert gc["generated"] == oc["generated"] == int(o["counts"].astype(np.uint64).sum())
    assert gc["invalid"] == oc["invalid"]
    if check_upward:       # a culled run counts the upward bunches of the propagated segments only
        assert abs(gc["upward"] - oc["upward"]) <= max(2, int(1e-5 * oc["generated"])), (gc["upward"], oc["upward"])
    assert gc["hits"] == int(g["tallies"]["hits"].sum())
    rep.update(generated=gc["generated"], hits_gpu=gc["hits"], hits_oracle=oc["hits"])

    flips = []
    if check_records:
        gr, orr = g["records"], o["records"]
        assert gr is not None and orr is not None
        assert gc["dropped"] == 0 and oc["dropped"] == 0
        assert len(gr) == gc["hits"], "records written != hits tallied"
        gkey = gr["id"].astype(np.uint64) * np.uint64(8192) + gr["tel"].astype(np.uint64)
        okey = orr["id"].astype(np.uint64) * np.uint64(8192) + orr["tel"].astype(np.uint64)
        assert len(np.unique(gkey)) == len(gkey), "duplicate GPU records"
        common, gi, oi = np.intersect1d(gkey, okey, return_indices=True)
        only_g = np.setdiff1d(np.arange(len(gkey)), gi)
        only_o = np.setdiff1d(np.arange(len(okey)), oi)
        # (b) every flip is enumerated and must sit on the sphere boundary
        for idx, src in [(only_g, gr), (only_o, orr)]:
            for i in idx:
                rid, k = int(src["id"][i]), int(src["tel"][i])
                hit, b, R, vz = oracle_impact(cfg, rid, k, first_id)
                flips.append((rid, k, b - R))
                assert abs(b - R) < TOL_FLIP_M, f"flip of photon {rid:#x} tel {k}: |b - R| = {abs(b - R):.3e} m"
        a, b_ = gr[gi], orr[oi]
        if len(a):
            dx, dy = np.abs(a["x"] - b_["x"]), np.abs(a["y"] - b_["y"])
            # 1 cm, plus half an fp32 ulp of the stored number: the record holds x, y as fp32, and the plane crossing of a
            # nearly horizontal photon that clips a sphere can lie > 131 km from the centre, where an ulp exceeds 1.5 cm
            tol_x, tol_y = TOL_XY_M + 2.0 ** -24 * np.abs(b_["x"]), TOL_XY_M + 2.0 ** -24 * np.abs(b_["y"])
            assert (dx <= tol_x).all() and (dy <= tol_y).all(), f"(c) position: {dx.max():.3e} {dy.max():.3e} m"
            rep.update(records_beyond_100km=int(((np.abs(b_["x"]) > 1e5) | (np.abs(b_["y"]) > 1e5)).sum()))
            # direction: the record stores (cos_x, cos_y) only.  The two stored components are compared
            # directly; the full angle (v_z rebuilt from the unit norm) is compared where the rebuild is
            # well conditioned, |v_z| >= 0.05 (a near-horizontal photon's v_z is not recoverable from fp32
            # cos_x, cos_y: d v_z = (cx dcx + cy dcy) / v_z).
            dcx = a["cx"].astype(np.float64) - b_["cx"]
            dcy = a["cy"].astype(np.float64) - b_["cy"]
            ang = np.sqrt(dcx ** 2 + dcy ** 2)
            gz = -np.sqrt(np.maximum(0.0, 1.0 - a["cx"].astype(np.float64) ** 2 - a["cy"].astype(np.float64) ** 2))
            oz = -np.sqrt(np.maximum(0.0, 1.0 - b_["cx"] ** 2 - b_["cy"] ** 2))
            steep = np.abs(oz) >= 0.05
            ang = np.where(steep, np.sqrt(dcx ** 2 + dcy ** 2 + (gz - oz) ** 2), ang)
            assert ang.max() <= TOL_DIR_RAD, f"(c) direction: {ang.max():.3e} rad"
            dt = np.abs(a["t"] - b_["t"])
            assert dt.max() <= TOL_T_NS, f"(d) time: {dt.max():.3e} ns"
            dl = np.abs(a["lam"] - b_["lam"]) / b_["lam"]
            assert dl.max() <= TOL_LAM_REL, f"wavelength: {dl.max():.3e}"
            # weight = w0 exp(-tau / |v_z|), plain relative error: the flat photons (|v_z| < 0.05), whose exponent reaches
            # hundreds, are evaluated in double on the GPU; for the others the exponent stays below 20 (2e-7 x 20 in fp32)
            dw = np.abs(a["w"] - b_["w"]) / np.maximum(np.abs(b_["w"]), 1e-300)
            assert dw.max() <= TOL_W_REL, f"weight: {dw.max():.3e}"
            rep.update(max_dxy_m=float(max(dx.max(), dy.max())), max_ang_rad=float(ang.max()), max_dt_ns=float(dt.max()),
                       max_dlam_rel=float(dl.max()), max_dw_rel=float(dw.max()),
                       flat_records_two_component_direction=int((~steep).sum()))
        rep.update(matched=len(common), flips=len(flips))
    # (b) per-telescope tallies: within 1e-3 relative, or explained by the enumerated boundary flips
    B = float(cfg["params"]["bunch_size"])
    n_flip_tel = np.zeros(len(g["tallies"]), dtype=np.int64)
    for _, k, _ in flips:
        n_flip_tel[k] += 1
    for k in range(len(g["tallies"])):
        hg, ho = int(g["tallies"]["hits"][k]), int(o["tallies"]["hits"][k])
        slack = int(n_flip_tel[k]) if check_records else 3
        assert abs(hg - ho) <= max(TOL_TALLY_REL * ho, slack), f"(b) telescope {k}: hits {hg} vs {ho}"
        wg, wo = float(g["tallies"]["sum_w"][k]), float(o["tallies"]["sum_w"][k])
        assert abs(wg - wo) <= TOL_TALLY_REL * abs(wo) + B * slack, f"(b) telescope {k} sum_w: {wg} vs {wo}"
        if hg == ho and (not check_records or n_flip_tel[k] == 0):
            tg, to = float(g["tallies"]["sum_wt"][k]), float(o["tallies"]["sum_wt"][k])
            assert abs(tg - to) <= TOL_TALLY_REL * abs(to) + TOL_T_NS * abs(wo), f"(d) telescope {k} sum_wt: {tg} vs {to}"
    rep["flip_list"] = flips
    return rep


def gpu_hist(cfg: dict, core, r_max: float, n_bins: int, first_id: int = 0, chunks: int = 1):
    """Ground-plane radial profile of cfg through the CUDA path (C8OPT_MODE_GROUND_HIST)."""
    import torch

    import paper_2309_15861_b200 as c8

    seg = cfg["segments"]
    n = len(seg)
    par = dict(cfg["params"])
    par["mode"] = c8.MODE_GROUND_HIST
    ctx = c8.Context(cfg["atmosphere"])
    ctx.set_ground_histogram(core[0], core[1], r_max, n_bins)
    dev = torch.device("cuda:0")
    d_counts = torch.zeros((n, 2), dtype=torch.int32, device=dev)
    d_seg = torch.from_numpy(seg.view(np.uint8).reshape(n, 48).copy()).to(dev)
    bounds = [n * i // chunks for i in range(chunks + 1)]
    for lo, hi in zip(bounds[:-1], bounds[1:]):
        ctx.propagate_segments(d_seg[lo:], par, n=hi - lo, first_segment_id=first_id + lo, counts=d_counts[lo:])
    bins, over, counters = ctx.read_ground_histogram()
    out = dict(hist=bins, overflow=over, counters=counters, counts=d_counts.cpu().numpy().astype(np.uint32),
               launches=ctx.launch_count)
    ctx.close()
    return out


def compare_hist(g: dict, o: dict, r_max: float, n_bins: int, edge_m: float = 2e-3) -> dict:
    """Per-bin parity of the radial profile.  A bunch within `edge_m` of a bin edge may fall on either side in fp32
    (positions agree to well under a millimetre, criterion (c)); those are counted from the oracle's radii and bound
    the per-bin difference.  Bins with at least 50 bunches (the paper's cut): sum of weights within 1e-3
    relative beyond the edge bunches, mean arrival time within 0.1 ns (criterion (d))."""
    assert np.array_equal(g["counts"], o["counts"]), "criterion (a): per-segment bunch counts differ"
    gh, oh = g["hist"], o["hist"]
    dr = r_max / n_bins
    r = o["r"]
    frac = r / dr - np.floor(r / dr)
    near = (np.minimum(frac, 1.0 - frac) * dr <= edge_m)
    b_lo = np.floor((r - edge_m) / dr).astype(np.int64)
    b_hi = np.floor((r + edge_m) / dr).astype(np.int64)
    slack = np.zeros(n_bins + 1, dtype=np.int64)
    for b in (b_lo[near], b_hi[near]):
        np.add.at(slack, np.clip(b, 0, n_bins), 1)
    dn = np.abs(gh["n"].astype(np.int64) - oh["n"].astype(np.int64))
    assert np.all(dn <= slack[:n_bins]), (np.nonzero(dn > slack[:n_bins])[0][:10], dn.max())
    total_g, total_o = int(gh["n"].sum()) + g["overflow"], int(oh["n"].sum()) + o["overflow"]
    assert abs(total_g - total_o) <= max(2, int(1e-5 * total_o)), (total_g, total_o)
    assert abs(g["overflow"] - o["overflow"]) <= slack[n_bins] + max(2, int(1e-5 * total_o))
    big = (oh["n"] >= 50) & (gh["n"] >= 50)
    w_mean = oh["sum_w"][big] / oh["n"][big]
    dw = np.abs(gh["sum_w"][big] - oh["sum_w"][big])
    assert np.all(dw <= 1e-3 * oh["sum_w"][big] + 2.0 * slack[:n_bins][big] * w_mean)
    # mean time: a bunch near an edge may sit in either bin, which moves that bin's mean by at most w |t - mean| / sum_w;
    # beyond the sum of those (enumerated from the oracle's records) the means agree within 0.1 ns
    rec = o["records"]
    w_all, t_all = rec["w"].astype(np.float64), rec["t"].astype(np.float64)
    mt_full = np.where(oh["sum_w"] > 0, oh["sum_wt"] / np.maximum(oh["sum_w"], 1e-300), 0.0)
    infl = np.zeros(n_bins + 1)
    for b in (b_lo[near], b_hi[near]):
        bc = np.clip(b, 0, n_bins)
        np.add.at(infl, bc, w_all[near] * np.abs(t_all[near] - np.append(mt_full, 0.0)[bc]))
    mt_g, mt_o = gh["sum_wt"][big] / gh["sum_w"][big], oh["sum_wt"][big] / oh["sum_w"][big]
    dt = np.abs(mt_g - mt_o) - 1.05 * infl[:n_bins][big] / oh["sum_w"][big]
    assert np.all(dt <= TOL_T_NS), dt.max()
    return dict(bunches=total_o, overflow_gpu=g["overflow"], overflow_oracle=o["overflow"], bins_ge50=int(big.sum()),
                bins_differing=int(np.count_nonzero(dn)), max_dn=int(dn.max()), edge_bunches=int(near.sum()),
                max_dmean_t_ns=float(dt.max()) if dt.size else 0.0,
                max_dsumw_rel=float(np.max(dw / oh["sum_w"][big])) if dw.size else 0.0)
