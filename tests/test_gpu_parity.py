"""GPU parity: the CUDA path (through the C-ABI binding) against the fp64 oracle, element by element,
on the seeded synthetic configs of BASELINE.json (workloads.make_config).  Criteria (a)-(d) of
north_star are asserted in tests/parity_util.compare with the tolerances written there.

Run on the B200 box:  python -m pytest tests -m gpu -x -q
"""
import numpy as np
import pytest

import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def c8():
    import torch
    assert torch.cuda.is_available(), "these tests need the B200"
    from paper_2309_15861_b200.build import build
    build()           # compiles libc8opt.so in-tree if it is missing or older than its sources (nvcc, sm_100a)
    import paper_2309_15861_b200 as c8
    c8.lib()          # fail loudly if the CUDA extension is missing
    return c8


def _report(name, rep):
    print(f"[parity {name}] " + " ".join(f"{k}={v}" for k, v in rep.items() if k != "flip_list"))
    for rid, k, d in rep.get("flip_list", []):
        print(f"[parity {name}] flip photon={rid:#x} tel={k} b-R={d:+.3e} m")


def test_config1_records_and_tallies(c8):
    """configs[0]: 10^4 electron segments, single-layer atmosphere, 1 telescope; every record compared."""
    import parity_util as pu
    cfg = wl.make_config("c1")
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("c1", rep)
    assert rep["matched"] > 100


def test_config1_tally_mode_equals_output_mode(c8):
    import parity_util as pu
    cfg = wl.make_config("c1")
    a = pu.gpu_run(cfg, c8.MODE_TALLY)
    b = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    assert np.array_equal(a["tallies"]["hits"], b["tallies"]["hits"])
    assert np.allclose(a["tallies"]["sum_w"], b["tallies"]["sum_w"], rtol=1e-12)
    assert a["counters"]["generated"] == b["counters"]["generated"]
    assert a["counters"]["records"] == 0 and b["counters"]["records"] == b["counters"]["hits"]


@pytest.mark.parametrize("n", [0, 1, 31, 257, 1000])
def test_ragged_sizes(c8, n):
    """Empty input, less than a warp, a tile plus one, several tiles with a ragged tail."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=max(n, 1))
    cfg["segments"] = cfg["segments"][:n]
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report(f"ragged{n}", rep)


def test_config2_subset_records(c8):
    """configs[1] shape (5-layer atmosphere, 4 telescopes) on 50k segments: every record compared."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=50_000)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("c2-50k", rep)
    assert rep["matched"] > 5000


def test_config2_full_size_tally(c8):
    """configs[1] at full size (10^6 segments) in the launch configuration bench.py times (tally mode)."""
    import parity_util as pu
    cfg = wl.make_config("c2")
    g = pu.gpu_run(cfg, c8.MODE_TALLY)
    o = pu.oracle_run(cfg, record_capacity=0)
    rep = pu.compare(cfg, g, o, check_records=False)
    _report("c2-full", rep)


def test_batching_and_host_path_invariance(c8):
    """Results do not depend on how segments are batched (R20), nor on the host-buffer entry point."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=100_000)
    a = pu.gpu_run(cfg, c8.MODE_OUTPUT, first_id=7)
    b = pu.gpu_run(cfg, c8.MODE_OUTPUT, first_id=7, chunks=3)
    c = pu.gpu_run(cfg, c8.MODE_OUTPUT, first_id=7, host_segments=True)
    for other in (b, c):
        assert np.array_equal(a["counts"], other["counts"])
        assert np.array_equal(a["tallies"]["hits"], other["tallies"]["hits"])
        assert np.array_equal(a["records"]["id"], other["records"]["id"])
        for f in ("x", "y", "cx", "cy", "t", "lam", "w"):
            assert np.array_equal(a["records"][f], other["records"][f])
        assert np.allclose(a["tallies"]["sum_w"], other["tallies"]["sum_w"], rtol=1e-12)
    assert b["launches"] == 3 and c["launches"] >= 1


def test_config3_fluorescence_isotropic_and_beamed(c8):
    """configs[2] at its full size (10^6 segments): fluorescence only, telescope at 10 km; isotropic (hit list identical)
    and beamed 2 deg; every record compared."""
    import parity_util as pu
    for name in ("c3a", "c3b"):
        cfg = wl.make_config(name)
        g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
        o = pu.oracle_run(cfg)
        rep = pu.compare(cfg, g, o)
        _report(name, rep)
        if name == "c3b":
            assert rep["matched"] > 100


def test_isotropic_near_telescope(c8):
    """Isotropic fluorescence with a big sphere nearby, so that the isotropic branch has many hits."""
    import parity_util as pu
    cfg = wl.make_config("c3a", n_segments=20_000)
    cfg["telescopes"] = np.array([[300.0, 0.0, 2000.0, 150.0]], dtype=np.float32)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("iso-near", rep)
    assert rep["matched"] > 200


def test_config4_subsample(c8):
    """configs[3] shape: both processes, 100 telescopes, 5 layers + transmission table; 1 % subsample."""
    import parity_util as pu
    cfg = wl.make_config("c4", n_segments=100_000)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("c4-1pct", rep)
    assert rep["matched"] > 5000


def test_non_coplanar_and_generic_tracks(c8):
    """Telescopes at different altitudes (general q_z != 0 test) and tracks that are horizontal / upward
    (generic Cherenkov projection), plus invalid segments."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=30_000)
    tel = cfg["telescopes"].copy()
    tel[:, 2] += np.array([0.0, 35.0, -20.0, 60.0], dtype=np.float32)
    tel[:, 3] = np.array([6.0, 12.0, 25.0, 40.0], dtype=np.float32)
    cfg["telescopes"] = tel
    seg = cfg["segments"]
    rng = np.random.Generator(np.random.PCG64(99))
    # every 7th track gets a random direction (isotropic), so some are horizontal or upward
    idx = np.arange(0, len(seg), 7)
    v = rng.normal(size=(len(idx), 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    v = v.astype(np.float32).astype(np.float64)
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    seg["dx"][idx], seg["dy"][idx], seg["dz"][idx] = v[:, 0], v[:, 1], v[:, 2]
    seg["length"][idx] = np.minimum(seg["length"][idx], 5.0)
    # invalid ones
    seg["gamma"][11] = 0.5
    seg["dx"][12] = np.nan
    seg["length"][13] = -1.0
    seg["dz"][14] *= 1.01
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("noncoplanar", rep)
    assert g["counters"]["invalid"] == 4
    assert rep["matched"] > 1000


def test_segment_invalid_for_one_process_only(c8):
    """Both processes (two launches): a segment whose fluorescence bunch count alone is out of range (n_b >= 2^24), one
    whose Cherenkov count alone is, and one that is invalid for both are each counted once, as the oracle counts them."""
    import parity_util as pu
    cfg = wl.make_config("c4", n_segments=4000)
    seg = cfg["segments"]
    seg["dE"][100] = np.float32(1.0e7)              # 4 / MeV x 1e7 MeV = 4e7 bunches >= 2^24: fluorescence only
    seg["length"][200] = np.float32(1.0e6)          # ~ 34 / m x 1e6 m along a horizontal track at 2.5 km: Cherenkov only
    seg["z0"][200], seg["dz"][200], seg["dx"][200], seg["dy"][200] = 2500.0, 0.0, 1.0, 0.0
    seg["gamma"][200] = np.float32(1e4)
    seg["gamma"][300] = np.float32(0.5)             # both
    seg["dE"][301] = np.float32(1.0e7)
    seg["gamma"][301] = np.float32(np.nan)          # both, and the fluorescence count out of range as well
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("invalid-one-process", rep)
    assert g["counters"]["invalid"] == 4


def test_output_capacity_overflow(c8):
    """The kernel never writes past tel_capacity; the overflow is counted and reported as error -3."""
    import parity_util as pu
    cfg = wl.make_config("c1")
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=100)
    assert g["counters"]["records"] == 100
    assert g["counters"]["dropped"] == g["counters"]["hits"] - 100 > 0
    assert len(g["records"]) == 100


def test_accept_all_output(c8):
    """config 5g shape (every downward photon is written) on 3000 segments: the dense record path."""
    import parity_util as pu
    cfg = wl.make_config("c5g", n_segments=3000)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=1 << 20)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("c5g-3k", rep)
    assert rep["matched"] == rep["hits_oracle"] >= 0.999 * (g["counters"]["generated"] - g["counters"]["upward"])


@pytest.mark.parametrize("shift", [0, 1, 2, 3])
def test_dense_output_without_ids_equals_with_ids(c8, shift):
    """The launch bench.py times for the HBM roofline passes no id side buffer and takes the dense loop's fast path;
    its records must be the same set, bit for bit, as those of the general path that the parity tests check by id.
    The region starts 0..3 records into the buffer, so the 16-byte body of every block sees each alignment."""
    import parity_util as pu
    cfg = wl.make_config("c5g", n_segments=3000)
    a = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=1 << 20, region_shift=shift)
    b = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=1 << 20, with_ids=False, region_shift=shift)
    assert a["counters"] == b["counters"] and len(a["records"]) == len(b["records"]) > 400_000
    assert np.array_equal(a["tallies"]["hits"], b["tallies"]["hits"])
    assert np.allclose(a["tallies"]["sum_w"], b["tallies"]["sum_w"], rtol=1e-6)
    fields = ["x", "y", "cx", "cy", "t", "lam", "w"]
    ra = np.stack([a["records"][f] for f in fields], axis=1).view(np.uint32)
    rb = np.stack([b["records"][f] for f in fields], axis=1).view(np.uint32)
    ra = ra[np.lexsort(ra.T[::-1])]
    rb = rb[np.lexsort(rb.T[::-1])]
    assert np.array_equal(ra, rb)


def test_dense_hits_several_telescopes_misaligned_regions(c8):
    """Large overlapping spheres: most warp iterations are dense, the lanes of a warp hit different telescopes,
    a photon hits several; odd capacities make every region start off a 16-byte boundary."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=3000)
    cfg["telescopes"] = np.array([[0.0, 0.0, 2000.0, 300.0], [40.0, -30.0, 2000.0, 150.0],
                                  [-60.0, 20.0, 2000.0, 80.0], [10.0, 90.0, 2000.0, 6.0]], dtype=np.float32)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=(1 << 20) + 3)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("dense-4tel", rep)
    assert rep["matched"] > 0.5 * g["counters"]["generated"]
    t = pu.gpu_run(cfg, c8.MODE_TALLY)
    assert np.array_equal(t["tallies"]["hits"], g["tallies"]["hits"])


def test_dense_output_capacity_overflow(c8):
    """Accept-all output into a region that is too small: exactly `capacity` records, each a true hit, rest counted."""
    import parity_util as pu
    cfg = wl.make_config("c5g", n_segments=3000)
    cap = 100_001
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=cap)
    o = pu.oracle_run(cfg)
    assert g["counters"]["records"] == cap == len(g["records"])
    assert g["counters"]["dropped"] == g["counters"]["hits"] - cap > 0
    ids = g["records"]["id"]
    assert len(np.unique(ids)) == cap
    pos = np.searchsorted(o["records"]["id"], ids)
    assert np.array_equal(o["records"]["id"][pos], ids)
    assert np.max(np.abs(o["records"]["x"][pos] - g["records"]["x"].astype(np.float64))) < pu.TOL_XY_M
    assert np.max(np.abs(o["records"]["t"][pos] - g["records"]["t"].astype(np.float64))) < pu.TOL_T_NS


@pytest.mark.parametrize("name,n", [("c1", None), ("c2", 50_000), ("c4", 100_000), ("c3b", 50_000)])
def test_segment_culling_changes_nothing(c8, name, n):
    """C8OPT_FLAG_CULL (PAPER.md:57 in its exact form): the culled run must give the same records, bit for bit, and
    the same tallies as the full run; only the work differs."""
    import parity_util as pu
    cfg = wl.make_config(name) if n is None else wl.make_config(name, n_segments=n)
    a = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_CULL)
    b = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    assert np.array_equal(a["counts"], b["counts"])
    assert a["counters"]["generated"] == b["counters"]["generated"]
    assert np.array_equal(a["tallies"]["hits"], b["tallies"]["hits"])
    assert np.array_equal(a["records"]["id"], b["records"]["id"]) and np.array_equal(a["records"]["tel"], b["records"]["tel"])
    for f in ("x", "y", "cx", "cy", "t", "lam", "w"):
        assert np.array_equal(a["records"][f], b["records"][f])
    assert np.allclose(a["tallies"]["sum_w"], b["tallies"]["sum_w"], rtol=1e-12)
    assert a["counters"]["culled"] == 0
    frac = b["counters"]["culled"] / max(1, b["counters"]["generated"])
    print(f"[cull {name}] culled {b['counters']['culled']} of {b['counters']['generated']} bunches ({100 * frac:.1f} %)")
    if name != "c3b":
        assert frac > 0.2          # fluorescence (c3b) is never culled


@pytest.mark.parametrize("name,n,flag,deg", [("c2", 50_000, "centre", 6.0), ("c2", 50_000, "telescopes", 2.0), ("c4", 60_000, "centre", 4.0),
                                             ("c4", 60_000, "telescopes", 1.5), ("c1", None, "centre", 1.0)])
def test_angular_particle_cut(c8, name, n, flag, deg):
    """C8OPT_FLAG_CUT_CENTRE / _TELESCOPES (the paper's own lossy cut, R29) against the oracle with the same
    cut: the same segments are cut on both sides (decided in double, same operation order), so counts, tallies and
    records are compared exactly as without it; the bunches of the cut segments are reported."""
    import parity_util as pu
    cfg = wl.make_config(name) if n is None else wl.make_config(name, n_segments=n)
    full = pu.gpu_run(cfg, c8.MODE_TALLY)
    fl = c8.FLAG_CUT_CENTRE if flag == "centre" else c8.FLAG_CUT_TELESCOPES
    cfg["params"] = dict(cfg["params"], flags=fl, cut_angle=float(np.radians(deg)))
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o, check_upward=False)
    _report(f"cut-{name}-{flag}-{deg}", rep)
    assert g["counters"]["culled"] == int(o["counters"][7]) > 0
    lost = 1.0 - g["counters"]["hits"] / full["counters"]["hits"]
    print(f"[cut {name} {flag} {deg} deg] bunches skipped {g['counters']['culled'] / g['counters']['generated']:.3f}, hits lost {lost:.4f}")
    assert 0.0 <= lost < 1.0 and rep["matched"] > 50


def test_segment_culling_non_coplanar_big_spheres(c8):
    """Culling with telescopes of different sizes at different altitudes, against the oracle (which never culls)."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=30_000)
    tel = cfg["telescopes"].copy()
    tel[:, 2] += np.array([0.0, 35.0, -20.0, 60.0], dtype=np.float32)
    tel[:, 3] = np.array([6.0, 12.0, 25.0, 40.0], dtype=np.float32)
    cfg["telescopes"] = tel
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_CULL)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o, check_upward=False)
    _report("cull-noncoplanar", rep)
    assert g["counters"]["culled"] > 0 and rep["matched"] > 1000


@pytest.mark.parametrize("name,n,r_max,n_bins,core", [("c2", 30_000, 500.0, 1000, (0.0, 0.0)),
                                                      ("c4", 20_000, 2000.0, 500, (15.0, -25.0)),
                                                      ("c1", 2_000, 300.0, 64, (0.0, 0.0)),
                                                      ("c2", 1, 500.0, 1024, (0.0, 0.0))])
def test_ground_histogram(c8, name, n, r_max, n_bins, core):
    """C8OPT_MODE_GROUND_HIST (Fig. 3): radial photon density and arrival-time profile on the
    observation level against the oracle's binning of the accept-all plane records."""
    import oracle
    import parity_util as pu
    cfg = wl.make_config(name, n_segments=n)
    g = pu.gpu_hist(cfg, core, r_max, n_bins, chunks=2 if n > 1 else 1)
    o = oracle.ground_histogram(cfg["atmosphere"], cfg["segments"], cfg["params"], core, r_max, n_bins, threads=pu.n_threads())
    rep = pu.compare_hist(g, o, r_max, n_bins)
    print(f"[hist {name}-{n}] " + " ".join(f"{k}={v}" for k, v in rep.items()))
    assert g["counters"]["generated"] == int(o["counts"].astype(np.uint64).sum())
    if n > 1000:
        assert rep["bins_ge50"] > 20


def test_ground_histogram_needs_configuration_and_resets(c8):
    import torch
    cfg = wl.make_config("c1", n_segments=500)
    par = dict(cfg["params"], mode=c8.MODE_GROUND_HIST)
    ctx = c8.Context(cfg["atmosphere"])
    d_seg = torch.from_numpy(cfg["segments"].view(np.uint8).reshape(-1, 48).copy()).to("cuda:0")
    with pytest.raises(c8.C8optError):
        ctx.propagate_segments(d_seg, par, n=500, first_segment_id=0)          # no histogram configured
    ctx.set_ground_histogram(0.0, 0.0, 300.0, 30)
    with pytest.raises(c8.C8optError):
        ctx.propagate_segments(d_seg, dict(par, flags=c8.FLAG_CULL), n=500, first_segment_id=0)
    ctx.propagate_segments(d_seg, par, n=500, first_segment_id=0)
    a, over_a, cnt = ctx.read_ground_histogram()
    assert int(a["n"].sum()) + over_a == cnt["generated"] - cnt["upward"] == cnt["hits"] > 1000
    ctx.propagate_segments(d_seg, par, n=500, first_segment_id=0)                # accumulates
    b, over_b, _ = ctx.read_ground_histogram()
    assert np.array_equal(b["n"], 2 * a["n"]) and over_b == 2 * over_a
    ctx.reset_tallies()
    c, over_c, _ = ctx.read_ground_histogram()
    assert int(c["n"].sum()) == 0 and over_c == 0
    ctx.close()


def test_no_grid_possible_many_overlapping_spheres(c8):
    """12 large overlapping spheres: more than 4 reach discs cover every cell, no grid can be built, and every photon
    takes the wide test (TEL_GLOBAL), one photon per lane against all telescopes."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=1500)
    rng = np.random.Generator(np.random.PCG64(5))
    tel = np.zeros((12, 4), dtype=np.float32)
    tel[:, 0] = rng.uniform(-40, 40, 12); tel[:, 1] = rng.uniform(-40, 40, 12)
    tel[:, 2] = 2000.0 + rng.uniform(-10, 10, 12); tel[:, 3] = rng.uniform(30, 60, 12)
    cfg["telescopes"] = tel
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("no-grid-12tel", rep)
    assert rep["matched"] > 10000


def test_large_array_1600_telescopes(c8):
    """A 40 x 40 array (more than the 128 telescopes tallied in shared memory, more than culling tests one by one):
    global-memory tallies, grid lookup, bounding-sphere culling only."""
    import parity_util as pu
    cfg = wl.make_config("c4", n_segments=3000)
    cfg["telescopes"] = wl.telescopes_grid(n=40, spacing=35.0, r=6.0)
    a = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=1 << 15)
    o = pu.oracle_run(cfg, record_capacity=1 << 23)
    rep = pu.compare(cfg, a, o)
    _report("grid-1600tel", rep)
    assert rep["matched"] > 10000
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_CULL)
    b = pu.gpu_run(cfg, c8.MODE_TALLY)
    assert np.array_equal(a["tallies"]["hits"], b["tallies"]["hits"])


def test_eight_layers_and_segments_across_layer_boundaries(c8):
    """8 atmosphere layers (the maximum) with long segments, so that many tracks cross a layer boundary and the
    photons' layer is looked up per photon instead of taken from the frame."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=1500)
    l5 = cfg["atmosphere"]["layers"]
    # split the three lowest layers in two: same coefficients on both sides, so T(h) is unchanged but the index is not
    layers = [l5[0], (2000.5, l5[0][1], l5[0][2], l5[0][3]), l5[1], (7000.0, l5[1][1], l5[1][2], l5[1][3]),
              l5[2], (25000.0, l5[2][1], l5[2][2], l5[2][3]), l5[3], l5[4]]
    cfg["atmosphere"] = dict(cfg["atmosphere"], layers=layers)
    seg = cfg["segments"]
    seg["length"] = np.minimum(seg["length"] * 40.0, (seg["z0"] - 2000.0) / np.maximum(-seg["dz"], 0.05) * 0.999).astype(np.float32)
    cfg["telescopes"] = np.array([[0.0, 0.0, 2000.0, 25.0], [80.0, -40.0, 2000.0, 12.0]], dtype=np.float32)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("8-layers", rep)
    assert rep["matched"] > 5000


def test_one_segment_with_a_million_bunches(c8):
    """The photon index of one emitter far beyond a tile's usual size (n_b ~ 1.5e6 < 2^24): index arithmetic, the
    24-bit photon index of the record id, one warp share spanning a single emitter."""
    import parity_util as pu
    cfg = wl.make_config("c1", n_segments=3)
    seg = cfg["segments"]
    seg["x0"], seg["y0"], seg["z0"] = 0.0, 0.0, 9000.0
    seg["dx"], seg["dy"], seg["dz"] = 0.0, 0.0, -1.0
    seg["length"], seg["gamma"] = np.float32(50.0), np.float32(1e5)
    seg["t0"] = -(seg["z0"] - 2000.0) / 0.299792458
    cfg["params"] = dict(cfg["params"], bunch_size=5e-4)
    cfg["telescopes"] = np.array([[70.0, 60.0, 2000.0, 8.0]], dtype=np.float32)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("1e6-bunches", rep)
    assert g["counts"][:, 0].max() > 1_000_000 and rep["matched"] > 1000


@pytest.mark.parametrize("name,n", [("c1", None), ("c2", 50_000), ("c4", 60_000)])
def test_refraction_corrections(c8, name, n):
    """C8OPT_FLAG_REFRACT (R27): arrival point and direction corrected to first order on the GPU against
    the oracle with the same flag; the corrections are visible (the records differ from the straight-line run)."""
    import parity_util as pu
    cfg = wl.make_config(name) if n is None else wl.make_config(name, n_segments=n)
    plain = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_REFRACT)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report(f"refract-{name}", rep)
    assert rep["matched"] > 100
    common, ia, ib = np.intersect1d(plain["records"]["id"] * 4096 + plain["records"]["tel"],
                                    g["records"]["id"] * 4096 + g["records"]["tel"], return_indices=True)
    shift = np.hypot(plain["records"]["x"][ia] - g["records"]["x"][ib], plain["records"]["y"][ia] - g["records"]["y"][ib])
    print(f"[refract-{name}] median shift of the arrival point {np.median(shift):.4f} m, max {shift.max():.3f} m")
    assert len(common) > 0.9 * len(g["records"]) and 1e-3 < np.median(shift) < 1.0


@pytest.mark.parametrize("layout", ["4 telescopes", "4 x 4 grid"])
def test_refraction_inclined_showers(c8, layout):
    """C8OPT_FLAG_REFRACT beyond 60 degrees: half of the tracks are tilted to zenith angles of 58 .. 78 degrees and aimed
    at the array, so that photons on both sides of |v_z| = 0.5 (the steep candidate grid's limit) and of the cut-off
    |v_z| = 0.25 (R27) are corrected / kept and tested with the right slack, with and without culling."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=40_000)
    seg = cfg["segments"]
    rng = np.random.Generator(np.random.PCG64(321))
    idx = np.arange(0, len(seg), 2)
    zen = np.radians(rng.uniform(58.0, 78.0, len(idx)))
    az = rng.uniform(0.0, 2.0 * np.pi, len(idx))
    d = np.stack([np.sin(zen) * np.cos(az), np.sin(zen) * np.sin(az), -np.cos(zen)], axis=1)
    d = d.astype(np.float32).astype(np.float64)
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    h = seg["z0"][idx].astype(np.float64) - 2000.0
    aim = rng.normal(0.0, 30.0, (len(idx), 2))
    seg["x0"][idx] = aim[:, 0] - h * d[:, 0] / -d[:, 2]
    seg["y0"][idx] = aim[:, 1] - h * d[:, 1] / -d[:, 2]
    seg["dx"][idx], seg["dy"][idx], seg["dz"][idx] = d[:, 0], d[:, 1], d[:, 2]
    seg["length"][idx] = np.minimum(seg["length"][idx], 0.5 * h / -d[:, 2]).astype(np.float32)
    seg["t0"][idx] = (-(h / -d[:, 2]) / 0.299792458).astype(np.float32)
    if layout == "4 telescopes":
        tel = cfg["telescopes"].copy(); tel[:, 3] = 25.0
    else:
        tel = wl.telescopes_grid(n=4, spacing=60.0, r=12.0)
    cfg["telescopes"] = tel
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_REFRACT)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report(f"refract-inclined {layout}", rep)
    vz = -np.sqrt(np.maximum(0.0, 1.0 - g["records"]["cx"].astype(np.float64) ** 2 - g["records"]["cy"].astype(np.float64) ** 2))
    n_mid, n_flat = int(((vz > -0.5) & (vz <= -0.25)).sum()), int((vz > -0.25).sum())
    print(f"[refract-inclined {layout}] records with 0.25 <= |v_z| < 0.5: {n_mid}, flatter: {n_flat}")
    assert rep["matched"] > 5000 and n_mid > 500 and n_flat > 50
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_REFRACT | c8.FLAG_CULL)
    gc = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    assert np.array_equal(gc["records"]["id"], g["records"]["id"]) and np.array_equal(gc["records"]["x"], g["records"]["x"])
    assert gc["counters"]["culled"] > 0


def test_refraction_with_culling_non_coplanar(c8):
    """Both flags, spheres of different sizes at different altitudes: the culling test carries the refraction reach."""
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=30_000)
    tel = cfg["telescopes"].copy()
    tel[:, 2] += np.array([0.0, 35.0, -20.0, 60.0], dtype=np.float32)
    tel[:, 3] = np.array([6.0, 12.0, 25.0, 40.0], dtype=np.float32)
    cfg["telescopes"] = tel
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_REFRACT | c8.FLAG_CULL)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o, check_upward=False)
    _report("refract-cull-noncoplanar", rep)
    assert g["counters"]["culled"] > 0 and rep["matched"] > 1000


def test_refraction_in_ground_histogram(c8):
    import oracle
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=20_000)
    cfg["params"] = dict(cfg["params"], flags=c8.FLAG_REFRACT)
    g = pu.gpu_hist(cfg, (0.0, 0.0), 500.0, 500)
    o = oracle.ground_histogram(cfg["atmosphere"], cfg["segments"], cfg["params"], (0.0, 0.0), 500.0, 500, threads=pu.n_threads())
    rep = pu.compare_hist(g, o, 500.0, 500)
    print("[hist refract] " + " ".join(f"{k}={v}" for k, v in rep.items()))


def test_fluorescence_beamed_at_the_array(c8):
    """fl_beam_telescope = C8OPT_BEAM_ARRAY (R28): per-segment cone around the whole array with the photon
    number scaled; counts bit-exact against the oracle, records compared; far array (every segment beamed) and the
    c4 array (segments inside the array's sphere stay isotropic)."""
    import parity_util as pu
    cfg = wl.make_config("c3a", n_segments=100_000)
    tel = wl.telescopes_square().copy()
    tel[:, 0] += 2500.0; tel[:, 1] -= 1500.0        # 2.9 km off the shower axis
    tel[:, 3] = 12.0
    cfg["telescopes"] = tel
    cfg["params"] = dict(cfg["params"], fl_beam_telescope=c8.BEAM_ARRAY, fl_yield=4000.0)
    # (tracks a few metres above the telescopes' plane reach them 2.9 km away along nearly horizontal rays, v_z ~ 0.003:
    # those photons are evaluated in double on the GPU, flat_hit_f64)
    iso_generated = int(np.ceil(4000.0 * cfg["segments"]["dE"].astype(np.float64)).sum())
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("beam-array-far", rep)
    assert rep["matched"] > 300          # (cones of tracks just above the telescopes' plane reach above the horizontal: upward > 0)
    assert g["counters"]["generated"] < 1e-3 * iso_generated          # the paper's gain: the number of photons

    cfg = wl.make_config("c4", n_segments=20_000)
    cfg["params"] = dict(cfg["params"], fl_beam_telescope=c8.BEAM_ARRAY, fl_yield=400.0)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("beam-array-c4", rep)
    fl = rep  # both processes: compare() has already checked the per-process counts
    assert rep["matched"] > 20000


@pytest.mark.parametrize("name,n,mode_out", [("c2", 40_000, True), ("c4", 30_000, True), ("c5g", 2_000, True), ("c4", 30_000, False)])
def test_runs_are_repeatable(c8, name, n, mode_out):
    """Three runs of the same input: identical hit counts and (after sorting by id) bit-identical records -- the queues,
    staging areas and round flushes leave no room for a race to change a result; only the fp64 sums may differ in
    their last bits (atomic order)."""
    import parity_util as pu
    cfg = wl.make_config(name, n_segments=n)
    mode = c8.MODE_OUTPUT if mode_out else c8.MODE_TALLY
    runs = [pu.gpu_run(cfg, mode, capacity_per_tel=1 << 20) for _ in range(3)]
    for other in runs[1:]:
        assert np.array_equal(runs[0]["tallies"]["hits"], other["tallies"]["hits"])
        assert np.array_equal(runs[0]["counts"], other["counts"])
        assert runs[0]["counters"] == other["counters"]
        assert np.allclose(runs[0]["tallies"]["sum_w"], other["tallies"]["sum_w"], rtol=1e-12)
        if mode_out:
            for f in ("id", "tel", "x", "y", "cx", "cy", "t", "lam", "w"):
                assert np.array_equal(runs[0]["records"][f], other["records"][f])


def test_config5_full_size_one_percent_block(c8):
    """configs[4] at its full size (10^7 segments, photon-output mode, the launch bench.py times): the records of a
    contiguous 1 % block of segments, found by their ids among the 6.7e6 records of the run, against the oracle run on
    that block alone (its random streams are keyed by the global segment ids)."""
    import parity_util as pu
    cfg = wl.make_config("c5")
    lo, n_blk = 5_000_000, 100_000
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT, capacity_per_tel=2_500_000)
    assert g["counters"]["dropped"] == 0 and g["counters"]["records"] == g["counters"]["hits"] > 6_000_000
    import oracle
    o = oracle.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"][lo:lo + n_blk], cfg["params"], first_id=lo,
                   want_counts=True, record_capacity=1 << 20, threads=pu.n_threads())
    assert np.array_equal(g["counts"][lo:lo + n_blk], o["counts"])                      # (a) bit-exact counts
    gr = g["records"]
    seg_of = gr["id"] >> 25
    gb = gr[(seg_of >= lo) & (seg_of < lo + n_blk)]
    orr = o["records"]
    orr = orr[np.lexsort((orr["tel"], orr["id"]))]
    gk = gb["id"].astype(np.uint64) * 16 + gb["tel"].astype(np.uint64)
    ok = orr["id"].astype(np.uint64) * 16 + orr["tel"].astype(np.uint64)
    common, ia, ib = np.intersect1d(gk, ok, return_indices=True)
    assert len(gk) + len(ok) - 2 * len(common) <= 3 and len(common) > 50_000             # (b) at most a few edge flips ...
    blk_cfg = dict(cfg, segments=cfg["segments"][lo:lo + n_blk])
    for key in np.concatenate([np.setdiff1d(gk, ok), np.setdiff1d(ok, gk)]):            # ... each within 5 mm of the rim (R22)
        hit, b, R, _ = pu.oracle_impact(blk_cfg, int(key) >> 4, int(key) & 15, first_id=lo)
        print(f"[parity c5-full-1pct] flip photon={int(key) >> 4:#x} tel={int(key) & 15} b-R={b - R:+.3e} m")
        assert abs(b - R) < pu.TOL_FLIP_M
    a, b = gb[ia], orr[ib]
    assert np.max(np.abs(a["x"] - b["x"])) <= pu.TOL_XY_M and np.max(np.abs(a["y"] - b["y"])) <= pu.TOL_XY_M      # (c)
    assert np.max(np.abs(a["cx"] - b["cx"])) <= 1e-5 and np.max(np.abs(a["cy"] - b["cy"])) <= 1e-5
    assert np.max(np.abs(a["t"] - b["t"])) <= pu.TOL_T_NS                                                        # (d)
    assert np.max(np.abs(a["lam"] - b["lam"]) / b["lam"]) <= pu.TOL_LAM_REL
    print(f"[parity c5-full-1pct] records_total={len(gr)} block_gpu={len(gk)} block_oracle={len(ok)} matched={len(common)} "
          f"max_dxy_m={max(np.max(np.abs(a['x'] - b['x'])), np.max(np.abs(a['y'] - b['y']))):.3e} "
          f"max_dt_ns={np.max(np.abs(a['t'] - b['t'])):.3e}")


def test_config4_full_size_tally(c8):
    """configs[3] at its full size (10^7 segments, 100 telescopes, both processes, transmission table) in the launch
    configuration bench.py times (tally mode): per-segment counts of both processes bit-exact, per-telescope hits and
    weight sums against the oracle's (about a minute of host time on 16 cores)."""
    import parity_util as pu
    cfg = wl.make_config("c4")
    g = pu.gpu_run(cfg, c8.MODE_TALLY)
    o = pu.oracle_run(cfg, record_capacity=0)
    rep = pu.compare(cfg, g, o, check_records=False)
    _report("c4-full", rep)
    assert g["counters"]["generated"] > 2_000_000_000 and g["counters"]["hits"] > 10_000_000
    d = np.abs(g["tallies"]["hits"].astype(np.int64) - o["tallies"]["hits"].astype(np.int64))
    print(f"[parity c4-full] per-telescope hit differences: max {d.max()}, total {d.sum()} of {int(o['tallies']['hits'].sum())}")
    assert d.max() <= 3


@pytest.mark.parametrize("name,n,B", [("c2", 40_000, 8.0), ("c4", 30_000, 3.5), ("c3b", 100_000, 2.0)])
def test_bunch_size_above_one(c8, name, n, B):
    """R1 with B > 1: n_b = ceil(mu / B) bunches of weight mu / n_b <= B; counts bit-exact, records and weights compared."""
    import parity_util as pu
    cfg = wl.make_config(name, n_segments=n)
    cfg["params"] = dict(cfg["params"], bunch_size=B)
    if name == "c2":
        cfg["telescopes"][:, 3] = 15.0
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report(f"bunch-{name}-{B}", rep)
    w = g["records"]["w"]
    assert rep["matched"] > 100 and w.max() <= B * (1 + 1e-6)
    if name != "c3b":                       # (beamed bunches carry the factor Omega / 4 pi = 3e-4)
        assert w.max() > 1.0


def test_full_tile_of_emitters_near_the_bunch_limit(c8):
    """the tile's photon index space is 32 bits wide.  300 segments of ~1.6e7 bunches each (the limit is 2^24 - 1)
    fill one tile of 255 segments with 4.1e9 photon slots (255 x 2^24 < 2^32) and start a second one; counts bit-exact,
    tallies against the oracle (about half a minute of host time)."""
    import parity_util as pu
    cfg = wl.make_config("c1", n_segments=300)
    seg = cfg["segments"]
    seg["x0"], seg["y0"], seg["z0"] = 0.0, 0.0, 9000.0
    seg["dx"], seg["dy"], seg["dz"] = 0.0, 0.0, -1.0
    seg["length"], seg["gamma"] = np.float32(50.0), np.float32(1e5)
    seg["z0"] += np.arange(300, dtype=np.float32)                     # (distinct emitters)
    seg["t0"] = -(seg["z0"] - 2000.0) / 0.299792458
    cfg["params"] = dict(cfg["params"], bunch_size=4.7e-5)
    cfg["telescopes"] = np.array([[70.0, 60.0, 2000.0, 8.0]], dtype=np.float32)
    g = pu.gpu_run(cfg, c8.MODE_TALLY)
    assert g["counts"][:, 0].min() > 12_000_000 and g["counts"][:, 0].max() < (1 << 24)
    assert g["counters"]["generated"] > 4_000_000_000
    o = pu.oracle_run(cfg, record_capacity=0)
    rep = pu.compare(cfg, g, o, check_records=False)
    _report("255-big-emitters", rep)


def test_many_flat_photons_in_one_tile(c8):
    """Isotropic fluorescence at 250 photons per segment beside a 150 m sphere 300 m away: every tile sets tens of flat
    (|v_z| < 0.05) photons aside for its double-precision pass, some of them so flat that they cross the telescope's plane
    hundreds of kilometres away (the fp32 record then carries half an ulp of rounding on top of the 1 cm)."""
    import parity_util as pu
    cfg = wl.make_config("c3a", n_segments=3000)
    cfg["telescopes"] = np.array([[300.0, 0.0, 2000.0, 150.0]], dtype=np.float32)
    cfg["params"] = dict(cfg["params"], fl_yield=250.0)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("flat-many", rep)
    assert rep["flat_records_two_component_direction"] > 150 and rep["matched"] > 10_000


@pytest.mark.parametrize("name,n,b", [("c2", 40_000, 5670.0), ("c1", None, 5670.0), ("c4", 60_000, 5670.0), ("c2", 30_000, 60_000.0)])
def test_wavelength_dependent_refractive_index(c8, name, n, b):
    """R30 (PAPER.md:45 with n(lambda)): n - 1 = eta(h) (1 + b / lambda^2).  The yield is the Simpson integral over the
    band (bunch counts bit-exact), every photon leaves at the Cherenkov angle of its own wavelength with the weight
    factor sin^2 / <sin^2>; records against the oracle on one telescope, on configs[1]'s array, with both processes
    on configs[3]'s array, and with a dispersion ten times that of air (thresholds inside the band for many emitters)."""
    import parity_util as pu
    cfg = wl.make_config(name, n_segments=n)
    base = pu.gpu_run(cfg, c8.MODE_TALLY)
    cfg["params"] = dict(cfg["params"], cauchy_b=b)
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report(f"dispersion-{name}-b{b:g}", rep)
    assert rep["matched"] > 100
    # more light than with the long-wavelength n (n grows towards the blue), and tally mode sees the same photons
    assert g["counters"]["generated"] > base["counters"]["generated"]
    t = pu.gpu_run(cfg, c8.MODE_TALLY)
    assert np.array_equal(t["tallies"]["hits"], g["tallies"]["hits"])
    assert np.allclose(t["tallies"]["sum_w"], g["tallies"]["sum_w"], rtol=1e-12)
    assert t["counters"]["generated"] == g["counters"]["generated"] and t["counters"]["upward"] == g["counters"]["upward"]


def test_wavelength_dependent_refractive_index_argument_errors(c8):
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=1000)
    for over, msg in ((dict(cauchy_b=-1.0), "cauchy_b_nm2"), (dict(cauchy_b=5670.0, flags=c8.FLAG_CULL), "culling")):
        cfg["params"] = dict(cfg["params"], **over)
        with pytest.raises(c8.C8optError) as ei:
            pu.gpu_run(cfg, c8.MODE_TALLY)
        assert ei.value.code == -1 and msg in str(ei.value)
        cfg["params"].pop("flags", None)


def test_wavelength_dependent_refractive_index_with_refraction_and_cut(c8):
    """R30 together with the refraction corrections (R27) and the paper's angular cut (R29), through the host-segment
    entry point; and through c8opt_tally_static (same tallies as the context path)."""
    import torch
    import parity_util as pu
    cfg = wl.make_config("c2", n_segments=30_000)
    cfg["params"] = dict(cfg["params"], cauchy_b=5670.0, flags=c8.FLAG_REFRACT | c8.FLAG_CUT_TELESCOPES, cut_angle=float(np.radians(5.0)))
    g = pu.gpu_run(cfg, c8.MODE_OUTPUT, host_segments=True)
    o = pu.oracle_run(cfg)
    rep = pu.compare(cfg, g, o)
    _report("dispersion-refract-cut-c2", rep)
    assert rep["matched"] > 100 and g["counters"]["culled"] > 0
    dev = torch.device("cuda:0")
    n = len(cfg["segments"])
    d_seg = torch.from_numpy(cfg["segments"].view(np.uint8).reshape(n, 48).copy()).to(dev)
    tau = cfg["atmosphere"].get("tau")
    d_tau = None if tau is None else torch.from_numpy(np.ascontiguousarray(tau, dtype=np.float32)).to(dev)
    n_tel = len(cfg["telescopes"])
    d_tal = torch.zeros((n_tel, 3), dtype=torch.int64, device=dev)
    d_cnt = torch.zeros(8, dtype=torch.int64, device=dev)
    c8.tally_static(cfg["atmosphere"], cfg["telescopes"], d_seg, dict(cfg["params"], mode=c8.MODE_TALLY), d_tal, d_cnt, d_tau=d_tau, n=n)
    torch.cuda.synchronize()
    tallies = d_tal.cpu().numpy().view(np.uint8).reshape(-1).view(c8.TALLY_DTYPE)
    assert np.array_equal(tallies["hits"], g["tallies"]["hits"])
    assert np.allclose(tallies["sum_w"], g["tallies"]["sum_w"], rtol=1e-12)
