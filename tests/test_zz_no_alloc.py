"""GPU test of c8opt_tally_static, the entry point that allocates nothing (include/c8opt.h): its tallies and counters
against the context path's (c8opt_propagate_segments, tally mode) on the same seeded inputs, on two calls in a row that
share the library's static scratch array.  Collected last on purpose (the suite runs with pytest -x).

Run on the B200 box:  python -m pytest tests/test_zz_no_alloc.py -m gpu -x -q
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
    build()
    import paper_2309_15861_b200 as c8
    c8.lib()
    return c8


def _context_path(c8, cfg, par, d_seg, n):
    ctx = c8.Context(cfg["atmosphere"])
    ctx.add_telescopes(cfg["telescopes"])
    ctx.propagate_segments(d_seg, par, n=n)
    tallies, counters, _ = ctx.read_tallies()
    ctx.close()
    return tallies, counters


def _prepare(c8, name, n_segments, **over):
    import torch
    cfg = wl.make_config(name, n_segments=n_segments)
    seg = cfg["segments"]
    n = len(seg)
    dev = torch.device("cuda:0")
    d_seg = torch.from_numpy(seg.view(np.uint8).reshape(n, 48).copy()).to(dev)
    tau = cfg["atmosphere"].get("tau")
    d_tau = None if tau is None else torch.from_numpy(np.ascontiguousarray(tau, dtype=np.float32)).to(dev)
    par = dict(cfg["params"], mode=c8.MODE_TALLY, **over)
    n_tel = len(cfg["telescopes"])
    d_tal = torch.full((n_tel, 3), -1, dtype=torch.int64, device=dev)          # 24 bytes per telescope, pre-filled with junk
    d_cnt = torch.full((8,), -1, dtype=torch.int64, device=dev)
    return cfg, par, d_seg, n, d_tau, d_tal, d_cnt


def _static_path(c8, prep):
    import torch
    cfg, par, d_seg, n, d_tau, d_tal, d_cnt = prep
    c8.tally_static(cfg["atmosphere"], cfg["telescopes"], d_seg, par, d_tal, d_cnt, d_tau=d_tau, n=n)
    torch.cuda.synchronize()
    tallies = d_tal.cpu().numpy().view(np.uint8).reshape(-1).view(c8.TALLY_DTYPE).copy()
    counters = dict(zip(c8.COUNTER_NAMES, (int(c) for c in d_cnt.cpu().numpy().view(np.uint64))))
    return tallies, counters


def _same(a, b):
    (ta, ca), (tb, cb) = a, b
    assert ca == cb, (ca, cb)
    assert np.array_equal(ta["hits"], tb["hits"])
    assert ta["hits"].sum() > 0
    # the tolerance of the other invariance tests (test_batching_and_host_path_invariance): order of the fp64 atomics
    assert np.allclose(ta["sum_w"], tb["sum_w"], rtol=1e-12)
    assert np.allclose(ta["sum_wt"], tb["sum_wt"], rtol=1e-12)


def test_static_entry_point_equals_context_path_two_calls_in_a_row(c8):
    """Call 1: configs[1]'s array (4 telescopes, transmission table, 50 000 segments); call 2, straight after it on the
    same stream: configs[0] (one telescope, single layer, no table) -- the scratch of call 1 must not leak into call 2
    -- and call 3 the first again, with culling and the refraction corrections."""
    import torch
    p1 = _prepare(c8, "c2", 50_000)
    p2 = _prepare(c8, "c1", None)
    p3 = _prepare(c8, "c2", 50_000, flags=c8.FLAG_CULL | c8.FLAG_REFRACT)
    want = [_context_path(c8, p[0], p[1], p[2], p[3]) for p in (p1, p2, p3)]
    got1 = _static_path(c8, p1)
    got2 = _static_path(c8, p2)
    got3 = _static_path(c8, p3)
    for got, exp in zip((got1, got2, got3), want):
        _same(got, exp)
    # two calls back to back without a host synchronisation between them, and no device memory taken by either
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for p in (p1, p2):
        c8.tally_static(p[0]["atmosphere"], p[0]["telescopes"], p[2], p[1], p[5], p[6], d_tau=p[4], n=p[3])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    for p, exp in zip((p1, p2), want):
        tallies = p[5].cpu().numpy().view(np.uint8).reshape(-1).view(c8.TALLY_DTYPE)
        assert np.array_equal(tallies["hits"], exp[0]["hits"])
        assert np.allclose(tallies["sum_w"], exp[0]["sum_w"], rtol=1e-12)


def test_static_entry_point_both_processes_and_empty_input(c8):
    import torch
    cfg = wl.make_config("c4", n_segments=20_000)
    cfg["telescopes"] = np.asarray(cfg["telescopes"])[:8]                       # the stated maximum
    n = len(cfg["segments"])
    dev = torch.device("cuda:0")
    d_seg = torch.from_numpy(cfg["segments"].view(np.uint8).reshape(n, 48).copy()).to(dev)
    tau = cfg["atmosphere"].get("tau")
    d_tau = None if tau is None else torch.from_numpy(np.ascontiguousarray(tau, dtype=np.float32)).to(dev)
    par = dict(cfg["params"], mode=c8.MODE_TALLY, fl_beam_telescope=-1)
    d_tal = torch.zeros((8, 3), dtype=torch.int64, device=dev)
    d_cnt = torch.zeros(8, dtype=torch.int64, device=dev)
    prep = (cfg, par, d_seg, n, d_tau, d_tal, d_cnt)
    _same(_static_path(c8, prep), _context_path(c8, cfg, par, d_seg, n))
    empty = (cfg, par, d_seg, 0, d_tau, d_tal, d_cnt)
    tallies, counters = _static_path(c8, empty)
    assert tallies["hits"].sum() == 0 and tallies["sum_w"].sum() == 0.0 and counters["generated"] == 0 and counters["segments"] == 0


def test_static_entry_point_rejects_what_it_cannot_hold(c8):
    import torch
    cfg = wl.make_config("c4", n_segments=1000)
    tel = np.asarray(cfg["telescopes"])
    assert len(tel) > c8.STATIC_MAX_TELESCOPES
    dev = torch.device("cuda:0")
    d_seg = torch.zeros((1000, 48), dtype=torch.uint8, device=dev)
    d_tal = torch.zeros((len(tel), 3), dtype=torch.int64, device=dev)
    par = dict(cfg["params"], mode=c8.MODE_TALLY)
    with pytest.raises(c8.C8optError) as ei:
        c8.tally_static(cfg["atmosphere"], tel, d_seg, par, d_tal)
    assert ei.value.code == -1 and "at most 8" in str(ei.value)
    with pytest.raises(c8.C8optError) as ei:
        c8.tally_static(cfg["atmosphere"], tel[:4], d_seg, dict(par, mode=c8.MODE_OUTPUT), d_tal)
    assert ei.value.code == -1 and "C8OPT_MODE_TALLY" in str(ei.value)
