"""ctypes front end of the fp64 CPU oracle (oracle/c8opt_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this package.  It
does not import, link or read anything of the CUDA path.

The C file is compiled on first use with plain gcc (-O2, no fast-math, no FMA
contraction) into oracle/liboracle.so.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "c8opt_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc; returns the path of the shared object."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fPIC", "-shared",
                               "-Wall", "-Wno-misleading-indentation", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class Layer(C.Structure):
    _fields_ = [("h_lo", C.c_double), ("a", C.c_double), ("b", C.c_double), ("c", C.c_double)]


class Atmosphere(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("layers", Layer * 8),
                ("eta0", C.c_double), ("rho0", C.c_double), ("h_obs", C.c_double),
                ("tau_nh", C.c_int), ("tau_nl", C.c_int),
                ("tau_h0", C.c_double), ("tau_dh", C.c_double), ("tau_l0", C.c_double), ("tau_dl", C.c_double),
                ("tau", C.POINTER(C.c_float))]


class Params(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("processes", C.c_uint32),
                ("lam1", C.c_double), ("lam2", C.c_double), ("bunch_size", C.c_double),
                ("fl_yield", C.c_double), ("fl_lam1", C.c_double), ("fl_lam2", C.c_double),
                ("fl_beam_telescope", C.c_int), ("fl_beam_halfangle", C.c_double), ("refract", C.c_int),
                ("cut_mode", C.c_int), ("cut_angle", C.c_double), ("cauchy_b", C.c_double)]


FLAG_REFRACT = 2      # the bit of params["flags"] that asks for the refraction corrections (R27)
FLAG_CUT_CENTRE = 4   # R29: angular particle cut against the experiment centre ...
FLAG_CUT_TELESCOPES = 8   # ... or against the nearest telescope; params["cut_angle"] in rad


class Frame(C.Structure):
    _fields_ = [("n_b", C.c_uint32), ("mu", C.c_double), ("w0", C.c_double),
                ("p0", C.c_double * 3), ("d", C.c_double * 3),
                ("L", C.c_double), ("t0", C.c_double), ("inv_beta_c", C.c_double),
                ("sin_c", C.c_double), ("cos_c", C.c_double),
                ("A", C.c_double * 3), ("M", (C.c_double * 3) * 3),
                ("one_minus_cos_ab", C.c_double), ("kind", C.c_int),
                ("disp_eta", C.c_double), ("disp_beta2", C.c_double), ("disp_mean", C.c_double)]


class Photon(C.Structure):
    _fields_ = [("e", C.c_double * 3), ("v", C.c_double * 3),
                ("t_e", C.c_double), ("lam", C.c_double), ("w", C.c_double)]


TALLY_DTYPE = np.dtype([("hits", "<u8"), ("sum_w", "<f8"), ("sum_wt", "<f8")])
RECORD_DTYPE = np.dtype([("x", "<f8"), ("y", "<f8"), ("cx", "<f8"), ("cy", "<f8"), ("t", "<f8"),
                         ("lam", "<f8"), ("w", "<f8"), ("id", "<u8"), ("tel", "<i4"), ("pad", "<i4")])
COUNTER_NAMES = ("segments", "generated", "upward", "hits", "records", "dropped", "invalid", "cut")


def lib():
    global _lib
    if _lib is None:
        # C8OPT_ORACLE_LIB: a build of the same source made elsewhere (the sanitizer test's ASan / UBSan build)
        L = C.CDLL(os.environ.get("C8OPT_ORACLE_LIB") or build())
        u32p, dp = C.POINTER(C.c_uint32), C.POINTER(C.c_double)
        L.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.orc_philox4x32_10.restype = None
        L.orc_uniform.argtypes = [C.c_uint32]
        L.orc_uniform.restype = C.c_double
        for name in ("orc_depth", "orc_density", "orc_refractivity"):
            f = getattr(L, name)
            f.argtypes = [C.POINTER(Atmosphere), C.c_double]
            f.restype = C.c_double
        L.orc_preamble.argtypes = [C.POINTER(Atmosphere), C.POINTER(Params), C.c_void_p, C.c_int, dp, C.POINTER(Frame)]
        L.orc_preamble.restype = C.c_int
        L.orc_make_photon.argtypes = [C.POINTER(Frame), C.POINTER(Params), C.c_uint64, C.c_uint32, C.c_int,
                                      C.POINTER(Photon)]
        L.orc_make_photon.restype = None
        L.orc_intersect.argtypes = [dp, dp, dp, dp, dp, dp, dp]
        L.orc_intersect.restype = C.c_int
        L.orc_arrival_time.argtypes = [C.POINTER(Atmosphere)] + [C.c_double] * 5
        L.orc_arrival_time.restype = C.c_double
        L.orc_optical_depth.argtypes = [C.POINTER(Atmosphere), C.c_double, C.c_double]
        L.orc_optical_depth.restype = C.c_double
        L.orc_transmission.argtypes = [C.POINTER(Atmosphere), C.c_double, C.c_double, C.c_double]
        L.orc_refraction.argtypes = [C.POINTER(Atmosphere), C.c_double, C.c_double, C.c_double,
                                     C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.orc_refraction.restype = None
        L.orc_array_sphere.argtypes = [C.POINTER(C.c_double), C.c_int, C.POINTER(C.c_double)]
        L.orc_array_sphere.restype = None
        L.orc_transmission.restype = C.c_double
        L.orc_run.argtypes = [C.POINTER(Atmosphere), dp, C.c_int, C.c_void_p, C.c_uint64, C.c_uint64,
                              C.POINTER(Params), C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint64,
                              C.POINTER(C.c_uint64)]
        L.orc_run.restype = None
        _lib = L
    return _lib


# ------------------------------------------------------------------ marshalling
def make_atmosphere(atm: dict) -> Atmosphere:
    a = Atmosphere()
    layers = atm["layers"]
    assert 1 <= len(layers) <= 8
    a.n_layers = len(layers)
    for i, (h_lo, aa, bb, cc) in enumerate(layers):
        a.layers[i] = Layer(h_lo, aa, bb, cc)
    a.eta0, a.rho0, a.h_obs = atm["eta0"], atm["rho0"], atm["h_obs"]
    tau = atm.get("tau")
    if tau is not None:
        tau = np.ascontiguousarray(tau, dtype=np.float32)
        a.tau_nh, a.tau_nl = tau.shape
        a.tau_h0, a.tau_dh, a.tau_l0, a.tau_dl = atm["tau_h0"], atm["tau_dh"], atm["tau_l0"], atm["tau_dl"]
        a.tau = tau.ctypes.data_as(C.POINTER(C.c_float))
        a._keep = tau
    else:
        a.tau_nh = a.tau_nl = 0
        a.tau = None
    return a


def make_params(p: dict) -> Params:
    return Params(int(p["seed"]), int(p["processes"]), p["lam1"], p["lam2"], p["bunch_size"],
                  p["fl_yield"], p["fl_lam1"], p["fl_lam2"], int(p["fl_beam_telescope"]), p["fl_beam_halfangle"],
                  1 if (int(p.get("flags", 0)) & FLAG_REFRACT) else 0,
                  2 if (int(p.get("flags", 0)) & FLAG_CUT_TELESCOPES) else 1 if (int(p.get("flags", 0)) & FLAG_CUT_CENTRE) else 0,
                  float(p.get("cut_angle", 0.0)), float(p.get("cauchy_b", 0.0)))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


# ------------------------------------------------------------------ small pieces (for the pins)
def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr])
    k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(x) for x in o]


def uniform(r: int) -> float:
    return lib().orc_uniform(int(r) & 0xFFFFFFFF)


def depth(atm: dict, h: float) -> float:
    return lib().orc_depth(C.byref(make_atmosphere(atm)), float(h))


def density(atm: dict, h: float) -> float:
    return lib().orc_density(C.byref(make_atmosphere(atm)), float(h))


def refractivity(atm: dict, h: float) -> float:
    return lib().orc_refractivity(C.byref(make_atmosphere(atm)), float(h))


def preamble(atm: dict, params: dict, segment, tag: int, beam_tel=None):
    """Returns (status, Frame) for one segment record (numpy void / 1-element array)."""
    seg = np.ascontiguousarray(segment).reshape(1)
    f = Frame()
    bt = np.ascontiguousarray(beam_tel, dtype=np.float64) if beam_tel is not None else np.zeros(4)
    st = lib().orc_preamble(C.byref(make_atmosphere(atm)), C.byref(make_params(params)),
                            seg.ctypes.data, int(tag), _dp(bt), C.byref(f))
    return st, f


BEAM_ARRAY = -2       # params["fl_beam_telescope"]: one emission cone around the whole array, photon number scaled (R28)


def array_sphere(telescopes) -> np.ndarray:
    """(centre_x, centre_y, centre_z, R_b) of R28: the sphere that holds every telescope sphere."""
    tel64 = np.ascontiguousarray(np.asarray(telescopes, dtype=np.float32).astype(np.float64).reshape(-1))
    out = np.zeros(4)
    lib().orc_array_sphere(_dp(tel64), len(tel64) // 4, _dp(out))
    return out


def make_photon(frame: Frame, params: dict, S: int, j: int, tag: int) -> Photon:
    ph = Photon()
    lib().orc_make_photon(C.byref(frame), C.byref(make_params(params)), int(S), int(j), int(tag), C.byref(ph))
    return ph


def intersect(e, v, tel):
    """Returns (hit, b2, s_c, s_pl, x, y)."""
    e = np.ascontiguousarray(e, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    t = np.ascontiguousarray(tel, dtype=np.float64)
    b2, sc, sp = C.c_double(), C.c_double(), C.c_double()
    xy = np.zeros(2)
    hit = lib().orc_intersect(_dp(e), _dp(v), _dp(t), C.byref(b2), C.byref(sc), C.byref(sp), _dp(xy))
    return bool(hit), b2.value, sc.value, sp.value, float(xy[0]), float(xy[1])


def arrival_time(atm: dict, e_z, c_z, v_z, s_pl, t_e) -> float:
    return lib().orc_arrival_time(C.byref(make_atmosphere(atm)), e_z, c_z, v_z, s_pl, t_e)


def refraction(atm: dict, e_z, c_z, v_z):
    """(dr [m], dtheta [rad]) of R27 for a ray from altitude e_z down to c_z with direction cosine v_z < 0."""
    dr, dth = C.c_double(0.0), C.c_double(0.0)
    lib().orc_refraction(C.byref(make_atmosphere(atm)), float(e_z), float(c_z), float(v_z), C.byref(dr), C.byref(dth))
    return dr.value, dth.value


def intersect_refracted(atm: dict, e, v, tel):
    """R10 / R11 with the corrections of R27.  Returns (hit, b2, s_c, s_pl, x, y, v_out[3])."""
    e = np.ascontiguousarray(e, dtype=np.float64)
    v = np.ascontiguousarray(v, dtype=np.float64)
    t = np.ascontiguousarray(tel, dtype=np.float64)
    b2, sc, sp = C.c_double(), C.c_double(), C.c_double()
    xy, vo = np.zeros(2), np.zeros(3)
    f = lib().orc_intersect_refracted
    f.argtypes = [C.POINTER(Atmosphere)] + [C.POINTER(C.c_double)] * 3 + [C.POINTER(C.c_double)] * 3 + [C.POINTER(C.c_double)] * 2
    f.restype = C.c_int
    hit = f(C.byref(make_atmosphere(atm)), _dp(e), _dp(v), _dp(t), C.byref(b2), C.byref(sc), C.byref(sp), _dp(xy), _dp(vo))
    return bool(hit), b2.value, sc.value, sp.value, float(xy[0]), float(xy[1]), vo


def particle_cut(p0, d, L, telescopes, mode: int, cut_angle: float) -> bool:
    """R29: is the Cherenkov segment (start p0, unit direction d, length L) cut?  mode 1 = angle to the
    experiment centre, 2 = smallest angle to a telescope."""
    tel = np.ascontiguousarray(np.asarray(telescopes, dtype=np.float32).astype(np.float64))
    centre = array_sphere(telescopes)
    f = lib().orc_particle_cut
    f.argtypes = [C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_double, C.POINTER(C.c_double), C.c_int,
                  C.POINTER(C.c_double), C.c_int, C.c_double]
    f.restype = C.c_int
    p0 = np.ascontiguousarray(p0, dtype=np.float64)
    d = np.ascontiguousarray(d, dtype=np.float64)
    return bool(f(_dp(p0), _dp(d), float(L), _dp(tel), len(tel), _dp(np.ascontiguousarray(centre[:3])), int(mode), float(cut_angle)))


def dispersion_integral(eta: float, beta2: float, b: float, x1: float, x2: float) -> float:
    """R30: int_{x2}^{x1} max(0, sin^2 theta_c(x)) dx by the oracle's 16-interval Simpson rule (x = 1 / lambda)."""
    f = lib().orc_dispersion_integral
    f.argtypes = [C.c_double] * 5
    f.restype = C.c_double
    return f(eta, beta2, b, x1, x2)


def optical_depth(atm: dict, h, lam) -> float:
    return lib().orc_optical_depth(C.byref(make_atmosphere(atm)), float(h), float(lam))


def transmission(atm: dict, h, lam, v_z) -> float:
    return lib().orc_transmission(C.byref(make_atmosphere(atm)), float(h), float(lam), float(v_z))


# ------------------------------------------------------------------ the whole path
def _run_range(atm, tel64, seg, first_id, par, want_counts, rec_cap):
    n = len(seg)
    n_tel = len(tel64) // 4
    counts = np.zeros((n, 2), dtype=np.uint32) if want_counts else None
    tallies = np.zeros(n_tel, dtype=TALLY_DTYPE)
    counters = np.zeros(8, dtype=np.uint64)
    records = np.zeros(rec_cap, dtype=RECORD_DTYPE) if rec_cap else None
    n_rec = C.c_uint64(0)
    lib().orc_run(C.byref(atm), _dp(tel64), n_tel, seg.ctypes.data, n, int(first_id), C.byref(par),
                  counts.ctypes.data if want_counts else None, tallies.ctypes.data, counters.ctypes.data,
                  records.ctypes.data if rec_cap else None, rec_cap, C.byref(n_rec))
    return counts, tallies, counters, (records[: n_rec.value] if rec_cap else None)


def run(atmosphere: dict, telescopes, segments, params: dict, first_id: int = 0, want_counts: bool = True,
        record_capacity: int = 0, threads: int = 1) -> dict:
    """Run the whole path over `segments` (global ids first_id + i).

    Splitting the segment range over threads is legal because the random stream
    is keyed by the global segment id; records are concatenated in segment
    order, tallies summed in range order.  Returns dict(counts, tallies,
    counters, records).  record_capacity is per call (split evenly per thread
    range is NOT done: each range gets the full capacity).
    """
    lib()
    atm = make_atmosphere(atmosphere)
    par = make_params(params)
    seg = np.ascontiguousarray(segments)
    assert seg.dtype.itemsize == 48
    tel64 = np.ascontiguousarray(np.asarray(telescopes, dtype=np.float32).astype(np.float64).reshape(-1))
    n = len(seg)
    threads = max(1, min(int(threads), n if n else 1))
    bounds = [n * i // threads for i in range(threads + 1)]
    jobs = [(bounds[i], bounds[i + 1]) for i in range(threads)]

    def work(j):
        lo, hi = j
        return _run_range(atm, tel64, seg[lo:hi], first_id + lo, par, want_counts, record_capacity)

    if threads == 1:
        parts = [work(jobs[0])]
    else:
        with ThreadPoolExecutor(threads) as ex:
            parts = list(ex.map(work, jobs))
    counts = np.concatenate([p[0] for p in parts]) if want_counts else None
    tallies = np.zeros(len(tel64) // 4, dtype=TALLY_DTYPE)
    counters = np.zeros(8, dtype=np.uint64)
    for p in parts:
        for name in ("hits", "sum_w", "sum_wt"):
            tallies[name] += p[1][name]
        counters += p[2]
    records = np.concatenate([p[3] for p in parts]) if record_capacity else None
    return dict(counts=counts, tallies=tallies, counters=counters, records=records)


# ------------------------------------------------------------------ ground-plane radial profile
HIST_DTYPE = np.dtype([("n", "<u8"), ("sum_w", "<f8"), ("sum_wt", "<f8")])


def ground_histogram(atmosphere: dict, segments, params: dict, core_xy, r_max: float, n_bins: int,
                     first_id: int = 0, threads: int = 1, record_capacity: int = 1 << 24) -> dict:
    """Radial intensity and timing profile on the observation level (section 3.1, Fig. 3a/3b:
    photon density and mean arrival time against the distance from the shower core; R26).

    Definition written out: every bunch that crosses the plane z = h_obs going down (R10 with an accept-all
    detector: a sphere of radius 1e9 m centred on the core at h_obs, so its record holds the crossing point
    relative to the core, R11, the arrival time, R8, and the weight, R17) falls into the bin
    floor(r / (r_max / n_bins)), r = sqrt(x^2 + y^2); bins hold {n, sum w, sum w t}; r >= r_max counts as overflow.
    Density = sum_w / annulus area and mean time = sum_wt / sum_w are formed by `profile()`.
    """
    tel = np.array([[float(core_xy[0]), float(core_xy[1]), float(atmosphere["h_obs"]), 1.0e9]], dtype=np.float32)
    res = run(atmosphere, tel, segments, params, first_id=first_id, want_counts=True,
              record_capacity=record_capacity, threads=threads)
    rec = res["records"]
    assert int(res["counters"][COUNTER_NAMES.index("dropped")]) == 0, "record_capacity too small for the histogram"
    r = np.sqrt(rec["x"].astype(np.float64) ** 2 + rec["y"].astype(np.float64) ** 2)
    dr = float(r_max) / int(n_bins)
    b = np.floor(r / dr).astype(np.int64)
    inside = b < n_bins
    hist = np.zeros(n_bins, dtype=HIST_DTYPE)
    w = rec["w"].astype(np.float64)
    t = rec["t"].astype(np.float64)
    hist["n"] = np.bincount(b[inside], minlength=n_bins).astype(np.uint64)
    hist["sum_w"] = np.bincount(b[inside], weights=w[inside], minlength=n_bins)
    hist["sum_wt"] = np.bincount(b[inside], weights=(w * t)[inside], minlength=n_bins)
    return dict(hist=hist, overflow=int(np.count_nonzero(~inside)), r=r, records=rec, counters=res["counters"],
                counts=res["counts"])


def profile(hist, r_max: float, min_photons: int = 50):
    """Fig. 3a / 3b quantities: photon density [1/m^2] and mean arrival time [ns] per radial bin; bins with fewer than
    `min_photons` bunches are masked (NaN), the paper's cut of at least 50 photons per bin."""
    n_bins = len(hist)
    edges = np.linspace(0.0, float(r_max), n_bins + 1)
    area = np.pi * (edges[1:] ** 2 - edges[:-1] ** 2)
    ok = hist["n"] >= min_photons
    dens = np.where(ok, hist["sum_w"] / area, np.nan)
    with np.errstate(invalid="ignore", divide="ignore"):
        mean_t = np.where(ok & (hist["sum_w"] > 0), hist["sum_wt"] / hist["sum_w"], np.nan)
    return 0.5 * (edges[1:] + edges[:-1]), dens, mean_t
