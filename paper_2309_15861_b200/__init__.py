"""paper_2309_15861_b200 -- thin Python binding of the C-ABI library libc8opt.so.

Argument marshalling only: every step of the photon path (preamble, Philox draw,
generation, propagation, sphere test, tally / record output) runs in the CUDA
kernels behind include/c8opt.h.  There is no CPU fallback: if the shared library
is missing or no B200 is present, calls raise.

    ctx = Context(atmosphere_dict)            # c8opt_create_atmosphere
    ctx.add_telescopes(xyzr)                  # c8opt_add_telescopes
    ctx.propagate_segments(d_seg, params)     # c8opt_propagate_segments (device tensor)
    ctx.propagate_segments_host(h_seg, params)  # c8opt_propagate_segments_host (numpy / pinned tensor)
    tallies, counters, tel_count = ctx.read_tallies()   # c8opt_read_tallies

`atmosphere_dict` / `params` use the same plain-dict layout as workloads/ (inputs only).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

from .build import LIB_PATH, build  # noqa: F401

MAX_LAYERS = 8
PROC_CHERENKOV, PROC_FLUORESCENCE = 1, 2
MODE_TALLY, MODE_OUTPUT, MODE_GROUND_HIST = 0, 1, 2
BEAM_ARRAY = -2
FLAG_CULL = 1
FLAG_REFRACT = 2
FLAG_CUT_CENTRE = 4
FLAG_CUT_TELESCOPES = 8
COUNTER_NAMES = ("segments", "generated", "upward", "hits", "records", "dropped", "invalid", "culled")
TALLY_DTYPE = np.dtype([("hits", "<u8"), ("sum_w", "<f8"), ("sum_wt", "<f8")])
HIST_DTYPE = np.dtype([("n", "<u8"), ("sum_w", "<f8"), ("sum_wt", "<f8")])
RECORD_FLOATS = 7

EXPORTS = ("c8opt_create_atmosphere", "c8opt_add_telescopes", "c8opt_propagate_segments",
           "c8opt_propagate_segments_host", "c8opt_read_tallies", "c8opt_reset_tallies", "c8opt_destroy",
           "c8opt_last_error", "c8opt_launch_count", "c8opt_set_ground_histogram", "c8opt_read_ground_histogram",
           "c8opt_reserve_host_staging", "c8opt_tally_static")
STATIC_MAX_TELESCOPES = 8


class C8optError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"c8opt error {code}: {message}")
        self.code = code


class _Layer(C.Structure):
    _fields_ = [("h_lo_m", C.c_double), ("a_gcm2", C.c_double), ("b_gcm2", C.c_double), ("c_m", C.c_double)]


class _AtmosphereDesc(C.Structure):
    _fields_ = [("n_layers", C.c_int32), ("layers", _Layer * MAX_LAYERS),
                ("eta0", C.c_double), ("rho0_gcm3", C.c_double), ("h_obs_m", C.c_double),
                ("tau_nh", C.c_int32), ("tau_nl", C.c_int32),
                ("tau_h0_m", C.c_double), ("tau_dh_m", C.c_double), ("tau_l0_nm", C.c_double), ("tau_dl_nm", C.c_double),
                ("tau", C.POINTER(C.c_float))]


class _RunParams(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("processes", C.c_uint32), ("mode", C.c_uint32),
                ("lam1_nm", C.c_double), ("lam2_nm", C.c_double), ("bunch_size", C.c_double),
                ("fl_yield_per_MeV", C.c_double), ("fl_lam1_nm", C.c_double), ("fl_lam2_nm", C.c_double),
                ("fl_beam_telescope", C.c_int32), ("flags", C.c_uint32), ("fl_beam_halfangle_rad", C.c_double),
                ("cut_angle_rad", C.c_double), ("cauchy_b_nm2", C.c_double)]


class _Output(C.Structure):
    _fields_ = [("records", C.c_void_p), ("tel_offset", C.c_void_p), ("tel_capacity", C.c_void_p),
                ("ids", C.c_void_p), ("counts", C.c_void_p)]


_lib = None


def lib():
    """Load libc8opt.so (built in-tree by build()); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.c8opt_create_atmosphere.argtypes = [C.POINTER(_AtmosphereDesc), C.POINTER(vp)]
        L.c8opt_add_telescopes.argtypes = [vp, C.POINTER(C.c_float), C.c_int32]
        L.c8opt_propagate_segments.argtypes = [vp, vp, C.c_uint64, C.c_uint64, C.POINTER(_RunParams), C.POINTER(_Output), vp]
        L.c8opt_propagate_segments_host.argtypes = L.c8opt_propagate_segments.argtypes
        L.c8opt_read_tallies.argtypes = [vp, vp, C.c_int32, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.c8opt_reset_tallies.argtypes = [vp, vp]
        L.c8opt_destroy.argtypes = [vp]
        L.c8opt_destroy.restype = None
        L.c8opt_last_error.argtypes = [vp]
        L.c8opt_last_error.restype = C.c_char_p
        L.c8opt_launch_count.argtypes = [vp]
        L.c8opt_launch_count.restype = C.c_uint64
        L.c8opt_set_ground_histogram.argtypes = [vp, C.c_double, C.c_double, C.c_double, C.c_int32]
        L.c8opt_read_ground_histogram.argtypes = [vp, vp, C.c_int32, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
        L.c8opt_reserve_host_staging.argtypes = [vp, C.c_uint64]
        L.c8opt_tally_static.argtypes = [C.POINTER(_AtmosphereDesc), vp, C.POINTER(C.c_float), C.c_int32, vp, C.c_uint64,
                                         C.c_uint64, C.POINTER(_RunParams), vp, vp, vp]
        for name in EXPORTS[:6] + EXPORTS[9:]:
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def _ptr(x) -> int:
    """Device / host address of a torch tensor, numpy array, int or None."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    raise TypeError(type(x))


def _stream(stream) -> int:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    return int(getattr(stream, "cuda_stream", stream))


def make_run_params(p: dict) -> _RunParams:
    return _RunParams(int(p["seed"]), int(p["processes"]), int(p.get("mode", MODE_TALLY)),
                      float(p["lam1"]), float(p["lam2"]), float(p["bunch_size"]),
                      float(p["fl_yield"]), float(p["fl_lam1"]), float(p["fl_lam2"]),
                      int(p["fl_beam_telescope"]), int(p.get("flags", 0)), float(p["fl_beam_halfangle"]),
                      float(p.get("cut_angle", 0.0)), float(p.get("cauchy_b", 0.0)))


def _atmosphere_desc(atmosphere: dict):
    """(c8opt_atmosphere_desc, the float32 table it points at or None)."""
    d = _AtmosphereDesc()
    layers = atmosphere["layers"]
    d.n_layers = len(layers)
    for i, (h_lo, a, b, c) in enumerate(layers[:MAX_LAYERS]):
        d.layers[i] = _Layer(h_lo, a, b, c)
    d.eta0, d.rho0_gcm3, d.h_obs_m = atmosphere["eta0"], atmosphere["rho0"], atmosphere["h_obs"]
    tau = atmosphere.get("tau")
    if tau is not None:
        tau = np.ascontiguousarray(tau, dtype=np.float32)
        d.tau_nh, d.tau_nl = tau.shape
        d.tau_h0_m, d.tau_dh_m = atmosphere["tau_h0"], atmosphere["tau_dh"]
        d.tau_l0_nm, d.tau_dl_nm = atmosphere["tau_l0"], atmosphere["tau_dl"]
        d.tau = tau.ctypes.data_as(C.POINTER(C.c_float))
    return d, tau


def tally_static(atmosphere: dict, xyzr, d_seg, params: dict, d_tallies_out, d_counters_out=None, d_tau=None,
                 n: int | None = None, first_segment_id: int = 0, stream=None):
    """c8opt_tally_static: the tally pass with no context and no allocation (asynchronous on `stream`).
    d_seg, d_tallies_out ([n_tel] x 24 bytes), d_counters_out ([8] uint64) and d_tau (the transmission table, float32
    [tau_nh, tau_nl], or None) are the caller's CUDA tensors; atmosphere["tau"] only gives the table's shape."""
    d, _tau = _atmosphere_desc(atmosphere)
    d.tau = None
    t = np.ascontiguousarray(xyzr, dtype=np.float32).reshape(-1, 4)
    if n is None:
        n = d_seg.numel() * d_seg.element_size() // 48
    rp = make_run_params(params)
    rc = lib().c8opt_tally_static(C.byref(d), _ptr(d_tau), t.ctypes.data_as(C.POINTER(C.c_float)), len(t), _ptr(d_seg), n,
                                  first_segment_id, C.byref(rp), _ptr(d_tallies_out), _ptr(d_counters_out), _stream(stream))
    if rc != 0:
        raise C8optError(rc, lib().c8opt_last_error(None).decode())


class Context:
    """Owns one c8opt_ctx."""

    def __init__(self, atmosphere: dict):
        d, _tau = _atmosphere_desc(atmosphere)
        self._h = C.c_void_p()
        self.n_tel = 0
        self.hist_bins = 0
        rc = lib().c8opt_create_atmosphere(C.byref(d), C.byref(self._h))
        if rc != 0:
            raise C8optError(rc, lib().c8opt_last_error(None).decode())

    def _check(self, rc: int, allow=()):
        if rc != 0 and rc not in allow:
            raise C8optError(rc, lib().c8opt_last_error(self._h).decode())
        return rc

    def add_telescopes(self, xyzr):
        t = np.ascontiguousarray(xyzr, dtype=np.float32).reshape(-1, 4)
        self._check(lib().c8opt_add_telescopes(self._h, t.ctypes.data_as(C.POINTER(C.c_float)), len(t)))
        self.n_tel = len(t)

    @staticmethod
    def _output(records, tel_offset, tel_capacity, ids, counts):
        if records is None and counts is None:
            return None
        return _Output(_ptr(records), _ptr(tel_offset), _ptr(tel_capacity), _ptr(ids), _ptr(counts))

    def propagate_segments(self, d_seg, params: dict, n: int | None = None, first_segment_id: int = 0,
                           records=None, tel_offset=None, tel_capacity=None, ids=None, counts=None, stream=None):
        """d_seg: CUDA tensor holding n 48-byte segment records (any dtype, contiguous)."""
        if n is None:
            n = d_seg.numel() * d_seg.element_size() // 48
        out = self._output(records, tel_offset, tel_capacity, ids, counts)
        rp = make_run_params(params)
        self._check(lib().c8opt_propagate_segments(self._h, _ptr(d_seg), n, first_segment_id, C.byref(rp),
                                                   C.byref(out) if out is not None else None, _stream(stream)))

    def propagate_segments_host(self, h_seg, params: dict, n: int | None = None, first_segment_id: int = 0,
                                records=None, tel_offset=None, tel_capacity=None, ids=None, counts=None, stream=None):
        """h_seg: HOST buffer (numpy structured array or pinned torch tensor) of 48-byte segment records."""
        if n is None:
            n = (h_seg.nbytes if isinstance(h_seg, np.ndarray) else h_seg.numel() * h_seg.element_size()) // 48
        out = self._output(records, tel_offset, tel_capacity, ids, counts)
        rp = make_run_params(params)
        self._check(lib().c8opt_propagate_segments_host(self._h, _ptr(h_seg), n, first_segment_id, C.byref(rp),
                                                        C.byref(out) if out is not None else None, _stream(stream)))

    def reserve_host_staging(self, max_segments: int):
        """Pre-allocate the device staging of propagate_segments_host (c8opt_reserve_host_staging)."""
        self._check(lib().c8opt_reserve_host_staging(self._h, int(max_segments)))

    def read_tallies(self, allow_overflow: bool = False):
        """Synchronises; returns (tallies[n_tel], counters dict, records written per telescope)."""
        tallies = np.zeros(self.n_tel, dtype=TALLY_DTYPE)
        counters = np.zeros(8, dtype=np.uint64)
        tel_count = np.zeros(self.n_tel, dtype=np.uint64)
        self._check(lib().c8opt_read_tallies(self._h, tallies.ctypes.data, self.n_tel,
                                             counters.ctypes.data_as(C.POINTER(C.c_uint64)),
                                             tel_count.ctypes.data_as(C.POINTER(C.c_uint64))),
                    allow=(-3,) if allow_overflow else ())
        return tallies, dict(zip(COUNTER_NAMES, (int(c) for c in counters))), tel_count

    def set_ground_histogram(self, core_x: float, core_y: float, r_max: float, n_bins: int):
        self._check(lib().c8opt_set_ground_histogram(self._h, float(core_x), float(core_y), float(r_max), int(n_bins)))
        self.hist_bins = int(n_bins)

    def read_ground_histogram(self):
        """Synchronises; returns (bins[n_bins] of {n, sum_w, sum_wt}, overflow, counters dict)."""
        bins = np.zeros(self.hist_bins, dtype=HIST_DTYPE)
        over = C.c_uint64(0)
        counters = np.zeros(8, dtype=np.uint64)
        self._check(lib().c8opt_read_ground_histogram(self._h, bins.ctypes.data, self.hist_bins, C.byref(over),
                                                      counters.ctypes.data_as(C.POINTER(C.c_uint64))))
        return bins, int(over.value), dict(zip(COUNTER_NAMES, (int(c) for c in counters)))

    def reset_tallies(self, stream=None):
        self._check(lib().c8opt_reset_tallies(self._h, _stream(stream)))

    @property
    def launch_count(self) -> int:
        return int(lib().c8opt_launch_count(self._h))

    def close(self):
        if self._h:
            lib().c8opt_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
