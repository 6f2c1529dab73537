"""Seeded synthetic inputs shared by the fp64 oracle and the CUDA path.

This module holds NO arithmetic of the method (no photon yield, no Cherenkov
angle, no ray tracing, no RNG of the method).  It only manufactures *inputs*:
track-segment tables, telescope layouts, atmosphere descriptors and the
optical-depth table, with the shapes and distributions of the workloads that
BASELINE.json `configs[0..4]` name (called config 1..5 there and here) and that
SURVEY.md §8(d) "Synthetic inputs" spells out.  The paper's real workloads are
CORSIKA air showers (PAPER.md:87, 100 x 500 GeV gamma showers) which are not
available; these seeded segment sets stand in for them.

Everything is written once to fp32 so that the oracle and the GPU read the
same quantised numbers.

Inputs are plain Python / numpy objects:

* segments   : structured array, dtype SEGMENT_DTYPE (48 bytes / record)
* telescopes : float32 array [n_tel, 4] = (x, y, z, R) in metres
* atmosphere : dict(layers=[(h_lo, a, b, c), ...], eta0, rho0, h_obs,
                    tau=None | float32[nh, nl], tau_h0, tau_dh, tau_l0, tau_dl)
* params     : dict with the run parameters (seed, processes, bands, ...)
"""
from __future__ import annotations

import math

import numpy as np

C_M_PER_NS = 0.299792458  # speed of light, used only for the front-relative clock t0 (R12)

SEGMENT_DTYPE = np.dtype(
    [
        ("x0", "<f4"), ("y0", "<f4"), ("z0", "<f4"), ("t0", "<f4"),
        ("dx", "<f4"), ("dy", "<f4"), ("dz", "<f4"), ("length", "<f4"),
        ("gamma", "<f4"), ("charge", "<f4"), ("dE", "<f4"), ("flags", "<u4"),
    ]
)
assert SEGMENT_DTYPE.itemsize == 48

PROC_CHERENKOV = 1
PROC_FLUORESCENCE = 2
MODE_TALLY = 0
MODE_OUTPUT = 1

H_OBS = 2000.0
RHO0 = 1.225e-3  # g/cm^3, sea level
ETA0 = 2.83e-4   # n(0) - 1, BASELINE.json configs[0]


# --------------------------------------------------------------------------
# atmospheres (inputs: coefficient tables only)
# --------------------------------------------------------------------------
def atmosphere_single_layer(h_scale: float = 8400.0, h_obs: float = H_OBS) -> dict:
    """Config 1: isothermal layer, n(h) = 1 + 2.83e-4 exp(-h / 8.4 km).

    T(h) = a + b exp(-h/c) with a = 0, c = H, b = rho0 * H (g/cm^2; the factor
    100 converts m to cm).  SURVEY.md §8(c) "Atmosphere".
    """
    b = RHO0 * h_scale * 100.0
    return dict(layers=[(0.0, 0.0, b, h_scale)], eta0=ETA0, rho0=RHO0, h_obs=h_obs,
                tau=None, tau_h0=0.0, tau_dh=1.0, tau_l0=0.0, tau_dl=1.0)


def five_layer_coefficients():
    """Stand-in 5-layer table of SURVEY.md §8(c) R18 (all layers exponential).

    Boundaries 0/4/10/40/100 km, scale heights 9.5/8.5/6.5/7.5/7.5 km,
    rho(0) = 1.225e-3 g/cm^3; b_{i+1} from density continuity, a_{i+1} from
    depth continuity, and a constant shift so that T(112.8 km) = 0.
    """
    h_lo = [0.0, 4000.0, 10000.0, 40000.0, 100000.0]
    c = [9500.0, 8500.0, 6500.0, 7500.0, 7500.0]
    b = [RHO0 * c[0] * 100.0]
    a = [0.0]
    for i in range(4):
        h = h_lo[i + 1]
        dens = b[i] / c[i] * math.exp(-h / c[i])
        b.append(dens * c[i + 1] * math.exp(h / c[i + 1]))
        t_below = a[i] + b[i] * math.exp(-h / c[i])
        a.append(t_below - b[i + 1] * math.exp(-h / c[i + 1]))
    shift = a[4] + b[4] * math.exp(-112800.0 / c[4])
    a = [ai - shift for ai in a]
    return [(h_lo[i], a[i], b[i], c[i]) for i in range(5)]


def atmosphere_five_layer(h_obs: float = H_OBS, tau: np.ndarray | None = None,
                          lam1: float = 300.0, lam2: float = 600.0) -> dict:
    atm = dict(layers=five_layer_coefficients(), eta0=ETA0, rho0=RHO0, h_obs=h_obs,
               tau=None, tau_h0=0.0, tau_dh=1.0, tau_l0=0.0, tau_dl=1.0)
    if tau is not None:
        nh, nl = tau.shape
        atm.update(tau=np.ascontiguousarray(tau, dtype=np.float32), tau_h0=h_obs, tau_dh=500.0,
                   tau_l0=lam1, tau_dl=(lam2 - lam1) / (nl - 1))
    return atm


def transmission_table(seed: int, nh: int = 64, nl: int = 32) -> np.ndarray:
    """Config 4: tau(h, lambda), uniform 0..1, every wavelength column sorted
    ascending in h (BASELINE.json configs[3] "rows monotone in h")."""
    rng = np.random.Generator(np.random.PCG64(seed + 1000))
    tau = np.sort(rng.random((nh, nl)), axis=0)
    return tau.astype(np.float32)


def depth_of(atm: dict, h: np.ndarray) -> np.ndarray:
    """T(h) of the input atmosphere (needed to place segments at a depth X)."""
    h = np.asarray(h, dtype=np.float64)
    out = np.zeros_like(h)
    layers = atm["layers"]
    for i, (h_lo, a, b, c) in enumerate(layers):
        hi = layers[i + 1][0] if i + 1 < len(layers) else np.inf
        lo = -np.inf if i == 0 else h_lo
        m = (h >= lo) & (h < hi)
        out[m] = a + b * np.exp(-h[m] / c)
    return out


def altitude_of(atm: dict, x: np.ndarray) -> np.ndarray:
    """Inverse of depth_of: altitude h with T(h) = X."""
    x = np.asarray(x, dtype=np.float64)
    out = np.full_like(x, np.nan)
    layers = atm["layers"]
    for i, (h_lo, a, b, c) in enumerate(layers):
        t_lo = a + b * math.exp(-h_lo / c) if i > 0 else np.inf
        t_hi = (a + b * math.exp(-layers[i + 1][0] / c)) if i + 1 < len(layers) else -np.inf
        m = (x <= t_lo) & (x > t_hi) & (x > a)
        out[m] = -c * np.log((x[m] - a) / b)
    return out


# --------------------------------------------------------------------------
# telescopes
# --------------------------------------------------------------------------
def telescopes_single(z: float = H_OBS, r: float = 6.0) -> np.ndarray:
    return np.array([[0.0, 0.0, z, r]], dtype=np.float32)


def telescopes_square(half: float = 50.0, z: float = H_OBS, r: float = 6.0) -> np.ndarray:
    return np.array([[sx * half, sy * half, z, r] for sy in (-1, 1) for sx in (-1, 1)], dtype=np.float32)


def telescopes_far(dist: float = 10000.0, z: float = H_OBS, r: float = 6.0) -> np.ndarray:
    return np.array([[dist, 0.0, z, r]], dtype=np.float32)


def telescopes_grid(n: int = 10, spacing: float = 120.0, z: float = H_OBS, r: float = 6.0) -> np.ndarray:
    c = (n - 1) / 2.0
    return np.array([[(i - c) * spacing, (j - c) * spacing, z, r] for j in range(n) for i in range(n)],
                    dtype=np.float32)


def telescope_accept_all(z: float = H_OBS) -> np.ndarray:
    """Config 5g: one "telescope" so large that every downward photon is inside
    it: every photon reaching the plane z is written."""
    return np.array([[0.0, 0.0, z, 1.0e9]], dtype=np.float32)


# --------------------------------------------------------------------------
# segment sets
# --------------------------------------------------------------------------
def _finish(x0, y0, z0, polar, azim, length, gamma, charge, dE, flags, h_obs):
    n = len(z0)
    sinp = np.sin(polar)
    dx = sinp * np.cos(azim)
    dy = sinp * np.sin(azim)
    dz = -np.cos(polar)
    # keep the whole track above the observation level (R21)
    lmax = np.maximum((z0 - h_obs - 1.0) / np.maximum(-dz, 1e-9), 0.0)
    length = np.minimum(length, lmax)
    seg = np.zeros(n, dtype=SEGMENT_DTYPE)
    seg["x0"], seg["y0"], seg["z0"] = x0, y0, z0
    seg["t0"] = -(z0 - h_obs) / C_M_PER_NS  # shower-front-relative clock (R12)
    d = np.stack([dx, dy, dz], axis=1).astype(np.float32).astype(np.float64)
    d /= np.linalg.norm(d, axis=1, keepdims=True)  # re-normalise after fp32 quantisation
    seg["dx"], seg["dy"], seg["dz"] = d[:, 0], d[:, 1], d[:, 2]
    seg["length"], seg["gamma"], seg["charge"], seg["dE"], seg["flags"] = length, gamma, charge, dE, flags
    return seg


def _log_uniform(rng, lo, hi, n):
    return np.exp(rng.uniform(math.log(lo), math.log(hi), n))


def segments_config1(n: int = 10_000, seed: int = 1, h_obs: float = H_OBS) -> np.ndarray:
    """BASELINE.json configs[0]: 10^4 electron segments, 6-12 km, +-200 m, within 3 deg."""
    rng = np.random.Generator(np.random.PCG64(seed))
    z0 = rng.uniform(6000.0, 12000.0, n)
    x0 = rng.uniform(-200.0, 200.0, n)
    y0 = rng.uniform(-200.0, 200.0, n)
    cosp = rng.uniform(math.cos(math.radians(3.0)), 1.0, n)  # uniform in cos(theta)
    polar = np.arccos(cosp)
    azim = rng.uniform(0.0, 2.0 * math.pi, n)
    length = rng.exponential(10.0, n)
    gamma = _log_uniform(rng, 1e2, 1e4, n)
    charge = np.full(n, -1.0)
    dE = np.zeros(n)
    flags = np.zeros(n, dtype=np.uint32)
    return _finish(x0, y0, z0, polar, azim, length, gamma, charge, dE, flags, h_obs)


def segments_shower(n: int, seed: int, atm: dict, xmax: float = 350.0, lam_gh: float = 70.0,
                    lateral=(30.0,), gamma_range=(50.0, 1e5), muon_fraction: float = 0.2,
                    dE_range=(0.1, 10.0), mean_angle_deg: float = 4.0, h_obs: float = H_OBS) -> np.ndarray:
    """Shower-shaped segment set (BASELINE.json configs[1..4]).

    Depth X ~ Gamma(Xmax/lambda + 1, lambda), i.e. a Gaisser-Hillas profile with
    X0 = 0; redrawn while X >= 0.999 T(h_obs).  z0 = T^-1(X).  Lateral offset is
    Gaussian per axis (a 50/50 mixture when two sigmas are given).  Angle to the
    (vertical) shower axis ~ Exp(mean 4 deg) clamped at 60 deg.
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    t_obs = float(depth_of(atm, np.array([h_obs]))[0])
    x = rng.gamma(xmax / lam_gh + 1.0, lam_gh, n)
    bad = x >= 0.999 * t_obs
    while bad.any():
        x[bad] = rng.gamma(xmax / lam_gh + 1.0, lam_gh, int(bad.sum()))
        bad = x >= 0.999 * t_obs
    z0 = altitude_of(atm, x)
    assert np.isfinite(z0).all()
    if len(lateral) == 1:
        sig = np.full(n, lateral[0])
    else:
        sig = np.where(rng.random(n) < 0.5, lateral[0], lateral[1])
    x0 = rng.normal(0.0, 1.0, n) * sig
    y0 = rng.normal(0.0, 1.0, n) * sig
    polar = np.minimum(rng.exponential(math.radians(mean_angle_deg), n), math.radians(60.0))
    azim = rng.uniform(0.0, 2.0 * math.pi, n)
    length = rng.exponential(10.0, n)
    gamma = _log_uniform(rng, gamma_range[0], gamma_range[1], n)
    charge = np.where(rng.random(n) < 0.5, -1.0, 1.0)
    flags = (rng.random(n) < muon_fraction).astype(np.uint32)  # bit 0: muon label (R21: label only)
    dE = _log_uniform(rng, dE_range[0], dE_range[1], n)
    return _finish(x0, y0, z0, polar, azim, length, gamma, charge, dE, flags, h_obs)


# --------------------------------------------------------------------------
# run parameters and the five configurations
# --------------------------------------------------------------------------
def default_params(**kw) -> dict:
    p = dict(seed=1, processes=PROC_CHERENKOV, lam1=300.0, lam2=600.0, bunch_size=1.0,
             fl_yield=4.0, fl_lam1=340.0, fl_lam2=450.0, fl_beam_telescope=-1,
             fl_beam_halfangle=math.radians(2.0), mode=MODE_TALLY)
    p.update(kw)
    return p


def make_config(name: str, n_segments: int | None = None, seed_offset: int = 0) -> dict:
    """Return dict(segments, telescopes, atmosphere, params, name) for
    'c1', 'c2', 'c3a', 'c3b', 'c4', 'c5', 'c5g' (BASELINE.json configs[0..4];
    'c5g' is the accept-all variant SURVEY.md §8(d) adds).  seed_offset != 0
    draws a different, equally distributed segment set (one per rank when the
    job is sharded); the Philox seed of the run is left unchanged."""
    so = 7919 * int(seed_offset)
    if name == "c1":
        atm = atmosphere_single_layer()
        seg = segments_config1(n_segments or 10_000, seed=1 + so)
        tel = telescopes_single()
        par = default_params(seed=1)
    elif name in ("c2", "c5", "c5g"):
        atm = atmosphere_five_layer()
        n = n_segments or (1_000_000 if name == "c2" else 10_000_000)
        seg = segments_shower(n, seed=2 + so, atm=atm, xmax=350.0, lateral=(30.0,))
        tel = telescope_accept_all() if name == "c5g" else telescopes_square()
        par = default_params(seed=2, mode=MODE_TALLY if name == "c2" else MODE_OUTPUT)
    elif name in ("c3a", "c3b"):
        atm = atmosphere_five_layer()
        seg = segments_shower(n_segments or 1_000_000, seed=3 + so, atm=atm, xmax=700.0, lateral=(30.0,),
                              muon_fraction=0.0)
        seg["charge"] = -1.0
        tel = telescopes_far()
        par = default_params(seed=3, processes=PROC_FLUORESCENCE,
                             fl_beam_telescope=(0 if name == "c3b" else -1))
    elif name == "c4":
        tau = transmission_table(seed=4)
        atm = atmosphere_five_layer(tau=tau)
        seg = segments_shower(n_segments or 10_000_000, seed=4 + so, atm=atm, xmax=500.0, lateral=(20.0, 200.0))
        tel = telescopes_grid()
        par = default_params(seed=4, processes=PROC_CHERENKOV | PROC_FLUORESCENCE)
    else:
        raise ValueError(name)
    return dict(name=name, segments=seg, telescopes=tel, atmosphere=atm, params=par)
