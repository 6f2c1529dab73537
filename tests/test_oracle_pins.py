"""Pins of the fp64 oracle against what the paper and the mathematics fix.

The paper (arxiv 2309.15861) prints no worked numerical example, so the oracle
is pinned to closed forms, invariants, special cases that reduce to textbook
results, statistical laws with a known expectation, and brute force on tiny
inputs (SURVEY.md §8(c) "Pins").  None of these tests touches the CUDA path.
"""
import math
import os

import numpy as np
import pytest

import oracle as O
import workloads as W
from conftest import ROOT

C = 0.299792458
ALPHA = 7.2973525693e-3


def one_segment(x0=0.0, y0=0.0, z0=10000.0, t0=0.0, d=(0.0, 0.0, -1.0), length=1.0, gamma=1e7,
                charge=-1.0, dE=1.0):
    s = np.zeros(1, dtype=W.SEGMENT_DTYPE)
    d = np.asarray(d, dtype=np.float64)
    d = d / np.linalg.norm(d)
    s["x0"], s["y0"], s["z0"], s["t0"] = x0, y0, z0, t0
    s["dx"], s["dy"], s["dz"] = d
    s["length"], s["gamma"], s["charge"], s["dE"] = length, gamma, charge, dE
    return s


ATM1 = W.atmosphere_single_layer()
ATM5 = W.atmosphere_five_layer()
PAR = W.default_params()


# ------------------------------------------------------------------ Philox / uniforms
def test_philox_known_answer_vectors():
    n = 0
    with open(os.path.join(ROOT, "tests", "golden", "philox4x32_10_kat.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            w = [int(x, 16) for x in line.split()]
            assert O.philox4x32_10(w[0:4], w[4:6]) == w[6:10]
            n += 1
    assert n == 3


def test_philox_is_a_bijection_of_the_counter_on_a_sample():
    # distinct counters -> distinct outputs (Philox is a keyed permutation of the 128-bit counter)
    outs = {tuple(O.philox4x32_10([j, 7, 0, t], [5, 9])) for j in range(2000) for t in (0, 1)}
    assert len(outs) == 4000


def test_uniform_construction_R19():
    assert O.uniform(0) == 2.0 ** -24
    assert O.uniform(0xFFFFFFFF) == 1.0 - 2.0 ** -24
    assert O.uniform(0x1FF) == 2.0 ** -24            # low 9 bits are dropped
    assert O.uniform(0x200) == 1.5 * 2.0 ** -23
    rng = np.random.default_rng(0)
    for r in rng.integers(0, 2 ** 32, 200):
        u = O.uniform(int(r))
        assert 0.0 < u < 1.0 and float(np.float32(u)) == u   # exactly representable in fp32


def test_uniform_stream_mean_and_variance():
    u = np.array([O.uniform(x) for j in range(4000) for x in O.philox4x32_10([j, 1, 0, 0], [42, 0])])
    assert abs(u.mean() - 0.5) < 4 * math.sqrt(1 / 12 / len(u))
    assert abs(u.var() - 1 / 12) < 0.003


# ------------------------------------------------------------------ atmosphere
def test_column_depth_single_layer(golden_closed_forms):
    g = golden_closed_forms
    assert O.depth(ATM1, 0.0) == pytest.approx(g["depth_h0_gcm2"], rel=1e-6)
    assert O.depth(ATM1, 2000.0) == pytest.approx(g["depth_h2000_gcm2"], rel=1e-5)
    for h in (0.0, 1234.0, 8400.0, 30000.0):
        assert O.depth(ATM1, h) == pytest.approx(1.225e-3 * 840000.0 * math.exp(-h / 8400.0), rel=1e-14)
        assert O.refractivity(ATM1, h) == pytest.approx(2.83e-4 * math.exp(-h / 8400.0), rel=1e-14)


def test_five_layer_check_values_and_continuity(golden_closed_forms):
    g = golden_closed_forms
    for h, key in ((0, "five_layer_T_h0"), (2000, "five_layer_T_h2000"), (10000, "five_layer_T_h10000"),
                   (40000, "five_layer_T_h40000")):
        assert O.depth(ATM5, float(h)) == pytest.approx(g[key], rel=2e-4)
    assert O.density(ATM5, 0.0) == pytest.approx(1.225e-3, rel=1e-12)
    assert O.depth(ATM5, 112800.0) == pytest.approx(0.0, abs=1e-9)
    for hb in (4000.0, 10000.0, 40000.0, 100000.0):          # T and rho continuous across boundaries
        assert O.depth(ATM5, hb - 1e-6) == pytest.approx(O.depth(ATM5, hb), rel=1e-9)
        assert O.density(ATM5, hb - 1e-6) == pytest.approx(O.density(ATM5, hb), rel=1e-9)


def test_density_is_minus_dT_dh():
    for atm in (ATM1, ATM5):
        for h in (500.0, 3000.0, 7000.0, 25000.0, 60000.0):
            dT = (O.depth(atm, h + 0.5) - O.depth(atm, h - 0.5)) / 1.0   # g/cm^2 per m
            assert O.density(atm, h) == pytest.approx(-dT / 100.0, rel=1e-6)


# ------------------------------------------------------------------ Cherenkov closed forms
@pytest.mark.parametrize("h", [0, 2000, 8400, 10000])
def test_cherenkov_angle_yield_and_threshold(golden_closed_forms, h):
    g = golden_closed_forms
    n = 1.0 + 2.83e-4 * math.exp(-h / 8400.0)
    L = 2.0
    seg = one_segment(z0=h + L / 2, length=L, gamma=1e7)       # midpoint altitude = h (R3)
    st, f = O.preamble(ATM1, PAR, seg[0], 0)
    assert st == 0
    theta = math.atan2(f.sin_c, f.cos_c)
    assert math.degrees(theta) == pytest.approx(g[f"theta_c_deg_h{h}"], abs=2e-5)
    assert theta == pytest.approx(math.acos(1.0 / n), rel=1e-9)
    assert f.sin_c ** 2 + f.cos_c ** 2 == pytest.approx(1.0, abs=1e-15)
    # photons per metre at beta = 1, 300-600 nm
    assert f.mu / L == pytest.approx(g[f"photons_per_m_h{h}"], rel=2e-4)
    c_ft = 2 * math.pi * ALPHA * (1 / 300e-9 - 1 / 600e-9)
    assert f.mu / L == pytest.approx(c_ft * (1.0 - 1.0 / n ** 2), rel=1e-9)
    assert f.n_b == math.ceil(f.mu) and f.w0 == pytest.approx(f.mu / f.n_b, rel=1e-15)
    # threshold: no photons just below gamma_th, photons just above
    gth = (1.0 - 1.0 / n ** 2) ** -0.5
    assert gth == pytest.approx(g[f"gamma_th_h{h}"], rel=2e-5)
    st, f_lo = O.preamble(ATM1, PAR, one_segment(z0=h + L / 2, length=L, gamma=gth * (1 - 1e-4))[0], 0)
    st, f_hi = O.preamble(ATM1, PAR, one_segment(z0=h + L / 2, length=100.0, gamma=gth * (1 + 1e-2),
                                                 d=(1, 0, 0))[0], 0)
    assert f_lo.n_b == 0 and f_hi.n_b > 0


def test_theta_c_rad_sea_level(golden_closed_forms):
    st, f = O.preamble(ATM1, PAR, one_segment(z0=0.5, length=1.0)[0], 0)
    assert math.atan2(f.sin_c, f.cos_c) == pytest.approx(golden_closed_forms["theta_c_rad_h0"], abs=2e-7)


def test_frank_tamm_constant(golden_closed_forms):
    g = golden_closed_forms
    assert 2 * math.pi * ALPHA == pytest.approx(g["two_pi_alpha"], rel=1e-9)
    # the prefactor printed in PAPER.md:45, pi e^2 / (h eps0 c), from CODATA constants
    e, hp, eps0, c0 = 1.602176634e-19, 6.62607015e-34, 8.8541878128e-12, 299792458.0
    assert math.pi * e * e / (hp * eps0 * c0) == pytest.approx(g["two_pi_alpha"], rel=1e-8)
    for lam1, lam2, key, scale in ((300.0, 600.0, "frank_tamm_per_m_300_600", 1.0),
                                   (400.0, 700.0, "frank_tamm_per_cm_400_700", 0.01)):
        par = W.default_params(lam1=lam1, lam2=lam2)
        st, f = O.preamble(ATM1, par, one_segment(z0=0.5, length=1.0)[0], 0)
        assert f.mu / f.sin_c ** 2 * scale == pytest.approx(g[key], abs=5.1e-3)   # fixture printed to 2 decimals
    # charge enters as z^2, length linearly
    st, f1 = O.preamble(ATM1, PAR, one_segment(z0=5000.0, length=1.0, d=(1, 0, 0))[0], 0)
    st, f2 = O.preamble(ATM1, PAR, one_segment(z0=5000.0, length=3.0, d=(1, 0, 0), charge=2.0)[0], 0)
    assert f2.mu == pytest.approx(12.0 * f1.mu, rel=1e-14)


def test_bunching_R1():
    seg = one_segment(z0=5000.0, length=10.0, d=(1, 0, 0))
    st, f1 = O.preamble(ATM1, PAR, seg[0], 0)
    st, f5 = O.preamble(ATM1, W.default_params(bunch_size=5.0), seg[0], 0)
    assert f1.mu == f5.mu
    assert f5.n_b == math.ceil(f5.mu / 5.0) and f5.w0 == pytest.approx(f5.mu / f5.n_b) and f5.w0 <= 5.0
    assert f1.w0 <= 1.0


def test_invalid_segments_are_rejected():
    for kw in (dict(gamma=0.5), dict(length=-1.0), dict(gamma=float("nan")), dict(z0=float("inf"))):
        st, f = O.preamble(ATM1, PAR, one_segment(**kw)[0], 0)
        assert st == -1 and f.n_b == 0
    s = one_segment()
    s["dx"] = 0.1                                       # |d| off unity by more than 1e-3
    st, f = O.preamble(ATM1, PAR, s[0], 0)
    assert st == -1


# ------------------------------------------------------------------ rotation
def _random_dirs(n, seed):
    rng = np.random.default_rng(seed)
    v = rng.normal(size=(n, 3))
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def test_rodrigues_matrix_invariants():
    dirs = list(_random_dirs(50, 1)) + [np.array([0, 0, -1.0]), np.array([0, 0, 1.0]), np.array([1.0, 0, 0])]
    for d in dirs:
        st, f = O.preamble(ATM1, PAR, one_segment(z0=8000.0, d=d, length=1.0)[0], 0)
        M = np.array([[f.M[i][j] for j in range(3)] for i in range(3)])
        A = np.array(list(f.A))
        dd = np.array(list(f.d))
        assert np.allclose(M, M.T, atol=0)                         # symmetric
        assert np.allclose(M @ M, np.eye(3), atol=1e-14)           # involution
        assert np.linalg.det(M) == pytest.approx(1.0, abs=1e-14)   # proper rotation
        assert np.allclose(M @ np.array([0, 0, -1.0]), dd, atol=1e-14)   # downward normal -> track direction
        assert np.linalg.norm(A) == pytest.approx(1.0, abs=1e-15)
        # geometric definition: rotation by pi about A (general axis-angle formula)
        K = np.array([[0, -A[2], A[1]], [A[2], 0, -A[0]], [-A[1], A[0], 0]])
        Rpi = np.eye(3) + math.sin(math.pi) * K + (1 - math.cos(math.pi)) * (K @ K)
        assert np.allclose(M, Rpi, atol=1e-14)
        if 1 - dd[2] >= 1e-12:                                     # A bisects d and -z
            assert A @ dd == pytest.approx(A @ np.array([0, 0, -1.0]), abs=1e-14)


def test_every_cherenkov_photon_lies_on_the_cone():
    for d in _random_dirs(20, 2):
        if d[2] > 0:
            d = -d
        seg = one_segment(z0=8000.0, d=d, length=25.0)
        st, f = O.preamble(ATM1, PAR, seg[0], 0)
        dd = np.array(list(f.d))
        for j in range(0, f.n_b, max(1, f.n_b // 40)):
            ph = O.make_photon(f, PAR, 11, j, 0)
            v = np.array(list(ph.v))
            e = np.array(list(ph.e))
            assert v @ dd == pytest.approx(f.cos_c, abs=1e-14)     # v . d = cos(theta_c)
            assert np.linalg.norm(v) == pytest.approx(1.0, abs=1e-14)
            s = (e - np.array([seg["x0"][0], seg["y0"][0], seg["z0"][0]], dtype=np.float64)) @ dd
            assert 0.0 < s < float(seg["length"][0])               # on the track
            assert np.allclose(np.cross(e - np.array(list(f.p0)), dd), 0, atol=1e-8)
            assert ph.t_e == pytest.approx(s * f.inv_beta_c, abs=1e-9)  # t0 = 0, moves at beta c
            assert 300.0 < ph.lam < 600.0


def test_azimuth_is_uniform_around_the_track():
    seg = one_segment(z0=8000.0, d=(0.3, -0.2, -0.93), length=200.0)
    st, f = O.preamble(ATM1, PAR, seg[0], 0)
    dd = np.array(list(f.d))
    e1 = np.cross(dd, [0, 0, 1.0]); e1 /= np.linalg.norm(e1)
    e2 = np.cross(dd, e1)
    phis = []
    for j in range(f.n_b):
        v = np.array(list(O.make_photon(f, PAR, 3, j, 0).v))
        phis.append(math.atan2(v @ e2, v @ e1))
    hist, _ = np.histogram(phis, bins=8, range=(-math.pi, math.pi))
    exp = len(phis) / 8
    assert ((hist - exp) ** 2 / exp).sum() < 24.3                 # chi2, 7 dof, p ~ 1e-3


def test_wavelength_law_R4():
    seg = one_segment(z0=3000.0, d=(1, 0, 0), length=300.0)
    st, f = O.preamble(ATM1, PAR, seg[0], 0)
    lam = np.array([O.make_photon(f, PAR, 5, j, 0).lam for j in range(f.n_b)])
    n = len(lam)
    assert n > 5000
    inv = 1.0 / lam                                                # uniform on [1/600, 1/300]
    lo, hi = 1 / 600.0, 1 / 300.0
    assert abs(inv.mean() - (lo + hi) / 2) < 4 * (hi - lo) / math.sqrt(12 * n)
    assert abs(np.median(lam) - 400.0) < 400.0 * 4 * 0.5 / math.sqrt(n) * 1.5   # median = 2/(1/l1 + 1/l2)
    # fluorescence: uniform on [340, 450]
    par = W.default_params(processes=W.PROC_FLUORESCENCE)
    st, ff = O.preamble(ATM1, par, one_segment(dE=2000.0)[0], 1)
    lf = np.array([O.make_photon(ff, par, 5, j, 1).lam for j in range(ff.n_b)])
    assert ff.n_b == 8000 and lf.min() > 340 and lf.max() < 450
    assert abs(lf.mean() - 395.0) < 4 * 110 / math.sqrt(12 * 8000)


# ------------------------------------------------------------------ ray - sphere (R10)
def _quadratic_hit(e, v, c, R):
    """Independent formulation: |e + s v - c|^2 = R^2 has real roots and their mean is > 0."""
    oc = e - c
    b = 2.0 * (oc @ v)
    cc = oc @ oc - R * R
    disc = b * b - 4.0 * cc
    return disc >= 0.0 and (-b / 2.0) > 0.0


def test_ray_sphere_against_quadratic_solver_and_sampling():
    rng = np.random.default_rng(3)
    n_hit = 0
    for i in range(1000):
        c = np.array([rng.uniform(-50, 50), rng.uniform(-50, 50), 2000.0])
        R = rng.uniform(1.0, 30.0)
        e = c + np.array([rng.uniform(-200, 200), rng.uniform(-200, 200), rng.uniform(1.0, 3000.0)])
        aim = c + rng.normal(size=3) * R * 0.8                     # aim near the sphere so ~half hit
        v = aim - e
        v /= np.linalg.norm(v)
        if i % 10 == 0:
            v = -v                                                 # upward rays never hit
        hit, b2, s_c, s_pl, x, y = O.intersect(e, v, list(c) + [R])
        expect = v[2] < 0 and _quadratic_hit(e, v, c, R)
        assert hit == expect
        # dense sampling of the ray: the smallest distance to the centre
        s = np.linspace(0.0, 2 * np.linalg.norm(c - e), 20001)
        dist = np.linalg.norm(e[None, :] + s[:, None] * v[None, :] - c[None, :], axis=1)
        if abs(math.sqrt(max(b2, 0)) - R) > 0.05 and s_c > 1.0:
            assert (dist.min() <= R) == (b2 <= R * R)
        if v[2] < 0:
            g = e + s_pl * v
            assert g[2] == pytest.approx(c[2], abs=1e-9)
            assert (x, y) == (pytest.approx(g[0] - c[0], abs=1e-9), pytest.approx(g[1] - c[1], abs=1e-9))
        n_hit += hit
    assert 200 < n_hit < 800


def test_vertical_ray_hits_iff_offset_le_R():
    for b, expect in ((5.999, True), (6.001, False), (0.0, True), (6.0, True)):
        hit, b2, s_c, s_pl, x, y = O.intersect([b, 0, 5000.0], [0, 0, -1.0], [0, 0, 2000.0, 6.0])
        assert hit == expect and b2 == pytest.approx(b * b, abs=1e-9) and s_pl == 3000.0 and x == b
    # emission inside the sphere moving away from the centre, and below the centre plane: miss (R10)
    assert not O.intersect([0, 0, 1999.0], [0, 0, -1.0], [0, 0, 2000.0, 6.0])[0]
    assert not O.intersect([0, 0, 2001.0], [0, 0, 1.0], [0, 0, 2000.0, 6.0])[0]


def test_impact_parameter_is_rotation_invariant():
    rng = np.random.default_rng(4)
    for _ in range(100):
        e, c = rng.normal(size=3) * 1000, rng.normal(size=3) * 10
        v = rng.normal(size=3); v /= np.linalg.norm(v)
        Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
        _, b2a, sca, *_ = O.intersect(e, v, list(c) + [6.0])
        _, b2b, scb, *_ = O.intersect(Q @ e, Q @ v, list(Q @ c) + [6.0])
        assert b2a == pytest.approx(b2b, rel=1e-9, abs=1e-6) and sca == pytest.approx(scb, rel=1e-12, abs=1e-9)


# ------------------------------------------------------------------ timing (R8)
def test_vertical_ray_optical_delay(golden_closed_forms):
    g = golden_closed_forms
    t = O.arrival_time(ATM1, 10000.0, 2000.0, -1.0, 8000.0, 0.0)
    vac = 8000.0 / C
    assert vac == pytest.approx(g["vertical_10km_2km_vacuum_ns"], abs=1e-3)
    assert t - vac == pytest.approx(g["vertical_10km_2km_excess_ns"], abs=1e-5)
    assert (t - vac) * C == pytest.approx(g["vertical_10km_2km_excess_m"], abs=1e-6)
    # slant: both the geometric and the excess path scale with 1/|v_z|
    vz = -0.8
    ts = O.arrival_time(ATM1, 10000.0, 2000.0, vz, 8000.0 / 0.8, 0.0)
    assert ts == pytest.approx(t / 0.8, rel=1e-14)


def test_optical_delay_equals_numerical_integral_five_layer():
    # integral of eta(h) dh from 2 km to 30 km by the trapezoid rule on a fine grid
    h = np.linspace(2000.0, 30000.0, 280001)
    eta = np.array([O.refractivity(ATM5, x) for x in h[::100]])
    integral = np.trapezoid(eta, h[::100])
    t = O.arrival_time(ATM5, 30000.0, 2000.0, -1.0, 28000.0, 0.0)
    assert (t - 28000.0 / C) * C == pytest.approx(integral, rel=1e-6)


# ------------------------------------------------------------------ transmission (R17)
def _atm_with_tau(tau):
    return W.atmosphere_five_layer(tau=np.asarray(tau, dtype=np.float32))


def test_transmission_special_cases():
    assert O.transmission(ATM5, 5000.0, 400.0, -0.7) == 1.0            # no table -> weights unchanged
    assert O.transmission(_atm_with_tau(np.zeros((64, 32))), 5000.0, 400.0, -0.7) == 1.0
    atm = _atm_with_tau(np.full((64, 32), 0.25))
    for vz in (-1.0, -0.5, -0.123):
        assert O.transmission(atm, 7000.0, 433.0, vz) == pytest.approx(math.exp(-0.25 / abs(vz)), rel=1e-7)


def test_optical_depth_is_bilinear_and_clamped():
    i, j = np.meshgrid(np.arange(64), np.arange(32), indexing="ij")
    atm = _atm_with_tau(0.5 * i + 0.25 * j)                             # linear table -> exact reproduction
    dl = 300.0 / 31
    for h, lam in ((2000.0, 300.0), (2750.0, 300.0 + 3.5 * dl), (33499.0, 599.0), (12345.0, 456.7)):
        fh, fl = (h - 2000.0) / 500.0, (lam - 300.0) / dl
        assert O.optical_depth(atm, h, lam) == pytest.approx(0.5 * fh + 0.25 * fl, rel=1e-6, abs=1e-6)
    assert O.optical_depth(atm, 0.0, 100.0) == pytest.approx(0.0, abs=1e-12)        # clamped low
    assert O.optical_depth(atm, 1e6, 1e4) == pytest.approx(0.5 * 63 + 0.25 * 31, rel=1e-7)  # clamped high
    rng = np.random.default_rng(5)
    tau = rng.random((64, 32)).astype(np.float32)
    atm = _atm_with_tau(tau)
    for _ in range(50):                                                # grid nodes are reproduced
        a, b = rng.integers(0, 64), rng.integers(0, 32)
        assert O.optical_depth(atm, 2000.0 + 500.0 * a, 300.0 + dl * b) == pytest.approx(float(tau[a, b]), abs=2e-6)


# ------------------------------------------------------------------ whole-path pins
def test_isotropic_acceptance_fraction():
    """Fraction of isotropic rays from distance D hitting a sphere R is (1 - sqrt(1 - R^2/D^2))/2 = 0.1
    for R = 600, D = 1000 (SURVEY.md §8(c) pin "Isotropic acceptance")."""
    par = W.default_params(processes=W.PROC_FLUORESCENCE, seed=77)
    seg = one_segment(z0=3000.0, length=1e-3, gamma=100.0, dE=250000.0)   # 1e6 photons, 1000 m above the centre
    tel = np.array([[0, 0, 2000.0, 600.0]], dtype=np.float32)
    r = O.run(ATM5, tel, seg, par)
    n = int(r["counters"][1])
    assert n == 1_000_000 and int(r["counts"][0, 1]) == n
    frac = int(r["tallies"]["hits"][0]) / n
    assert abs(frac - 0.1) < 4 * math.sqrt(0.1 * 0.9 / n)
    assert abs(int(r["counters"][2]) / n - 0.5) < 4 * 0.5 / math.sqrt(n)   # half go upward
    assert r["tallies"]["sum_w"][0] == pytest.approx(r["tallies"]["hits"][0] * 1.0, rel=1e-12)


def test_beaming_weight_and_equal_expectation(golden_closed_forms):
    g = golden_closed_forms
    par_b = W.default_params(processes=W.PROC_FLUORESCENCE, fl_beam_telescope=0)
    tel = np.array([[0, 0, 2000.0, 600.0]], dtype=np.float32)
    seg = one_segment(z0=3000.0, length=1e-3, gamma=100.0, dE=50000.0)     # 2e5 photons
    st, f = O.preamble(ATM5, par_b, seg[0], 1, beam_tel=tel[0].astype(np.float64))
    omega = 2 * math.pi * f.one_minus_cos_ab
    assert omega == pytest.approx(g["omega_2deg_sr"], rel=1e-6)
    assert f.w0 == pytest.approx(g["omega_2deg_over_4pi"], rel=1e-6)        # mu / n_b = 1 here
    # all beamed photons stay inside the cone around the line of sight (straight down here)
    for j in range(0, 2000, 7):
        v = np.array(list(O.make_photon(f, par_b, 0, j, 1).v))
        assert v @ np.array([0, 0, -1.0]) >= math.cos(math.radians(2.0)) - 1e-15
    # equal expectation of the weighted tally when the cone (40 deg) covers the sphere (36.87 deg)
    par_iso = W.default_params(processes=W.PROC_FLUORESCENCE, seed=5)
    par_40 = W.default_params(processes=W.PROC_FLUORESCENCE, seed=6, fl_beam_telescope=0,
                              fl_beam_halfangle=math.radians(40.0))
    ri = O.run(ATM5, tel, seg, par_iso)
    rb = O.run(ATM5, tel, seg, par_40)
    n = 200_000
    assert int(rb["counters"][2]) == 0                                       # none upward when beamed down
    exp = 0.1 * n
    sig_i = math.sqrt(n * 0.1 * 0.9)
    p_b = 0.2 / (1 - math.cos(math.radians(40.0)))                           # hit probability inside the cone
    w_b = (1 - math.cos(math.radians(40.0))) / 2
    sig_b = w_b * math.sqrt(n * p_b * (1 - p_b))
    assert abs(ri["tallies"]["sum_w"][0] - exp) < 4 * sig_i
    assert abs(rb["tallies"]["sum_w"][0] - exp) < 4 * sig_b
    assert rb["tallies"]["hits"][0] > 3 * ri["tallies"]["hits"][0]           # beaming buys statistics


def test_beamed_line_of_sight_points_at_the_telescope():
    par_b = W.default_params(processes=W.PROC_FLUORESCENCE, fl_beam_telescope=0, fl_beam_halfangle=1e-4)
    tel = np.array([10000.0, 0.0, 2000.0, 6.0])
    seg = one_segment(x0=100.0, y0=-50.0, z0=9000.0, d=(0.1, 0.2, -0.97), length=10.0, dE=100.0)
    st, f = O.preamble(ATM5, par_b, seg[0], 1, beam_tel=tel)
    mid = np.array(list(f.p0)) + 0.5 * f.L * np.array(list(f.d))
    los = tel[:3] - mid
    los /= np.linalg.norm(los)
    for j in range(20):
        v = np.array(list(O.make_photon(f, par_b, 9, j, 1).v))
        assert math.acos(min(1.0, v @ los)) <= 1.0001e-4


def test_cherenkov_ring_geometry():
    """Vertical track, emission ~ point-like at dh above the plane: every ground point lies on the
    circle of radius dh tan(theta_c) (SURVEY.md §8(c) pin "Ring geometry")."""
    seg = one_segment(z0=10000.0, length=1e-2, gamma=1e6)
    seg["t0"] = 0.0
    par = W.default_params(bunch_size=1e-4, seed=3)                  # many bunches from a short track
    tel = W.telescope_accept_all()
    r = O.run(ATM1, tel, seg, par, record_capacity=100000)
    rec = r["records"]
    st, f = O.preamble(ATM1, par, seg[0], 0)
    assert len(rec) == f.n_b > 1000
    rad = np.hypot(rec["x"], rec["y"])
    tan_c = f.sin_c / f.cos_c
    assert np.all(np.abs(rad - 8000.0 * tan_c) <= 1e-2 * tan_c + 1e-9)
    # direction cosines are those of the cone, and times follow the optical path
    assert np.allclose(np.hypot(rec["cx"], rec["cy"]), f.sin_c, atol=1e-12)
    t_exp = (8000.0 / f.cos_c) / C + 0.01 * (2.83e-4 / 1.225e-3) * (O.depth(ATM1, 2000.0) - O.depth(ATM1, 10000.0)) \
        / f.cos_c / C
    assert np.all(np.abs(rec["t"] - t_exp) < 1e-3)
    assert np.allclose(rec["w"], f.w0, rtol=1e-15)


def test_conservation_laws_config1_sample():
    c = W.make_config("c1", 2000)
    r = O.run(c["atmosphere"], c["telescopes"], c["segments"], c["params"], record_capacity=10000)
    cnt = r["counters"]
    assert cnt[0] == 2000 and cnt[1] == r["counts"].sum()
    assert cnt[3] == r["tallies"]["hits"].sum() == cnt[4] == len(r["records"]) and cnt[5] == 0
    assert r["tallies"]["sum_w"][0] == pytest.approx(r["records"]["w"].sum(), rel=1e-12)
    assert r["tallies"]["sum_wt"][0] == pytest.approx((r["records"]["w"] * r["records"]["t"]).sum(), rel=1e-12)
    # closed-form count: ceil of the Frank-Tamm yield from its textbook definition, vectorised in numpy
    s = c["segments"]
    z0, L, dz, gam = (s[k].astype(np.float64) for k in ("z0", "length", "dz", "gamma"))
    n = 1.0 + 2.83e-4 * np.exp(-(z0 + 0.5 * L * dz) / 8400.0)
    beta2 = 1.0 - 1.0 / gam ** 2
    sin2 = np.maximum(1.0 - 1.0 / (beta2 * n * n), 0.0)
    mu = 2 * math.pi * ALPHA * (1 / 300e-9 - 1 / 600e-9) * L * sin2
    nb = np.ceil(mu).astype(np.int64)
    mismatch = np.nonzero(nb != r["counts"][:, 0])[0]
    # the naive 1 - 1/(beta n)^2 loses ~1e-12 relative: allow ceil() flips only where mu is within 1e-9 of an integer
    assert all(abs(mu[i] - round(mu[i])) < 1e-9 for i in mismatch) and len(mismatch) <= 1
    # segment ids are what the records say, and the split over threads changes nothing
    r2 = O.run(c["atmosphere"], c["telescopes"], c["segments"], c["params"], record_capacity=10000, threads=3)
    assert np.array_equal(r2["counts"], r["counts"]) and np.array_equal(r2["tallies"]["hits"], r["tallies"]["hits"])
    assert np.array_equal(r2["records"]["id"], r["records"]["id"])
    assert ((r["records"]["id"] >> 25) < 2000).all()


def test_first_segment_id_makes_batches_independent_of_batching():
    c = W.make_config("c1", 600)
    full = O.run(c["atmosphere"], c["telescopes"], c["segments"], c["params"], record_capacity=5000)
    a = O.run(c["atmosphere"], c["telescopes"], c["segments"][:250], c["params"], record_capacity=5000)
    b = O.run(c["atmosphere"], c["telescopes"], c["segments"][250:], c["params"], first_id=250, record_capacity=5000)
    assert np.array_equal(np.concatenate([a["records"]["id"], b["records"]["id"]]), full["records"]["id"])
    assert np.array_equal(a["tallies"]["hits"] + b["tallies"]["hits"], full["tallies"]["hits"])


def test_both_processes_and_record_capacity():
    c = W.make_config("c4", 300)
    c["telescopes"] = W.telescope_accept_all()
    r = O.run(c["atmosphere"], c["telescopes"], c["segments"], c["params"], record_capacity=1000)
    cnt = r["counters"]
    assert (r["counts"][:, 1] == np.ceil(4.0 * c["segments"]["dE"].astype(np.float64))).all()
    assert cnt[1] == r["counts"].sum() and cnt[4] == 1000 and cnt[5] == cnt[3] - 1000
    # accept-all sphere: every downward photon is a hit except those emitted (inside the sphere) with the
    # closest approach behind them, s_c <= 0 (R10) -- near-horizontal fluorescence photons flying outward
    down = int(cnt[1] - cnt[2])
    assert int(cnt[3]) <= down and down - int(cnt[3]) < 0.005 * down
    tags = (r["records"]["id"] >> 24) & 1
    assert set(np.unique(tags)) <= {0, 1}
    # transmission can only reduce the weight
    assert (r["records"]["w"] <= 1.0 + 1e-12).all() and (r["records"]["w"] > 0).all()


# ------------------------------------------------------------------ tiny brute-force case
def test_tiny_case_against_pure_python_restatement():
    """1 segment, <= 32 photons, 1 telescope, recomputed in pure Python with a different formulation:
    Python-int Philox, rotation by pi about the bisector through the generic axis-angle formula, and a
    quadratic-equation ray-sphere test."""
    M0, M1, W0, W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85

    def philox(ctr, key):
        c, k = list(ctr), list(key)
        for _ in range(10):
            p0, p1 = M0 * c[0], M1 * c[2]
            c = [(p1 >> 32) ^ c[1] ^ k[0], p1 & 0xFFFFFFFF, (p0 >> 32) ^ c[3] ^ k[1], p0 & 0xFFFFFFFF]
            k = [(k[0] + W0) & 0xFFFFFFFF, (k[1] + W1) & 0xFFFFFFFF]
        return c

    seg = one_segment(x0=3.0, y0=-2.0, z0=2600.0, d=(0.004, -0.003, -1.0), length=0.8, gamma=300.0)
    seg["t0"] = -2.0
    tel = np.array([[0.0, 0.0, 2000.0, 9.0]], dtype=np.float32)
    par = W.default_params(seed=(7 << 32) | 12345)
    r = O.run(ATM1, tel, seg, par, first_id=(1 << 33) + 5, record_capacity=100)
    nb = int(r["counts"][0, 0])
    assert 8 <= nb <= 32

    s = seg[0]
    p0 = np.array([s["x0"], s["y0"], s["z0"]], dtype=np.float64)
    d = np.array([s["dx"], s["dy"], s["dz"]], dtype=np.float64)
    d /= np.linalg.norm(d)
    L, gam = float(s["length"]), float(s["gamma"])
    n = 1.0 + 2.83e-4 * math.exp(-(p0[2] + 0.5 * L * d[2]) / 8400.0)
    beta = math.sqrt(1.0 - 1.0 / gam ** 2)
    theta = math.acos(1.0 / (beta * n))
    mu = 2 * math.pi * ALPHA * (1 / 300e-9 - 1 / 600e-9) * L * math.sin(theta) ** 2
    assert nb == math.ceil(mu)
    A = d + np.array([0, 0, -1.0]); A /= np.linalg.norm(A)
    K = np.array([[0, -A[2], A[1]], [A[2], 0, -A[0]], [-A[1], A[0], 0]])
    Rpi = np.eye(3) + 2.0 * (K @ K)
    S = (1 << 33) + 5
    hits = []
    for j in range(nb):
        rr = philox([j >> 1, S & 0xFFFFFFFF, S >> 32, 0], [12345, 7])       # R20: one block for the photons 2k, 2k + 1
        a, b = rr[2 * (j & 1)], rr[2 * (j & 1) + 1]
        u = [((a >> 9) + 0.5) / 2 ** 23, ((b >> 9) + 0.5) / 2 ** 23, ((((a & 511) << 9) | (b & 511)) + 0.5) / 2 ** 18]
        e = p0 + u[0] * L * d
        phi = 2 * math.pi * u[1]
        p = np.array([math.cos(phi) * math.sin(theta), math.sin(phi) * math.sin(theta), -math.cos(theta)])
        v = Rpi @ p
        if _quadratic_hit(e, v, tel[0, :3].astype(np.float64), 9.0):
            sp = (2000.0 - e[2]) / v[2]
            g = e + sp * v
            t = -2.0 + u[0] * L / (beta * C) + (sp + 2.83e-4 * 8400.0 * (math.exp(-2000 / 8400.0)
                                                                          - math.exp(-e[2] / 8400.0)) / abs(v[2])) / C
            lam = 1.0 / (1 / 300.0 - u[2] * (1 / 300.0 - 1 / 600.0))
            hits.append((j, g[0], g[1], v[0], v[1], t, lam, mu / nb))
    rec = r["records"]
    assert len(hits) == len(rec) >= 3
    for h, q in zip(hits, rec):
        assert (int(q["id"]) & 0xFFFFFF) == h[0] and (int(q["id"]) >> 25) == S
        assert q["x"] == pytest.approx(h[1], abs=1e-7) and q["y"] == pytest.approx(h[2], abs=1e-7)
        assert q["cx"] == pytest.approx(h[3], abs=1e-10) and q["cy"] == pytest.approx(h[4], abs=1e-10)
        assert q["t"] == pytest.approx(h[5], abs=1e-8) and q["lam"] == pytest.approx(h[6], rel=1e-12)
        assert q["w"] == pytest.approx(h[7], rel=1e-9)


# ------------------------------------------------------------------ ground-plane radial profile
def test_ground_histogram_vertical_track_closed_form():
    """A vertical track above the core: a photon emitted at path length s lands at r = (z0 - s - h_obs) tan(theta_c),
    uniform in s, so the radial histogram is flat between r(L) and r(0), empty elsewhere, holds all n_b bunches with
    total weight mu, and the mean arrival time of a bin lies between the closed-form times of its two edges."""
    z0, L, h_obs = 10000.0, 400.0, 2000.0
    seg = one_segment(x0=30.0, y0=-40.0, z0=z0, length=L, gamma=1e6)
    par = W.default_params(bunch_size=0.05, seed=11)
    st, f = O.preamble(ATM1, par, seg[0], 0)
    assert st == 0 and f.n_b > 100000
    r_max, n_bins = 120.0, 240
    res = O.ground_histogram(ATM1, seg, par, (30.0, -40.0), r_max, n_bins)
    h = res["hist"]
    tan_c = f.sin_c / f.cos_c
    r_hi, r_lo = (z0 - h_obs) * tan_c, (z0 - L - h_obs) * tan_c
    assert 95.0 < r_lo < r_hi < 110.0
    assert int(h["n"].sum()) == f.n_b and res["overflow"] == 0
    assert math.isclose(h["sum_w"].sum(), f.n_b * f.w0, rel_tol=1e-12)
    dr = r_max / n_bins
    edges = np.arange(n_bins + 1) * dr
    overlap = np.clip(np.minimum(edges[1:], r_hi) - np.maximum(edges[:-1], r_lo), 0.0, None)
    expect = f.n_b * overlap / (r_hi - r_lo)
    assert np.all(h["n"][overlap == 0.0] == 0)
    assert np.all(np.abs(h["n"].astype(np.float64) - expect) <= 5.0 * np.sqrt(expect) + 1.0)
    beta = math.sqrt(1.0 - 1e-12)
    kappa = 0.01 * ATM1["eta0"] / ATM1["rho0"]

    def t_of_r(r):                       # closed form along the vertical track: emission height from the landing radius
        hgt = r / tan_c + h_obs
        s = z0 - hgt
        return s / (beta * C) + ((hgt - h_obs) / f.cos_c + kappa * (O.depth(ATM1, h_obs) - O.depth(ATM1, hgt)) / f.cos_c) / C

    for b in np.nonzero(overlap > 0.5 * dr)[0]:
        ta, tb = t_of_r(max(edges[b], r_lo)), t_of_r(min(edges[b + 1], r_hi))
        mean_t = h["sum_wt"][b] / h["sum_w"][b]
        assert min(ta, tb) - 1e-9 <= mean_t <= max(ta, tb) + 1e-9


def test_ground_histogram_overflow_core_offset_and_profile_cut():
    seg = one_segment(z0=10000.0, length=10.0, gamma=1e6)
    par = W.default_params(bunch_size=0.05, seed=5)
    st, f = O.preamble(ATM1, par, seg[0], 0)
    # the ring (radius ~106 m about (0, 0)) seen from a core 1 km away: everything overflows a 120 m histogram
    far = O.ground_histogram(ATM1, seg, par, (1000.0, 0.0), 120.0, 24)
    assert far["overflow"] == f.n_b and int(far["hist"]["n"].sum()) == 0
    # seen from a core 50 m away the distances spread over |106 - 50| .. 106 + 50
    off = O.ground_histogram(ATM1, seg, par, (50.0, 0.0), 200.0, 40)
    lo, hi = np.nonzero(off["hist"]["n"])[0][[0, -1]]
    tan_c = f.sin_c / f.cos_c
    assert lo == int(((8000.0 - 10.0) * tan_c - 50.0) // 5.0) and hi == int((8000.0 * tan_c + 50.0) // 5.0)
    # Fig. 3 quantities: density = sum_w / annulus area, mean time = sum_wt / sum_w, bins under 50 photons masked
    hist = np.zeros(3, dtype=O.HIST_DTYPE)
    hist["n"], hist["sum_w"], hist["sum_wt"] = [49, 50, 1000], [49.0, 100.0, 500.0], [490.0, 300.0, 2500.0]
    rc, dens, mt = O.profile(hist, 30.0)
    assert np.allclose(rc, [5.0, 15.0, 25.0])
    assert np.isnan(dens[0]) and np.isnan(mt[0])
    assert math.isclose(dens[1], 100.0 / (math.pi * (400.0 - 100.0))) and math.isclose(mt[1], 3.0)
    assert math.isclose(dens[2], 500.0 / (math.pi * (900.0 - 400.0))) and math.isclose(mt[2], 5.0)


def test_ground_histogram_counts_every_downward_bunch():
    """Conservation on a shower-shaped sample: bins + overflow = generated - upward."""
    cfg = W.make_config("c2", n_segments=300)
    res = O.ground_histogram(cfg["atmosphere"], cfg["segments"], cfg["params"], (0.0, 0.0), 500.0, 100)
    cnt = dict(zip(O.COUNTER_NAMES, (int(v) for v in res["counters"])))
    assert int(res["hist"]["n"].sum()) + res["overflow"] == cnt["generated"] - cnt["upward"] > 10000
    assert res["overflow"] > 0 and np.count_nonzero(res["hist"]["n"]) > 50


# ------------------------------------------------------------------ refraction corrections (R27)
def _snell_ray(atm, e_z, c_z, theta0, n_steps=200000):
    """Numerically integrated planar Snell ray: n(z) sin(theta(z)) = const, dx = tan(theta) dz (midpoint rule)."""
    edges = np.linspace(e_z, c_z, n_steps + 1)
    zm = 0.5 * (edges[1:] + edges[:-1])
    layers = atm["layers"]

    def eta(z):
        z = np.atleast_1d(np.asarray(z, dtype=np.float64))
        out = np.empty_like(z)
        for i, (h_lo, a, b, c) in enumerate(layers):
            h_hi = layers[i + 1][0] if i + 1 < len(layers) else np.inf
            m = (z >= h_lo) & (z < h_hi) if i else (z < h_hi)
            out[m] = atm["eta0"] * ((b / c) * np.exp(-z[m] / c) / 100.0) / atm["rho0"]
        return out

    k = (1.0 + eta(e_z)[0]) * math.sin(theta0)
    sin_t = k / (1.0 + eta(zm))
    x = np.sum(sin_t / np.sqrt(1.0 - sin_t ** 2)) * (e_z - c_z) / n_steps
    theta1 = math.asin(k / (1.0 + eta(c_z)[0]))
    return x - (e_z - c_z) * math.tan(theta0), theta1 - theta0


@pytest.mark.parametrize("atm", [ATM1, ATM5], ids=["one-layer", "five-layer"])
@pytest.mark.parametrize("theta_deg,e_z", [(4.0, 10000.0), (20.0, 6000.0), (45.0, 12000.0), (1.0, 3000.0)])
def test_refraction_corrections_against_integrated_snell_ray(atm, theta_deg, e_z):
    """R27's closed forms against a ray traced through the same n(z) in 2e5 altitude steps: they are first order in
    eta (3e-4 at most), so the agreement is to a few 1e-3 relative; both are negative (bending towards the vertical)."""
    th = math.radians(theta_deg)
    dr, dth = O.refraction(atm, e_z, 2000.0, -math.cos(th))
    dr_num, dth_num = _snell_ray(atm, e_z, 2000.0, th)
    assert dr < 0.0 and dth < 0.0
    assert math.isclose(dr, dr_num, rel_tol=3e-3), (dr, dr_num)
    assert math.isclose(dth, dth_num, rel_tol=3e-3), (dth, dth_num)


@pytest.mark.parametrize("atm", [ATM1, ATM5], ids=["one-layer", "five-layer"])
def test_refraction_first_order_validity_bound(atm):
    """Where R27's first-order forms hold: they drop terms of relative size O(eta tan^2 theta0).  Against the integrated
    Snell ray they stay within 3e-3 at zenith angles 55, 60, 65 and 75 degrees for emission at 12 and 30 km, and they
    have left that bound at 80 and 85 degrees -- which is where the oracle's cut-off |v_z| >= 0.25 (75.5 degrees) comes
    from: it is set by this error, not by any data structure of the GPU path."""
    for e_z in (12000.0, 30000.0):
        for deg in (55.0, 60.0, 65.0, 75.0):
            th = math.radians(deg)
            dr, dth = O.refraction(atm, e_z, 2000.0, -math.cos(th))
            dr_num, dth_num = _snell_ray(atm, e_z, 2000.0, th)
            assert math.isclose(dr, dr_num, rel_tol=3e-3) and math.isclose(dth, dth_num, rel_tol=3e-3), (e_z, deg, dr, dr_num)
        for deg in (80.0, 85.0):
            th = math.radians(deg)
            dr, _ = O.refraction(atm, e_z, 2000.0, -math.cos(th))
            dr_num, _ = _snell_ray(atm, e_z, 2000.0, th)
            assert abs(dr / dr_num - 1.0) > 3e-3, (e_z, deg, dr, dr_num)
    assert math.isclose(math.degrees(math.acos(0.25)), 75.52, abs_tol=0.01)


def _ray(zenith_deg, azimuth_deg=30.0):
    th, ph = math.radians(zenith_deg), math.radians(azimuth_deg)
    return np.array([math.sin(th) * math.cos(ph), math.sin(th) * math.sin(ph), -math.cos(th)])


def test_refraction_cutoff_moves_rays_inside_and_keeps_rays_outside():
    """A ray just steeper than the cut-off (|v_z| = 0.2501) arrives moved by dr along its horizontal flight direction and
    turned by dtheta; a ray just flatter (|v_z| = 0.2499) arrives where the straight line does, direction unchanged."""
    tel = np.array([0.0, 0.0, 2000.0, 1e9])
    e = np.array([100.0, -50.0, 9000.0])
    for vz, moved in ((0.2501, True), (0.2499, False), (0.5001, True), (0.4999, True), (0.9, True)):
        v = _ray(math.degrees(math.acos(vz)))
        hit0, _, _, sp0, x0, y0 = O.intersect(e, v, tel)
        hit1, _, _, sp1, x1, y1, vo = O.intersect_refracted(ATM5, e, v, tel)
        assert hit0 and hit1 and sp0 == sp1
        if moved:
            dr, dth = O.refraction(ATM5, e[2], 2000.0, v[2])
            hx, hy = v[0] / math.hypot(v[0], v[1]), v[1] / math.hypot(v[0], v[1])
            assert math.isclose(x1 - x0, dr * hx, rel_tol=1e-9) and math.isclose(y1 - y0, dr * hy, rel_tol=1e-9)
            assert math.isclose(math.acos(-vo[2]) - math.acos(-v[2]), dth, rel_tol=1e-6)
            assert abs(dr) > 0.05
        else:
            assert x1 == x0 and y1 == y0 and np.array_equal(vo, v)


def test_refraction_flips_the_hit_decision_on_a_small_sphere():
    """The sphere test runs on the corrected values: a 45-degree ray from 10 km above the plane lands 1.4 m short of its
    straight line, so a 0.9 m sphere centred 2 m behind the straight-line point (b = 2 cos 45 = 1.41 m: a miss) is hit
    once the correction is applied (b = 0.43 m), and a sphere centred on the straight-line point (a hit) is missed
    (b = 0.98 m)."""
    v = _ray(45.0, azimuth_deg=0.0)                                    # flies towards +x
    e = np.array([0.0, 0.0, 12000.0])
    dr, _ = O.refraction(ATM5, 12000.0, 2000.0, v[2])
    assert -1.6 < dr < -1.2
    x_line = 10000.0                                                   # straight-line plane crossing
    behind = np.array([x_line - 2.0, 0.0, 2000.0, 0.9])
    on_line = np.array([x_line, 0.0, 2000.0, 0.9])
    assert not O.intersect(e, v, behind)[0] and O.intersect(e, v, on_line)[0]
    hit_b, b2_b, *_ = O.intersect_refracted(ATM5, e, v, behind)
    hit_o, b2_o, *_ = O.intersect_refracted(ATM5, e, v, on_line)
    assert hit_b and math.isclose(math.sqrt(b2_b), abs(2.0 + dr) * math.cos(math.radians(45.0)), rel_tol=1e-3)
    assert not hit_o and math.isclose(math.sqrt(b2_o), abs(dr) * math.cos(math.radians(45.0)), rel_tol=1e-3)


def test_refraction_magnitude_and_vertical_ray():
    """SURVEY.md §8(f) quotes ~3 cm and ~7e-6 rad at 4 degrees from 8 km above the plane; a vertical ray is not moved."""
    dr, dth = O.refraction(ATM1, 10000.0, 2000.0, -math.cos(math.radians(4.0)))
    assert 0.01 < -dr < 0.06 and 3e-6 < -dth < 1.5e-5
    dr0, dth0 = O.refraction(ATM1, 10000.0, 2000.0, -1.0)
    assert dr0 == 0.0 and dth0 == 0.0


def test_refracted_records_move_by_the_corrections():
    """Whole path with the flag: every record of an accept-all plane detector is the unrefracted record moved by dr
    along the horizontal flight direction and turned by dtheta; times, wavelengths and weights are unchanged."""
    seg = one_segment(z0=9000.0, d=(0.3, -0.1, -1.0), length=5.0, gamma=1e6)
    par = W.default_params(bunch_size=0.5, seed=9)
    tel = W.telescope_accept_all()
    a = O.run(ATM5, tel, seg, par, record_capacity=10000)["records"]
    b = O.run(ATM5, tel, seg, dict(par, flags=O.FLAG_REFRACT), record_capacity=10000)["records"]
    assert len(a) == len(b) > 100 and np.array_equal(a["id"], b["id"])
    assert np.array_equal(a["t"], b["t"]) and np.array_equal(a["lam"], b["lam"]) and np.array_equal(a["w"], b["w"])
    for ra, rb in zip(a[:50], b[:50]):
        vz = -math.sqrt(1.0 - ra["cx"] ** 2 - ra["cy"] ** 2)
        sin0 = math.hypot(ra["cx"], ra["cy"])
        st, f = O.preamble(ATM5, par, seg[0], 0)
        ph = O.make_photon(f, par, 0, int(ra["id"]) & 0xFFFFFF, 0)
        dr, dth = O.refraction(ATM5, ph.e[2], 2000.0, vz)
        assert math.isclose(rb["x"] - ra["x"], dr * ra["cx"] / sin0, rel_tol=1e-6, abs_tol=1e-9)
        assert math.isclose(rb["y"] - ra["y"], dr * ra["cy"] / sin0, rel_tol=1e-6, abs_tol=1e-9)
        th_b = math.asin(math.hypot(rb["cx"], rb["cy"]))
        assert math.isclose(th_b - math.asin(sin0), dth, rel_tol=1e-5, abs_tol=1e-12)


# ------------------------------------------------------------------ beaming at the whole array (R28)
def test_array_beaming_solid_angle_and_photon_number():
    """Cone around the whole array with the paper's scaling of the photon NUMBER: closed-form solid angle, n_b and
    weight; inside the array (D <= R_b + L/2) the emission stays isotropic and unscaled."""
    tel = W.telescopes_square()                                     # (+-50, +-50, 2000), R = 6
    sph = O.array_sphere(tel)
    assert np.allclose(sph[:3], [0.0, 0.0, 2000.0]) and math.isclose(sph[3], math.hypot(50.0, 50.0) + 6.0, rel_tol=1e-12)
    par = W.default_params(processes=W.PROC_FLUORESCENCE, fl_beam_telescope=O.BEAM_ARRAY, bunch_size=1.0)
    seg = one_segment(x0=3000.0, y0=4000.0, z0=2000.0 + 12000.0, d=(0.0, 0.6, -0.8), length=20.0, dE=2.5e6)   # mu = 1e7
    st, f = O.preamble(ATM5, par, seg[0], 1, beam_tel=sph)
    mid = np.array([3000.0, 4000.0, 14000.0]) + 10.0 * np.array([0.0, 0.6, -0.8])
    D = np.linalg.norm(sph[:3] - mid)
    alpha = math.asin((sph[3] + 10.0) / D)
    frac = (1.0 - math.cos(alpha)) / 2.0
    assert st == 0 and f.kind == 2
    assert math.isclose(f.one_minus_cos_ab, 1.0 - math.cos(alpha), rel_tol=1e-9)
    mu = 4.0 * 2.5e6
    assert f.n_b == math.ceil(mu * frac / 1.0) and math.isclose(f.w0, mu * frac / f.n_b, rel_tol=1e-9)
    assert 0.5 < f.w0 <= 1.0 and f.n_b < 1e-4 * mu                   # the gain: far fewer bunches of about unit weight
    # inside the array: isotropic, unscaled
    seg_in = one_segment(x0=10.0, y0=0.0, z0=2030.0, length=5.0, dE=250.0)
    st, fi = O.preamble(ATM5, par, seg_in[0], 1, beam_tel=sph)
    assert st == 0 and fi.kind == 1 and fi.n_b == 1000 and fi.w0 == 1.0


def test_array_beaming_cone_holds_every_ray_to_every_telescope():
    """Brute force: from random points of the track to random points of every telescope sphere, the direction lies in
    the emission cone; and every emitted photon lies in it too."""
    tel = W.telescopes_grid(n=3, spacing=120.0)
    sph = O.array_sphere(tel)
    par = W.default_params(processes=W.PROC_FLUORESCENCE, fl_beam_telescope=O.BEAM_ARRAY, bunch_size=1.0, seed=21)
    seg = one_segment(x0=-900.0, y0=400.0, z0=4500.0, d=(0.5, 0.1, -0.86), length=300.0, dE=1e6)
    st, f = O.preamble(ATM5, par, seg[0], 1, beam_tel=sph)
    assert st == 0 and f.kind == 2
    p0, d, L = np.array(list(f.p0)), np.array(list(f.d)), f.L
    axis = sph[:3] - (p0 + 0.5 * L * d)
    axis /= np.linalg.norm(axis)
    cos_a = 1.0 - f.one_minus_cos_ab
    rng = np.random.Generator(np.random.PCG64(3))
    for k in range(len(tel)):
        c, R = tel[k, :3].astype(np.float64), float(tel[k, 3])
        for _ in range(200):
            e = p0 + rng.uniform(0.0, L) * d
            n = rng.normal(size=3)
            pt = c + R * rng.uniform(0.0, 1.0) ** (1 / 3) * n / np.linalg.norm(n)
            u = (pt - e) / np.linalg.norm(pt - e)
            assert u @ axis >= cos_a - 1e-12
    for j in range(0, f.n_b, max(1, f.n_b // 300)):
        v = np.array(list(O.make_photon(f, par, 0, j, 1).v))
        assert v @ axis >= cos_a - 1e-12


def test_array_beaming_keeps_the_expected_tally():
    """The scaled number of photons in the cone gives the same expected weighted tally as isotropic emission."""
    tel = np.array([[0.0, 0.0, 2000.0, 300.0], [500.0, 0.0, 2000.0, 200.0]], dtype=np.float32)
    seg = one_segment(x0=100.0, y0=50.0, z0=5000.0, length=1e-3, gamma=100.0, dE=2.5e5)      # mu = 1e6 at one point
    par_i = W.default_params(processes=W.PROC_FLUORESCENCE, seed=5)
    par_a = W.default_params(processes=W.PROC_FLUORESCENCE, seed=6, fl_beam_telescope=O.BEAM_ARRAY)
    ri = O.run(ATM5, tel, seg, par_i)
    ra = O.run(ATM5, tel, seg, par_a)
    assert int(ra["counters"][1]) < 0.1 * int(ri["counters"][1])      # far fewer photons generated
    for k in range(2):
        # isotropic: binomial with p_k = hits / n; the beamed run has the same expectation n p_k with unit-ish weights
        n_i = int(ri["counters"][1]); h_i = int(ri["tallies"]["hits"][k])
        sig = math.sqrt(h_i) + math.sqrt(ra["tallies"]["sum_w"][k])
        assert abs(ri["tallies"]["sum_w"][k] - ra["tallies"]["sum_w"][k]) < 5.0 * sig, (k, ri["tallies"][k], ra["tallies"][k])
        assert h_i > 500


def test_cherenkov_pair_shares_one_philox_block_R20():
    """R20: photons 2k and 2k + 1 of a Cherenkov emitter take the two halves of one Philox block; position and azimuth
    use the upper 23 bits of their two words, the wavelength the 18 lower bits left over.  Checked word by word on a
    few photons, and statistically: the three uniforms are uniform and mutually uncorrelated."""
    seg = one_segment(z0=9000.0, length=100.0, gamma=1e5)
    par = W.default_params(seed=(3 << 32) | 99, bunch_size=0.05)
    st, f = O.preamble(ATM1, par, seg[0], 0)
    S = 1234567
    inv1, inv2 = 1.0 / par["lam1"], 1.0 / par["lam2"]
    for j in (0, 1, 2, 7, 1000, 1001):
        ph = O.make_photon(f, par, S, j, 0)
        r = O.philox4x32_10([j >> 1, S & 0xFFFFFFFF, S >> 32, 0], [99, 3])
        a, b = int(r[2 * (j & 1)]), int(r[2 * (j & 1) + 1])
        u1 = ((a >> 9) + 0.5) / 2 ** 23
        u3 = ((((a & 511) << 9) | (b & 511)) + 0.5) / 2 ** 18
        assert math.isclose(ph.e[2], 9000.0 - u1 * 100.0, rel_tol=0, abs_tol=1e-9)
        assert math.isclose(ph.lam, 1.0 / (inv1 - u3 * (inv1 - inv2)), rel_tol=1e-13)
    n = min(f.n_b, 40000) & ~1
    u = np.empty((n, 3))
    for j in range(n):
        ph = O.make_photon(f, par, S, j, 0)
        u[j, 0] = (9000.0 - ph.e[2]) / 100.0
        u[j, 1] = (math.atan2(ph.v[1], ph.v[0]) / (2 * math.pi)) % 1.0
        u[j, 2] = (inv1 - 1.0 / ph.lam) / (inv1 - inv2)
    assert np.all(np.abs(u.mean(axis=0) - 0.5) < 5 * math.sqrt(1 / 12 / n))
    assert np.all(np.abs(u.var(axis=0) - 1 / 12) < 0.005)
    c = np.corrcoef(u.T)
    assert abs(c[0, 1]) < 0.03 and abs(c[0, 2]) < 0.03 and abs(c[1, 2]) < 0.03
    # neighbours 2k, 2k + 1 are as independent as any other two photons
    assert abs(np.corrcoef(u[0::2, 0], u[1::2, 0])[0, 1]) < 0.03 and abs(np.corrcoef(u[0::2, 2], u[1::2, 2])[0, 1]) < 0.03


# ------------------------------------------------------------------ angular particle cut (R29)
def _tilted(axis, deg, azimuth_deg=40.0):
    """Unit vector at `deg` degrees from the unit vector `axis` (independent construction: Gram-Schmidt + cos / sin)."""
    axis = np.asarray(axis, dtype=np.float64) / np.linalg.norm(axis)
    t = np.cross(axis, [0.3, -0.2, 0.9]); t /= np.linalg.norm(t)
    s = np.cross(axis, t)
    a, ph = math.radians(deg), math.radians(azimuth_deg)
    return math.cos(a) * axis + math.sin(a) * (math.cos(ph) * t + math.sin(ph) * s)


def test_particle_cut_hand_built_angles():
    """A segment whose midpoint is 8 km above and 3 km beside the experiment centre: kept while its direction is within the
    cut of the line to the centre, cut beyond; the angle is re-measured here with an inverse cosine (the oracle uses
    none).  The vector starts at the MIDPOINT of the segment (R29)."""
    tel = W.telescopes_square()                                       # centre (0, 0, 2000)
    mid = np.array([3000.0, -1000.0, 10000.0])
    to_centre = np.array([0.0, 0.0, 2000.0]) - mid
    cut = math.radians(6.0)
    for deg, expect_cut in ((0.0, False), (5.9, False), (5.999, False), (6.001, True), (6.1, True), (90.0, True), (170.0, True)):
        d = _tilted(to_centre, deg)
        L = 40.0
        p0 = mid - 0.5 * L * d
        ang = math.acos(np.clip(np.dot(d, to_centre) / np.linalg.norm(to_centre), -1.0, 1.0))
        assert math.isclose(ang, math.radians(deg), abs_tol=1e-9)
        assert O.particle_cut(p0, d, L, tel, 1, cut) is expect_cut
    # measured from the start point instead, a long segment would be judged differently: 2 km long, aimed at the centre from its midpoint
    d = to_centre / np.linalg.norm(to_centre)
    assert not O.particle_cut(mid - 1000.0 * d, d, 2000.0, tel, 1, math.radians(0.01))
    assert not O.particle_cut(mid, d, 0.0, tel, 0, 0.0)               # mode 0: never cut


def test_particle_cut_nearest_telescope_mode():
    """Mode 2 ("the minimum angle to each individual telescope"): a segment aimed at a telescope 400 m from
    the array centre, 3 km up, is 7.6 degrees off the centre (cut at 6 degrees in mode 1) but 0 degrees off that telescope
    (kept in mode 2); aimed 6.5 degrees off every telescope it is cut in both."""
    tel = np.array([[400.0, 0.0, 2000.0, 6.0], [-400.0, 0.0, 2000.0, 6.0], [0.0, 400.0, 2000.0, 6.0], [0.0, -400.0, 2000.0, 6.0]], dtype=np.float32)
    mid = np.array([400.0, 0.0, 5000.0])
    d = np.array([0.0, 0.0, -1.0])
    cut = math.radians(6.0)
    off_centre = math.degrees(math.atan2(400.0, 3000.0))
    assert 7.5 < off_centre < 7.7
    assert O.particle_cut(mid - 5.0 * d, d, 10.0, tel, 1, cut) and not O.particle_cut(mid - 5.0 * d, d, 10.0, tel, 2, cut)
    far = np.array([5000.0, 5000.0, 9000.0])
    assert O.particle_cut(far, d, 10.0, tel, 1, cut) and O.particle_cut(far, d, 10.0, tel, 2, cut)
    # brute force over random segments: mode 2 cuts exactly those whose smallest angle (arccos) exceeds the cut
    rng = np.random.Generator(np.random.PCG64(11))
    n_cut = 0
    for _ in range(300):
        p0 = np.array([rng.uniform(-2000, 2000), rng.uniform(-2000, 2000), rng.uniform(3000, 12000)])
        dd = _tilted([0.0, 0.0, -1.0], rng.uniform(0.0, 25.0), rng.uniform(0.0, 360.0))
        L = rng.uniform(0.0, 30.0)
        m = p0 + 0.5 * L * dd
        angs = [math.acos(np.clip(np.dot(dd, t[:3] - m) / np.linalg.norm(t[:3] - m), -1, 1)) for t in tel.astype(np.float64)]
        if abs(min(angs) - cut) < 1e-6:
            continue
        assert O.particle_cut(p0, dd, L, tel, 2, cut) is (min(angs) > cut)
        n_cut += min(angs) > cut
    assert 50 < n_cut < 280


def test_particle_cut_in_the_whole_path():
    """With the cut, the run is the uncut run restricted to the kept segments: same records for them, none for the
    others; every bunch still counts as generated, the bunches of cut segments are reported; fluorescence is never cut."""
    cfg = W.make_config("c2", n_segments=3000)
    cfg["telescopes"][:, 3] = 40.0
    par = dict(cfg["params"], processes=3, fl_yield=20.0)
    a = O.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"], par, record_capacity=1 << 20)
    cut = math.radians(3.0)
    b = O.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"], dict(par, flags=O.FLAG_CUT_CENTRE, cut_angle=cut), record_capacity=1 << 20)
    assert np.array_equal(a["counts"], b["counts"])
    ca, cb = (dict(zip(O.COUNTER_NAMES, (int(v) for v in r["counters"]))) for r in (a, b))
    assert ca["cut"] == 0 and cb["generated"] == ca["generated"]
    seg = cfg["segments"]
    dn = np.stack([seg["dx"], seg["dy"], seg["dz"]], axis=1).astype(np.float64)
    dn /= np.linalg.norm(dn, axis=1, keepdims=True)
    mid = np.stack([seg["x0"], seg["y0"], seg["z0"]], axis=1).astype(np.float64) + 0.5 * seg["length"].astype(np.float64)[:, None] * dn
    u = np.array([0.0, 0.0, 2000.0]) - mid
    ang = np.arccos(np.clip(np.sum(dn * u, axis=1) / np.linalg.norm(u, axis=1), -1, 1))
    is_cut = ang > cut
    assert 0.2 < is_cut.mean() < 0.95
    assert cb["cut"] == int(a["counts"][is_cut, 0].astype(np.int64).sum())
    ra, rb = a["records"], b["records"]
    keep = ~(is_cut[(ra["id"] >> 25).astype(np.int64)] & (((ra["id"] >> 24) & 1) == 0))
    ra = ra[keep]
    ka, kb = np.lexsort((ra["tel"], ra["id"])), np.lexsort((rb["tel"], rb["id"]))
    assert len(ra) == len(rb) and 0 < len(rb) < len(a["records"])
    for f in ("id", "tel", "x", "y", "t", "w"):
        assert np.array_equal(ra[f][ka], rb[f][kb])
    assert int(((rb["id"] >> 24) & 1).sum()) == int(((a["records"]["id"] >> 24) & 1).sum()) > 0      # fluorescence untouched


# ------------------------------------------------------------------ sanitizers
def test_oracle_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """The oracle's C built with -fsanitize=address,undefined (errors abort) runs every branch of the whole path on a
    small case -- both processes, transmission table, refraction, the particle cut, array beaming, records up to and
    beyond their capacity, the ground histogram, threads -- and gives the same result as the plain build."""
    import subprocess
    import sys
    src = os.path.join(os.path.dirname(O.__file__), "c8opt_oracle.c")
    san = str(tmp_path / "liboracle_san.so")
    subprocess.check_call(["gcc", "-std=c99", "-O1", "-g", "-ffp-contract=off", "-fPIC", "-shared", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=all", "-o", san, src, "-lm"])
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    script = r"""
import sys, numpy as np
sys.path.insert(0, %r)
import oracle as O, workloads as W
cfg = W.make_config("c4", n_segments=400)
par = dict(cfg["params"], flags=O.FLAG_REFRACT | O.FLAG_CUT_TELESCOPES, cut_angle=0.2)
a = O.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"], par, record_capacity=1 << 16, threads=3)
b = O.run(cfg["atmosphere"], cfg["telescopes"], cfg["segments"], dict(par, fl_beam_telescope=O.BEAM_ARRAY), record_capacity=8)
h = O.ground_histogram(cfg["atmosphere"], cfg["segments"], cfg["params"], (1.0, 2.0), 800.0, 40, threads=2)
c1 = W.make_config("c3b", n_segments=300)
c = O.run(c1["atmosphere"], c1["telescopes"], c1["segments"], c1["params"], record_capacity=1 << 12)
print(int(a["tallies"]["hits"].sum()), int(a["counters"][7]), int(b["counters"][5]), int(h["hist"]["n"].sum()), int(c["counters"][1]))
""" % os.path.dirname(os.path.dirname(O.__file__))
    outs = []
    for env_extra in ({"LD_PRELOAD": asan, "C8OPT_ORACLE_LIB": san, "ASAN_OPTIONS": "detect_leaks=0"}, {}):
        env = dict(os.environ, **env_extra)
        r = subprocess.run([sys.executable, "-c", script], env=env, capture_output=True, text=True, timeout=600)
        assert r.returncode == 0, r.stderr[-2000:]
        outs.append(r.stdout.strip().splitlines()[-1])
    assert outs[0] == outs[1] and int(outs[0].split()[0]) > 100 and int(outs[0].split()[2]) > 0


# ------------------------------------------------------------------ wavelength-dependent refractive index (R30)
def _sin2_disp(eta, beta2, b, x):
    n = 1.0 + eta * (1.0 + b * x * x)
    return 1.0 - 1.0 / (beta2 * n * n)


def test_dispersion_integral_against_fine_quadrature_and_the_closed_form():
    """The Frank-Tamm lambda integral with n(lambda) - 1 = eta (1 + b / lambda^2): the oracle's 16-interval Simpson rule
    against a 2e5-point trapezoid of the same integrand (1e-9 relative: the integrand is a smooth, nearly quadratic
    function of x = 1 / lambda), and with b -> 0 against the closed form sin^2 theta_c (1/lam1 - 1/lam2) of R2."""
    x1, x2 = 1.0 / 300.0, 1.0 / 600.0
    for eta, gamma, b in ((2.83e-4, 1e4, 5670.0), (1.0e-4, 200.0, 5670.0), (2.2e-4, 80.0, 20000.0)):
        beta2 = 1.0 - 1.0 / gamma ** 2
        xs = np.linspace(x2, x1, 200001)
        ref = np.trapezoid(np.maximum(0.0, _sin2_disp(eta, beta2, b, xs)), xs)
        got = O.dispersion_integral(eta, beta2, b, x1, x2)
        assert ref > 0 and math.isclose(got, ref, rel_tol=1e-9), (got, ref)
    eta, beta2 = 2.83e-4, 1.0 - 1e-8
    closed = (1.0 - 1.0 / (beta2 * (1 + eta) ** 2)) * (x1 - x2)
    assert math.isclose(O.dispersion_integral(eta, beta2, 0.0, x1, x2), closed, rel_tol=1e-11)        # (1 - 1 / (beta n)^2 cancels 3 digits)
    # dispersion raises the yield: n is larger at every wavelength of the band
    assert O.dispersion_integral(eta, beta2, 5670.0, x1, x2) > closed * 1.03


def test_dispersion_threshold_inside_the_band():
    """A particle that is above the Cherenkov threshold only for the blue end of the band (n grows towards short
    wavelengths): the integrand is cut at 0 (the Theta of PAPER.md:45), the integral is that of the radiating part --
    to the accuracy of a 16-interval rule across a kink, a few 1e-3 -- and far below the no-threshold value."""
    eta, b = 2.0e-4, 5670.0
    x1, x2 = 1.0 / 300.0, 1.0 / 600.0
    n_mid = 1.0 + eta * (1.0 + b * (0.5 * (x1 + x2)) ** 2)
    beta2 = 1.0 / n_mid ** 2                                   # threshold exactly at the middle of the band in x
    xs = np.linspace(x2, x1, 400001)
    f = _sin2_disp(eta, beta2, b, xs)
    assert f[0] < 0 < f[-1]
    ref = np.trapezoid(np.maximum(0.0, f), xs)
    got = O.dispersion_integral(eta, beta2, b, x1, x2)
    assert math.isclose(got, ref, rel_tol=2e-2) and got < 0.3 * abs(np.trapezoid(np.abs(f), xs)) + ref


def test_dispersion_photons_leave_at_the_angle_of_their_wavelength():
    """R30 per photon: v . d = 1 / (beta n(lambda)) with n(lambda) - 1 = eta (1 + b / lambda^2), weight = w0 sin^2(lambda) /
    <sin^2>, so that the weights of all bunches sum to mu; blue photons open wider than red ones; with b = 0 the
    photons are those of R2 - R4 bit for bit."""
    seg = one_segment(z0=8000.0, d=(0.1, 0.2, -1.0), length=30.0, gamma=300.0)
    par0 = W.default_params(bunch_size=0.05, seed=5)
    par = dict(par0, cauchy_b=5670.0)
    st, f = O.preamble(ATM5, par, seg[0], 0)
    st0, f0 = O.preamble(ATM5, par0, seg[0], 0)
    assert st == 0 and f.n_b > f0.n_b > 2000
    eta = O.refractivity(ATM5, 8000.0 + 0.5 * 30.0 * f.d[2])
    beta2 = 1.0 - 1.0 / 300.0 ** 2
    assert math.isclose(f.mu, 2 * math.pi * 7.2973525693e-3 * 1e9 * 30.0 * O.dispersion_integral(eta, beta2, 5670.0, 1 / 300.0, 1 / 600.0), rel_tol=1e-12)
    sw, cs = 0.0, []
    for j in range(f.n_b):
        ph = O.make_photon(f, par, 0, j, 0)
        n = 1.0 + eta * (1.0 + 5670.0 / ph.lam ** 2)
        cos_c = 1.0 / (math.sqrt(beta2) * n)
        assert math.isclose(float(np.dot(ph.v, f.d)), cos_c, rel_tol=0, abs_tol=1e-12)
        assert math.isclose(ph.w, f.w0 * (1.0 - cos_c ** 2) / f.disp_mean, rel_tol=1e-9)
        sw += ph.w; cs.append((ph.lam, cos_c))
    assert math.isclose(sw, f.mu, rel_tol=0.02)                      # Monte-Carlo mean of sin^2 over the band
    cs.sort()
    assert cs[0][1] < cs[-1][1]                                      # shortest wavelength: smallest cos, widest cone
    for j in (0, 1, 17):
        a, b_ = O.make_photon(f0, par0, 0, j, 0), O.make_photon(f0, dict(par0, cauchy_b=0.0), 0, j, 0)
        assert tuple(a.v) == tuple(b_.v) and a.w == b_.w and a.lam == b_.lam
