"""Pins of the CPU oracle against what the paper and the mathematics fix (-m "not gpu").

Each pin is something other than the oracle itself: values the thesis prints
(tests/golden), closed forms, invariants, limits that reduce to textbook
results, brute force on tiny inputs.  P:n = PAPER.md line n.
"""
import copy
import ctypes as C
import math
import os

import numpy as np
import pytest
import scipy.constants as sc
from scipy import stats

from oracle import c8ph_oracle as O
from paper_2405_04229_b200 import workloads as W

C_LIGHT = sc.c * 1e-9  # m/ns


# ------------------------------------------------------------------ O0 RNG
def test_philox_known_answers(golden_dir):
    n = 0
    for line in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        w = [int(t, 16) for t in line.split()]
        assert O.philox4x32_10(w[0:4], w[4:6]) == w[6:10]
        n += 1
    assert n == 3


def test_philox_bijective_and_uniform():
    outs = set()
    words = []
    for j in range(1 << 12):
        r = O.philox4x32_10([j, 7, 0, 0], [1, 0])
        outs.add(tuple(r))
        words.append(r)
    assert len(outs) == 1 << 12                       # a bijection never collides
    words = np.array(words, dtype=np.uint64)
    for k in range(4):                                # equidistribution of the top byte
        cnt = np.bincount((words[:, k] >> 24).astype(int), minlength=256)
        assert stats.chisquare(cnt).pvalue > 1e-4


def test_uniform_is_exact_in_fp32_and_open_interval():
    for r in (0, 1, 511, 512, 0x7FFFFFFF, 0xFFFFFFFF, 123456789):
        u = O.uniform(r)
        assert 0.0 < u < 1.0
        assert float(np.float32(u)) == u              # (2m+1) 2^-24 is an fp32 number
        assert u == ((r >> 9) * 2 + 1) / 2.0 ** 24


# ------------------------------------------------------------------ O1 yield
def test_frank_tamm_closed_form():
    # Eq. 2.3: alpha = e^2 / (2 h eps0 c) from CODATA, not from the oracle's constant
    alpha = sc.e ** 2 / (2 * sc.h * sc.epsilon_0 * sc.c)
    n = 1.000293
    for beta in (1.0, 0.9999):
        want = 2 * math.pi * alpha * (1 / 300e-9 - 1 / 600e-9) * (1 - 1 / (beta * n) ** 2)
        got = O.cherenkov_yield(1.0, 1.0, beta, n, 300.0, 600.0)
        assert got == pytest.approx(want, rel=2e-8)
    assert O.cherenkov_yield(1.0, 1.0, 1.0, n, 300.0, 600.0) == pytest.approx(44.761, abs=2e-3)
    assert O.cherenkov_yield(-2.0, 3.0, 1.0, n, 300.0, 600.0) == pytest.approx(4 * 3 * 44.7611, rel=1e-5)


def test_cherenkov_threshold():
    n = 1.000293
    beta_th = 1.0 / n
    assert O.cherenkov_yield(1, 1, beta_th * (1 - 1e-9), n, 300, 600) == 0.0
    assert O.cherenkov_yield(1, 1, beta_th * (1 + 1e-9), n, 300, 600) > 0.0
    gamma_th = 1 / math.sqrt(1 - beta_th ** 2)
    assert gamma_th == pytest.approx(41.32, abs=0.01)  # sea-level electron threshold gamma


# ------------------------------------------------------------------ O4 rotation / cone
def test_rodrigues_properties():
    rng = np.random.default_rng(5)
    D = np.array([0.0, 0.0, -1.0])
    for _ in range(50):
        P = rng.normal(size=3)
        P /= np.linalg.norm(P)
        M = O.rodrigues(P)
        assert np.allclose(M @ D, P, atol=1e-14)       # maps the cone axis onto the particle
        assert np.allclose(M, M.T, atol=1e-15)
        assert np.allclose(M @ M, np.eye(3), atol=1e-14)
        assert np.linalg.det(M) == pytest.approx(1.0, abs=1e-13)
    M = O.rodrigues([0.0, 0.0, 1.0])                   # degenerate bisector
    assert np.allclose(M @ D, [0, 0, 1])
    # P = D: a half turn about the axis itself (M = 1 + 2 R^2 of P:706 with A = D)
    assert np.allclose(O.rodrigues([0.0, 0.0, -1.0]), np.diag([-1.0, -1.0, 1.0]))


def test_cone_direction_angle_norm_azimuth(golden_dir):
    facts = dict(l.split(None, 1) for l in open(os.path.join(golden_dir, "paper_facts.txt")) if not l.startswith("#"))
    rng = np.random.default_rng(6)
    P = np.array([0.3, -0.2, -0.9])
    P /= np.linalg.norm(P)
    M = O.rodrigues(P)
    cos_th = 1 / 1.000293
    sin_th = math.sqrt(1 - cos_th ** 2)
    # the thesis: opening angle in air "less than 1.4 deg"
    assert math.degrees(math.acos(cos_th)) < float(facts["cherenkov_angle_max_deg"])
    assert math.degrees(math.acos(cos_th)) == pytest.approx(1.3868, abs=1e-4)
    e1, e2 = M[:, 0], M[:, 1]
    az = []
    for phi in rng.uniform(0, 2 * math.pi, 4000):
        u = O.cone_direction(M, cos_th, sin_th, phi)
        assert abs(np.dot(u, P) - cos_th) < 1e-13
        assert abs(np.linalg.norm(u) - 1) < 1e-13
        az.append(math.atan2(np.dot(u, e2), np.dot(u, e1)))
    cnt = np.histogram(az, bins=16, range=(-math.pi, math.pi))[0]
    assert stats.chisquare(cnt).pvalue > 1e-4
    # local vector of P:680 for the un-rotated axis
    u = O.cone_direction(np.eye(3).ravel(), cos_th, sin_th, 0.25)
    assert np.allclose(u, [math.cos(0.25) * sin_th, math.sin(0.25) * sin_th, -cos_th])


# ------------------------------------------------------------------ O7 straight line, O2/O13 time
def _one_segment_cfg(z=10000.0, L=10.0, beta=1.0, d=(0.0, 0.0, -1.0), x=0.0, y=0.0):
    cfg = W.make_config(0, n_segments=1)
    s = cfg["segments"]
    s["x"][:], s["y"][:], s["z"][:] = x, y, z
    s["dx"][:], s["dy"][:], s["dz"][:] = d
    s["len"][:], s["beta"][:], s["t0"][:], s["charge"][:] = L, beta, 100.0, 1.0
    cfg["detector"].update(hist_nx=0, hist_ny=0)
    return cfg


def test_straight_line_plane_hit():
    I, t = O.straight_line([1.0, 2.0, 50.0], [0.6, 0.0, -0.8])
    assert np.allclose(I, [1 + 62.5 * 0.6, 2.0, 0.0]) and t == pytest.approx(62.5)


def test_constant_n_ring_and_arrival_time():
    """Exact constant-n limit: a vertical beta=1 particle lights the ring r = (Z-s) tan(theta_c)."""
    cfg = _one_segment_cfg()
    ph = O.run(cfg)["photons"]
    assert len(ph) > 300 and np.all(ph["status"] == O.ST_LANDED)
    n = float(np.float32(0.000293)) + 1.0
    tan_c = math.sqrt(n * n - 1.0)
    r = np.hypot(ph["x"], ph["y"])
    assert r.max() <= 10000.0 * tan_c + 1e-9 and r.min() >= 9990.0 * tan_c - 1e-9
    assert r.max() == pytest.approx(242.1, abs=0.3)    # 10 km * tan(1.3868 deg)
    # t = t0 + s/(beta c) + n D / c with D = (Z - s)/cos(theta_c)
    zs = r / tan_c
    s = 10000.0 - zs
    t = 100.0 + s / C_LIGHT + n * (zs * n) / C_LIGHT
    assert np.allclose(ph["t"], t, atol=1e-9, rtol=0)
    # direction keeps the cone angle
    assert np.allclose(-ph["uz"], 1 / n, atol=1e-13)
    assert abs(np.mean(s) - 5.0) < 5 * 10 / math.sqrt(12 * len(s))           # O2: uniform on the track


def test_emission_at_or_below_the_observation_level_is_dropped():
    """Reading R7 (Eq. 3.3 P:495 needs t* = -A_z/u_z > 0): a vertical track that straddles z = 0 lands the
    photons emitted above the plane on the analytic ring r = z_e tan(theta_c) and drops the others as up-going.  The
    emission point of every photon is re-derived here from the (known-answer pinned) Philox words, not from the run."""
    cfg = _one_segment_cfg(z=5.0, L=10.0)
    cfg["segments"]["charge"][:] = 3.0                                # 9x the photons
    res = O.run(cfg)
    ph = res["photons"]
    assert len(ph) > 3000
    n = float(np.float32(0.000293)) + 1.0
    tan_c = math.sqrt(n * n - 1.0)
    seed = cfg["seed"]
    s = np.array([O.uniform(O.philox4x32_10([int(j), 0, 0, 0], [seed & 0xFFFFFFFF, seed >> 32])[1]) * 10.0 for j in ph["j"]])
    z_e = 5.0 - s
    above = z_e > 0.0
    assert 0.4 < above.mean() < 0.6
    assert np.all(ph["status"][above] == O.ST_LANDED) and np.all(ph["status"][~above] == O.ST_UPGOING)
    assert np.allclose(np.hypot(ph["x"], ph["y"])[above], z_e[above] * tan_c, atol=1e-9, rtol=0)
    c = res["counters"]
    assert c["upgoing"] == int((~above).sum()) and c["landed"] == int(above.sum())
    # a track that ends exactly on the plane keeps every photon (z_e > 0 for s < L), one that starts on it keeps none
    assert np.all(O.run(_one_segment_cfg(z=10.0, L=10.0))["photons"]["status"] == O.ST_LANDED)
    assert np.all(O.run(_one_segment_cfg(z=0.0, L=10.0))["photons"]["status"] == O.ST_UPGOING)


def test_telescope_tie_break_earliest_entry_then_lowest_index():
    """O12 / R12: among several bounding spheres the ray enters, the earliest entry wins, then the lowest index.
    Two overlapping spheres (the second one raised, so that it is entered earlier by part of the rays) and an exact
    duplicate of each; entry parameters recomputed here in closed form from the photon records."""
    cfg = _one_segment_cfg(z=1000.0, L=200.0)
    cfg["segments"]["charge"][:] = 2.0
    tel = np.array([[20.0, 0.0, 0.0, 10.0], [25.0, 0.0, 5.0, 10.0], [25.0, 0.0, 5.0, 10.0], [20.0, 0.0, 0.0, 10.0]], dtype=np.float32)
    cfg["detector"]["tel_xyzr"] = tel
    ph = O.run(cfg)["photons"]
    ph = ph[ph["status"] == O.ST_LANDED]
    I = np.stack([ph["x"], ph["y"], np.zeros(len(ph))], axis=1)
    u = np.stack([ph["ux"], ph["uy"], ph["uz"]], axis=1)
    s_in = np.full((len(ph), 4), np.inf)
    for k in range(4):
        d = tel[k, :3].astype(np.float64) - I
        du = (d * u).sum(axis=1)
        m2 = (d * d).sum(axis=1) - du * du
        hit = m2 <= float(tel[k, 3]) ** 2
        s_in[hit, k] = du[hit] - np.sqrt(float(tel[k, 3]) ** 2 - m2[hit])
    want = np.where(np.isfinite(s_in.min(axis=1)), s_in.argmin(axis=1), -1)   # argmin returns the lowest index on ties
    both = np.isfinite(s_in[:, 0]) & np.isfinite(s_in[:, 1])
    gap = np.ones(len(ph))
    gap[both] = np.abs(s_in[both, 0] - s_in[both, 1])
    clear = gap > 1e-6                                                # not within rounding of an exact tie of k0 and k1
    assert np.array_equal(ph["tel"][clear], want[clear])
    assert not np.any(np.isin(ph["tel"], (2, 3)))                     # a duplicate never wins against its lower index
    print("both & k0 / both & k1 / k0 only / k1 only / none:", (both & (want == 0)).sum(), (both & (want == 1)).sum(),
          (~both & (want == 0)).sum(), (~both & (want == 1)).sum(), (want == -1).sum())
    assert (both & (want == 0)).sum() > 20 and (both & (want == 1)).sum() > 20 and (want == -1).sum() > 100
    assert (~both & (want >= 0)).sum() > 5                             # rays that enter one sphere only


def test_wavelength_law():
    cfg = _one_segment_cfg(L=200.0)
    ph = O.run(cfg)["photons"]
    lam = ph["lambda_nm"]
    assert lam.min() >= 300.0 and lam.max() <= 600.0
    # CDF of a 1/lambda^2 spectrum: F = (1/l1 - 1/l)/(1/l1 - 1/l2)
    cdf = lambda l: (1 / 300.0 - 1 / l) / (1 / 300.0 - 1 / 600.0)
    assert stats.kstest(lam, cdf).pvalue > 1e-3
    sig = (1 / 300 - 1 / 600) / math.sqrt(12 * len(lam))
    assert abs(np.mean(1 / lam) - 0.5 * (1 / 300 + 1 / 600)) < 5 * sig


# ------------------------------------------------------------------ O8 refraction
def _linear_atm(model="planar", n_g=1.5, n_top=1.0, h_top=100000.0):
    atm = W.make_atmosphere("planar_exp")
    h = atm["h0"] + atm["dh"] * np.arange(atm["n_nodes"])
    atm["refractivity"] = ((n_g - 1.0) + (n_top - n_g) * h / h_top).astype(np.float32)
    atm["model"] = model
    return atm


def test_trace_linear_profile_closed_form(golden_dir):
    """Thesis' test medium n = 1.5 -> 1.0 over 100 km; closed forms of the differential
    Snell law (Eq. 3.20, Eq. 3.23 with the integration constant's sign fixed)."""
    atm = _linear_atm()
    eta = atm["refractivity"].astype(np.float64)
    n_of = lambda h: 1.0 + np.interp(h, atm["dh"] * np.arange(len(eta)), eta)
    h_e, th = 50000.0, math.radians(45.0)
    n_e, n_g = n_of(h_e), n_of(0.0)
    b = abs((1.0 - 1.5) / 100000.0)
    K = n_e * math.sin(th)
    X = K / b * (math.acosh(n_g / K) - math.acosh(n_e / K))
    S = (math.sqrt(n_g ** 2 - K ** 2) - math.sqrt(n_e ** 2 - K ** 2)) / b
    F = lambda x: 0.5 * (x * math.sqrt(x * x - K * K) + K * K * math.acosh(x / K))
    cT = (F(n_g) - F(n_e)) / b
    assert X == pytest.approx(42375.7267, abs=0.05) and S == pytest.approx(65607.2976, abs=0.05)
    r1 = O.trace(atm, False, h_e, th, 0.0, sub=1)
    r4 = O.trace(atm, False, h_e, th, 0.0, sub=4)
    for key, want in (("disp", X), ("S", S), ("cT", cT)):
        e1, e4 = abs(r1[key] - want), abs(r4[key] - want)
        assert e1 / want < 1e-3                        # the thesis' own bound: <= 0.1 %
        assert e1 < 2e-3 and e4 < 2e-4, (key, e1, e4)  # second-order convergence to the closed form
    # Eq. 3.20: sin(nu) = c sin(alpha) / (c - y) -> arrival angle
    assert r1["sin_arr"] == pytest.approx(K / n_g, abs=1e-13)


def test_trace_invariants_and_limits():
    atm = W.make_atmosphere("spherical_5layer")
    R = atm["earth_radius"]
    for h_e, zen in ((10000.0, 20.0), (25000.0, 60.0), (5000.0, 75.0), (60000.0, 80.0)):
        th = math.radians(zen)
        n_e = 1 + O.refractivity(atm, h_e)
        n_g = 1 + O.refractivity(atm, 0.0)
        rp = O.trace(atm, False, h_e, th, 0.0)
        assert n_g * rp["sin_arr"] == pytest.approx(n_e * math.sin(th), rel=1e-13)          # Snell
        rs = O.trace(atm, True, h_e, th, 0.0)
        assert n_g * R * rs["sin_arr"] == pytest.approx(n_e * (R + h_e) * math.sin(th), rel=1e-12)  # Bouguer
        assert rs["S"] > rp["S"] * 0.999 and rs["cT"] > rs["S"]
    # constant n: the trace is the straight line
    hom = W.make_atmosphere("homogeneous")
    hom["model"] = "planar"
    r = O.trace(hom, False, 10000.0, math.radians(40), 0.0)
    assert r["disp"] == pytest.approx(10000 * math.tan(math.radians(40)), rel=1e-13)
    assert r["S"] == pytest.approx(10000 / math.cos(math.radians(40)), rel=1e-13)
    assert r["cT"] == pytest.approx(r["S"] * (1 + float(np.float32(0.000293))), rel=1e-13)
    hom["model"] = "spherical"
    r = O.trace(hom, True, 10000.0, math.radians(40), 0.0)
    re, rg, th = R + 10000.0, R, math.radians(40)
    assert r["disp"] == pytest.approx(math.asin(re * math.sin(th) / rg) - th, rel=1e-9)
    assert r["S"] == pytest.approx(re * math.cos(th) - math.sqrt(rg ** 2 - (re * math.sin(th)) ** 2), rel=1e-10)
    # R -> infinity: spherical -> planar
    big = copy.deepcopy(atm)
    big["earth_radius"] = 1e10
    rp = O.trace(atm, False, 12000.0, math.radians(50), 0.0)
    rs = O.trace(big, True, 12000.0, math.radians(50), 0.0)
    assert rs["disp"] * 1e10 == pytest.approx(rp["disp"], rel=2e-5)
    assert rs["S"] == pytest.approx(rp["S"], rel=2e-5) and rs["X"] == pytest.approx(rp["X"], rel=2e-5)
    # beyond the horizon: no ground
    assert O.trace(atm, True, 5000.0, math.radians(88.5), 0.0) is None
    assert O.trace(atm, True, 5000.0, math.radians(85.0), 0.0) is not None


def _brute_force_ray(atm, spherical, h_e, zen, h_g, ds=0.5):
    """Fine-step RK4 integration of the ray equation d/ds(n u) = grad n in the medium defined by
    the linearly interpolated table (independent numpy code)."""
    eta = atm["refractivity"].astype(np.float64)
    dh = atm["dh"]
    R = atm["earth_radius"]

    def n_and_grad(p):
        if spherical:
            r = math.hypot(p[0], p[1])
            h = r - R
            up = np.array([p[0] / r, p[1] / r])
        else:
            h = p[1]
            up = np.array([0.0, 1.0])
        f = min(max(h / dh, 0.0), len(eta) - 1.000001)
        i = int(f)
        return 1 + eta[i] + (f - i) * (eta[i + 1] - eta[i]), (eta[i + 1] - eta[i]) / dh * up, h

    def rhs(y):
        p, T = y[:2], y[2:4]
        n, g, _ = n_and_grad(p)
        return np.array([T[0] / n, T[1] / n, g[0], g[1], n])

    p0 = np.array([0.0, (R if spherical else 0.0) + h_e])
    n0, _, _ = n_and_grad(p0)
    y = np.array([p0[0], p0[1], n0 * math.sin(zen), -n0 * math.cos(zen), 0.0])
    S = 0.0
    while True:
        k1 = rhs(y); k2 = rhs(y + 0.5 * ds * k1); k3 = rhs(y + 0.5 * ds * k2); k4 = rhs(y + ds * k3)
        yn = y + ds / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        h_new = n_and_grad(yn[:2])[2]
        if h_new <= h_g:
            h_old = n_and_grad(y[:2])[2]
            f = (h_old - h_g) / (h_old - h_new)
            y = y + f * (yn - y)
            S += f * ds
            break
        y, S = yn, S + ds
    disp = math.atan2(y[0], y[1]) if spherical else y[0]
    return dict(disp=disp, S=S, cT=y[4])


@pytest.mark.parametrize("spherical", [False, True])
def test_trace_against_brute_force_integration(spherical):
    atm = W.make_atmosphere("spherical_5layer")
    scale = atm["earth_radius"] if spherical else 1.0
    for h_e, zen in ((3000.0, 30.0), (8000.0, 65.0)):
        th = math.radians(zen)
        want = _brute_force_ray(atm, spherical, h_e, th, 0.0, ds=1.0)
        got = O.trace(atm, spherical, h_e, th, 0.0, sub=1)
        assert abs(got["disp"] - want["disp"]) * scale < 2e-4
        assert abs(got["S"] - want["S"]) < 2e-4
        assert abs(got["cT"] - want["cT"]) < 2e-4


def test_trace_converged_at_table_spacing():
    """Reading R8: the integrator is converged to <= 0.1 mm / 0.3 ps at sub = 1."""
    atm = W.make_atmosphere("spherical_5layer")
    for h_e, zen in ((10000.0, 60.0), (30000.0, 75.0)):
        a = O.trace(atm, True, h_e, math.radians(zen), 0.0, sub=1)
        b = O.trace(atm, True, h_e, math.radians(zen), 0.0, sub=8)
        assert abs(a["disp"] - b["disp"]) * atm["earth_radius"] < 1e-4
        assert abs(a["cT"] - b["cT"]) / C_LIGHT < 3e-4


def test_refraction_magnitudes_sane():
    """The ray bends towards the vertical and lands short of the straight line (Fig. 3.3)."""
    cfg = W.make_config(2, n_segments=4)
    tab = O.table_for(cfg)
    v20 = O.table_lookup(cfg["table"], tab, 10000.0, math.radians(20))
    v60 = O.table_lookup(cfg["table"], tab, 10000.0, math.radians(60))
    assert v60[0] < v20[0] < 0 and -10.0 < v60[0] < -3.0
    assert 600 < v20[3] < 900 and 1200 < v60[3] < 1700            # slant depth g/cm^2 from 10 km
    assert 3.0 < v20[2] < 8.0                                       # ~ int (n-1) ds / c  [ns]


# ------------------------------------------------------------------ O9 table
def test_table_lookup_nodes_bilinear_and_sentinels():
    table = dict(n_h=9, n_zen=7, h_max=8000.0, zen_max_deg=60.0)
    hh = np.linspace(0, 8000.0, 9)[:, None]
    zz = np.linspace(0, math.radians(float(np.float32(60.0))), 7)[None, :]
    data = np.zeros((9, 7, 5), dtype=np.float32)
    coef = [(1.0, 2e-3, 3.0, 5e-4), (0.5, -1e-3, 1.0, 1e-4), (2, 0, 0, 0), (0, 1e-3, 0, 0), (0, 0, 1, 0)]
    for k, (a, b, c, d) in enumerate(coef):
        data[:, :, k] = a + b * hh + c * zz + d * hh * zz
    assert np.allclose(O.table_lookup(table, data, 3000.0, float(zz[0, 4])), data[3, 4], rtol=1e-6)   # node
    h, z = 3456.7, 0.61
    want = [a + b * h + c * z + d * h * z for a, b, c, d in coef]
    assert np.allclose(O.table_lookup(table, data, h, z), want, rtol=2e-6)                             # bilinear exact
    assert np.allclose(O.table_lookup(table, data, 8000.0, z)[0], want[0] + (8000 - h) * (2e-3 + 5e-4 * z), rtol=2e-6)
    assert O.table_lookup(table, data, 8000.1, z) is None and O.table_lookup(table, data, 100.0, 1.06) is None
    data[4, 5, :] = np.nan
    assert O.table_lookup(table, data, 3500.0, float(zz[0, 4]) + 0.01) is None                         # stencil touches NaN
    assert O.table_lookup(table, data, 2500.0, float(zz[0, 4]) + 0.01) is not None


def test_table_nodes_are_trace_minus_straight_line():
    cfg = W.make_config(2, n_segments=4)
    atm, table = cfg["atmosphere"], dict(n_h=17, n_zen=9, h_max=40000.0, zen_max_deg=80.0)
    tab = O.build_table(atm, table)
    assert np.all(tab[0] == 0)                                   # h_a <= h_obs
    assert np.all(tab[:, 0, 0] == 0)                             # vertical ray: no displacement
    R = atm["earth_radius"]
    a, b = 5, 6
    h, th = a * 40000.0 / 16, b * math.radians(float(np.float32(80.0))) / 8
    r = O.trace(atm, True, h, th, 0.0)
    p = (R + h) * math.sin(th)
    s_line = (R + h) * math.cos(th) - math.sqrt(R * R - p * p)
    psi_line = math.asin(p / R) - th
    assert tab[a, b, 0] == pytest.approx(R * (r["disp"] - psi_line), rel=1e-5)
    assert tab[a, b, 1] == pytest.approx(r["S"] - s_line, rel=1e-5)
    assert tab[a, b, 2] == pytest.approx((r["cT"] - s_line) / C_LIGHT, rel=1e-5)
    assert tab[a, b, 3] == pytest.approx(r["X"], rel=1e-6)


# ------------------------------------------------------------------ O11 transmission
def test_transmission_single_exponential_closed_form():
    atm = W.make_atmosphere("planar_exp", h_obs=2000.0, rayleigh=True)
    atm["refractivity"] = np.zeros_like(atm["refractivity"])          # straight ray
    th = math.radians(35.0)
    r = O.trace(atm, False, 9000.0, th, 2000.0)
    x_want = 1030.0 * (math.exp(-2000 / 8400.0) - math.exp(-9000 / 8400.0)) / math.cos(th)
    assert r["X"] == pytest.approx(x_want, rel=1e-6)
    lam = 350.0
    assert O.transmission(atm, r["X"], 0.0, lam) == pytest.approx(math.exp(-(400 / lam) ** 4 * x_want / 2970.0), rel=1e-6)
    atm["rayleigh_X"] = 0.0
    assert O.transmission(atm, r["X"], 0.3, lam) == 1.0               # alpha -> 0  =>  T = 1
    atm["aer_L"] = 15000.0
    ra = O.trace(atm, False, 9000.0, th, 2000.0)
    tau = 1200.0 / 15000.0 * (math.exp(-2000 / 1200.0) - math.exp(-9000 / 1200.0)) / math.cos(th)
    assert ra["tau_aer"] == pytest.approx(tau, rel=1e-12)
    assert O.transmission(atm, 0.0, ra["tau_aer"], 700.0) == pytest.approx(math.exp(-tau * 350.0 / 700.0), rel=1e-6)


# ------------------------------------------------------------------ O12 intersection
def test_ray_sphere_analytic_cases():
    u = np.array([0.0, 0.6, -0.8])
    hit, s = O.ray_sphere([0, 0, 0], u, [0, 0, 0], 6.0)
    assert hit and s == pytest.approx(-6.0)
    assert O.ray_sphere([7.5 - 1e-9, 0, 0], [0, 0, -1.0], [0, 0, 0], 7.5)[0]
    assert not O.ray_sphere([7.5 + 1e-9, 0, 0], [0, 0, -1.0], [0, 0, 0], 7.5)[0]
    # inclined ray: footprint stretches to r/|u_z| along the ray azimuth, stays r across it
    assert O.ray_sphere([0, 7.4, 0], u, [0, 0, 0], 6.0)[0] and not O.ray_sphere([0, 7.6, 0], u, [0, 0, 0], 6.0)[0]
    assert O.ray_sphere([5.9, 0, 0], u, [0, 0, 0], 6.0)[0] and not O.ray_sphere([6.1, 0, 0], u, [0, 0, 0], 6.0)[0]


def test_camera_pixel_centres_round_trip():
    det = W.make_config(3, n_segments=4)["detector"]
    az, el, p = math.radians(det["cam_az_deg"]), math.radians(det["cam_el_deg"]), math.radians(det["cam_pix_deg"])
    w = np.array([math.cos(el) * math.cos(az), math.cos(el) * math.sin(az), math.sin(el)])
    right = np.array([-math.sin(az), math.cos(az), 0.0])
    up = np.cross(w, right)
    for r, c in ((0, 0), (10, 7), (21, 19), (5, 0)):
        a = (c - 0.5 * (det["cam_cols"] - 1) + 0.5 * (r % 2)) * p
        e = (r - 0.5 * (det["cam_rows"] - 1)) * p * math.sqrt(3) / 2
        v = w + math.tan(a) * right + math.tan(e) * up
        v /= np.linalg.norm(v)
        assert O.camera_pixel(det, -v) == r * det["cam_cols"] + c
    assert O.camera_pixel(det, w) == -1                              # photon travelling along +axis: from behind
    v = w + math.tan(math.radians(25.0)) * right
    assert O.camera_pixel(det, -v / np.linalg.norm(v)) == -1         # outside the field of view


# ------------------------------------------------------------------ whole path: conservation, filters
def _check_conservation(res, w):
    c = res["counters"]
    assert c["emitted"] == res["total_bunches"] == int(res["n_bunch"].sum())
    assert c["emitted"] == c["upgoing"] + c["lv2"] + c["table_range"] + c["roulette"] + c["landed"]
    ph = res["photons"]
    assert len(ph) == c["emitted"] and int((ph["status"] == O.ST_LANDED).sum()) == c["landed"]
    assert c["segments"] == len(res["n_bunch"])
    assert c["in_grid"] == int((ph["bin"] >= 0).sum()) and c["tel_hit"] == int((ph["tel"] >= 0).sum())


def test_photon_count_conservation_cfg0():
    cfg = W.make_config(0)
    res = O.run(cfg)
    _check_conservation(res, 1.0)
    c = res["counters"]
    assert res["hist"].sum() == c["in_grid"] and c["landed"] == c["emitted"]
    # stochastic rounding is unbiased: sum N_i vs sum N_exp  (sigma^2 <= n_seg / 4)
    seg = cfg["segments"]
    n_exp = sum(O.cherenkov_yield(1.0, 10.0, float(b), 1 + float(np.float32(0.000293)), 300, 600) for b in seg["beta"])
    assert abs(c["emitted"] - n_exp) < 5 * math.sqrt(len(seg["beta"]) / 4)
    assert 3.5e5 < c["emitted"] < 3.9e5


def test_segment_order_and_batching_independence():
    cfg = W.make_config(0, n_segments=64)
    full = O.run(cfg)
    part = copy.deepcopy(cfg)
    part["segments"] = W.slice_segments(cfg["segments"], 40, 64)
    part["seg_id_base"] = 40
    sub = O.run(part)
    a = full["photons"][full["photons"]["seg"] >= 40]
    b = sub["photons"]
    assert len(a) == len(b)
    for f in ("x", "y", "t", "lambda_nm", "ux"):
        assert np.array_equal(a[f], b[f])


def test_explicit_segment_ids_make_the_order_irrelevant_and_non_finite_segments_are_dropped():
    """O0 / SURVEY 8(b): the Philox counter carries the segment id; handed over explicitly, a shuffled segment list gives
    the photons of the ordered one (mapped back by index).  A segment with a non-finite field or a zero direction is
    dropped and counted; the others keep their photons (ids unchanged)."""
    cfg = W.make_config(0, n_segments=96)
    full = O.run(cfg)
    perm = np.random.default_rng(3).permutation(96)
    sh = copy.deepcopy(cfg)
    sh["segments"] = {f: np.ascontiguousarray(v[perm]) for f, v in cfg["segments"].items()}
    sh["segments"]["id"] = perm.astype(np.uint64)
    got = O.run(sh)
    assert got["counters"] == full["counters"] and np.array_equal(got["hist"], full["hist"])
    a, b = full["photons"], got["photons"].copy()
    b["seg"] = perm[b["seg"]]
    a, b = a[np.lexsort((a["j"], a["seg"]))], b[np.lexsort((b["j"], b["seg"]))]
    for f in ("seg", "j", "x", "y", "t", "lambda_nm", "ux", "uy", "uz", "bin"):
        assert np.array_equal(a[f], b[f]), f
    # ids without shuffling = seg_id_base + i
    ident = copy.deepcopy(cfg)
    ident["segments"]["id"] = np.arange(96, dtype=np.uint64)
    assert np.array_equal(O.run(ident)["photons"], full["photons"])
    bad = copy.deepcopy(cfg)
    bad["segments"]["z"][5] = np.nan
    bad["segments"]["beta"][6] = np.inf
    for f in ("dx", "dy", "dz"):
        bad["segments"][f][7] = 0.0
    res = O.run(bad)
    assert res["counters"]["nonfinite"] == 3 and full["counters"]["nonfinite"] == 0
    assert res["counters"]["segments"] == 96
    keep = ~np.isin(full["photons"]["seg"], (5, 6, 7))
    assert np.array_equal(res["photons"], full["photons"][keep])
    assert np.isfinite(res["hist"]).all()


def test_filters_are_lossless_and_roulette_unbiased():
    cfg = W.make_config(2, n_segments=3000)
    on = O.run(cfg)
    _check_conservation(on, 5.0)
    off_cfg = copy.deepcopy(cfg)
    off_cfg["params"].update(lv1=False, lv2=False)
    off = O.run(off_cfg)
    _check_conservation(off, 5.0)
    assert on["counters"]["seg_lv1"] > 0 and on["counters"]["lv2"] > 0
    assert on["counters"]["tel_hit"] == off["counters"]["tel_hit"] > 50
    assert np.array_equal(on["tel_counts"], off["tel_counts"])
    hit_on = on["photons"][on["photons"]["tel"] >= 0]
    hit_off = off["photons"][off["photons"]["tel"] >= 0]
    key = lambda p: p["seg"] * (1 << 20) + p["j"]
    assert np.array_equal(np.sort(key(hit_on)), np.sort(key(hit_off)))
    # roulette: sum over survivors of w vs sum of w T over all that reached the roulette
    w_cfg = copy.deepcopy(off_cfg)
    w_cfg["params"]["trans"] = "weight"
    wres = O.run(w_cfg)
    ph = wres["photons"][wres["photons"]["status"] == O.ST_LANDED]
    exp, var = ph["T"].sum(), (ph["T"] * (1 - ph["T"])).sum()
    assert abs(off["counters"]["landed"] - exp) < 5 * math.sqrt(var)
    assert 0.2 < exp / len(ph) < 0.95


def test_planar_numeric_path_cfg1_small():
    cfg = W.make_config(1, n_segments=300)
    res = O.run(cfg)
    _check_conservation(res, 1.0)
    ph = res["photons"][res["photons"]["status"] == O.ST_LANDED]
    assert len(ph) > 1000
    assert res["hist"].sum() == pytest.approx(ph["weight"][ph["bin"] >= 0].sum(), rel=1e-12)
    assert np.all(ph["T"] < 1.0) and np.all(ph["T"] > 0.3)
    # refraction pulls the photon towards the vertical: it lands short of the straight line
    seg = cfg["segments"]
    ax = seg["x"][ph["seg"]] - seg["z"][ph["seg"]] * seg["dx"][ph["seg"]] / seg["dz"][ph["seg"]]
    assert np.all(np.hypot(ph["x"] - ph["x_line"], ph["y"] - ph["y_line"]) < 2.0)
    assert np.all(np.abs(np.hypot(ph["ux"], ph["uy"]) ** 2 + ph["uz"] ** 2 - 1) < 1e-12)


def test_fluorescence_sampling_isotropy_and_lines():
    cfg = W.make_config(3, n_segments=1)
    s = cfg["segments"]
    s["x"][:], s["y"][:], s["z"][:] = 0.0, 0.0, 10000.0
    s["dx"][:], s["dy"][:], s["dz"][:] = 0.0, 0.0, -1.0
    s["edep"][:] = 5000.0
    cfg["detector"]["tel_xyzr"] = np.array([[0.0, 0.0, 0.0, 1.9]], dtype=np.float32)
    cfg["params"].update(trace="straight", trans="off", lv2=False, aim_factor=1e9)   # psi -> 90 deg: half sphere
    res = O.run(cfg)
    ph = res["photons"]
    assert len(ph) == pytest.approx(4.0 * 5000.0 * 0.5, abs=1)                      # Y E Omega/4pi
    ph = ph[ph["status"] == O.ST_LANDED]
    mu = -ph["uz"]                                                                  # cos to the aim axis (-z)
    assert np.mean(mu) == pytest.approx(0.5, abs=5 * math.sqrt(1 / 12 / len(mu)))
    assert np.mean(mu ** 2) == pytest.approx(1 / 3, abs=0.02)
    assert abs(np.mean(ph["ux"])) < 0.03 and abs(np.mean(ph["uy"])) < 0.03
    lines, cdf = cfg["params"]["line_nm"], cfg["params"]["line_cdf"].astype(np.float64)
    prob = np.diff(np.concatenate([[0.0], cdf]))
    idx = np.searchsorted(lines, ph["lambda_nm"].astype(np.float32))
    cnt = np.bincount(idx, minlength=len(lines))
    keep = prob * len(ph) > 5
    assert stats.chisquare(cnt[keep], prob[keep] / prob[keep].sum() * cnt[keep].sum()).pvalue > 1e-4


def test_forced_cone_is_unbiased_in_margin():
    """hits/Omega independent of the aim factor (photon number scaled with the solid angle)."""
    hits = []
    for fac in (1.5, 3.0):
        cfg = W.make_config(3, n_segments=2000)
        cfg["segments"]["edep"][:] = 2.0e10
        cfg["params"].update(aim_factor=fac, trans="off")
        res = O.run(cfg, record=False)
        hits.append(res["counters"]["tel_hit"])
    assert hits[0] > 200
    assert abs(hits[0] - hits[1]) < 5 * math.sqrt(hits[0] + hits[1])


def test_thesis_model_array_fixtures(golden_dir):
    """Appendix B.3 layouts as parsed into tests/golden: counts, radii classes, and an
    oracle run of cfg4's shower on Array 1 whose telescope hits obey the bounding-sphere definition."""
    a1 = np.loadtxt(os.path.join(golden_dir, "telescope_array_1.txt"), comments="#").reshape(-1, 4)
    a2 = np.loadtxt(os.path.join(golden_dir, "telescope_array_2.txt"), comments="#").reshape(-1, 4)
    assert a1.shape == (13, 4) and sorted(set(a1[:, 3])) == [12.0, 23.0] and (a1[:, 3] == 23.0).sum() == 4
    assert a2.shape == (180, 4) and sorted(set(a2[:, 3])) == [2.1, 5.8, 11.1]
    assert [(a2[:, 3] == r).sum() for r in (11.1, 5.8, 2.1)] == [4, 56, 120]
    cfg = W.make_config(4, n_segments=300)
    cfg["detector"]["tel_xyzr"] = a1.astype(np.float32)
    res = O.run(cfg, record=True)
    ph = res["photons"]
    hit = ph[(ph["status"] == O.ST_LANDED) & (ph["tel"] >= 0)]
    assert len(hit) > 100 and res["counters"]["tel_hit"] == len(hit)
    c = a1[hit["tel"]]
    d = np.stack([c[:, 0] - hit["x"], c[:, 1] - hit["y"], c[:, 2]], axis=1)
    u = np.stack([hit["ux"], hit["uy"], hit["uz"]], axis=1)
    m2 = (d ** 2).sum(1) - ((d * u).sum(1)) ** 2
    assert np.all(m2 <= c[:, 3] ** 2 * (1 + 1e-9))


# ---------------------------------------------------------------------------------- dispersion (R13, row f4)
def _disp_integrand(k, beta, eta, b, l0):
    n = 1.0 + eta * (1.0 + b * (k * k - 1.0 / l0 ** 2))
    return np.maximum(0.0, 1.0 - 1.0 / (beta * n) ** 2)


def test_dispersive_yield_limits_closed_form_and_threshold():
    """P:318 yield integral with n(lambda): b -> 0 is Frank-Tamm's closed form; for b > 0 the integral has
    the closed form  k - [k/(2A(A+Bk^2)) + atan(k sqrt(B/A))/(2A sqrt(AB))]/beta^2  (A + B k^2 = n(k));
    with the Cherenkov threshold inside the band only the blue side of it contributes."""
    from scipy import integrate
    L = O.lib()
    a2pi = 2.0 * math.pi / 137.035999
    y0 = L.orc_cherenkov_yield(1.0, 7.0, 0.99995, 1.000293, 300.0, 600.0)
    assert abs(L.orc_cherenkov_yield_dispersive(1.0, 7.0, 0.99995, 0.000293, 300.0, 600.0, 0.0, 400.0) / y0 - 1) < 1e-12
    eta, b, l0, l1, l2 = 2.5e-4, 5700.0, 400.0, 250.0, 700.0
    A, B = 1.0 + eta * (1.0 - b / l0 ** 2), eta * b
    F = lambda k: k / (2 * A * (A + B * k * k)) + math.atan(k * math.sqrt(B / A)) / (2 * A * math.sqrt(A * B))
    for beta in (1.0, 0.99990):                                           # far above threshold
        want = a2pi * 3.0 * ((1 / l1 - 1 / l2) - (F(1 / l1) - F(1 / l2)) / beta ** 2) * 1e9
        got = L.orc_cherenkov_yield_dispersive(1.0, 3.0, beta, eta, l1, l2, b, l0)
        assert abs(got / want - 1) < 1e-9, (beta, got, want)
    # threshold inside the band: beta n(k_th) = 1
    k_th = 1.0 / 400.0
    beta = 1.0 / (1.0 + eta * (1.0 + b * (k_th ** 2 - 1 / l0 ** 2)))
    got = L.orc_cherenkov_yield_dispersive(1.0, 3.0, beta, eta, l1, l2, b, l0)
    want = a2pi * 3.0 * ((1 / l1 - k_th) - (F(1 / l1) - F(k_th)) / beta ** 2) * 1e9
    quad = a2pi * 3.0 * integrate.quad(_disp_integrand, 1 / l2, 1 / l1, args=(beta, eta, b, l0), points=[k_th], epsabs=0, epsrel=1e-12)[0] * 1e9
    assert 0 < got < 0.2 * L.orc_cherenkov_yield_dispersive(1.0, 3.0, 1.0, eta, l1, l2, b, l0)
    assert abs(got / want - 1) < 1e-6 and abs(quad / want - 1) < 1e-8
    # below threshold over the whole band
    assert L.orc_cherenkov_yield_dispersive(1.0, 3.0, 0.9997, eta, l1, l2, b, l0) == 0.0
    assert abs(L.orc_dispersion_factor(b, l0, l0) - 1.0) < 1e-15 and L.orc_dispersion_factor(b, l0, 300.0) > 1.0


def test_dispersive_photons_spectrum_and_cone_angle():
    """Photon level (cfg0: homogeneous n, straight line, so the record keeps the emission direction):
    u.P = 1/(beta n(lambda)) for every photon, and the wavelengths follow the density
    lambda^-2 sin^2 theta(lambda) (KS test) for particles just above threshold, where it is far from
    the non-dispersive 1/lambda-uniform law."""
    cfg = W.make_config(0, n_segments=400)
    eta, b, l0 = 0.000293, 5700.0, 400.0
    cfg["params"].update(disp_b_nm2=b, disp_lambda0_nm=l0, lambda_min_nm=300.0, lambda_max_nm=600.0)
    s = cfg["segments"]
    k_th = 1.0 / 520.0                                                    # threshold at 520 nm: only 300-520 nm emits
    s["beta"][:] = np.float32(1.0 / (1.0 + eta * (1.0 + b * (k_th ** 2 - 1 / l0 ** 2))))
    s["len"][:] = 400.0
    res = O.run(cfg, record=True)
    ph = res["photons"]
    assert len(ph) > 5000 and ph["lambda_nm"].max() < 520.5 and ph["lambda_nm"].min() >= 300.0
    P = np.stack([s["dx"], s["dy"], s["dz"]], axis=1).astype(np.float64)
    P /= np.linalg.norm(P, axis=1, keepdims=True)
    beta = s["beta"].astype(np.float64)[ph["seg"]]
    n_lam = 1.0 + float(np.float32(eta)) * (1.0 + float(np.float32(b)) * (1.0 / ph["lambda_nm"] ** 2 - 1.0 / l0 ** 2))
    cos_c = np.minimum(1.0, 1.0 / (beta * n_lam))
    up = ph["ux"] * P[ph["seg"], 0] + ph["uy"] * P[ph["seg"], 1] + ph["uz"] * P[ph["seg"], 2]
    assert np.abs(up - cos_c).max() < 1e-12
    # analytic CDF in k = 1/lambda of the density sin^2 theta(k)
    b0 = float(beta[0])
    ks = np.linspace(1 / 600.0, 1 / 300.0, 20001)
    dens = _disp_integrand(ks, b0, float(np.float32(eta)), float(np.float32(b)), l0)
    cdf = np.concatenate([[0.0], np.cumsum(0.5 * (dens[1:] + dens[:-1]) * np.diff(ks))])
    cdf /= cdf[-1]
    ks_stat = stats.kstest(1.0 / ph["lambda_nm"], lambda x: np.interp(x, ks, cdf))
    assert ks_stat.pvalue > 1e-3, ks_stat
    flat = stats.kstest(1.0 / ph["lambda_nm"], lambda x: np.clip((x - 1 / 600.0) / (1 / 300.0 - 1 / 600.0), 0, 1))
    assert flat.pvalue < 1e-12                                            # and clearly not the non-dispersive law
    # expected count: sum of the stochastic roundings reproduces the integral within 5 sigma
    want = sum(O.lib().orc_cherenkov_yield_dispersive(float(q), 400.0, float(bb), float(np.float32(eta)), 300.0, 600.0, float(np.float32(b)), l0)
               for q, bb in zip(s["charge"], s["beta"]))
    assert abs(len(ph) - want) < 5 * math.sqrt(len(s["beta"]) / 4.0) + 1


# ---------------------------------------------------------------------------------- detector efficiency (R14, row f4)
def test_detector_efficiency_folding():
    """eps(lambda) table folded into the survival probability: lookup is linear
    between nodes and held outside; eps = 1 changes nothing; a constant eps scales the roulette
    survivors by eps (binomial 5 sigma) and the weight-mode histogram exactly; a step eps(lambda)
    removes exactly the photons of the dark band."""
    keep = O._Keep()
    par = dict(W.make_config(4, n_segments=1)["params"])
    par.update(eff=np.array([0.0, 0.5, 1.0, 0.25], np.float32), eff_lambda0_nm=300.0, eff_dlambda_nm=100.0)
    ps = O.params_struct(par, keep)
    eff = lambda lam: O.lib().orc_efficiency(C.byref(ps), float(lam))
    assert eff(300.0) == 0.0 and eff(400.0) == 0.5 and eff(350.0) == 0.25 and abs(eff(575.0) - 0.4375) < 1e-12
    assert eff(100.0) == 0.0 and eff(900.0) == 0.25                     # end values held
    cfg = W.make_config(2, n_segments=6000)
    base = O.run(cfg, record=False)
    one = copy.deepcopy(cfg)
    one["params"].update(eff=np.ones(5, np.float32), eff_lambda0_nm=200.0, eff_dlambda_nm=150.0)
    r1 = O.run(one, record=False)
    assert r1["counters"] == base["counters"] and np.array_equal(r1["tel_counts"], base["tel_counts"])
    half = copy.deepcopy(cfg)
    half["params"].update(eff=np.full(2, 0.5, np.float32), eff_lambda0_nm=200.0, eff_dlambda_nm=600.0)
    rh = O.run(half, record=False)
    n0 = base["counters"]["landed"]
    assert n0 > 20000 and abs(rh["counters"]["landed"] - 0.5 * n0) < 5 * math.sqrt(0.25 * n0)
    assert rh["counters"]["roulette"] + rh["counters"]["landed"] == base["counters"]["roulette"] + n0
    # weight mode: hist scales exactly
    wcfg = W.make_config(1, n_segments=60)
    wb = O.run(wcfg, record=False)
    wh = copy.deepcopy(wcfg)
    wh["params"].update(eff=np.full(3, 0.25, np.float32), eff_lambda0_nm=100.0, eff_dlambda_nm=400.0)
    wr = O.run(wh, record=False)
    assert np.allclose(wr["hist"], 0.25 * wb["hist"], rtol=1e-12, atol=0) and wr["counters"] == wb["counters"]
    # step: dark below 450 nm (nodes at 449.9 / 450.1)
    st = copy.deepcopy(cfg)
    st["params"].update(eff=np.array([0, 0, 1, 1], np.float32), eff_lambda0_nm=449.7, eff_dlambda_nm=0.2)
    rs = O.run(st, record=True)
    ph = rs["photons"]
    landed = ph[ph["status"] == O.ST_LANDED]
    assert len(landed) > 1000 and landed["lambda_nm"].min() >= 449.9


# ---------------------------------------------------------------------------------- last mile (R15, row f3)
def _optics_det(az=30.0, el=70.0, f=17.0, rm=8.5, rc=0.735):
    det = dict(W.make_config(4, n_segments=1)["detector"])
    det.update(opt_enabled=True, opt_az_deg=az, opt_el_deg=el, opt_focal_m=f, opt_mirror_radius_m=rm, opt_camera_radius_m=rc)
    return det


def _last_mile(ds, I, u, c, r_sphere=12.0):
    arr = lambda v: (C.c_double * len(v))(*[float(x) for x in v])
    res = (C.c_double * 6)()
    rc = O.lib().orc_last_mile(C.byref(ds), arr(I), arr(u), arr(c), float(r_sphere), res)
    return rc, np.array(res[:])


def test_last_mile_parabolic_mirror_and_camera():
    """Thesis sec. 6.4, the MAGIC-like telescope it shows (17 m parabola, f = 17 m, camera
    1.47 m): rays parallel to the axis focus to the camera centre with the constant path length of the
    focus-directrix property; the camera shadows (R_c/R_m)^2 of the aperture; the ray through the vertex
    is shadowed exactly while f tan(delta) <= R_c; |u'| = 1; and an independent numerical intersection (root bracketing on the
    surface function, normal from its gradient) gives the same camera point for skew rays."""
    from scipy import optimize
    keep = O._Keep()
    az, el, f, rm, rc = 30.0, 70.0, 17.0, 8.5, 0.735
    ds = O.detector_struct(_optics_det(az, el, f, rm, rc), keep)
    a, e = np.radians(az), np.radians(el)
    w = np.array([np.cos(e) * np.cos(a), np.cos(e) * np.sin(a), np.sin(e)])
    er = np.array([-np.sin(a), np.cos(a), 0.0])
    eu = np.cross(w, er)
    c = np.array([120.0, -40.0, 9.0])
    V = c - 0.5 * f * w
    rng = np.random.default_rng(5)
    n_hit = n_shadow = 0
    for _ in range(4000):
        rho, ph = rm * np.sqrt(rng.uniform()), rng.uniform(0, 2 * np.pi)
        x, y = rho * np.cos(ph), rho * np.sin(ph)
        z_start = 30.0
        I = V + x * er + y * eu + z_start * w
        code, res = _last_mile(ds, I, -w, c)
        if rho <= rc:
            assert code == -1
            n_shadow += 1
        else:
            assert code == 1 and np.hypot(res[0], res[1]) < 1e-9
            assert abs(res[5] - (z_start + f)) < 1e-9                    # focus-directrix: constant path
            assert abs(np.linalg.norm(res[2:5]) - 1.0) < 1e-12
            n_hit += 1
    assert abs(n_shadow / 4000.0 - (rc / rm) ** 2) < 5 * math.sqrt((rc / rm) ** 2 / 4000.0)
    # outside the aperture / wrong way
    assert _last_mile(ds, V + (rm + 0.01) * er + 30.0 * w, -w, c)[0] == 0
    assert _last_mile(ds, V + 3.0 * er + 30.0 * w, w, c)[0] == 0
    # the ray through the vertex, tilted by delta, crosses the camera plane at f tan(delta) on its way in and
    # would image at the mirrored point: shadowed while that is inside the camera, a miss beyond it
    for delta in (0.002, 0.01, 0.03, 0.05, 0.08):
        d = np.sin(delta) * er - np.cos(delta) * w
        code, res = _last_mile(ds, V - 40.0 * d, d, c)
        assert code == (-1 if f * np.tan(delta) <= rc else 0)
    # skew rays against an independent numerical construction
    checked = 0
    for _ in range(300):
        tilt, pa = rng.uniform(0, 0.03), rng.uniform(0, 2 * np.pi)
        d = np.sin(tilt) * (np.cos(pa) * er + np.sin(pa) * eu) - np.cos(tilt) * w
        rho, ph = rm * np.sqrt(rng.uniform()), rng.uniform(0, 2 * np.pi)
        I = V + rho * np.cos(ph) * er + rho * np.sin(ph) * eu + 25.0 * w
        code, res = _last_mile(ds, I, d, c)
        loc = lambda s: np.array([(I + s * d - V) @ er, (I + s * d - V) @ eu, (I + s * d - V) @ w])
        g = lambda s: loc(s)[2] - (loc(s)[0] ** 2 + loc(s)[1] ** 2) / (4 * f)
        s_hit = optimize.brentq(g, 0.0, 60.0, xtol=1e-13)
        p = loc(s_hit)
        cam_cross = loc((f - (I - V) @ w) / (d @ w))
        if np.hypot(cam_cross[0], cam_cross[1]) <= rc:
            assert code == -1
            continue
        if np.hypot(p[0], p[1]) > rm:
            assert code == 0
            continue
        grad = np.array([-p[0] / (2 * f), -p[1] / (2 * f), 1.0])
        nrm = grad / np.linalg.norm(grad)
        dl = np.array([d @ er, d @ eu, d @ w])
        r = dl - 2 * (dl @ nrm) * nrm
        s2 = (f - p[2]) / r[2]
        xc, yc = p[0] + s2 * r[0], p[1] + s2 * r[1]
        if np.hypot(xc, yc) <= rc:
            assert code == 1 and abs(res[0] - xc) < 1e-9 and abs(res[1] - yc) < 1e-9 and abs(res[5] - (s_hit + s2)) < 1e-9
            checked += 1
        else:
            assert code == 0
    assert checked > 50


def test_last_mile_refracting_lens_total_internal_reflection_and_absorbers():
    """Reading R22 (thesis sec. 6.4: "light bending at a boundary layer (e.g. lens ...)", "absorption by
    objects"; Fig. 6.6a: total internal reflection).  Pins: vector Snell keeps n sin(angle) and the plane of incidence
    and fails exactly beyond the critical angle; paraxial rays through the plano-convex lens meet the axis at the
    thick-lens back focal distance R/(n-1) - t/n behind the plane face; a marginal ray of a fat lens is totally
    reflected at the plane face exactly where an independent 2-D angle construction says so; the optical path counts
    n inside the glass; the segment distance against brute force; a strut across the aperture of the MAGIC-like
    telescope removes the fraction of on-axis light that follows from its two shadows (incoming and reflected beam)."""
    from scipy.optimize import brentq as optimize_brentq
    L = O.lib()
    arr = lambda v: (C.c_double * len(v))(*[float(x) for x in v])
    rng = np.random.default_rng(11)
    # --- vector Snell
    for _ in range(200):
        N = rng.normal(size=3); N /= np.linalg.norm(N)
        u = rng.normal(size=3); u /= np.linalg.norm(u)
        n1, n2 = rng.uniform(1.0, 1.8, 2)
        out = (C.c_double * 3)()
        ok = L.orc_refract(arr(u), arr(N), n1, n2, out)
        si = math.sqrt(max(0.0, 1 - (u @ N) ** 2))
        assert bool(ok) == (n1 * si <= n2)                             # total internal reflection beyond the critical angle
        if ok:
            v = np.array(out[:])
            assert abs(np.linalg.norm(v) - 1) < 1e-12
            assert n2 * math.sqrt(max(0.0, 1 - (v @ N) ** 2)) == pytest.approx(n1 * si, abs=1e-12)
            assert abs(np.cross(u, N) @ v) < 1e-12 and (v @ N) * (u @ N) > 0           # same plane, same side
    # --- plano-convex lens, axis vertical (el = 90, az = -90: frame (right, up) = (x, y)): plane face at z = +f/2,
    #     camera at z = -f/2 about the centre
    n_l, R_l, t_l = 1.5, 3.0, 0.2
    bfd = R_l / (n_l - 1.0) - t_l / n_l                                # thick lens, curved side first
    det = _optics_det(az=-90.0, el=90.0, f=bfd, rm=0.8, rc=0.3)
    det.update(opt_kind=1, opt_lens_roc_m=R_l, opt_lens_thickness_m=t_l, opt_lens_index=n_l)
    keep = O._Keep()
    ds = O.detector_struct(det, keep)
    c = (0.0, 0.0, 10.0)
    for x in (1e-3, 5e-3, 0.02):
        rc, res = _last_mile(ds, (x, 0.0, 30.0), (0, 0, -1.0), c)
        assert rc == 1 and abs(res[0]) < 2e-3 * x + 40 * x ** 3 and abs(res[1]) < 1e-12   # paraxial focus (spherical aberration ~ x^3)
        rcf, resf = _last_mile(O.detector_struct(dict(det, opt_focal_m=0.5 * bfd), keep), (x, 0.0, 30.0), (0, 0, -1.0), c)
        assert rcf == 1 and resf[0] == pytest.approx(0.5 * x, rel=0.05)               # half way to the focus: half the height
    rc, res = _last_mile(ds, (1e-3, 0.0, 30.0), (0, 0, -1.0), c)
    sag = R_l - math.sqrt(R_l ** 2 - 1e-6)
    assert res[5] == pytest.approx((30.0 - (10.0 + 0.5 * bfd + t_l - sag)) + n_l * (t_l - sag) + bfd, abs=1e-6)   # n inside the glass
    # off-axis beam: the image height of a thin-lens-like system is efl * tan(field angle), efl = R/(n-1)
    ang = 0.01
    rc, res = _last_mile(ds, (1e-3 + 20.0 * math.tan(ang), 0.0, 30.0), (-math.sin(ang), 0, -math.cos(ang)), c)
    assert rc == 1 and res[0] == pytest.approx(-R_l / (n_l - 1.0) * math.tan(ang), rel=2e-2)
    # --- a fat lens (nearly a hemisphere): marginal rays meet the plane face beyond the critical angle; where that starts
    #     follows from an independent 2-D construction with angles (entry at polar angle a1, refracted by a1 - a2)
    n_l, R_l, t_l = 1.5, 1.0, 0.95
    det = _optics_det(az=-90.0, el=90.0, f=1.0, rm=0.998, rc=0.9)
    det.update(opt_kind=1, opt_lens_roc_m=R_l, opt_lens_thickness_m=t_l, opt_lens_index=n_l)
    keep = O._Keep()
    ds = O.detector_struct(det, keep)

    def tir_2d(x):
        a1 = math.asin(x / R_l)                                        # angle of incidence on the sphere = polar angle of the point
        a2 = math.asin(math.sin(a1) / n_l)
        return n_l * math.sin(a1 - a2) > 1.0                           # angle of the refracted ray against the axis
    seen = {1: 0, -3: 0}
    for x in np.concatenate([np.linspace(0.05, 0.98, 32), np.linspace(0.985, 0.9975, 26)]):
        rc, res = _last_mile(ds, (x, 0.0, 30.0), (0, 0, -1.0), c, r_sphere=3.0)
        if rc in (1, -3):
            assert (rc == -3) == tir_2d(x), x
            seen[rc] += 1
    assert seen[1] > 20 and seen[-3] > 5
    x_crit = optimize_brentq(lambda x: n_l * math.sin(math.asin(x) - math.asin(x / n_l)) - 1.0, 0.9, 0.999)
    assert _last_mile(ds, (x_crit - 1e-6, 0.0, 30.0), (0, 0, -1.0), c, r_sphere=3.0)[0] != -3
    assert _last_mile(ds, (x_crit + 1e-6, 0.0, 30.0), (0, 0, -1.0), c, r_sphere=3.0)[0] == -3
    # --- segment distance against brute force
    for _ in range(100):
        P0, P1, Q0, Q1 = rng.uniform(-1, 1, (4, 3))
        d = L.orc_segment_distance(arr(P0), arr(P1), arr(Q0), arr(Q1))
        s, tt = np.meshgrid(np.linspace(0, 1, 401), np.linspace(0, 1, 401))
        pts = (P0[None, None] + s[..., None] * (P1 - P0)) - (Q0[None, None] + tt[..., None] * (Q1 - Q0))
        assert d <= np.linalg.norm(pts, axis=2).min() + 1e-12 and d >= np.linalg.norm(pts, axis=2).min() - 0.01
    # --- a strut across the aperture of the MAGIC-like telescope (axis vertical), at height z_s above the sphere centre
    f, rm, rcam, r_s, z_s = 17.0, 8.5, 0.735, 0.05, 4.0
    det = _optics_det(az=-90.0, el=90.0, f=f, rm=rm, rc=rcam)
    det.update(opt_absorbers=np.array([[-9.0, 0.0, z_s, 9.0, 0.0, z_s, r_s]], np.float32))
    keep = O._Keep()
    ds = O.detector_struct(det, keep)
    det0 = _optics_det(az=-90.0, el=90.0, f=f, rm=rm, rc=rcam)
    keep0 = O._Keep()
    ds0 = O.detector_struct(det0, keep0)
    n_hit = n_abs = n_all = 0
    xs = np.linspace(-rm, rm, 341)
    for x in xs:
        for y in xs:
            if x * x + y * y > rm * rm:
                continue
            rc0, _ = _last_mile(ds0, (x, y, 40.0), (0, 0, -1.0), c, r_sphere=12.0)
            rc1, _ = _last_mile(ds, (x, y, 40.0), (0, 0, -1.0), c, r_sphere=12.0)
            if rc0 == 1:
                n_all += 1
                n_abs += rc1 == -2
                n_hit += rc1 == 1
                # the strut runs along x at y = 0: the incoming ray is blocked if |y| <= r_s; the reflected ray from the mirror
                # point (rho, rho^2/4f) to the focus passes the height of the strut at y (f - z_v)/(f - rho^2/4f)
                z_v = z_s + 0.5 * f                                  # height above the vertex
                blocked = abs(y) <= r_s or abs(y * (f - z_v) / (f - (x * x + y * y) / (4 * f))) <= r_s
                assert (rc1 == -2) == blocked or abs(abs(y) - r_s) < 1e-9, (x, y, rc1)
    assert n_all > 5e4 and n_hit + n_abs == n_all and 0.005 < n_abs / n_all < 0.03


def test_last_mile_in_the_run():
    """With optics on, camera hits are a subset of the sphere hits, the rest of the run is unchanged, and
    the recorded camera points lie inside the camera disc; arrival at the camera is later than at the
    bounding sphere's entry by at most the sphere diameter plus the focal length."""
    cfg = W.make_config(4, n_segments=400)
    tel = cfg["detector"]["tel_xyzr"].copy()
    tel[:, 3] = 12.0                                                      # sphere holds mirror and camera
    cfg["detector"]["tel_xyzr"] = tel
    base = O.run(cfg, record=True)
    cfg["detector"].update(opt_enabled=True, opt_az_deg=0.0, opt_el_deg=70.0, opt_focal_m=17.0,
                           opt_mirror_radius_m=8.5, opt_camera_radius_m=0.735)
    opt = O.run(cfg, record=True)
    for k in ("emitted", "landed", "in_grid", "tel_hit"):
        assert opt["counters"][k] == base["counters"][k]
    assert 0 < opt["counters"]["cam_hit"] < opt["counters"]["tel_hit"]
    ph = opt["photons"]
    cam = ph[ph["pix"] == 0]
    assert len(cam) == opt["counters"]["cam_hit"] and np.all(cam["tel"] >= 0)
    assert np.all(np.hypot(cam["x"], cam["y"]) <= 0.735 + 1e-12)
    b = base["photons"]
    kb = {(int(s), int(j)): t for s, j, t in zip(b["seg"], b["j"], b["t"])}
    dt = np.array([t - kb[(int(s), int(j))] for s, j, t in zip(cam["seg"], cam["j"], cam["t"])])
    assert np.all(np.abs(dt) < (24.0 + 17.0 + 20.0) / 0.299792458)


# ---------------------------------------------------------------------------------- sub-stepping (R16, row f2)
def test_substepping_follows_the_lorentz_helix():
    """Thesis sec. 4.2.1: chords of the magnetic path.  The chord end points agree with an
    independent RK4 integration of dP/ds = kappa P x B/|B|; every chord's sagitta is <= tol (and the
    piece count is the smallest that achieves it); chord lengths and clocks add up; no field or a stiff
    particle returns the track unchanged; opposite charges bend to opposite sides."""
    rng = np.random.default_rng(11)
    n = 40
    v = rng.normal(size=(n, 3)); v[:, 2] = -np.abs(v[:, 2]) - 0.5
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    trk = dict(x=rng.uniform(-100, 100, n), y=rng.uniform(-100, 100, n), z=rng.uniform(3e3, 2e4, n),
               dx=v[:, 0], dy=v[:, 1], dz=v[:, 2], len=rng.uniform(20, 300, n), beta=np.full(n, 0.9999),
               t0=rng.uniform(0, 1e4, n), charge=rng.choice([-1.0, 1.0], n), p_GeV=10 ** rng.uniform(-2, 0.5, n))
    trk = {k: np.asarray(a, dtype=np.float32) for k, a in trk.items()}
    B, tol = (2.0e-5, -0.5e-5, -4.3e-5), 0.01
    res = O.substep_tracks(trk, B, tol)
    seg, off = res["segments"], res["offsets"]
    assert off[-1] > 2 * n and np.all(np.diff(off) >= 1)
    Bv = np.array([float(np.float32(b)) for b in B]); bh = Bv / np.linalg.norm(Bv)
    for i in range(n):
        A = np.array([trk["x"][i], trk["y"][i], trk["z"][i]], dtype=np.float64)
        P = np.array([trk["dx"][i], trk["dy"][i], trk["dz"][i]], dtype=np.float64); P /= np.linalg.norm(P)
        L, q, p = float(trk["len"][i]), float(trk["charge"][i]), float(trk["p_GeV"][i])
        kappa = 0.299792458 * q * np.linalg.norm(Bv) / p
        m = off[i + 1] - off[i]
        # independent RK4 on (X, P)
        steps = 400 * m
        h = L / steps
        X, Pv = A.copy(), P.copy()
        f = lambda Pq: kappa * np.cross(Pq, bh)
        ends = [X.copy()]; mids = []
        for s in range(steps):
            k1 = f(Pv); k2 = f(Pv + 0.5 * h * k1); k3 = f(Pv + 0.5 * h * k2); k4 = f(Pv + h * k3)
            X = X + h * (Pv + (h / 6.0) * (k1 + k2 + k3))
            Pv = Pv + (h / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
            if (s + 1) % 400 == 0: ends.append(X.copy())
            if (s + 1) % 400 == 200: mids.append(X.copy())
        ends = np.array(ends)
        got0 = np.stack([seg[k][off[i]:off[i + 1]] for k in ("x", "y", "z")], axis=1).astype(np.float64)
        d = np.stack([seg[k][off[i]:off[i + 1]] for k in ("dx", "dy", "dz")], axis=1).astype(np.float64)
        ln = seg["len"][off[i]:off[i + 1]].astype(np.float64)
        got1 = got0 + d * ln[:, None]
        scale = 4e-7 * np.abs(A).max() + 1e-4                                # fp32 storage of km coordinates
        assert np.abs(got0 - ends[:-1]).max() < scale and np.abs(got1 - ends[1:]).max() < scale + 1e-5 * L
        sag = np.linalg.norm(0.5 * (ends[:-1] + ends[1:]) - np.array(mids), axis=1)
        assert sag.max() <= tol * 1.001 + 1e-9
        if m > 1:                                                            # one piece fewer would exceed tol
            curv = abs(kappa) * np.linalg.norm(P - (P @ bh) * bh)
            assert (L / (m - 1)) ** 2 * curv / 8.0 > tol * 0.999
        assert ln.sum() <= L * (1 + 1e-6) and ln.sum() > L * (1 - 1e-3)
        t_want = trk["t0"][i] + (L * np.arange(m) / m) / (float(trk["beta"][i]) * 0.299792458)
        assert np.allclose(seg["t0"][off[i]:off[i + 1]], t_want, rtol=2e-7, atol=1e-3)
        assert np.all(seg["charge"][off[i]:off[i + 1]] == q) and np.all(seg["beta"][off[i]:off[i + 1]] == trk["beta"][i])
    same = O.substep_tracks(trk, (0.0, 0.0, 0.0), tol)
    assert same["offsets"][-1] == n
    for k in ("x", "y", "z", "len", "t0"):
        assert np.allclose(same["segments"][k], trk[k], rtol=1e-6, atol=1e-6)
    stiff = dict(trk, p_GeV=np.full(n, 1e6, np.float32))
    assert O.substep_tracks(stiff, B, tol)["offsets"][-1] == n
    flip = dict(trk, charge=-trk["charge"])
    r2 = O.substep_tracks(flip, B, tol)
    assert np.array_equal(r2["offsets"], off)
    e0 = np.stack([seg[k] for k in ("x", "y", "z")], 1).astype(np.float64)
    e1 = np.stack([r2["segments"][k] for k in ("x", "y", "z")], 1).astype(np.float64)
    first = off[:-1]
    inner = np.setdiff1d(np.arange(off[-1]), first)
    assert np.abs(e0[first] - e1[first]).max() < 1e-3 and np.abs(e0[inner] - e1[inner]).max() > 1e-2


# ---------------------------------------------------------------------------------- tabulated extinction (R17, row f4)
def _rayleigh_ext_table(atm, lam):
    """tau_v(lambda, h) of the Rayleigh law of R11 on the atmosphere's height grid (vertical, obs level -> h)."""
    xv = atm["overburden"].astype(np.float64)
    h = atm["h0"] + atm["dh"] * np.arange(atm["n_nodes"])
    xg = np.interp(atm["h_obs"], h, xv)
    return ((400.0 / lam[:, None]) ** 4 * np.maximum(xg - xv[None, :], 0.0) / 2970.0).astype(np.float32)


def test_tabulated_extinction_reproduces_the_rayleigh_law():
    """A tau_v(lambda, h) table filled from the analytic Rayleigh law must reproduce R11's transmission:
    node values exactly, between wavelength nodes to the interpolation error of lambda^-4 on a 2 nm grid;
    the slant scaling by the air-mass factor X_slant / (X_v(h_obs) - X_v(h_e)) is exact for it; whole runs
    agree photon by photon (same roulette decisions up to ~1e-4 of the photons); tau scales linearly."""
    cfg = W.make_config(2, n_segments=3000)
    atm = cfg["atmosphere"]
    lam = np.arange(240.0, 711.0, 2.0)
    tab = copy.deepcopy(cfg)
    tab["atmosphere"].update(ext_tau_v=_rayleigh_ext_table(atm, lam), ext_lambda0_nm=240.0, ext_dlambda_nm=2.0)
    keep = O._Keep()
    a_tab, a_ana = O.atmosphere_struct(tab["atmosphere"], keep), O.atmosphere_struct(atm, keep)
    L = O.lib()
    for lam_q, h in ((300.0, 8000.0), (452.0, 12340.0), (601.0, 30.0), (333.3, 5555.5)):
        xs = 1.7 * (L.orc_overburden(C.byref(a_ana), 0.0) - L.orc_overburden(C.byref(a_ana), h))   # some slant path
        t_tab = L.orc_transmission_tabulated(C.byref(a_tab), xs, h, lam_q)
        t_ana = L.orc_transmission(C.byref(a_ana), xs, 0.0, lam_q)
        tol = 2e-6 if lam_q % 2 == 0 else 3e-4                           # on / between wavelength nodes
        assert abs(t_tab - t_ana) < tol * max(1.0, -math.log(t_ana)), (lam_q, h, t_tab, t_ana)
    assert L.orc_transmission_tabulated(C.byref(a_tab), 10.0, 0.0, 400.0) == 1.0   # emission at the observation level
    r_ana, r_tab = O.run(cfg, record=True), O.run(tab, record=True)
    assert r_ana["counters"]["emitted"] == r_tab["counters"]["emitted"]
    flips = int((r_ana["photons"]["status"] != r_tab["photons"]["status"]).sum())
    assert flips <= 3e-4 * r_ana["counters"]["emitted"] + 3
    same = r_ana["photons"]["status"] == r_tab["photons"]["status"]
    assert np.abs(r_ana["photons"]["T"][same] - r_tab["photons"]["T"][same]).max() < 3e-4
    dbl = copy.deepcopy(tab)
    dbl["atmosphere"]["ext_tau_v"] = 2.0 * tab["atmosphere"]["ext_tau_v"]
    r_dbl = O.run(dbl, record=True)
    m = (r_tab["photons"]["T"] > 0) & (r_tab["photons"]["status"] >= O.ST_ROULETTE - 4) & (r_tab["photons"]["T"] < 1)
    both = m & (r_dbl["photons"]["T"] > 0) & (r_dbl["photons"]["T"] < 1)
    assert both.sum() > 1000 and np.allclose(r_dbl["photons"]["T"][both], r_tab["photons"]["T"][both] ** 2, rtol=1e-9)


# ---------------------------------------------------------------------------------- multiple scattering (R18, row f2)
def test_multiple_scattering_substeps():
    """Highland / PDG width, and the correlated (offset, angle) pair per plane: for one piece in a
    constant-density slab and no field, Var(theta_plane) = theta0^2, Var(y_plane) = ds^2 theta0^2 / 3,
    corr(y, theta) = sqrt(3)/2; after n pieces the angular variance adds up; zero density or a stiff
    particle reproduce R16's pieces; the draw depends on (seed, track id, piece) only."""
    L = O.lib()
    assert abs(L.orc_highland_theta0(1.0, 1.0, 1.0, 0.1) - 0.0136 * math.sqrt(0.1) * (1 + 0.038 * math.log(0.1))) < 1e-15
    assert abs(L.orc_highland_theta0(0.5, 2.0, 2.0, 0.01) - 0.0136 / (0.5 * 2.0) * 2.0 * 0.1 * (1 + 0.038 * math.log(0.01 * 4 / 0.25))) < 1e-15
    assert L.orc_highland_theta0(1.0, 1.0, 1.0, 0.0) == 0.0
    atm = W.make_atmosphere("planar_exp")
    n_nodes = atm["n_nodes"]
    rho = 0.1                                                             # g/cm^2 per m, constant
    atm["overburden"] = (rho * atm["dh"] * (n_nodes - 1 - np.arange(n_nodes))).astype(np.float32)
    n = 20000
    trk = dict(x=np.zeros(n), y=np.zeros(n), z=np.full(n, 20000.0), dx=np.zeros(n), dy=np.zeros(n), dz=-np.ones(n),
               len=np.full(n, 50.0), beta=np.ones(n), t0=np.zeros(n), charge=-np.ones(n), p_GeV=np.full(n, 0.05))
    trk = {k: np.asarray(v, np.float32) for k, v in trk.items()}
    one = O.substep_tracks_ms(atm, trk, (0, 0, 0), 0.01, 50.0, 36.62)
    assert one["offsets"][-1] == n
    th0 = L.orc_highland_theta0(1.0, float(np.float32(0.05)), -1.0, rho * 50.0 / float(np.float32(36.62)))
    s = one["segments"]
    # chord of a single piece: end point = start + (0,0,-ds) + (ya, yb, 0) -> transverse direction components = y/len
    yx, yy = s["dx"].astype(np.float64) * s["len"], s["dy"].astype(np.float64) * s["len"]
    for y in (yx, yy):
        assert abs(y.var() / (50.0 ** 2 * th0 ** 2 / 3.0) - 1.0) < 5 * math.sqrt(2.0 / n)
        assert abs(y.mean()) < 5 * 50.0 * th0 / math.sqrt(3.0 * n)
    # several pieces: direction of the last chord carries the accumulated deflection
    m = 8
    many = O.substep_tracks_ms(atm, trk, (0, 0, 0), 0.01, 50.0 / m, 36.62)
    assert many["offsets"][-1] == n * m
    th0m = L.orc_highland_theta0(1.0, float(np.float32(0.05)), -1.0, rho * (50.0 / m) / float(np.float32(36.62)))
    sm = many["segments"]
    last = np.arange(n) * m + (m - 1)
    # last chord direction = accumulated angle of m-1 pieces + own offset/len: Var = (m-1) th0m^2 + th0m^2/3
    want = (m - 1 + 1.0 / 3.0) * th0m ** 2
    assert abs(sm["dx"][last].astype(np.float64).var() / want - 1.0) < 6 * math.sqrt(2.0 / n)
    # continuity of the walk: piece 1 starts where piece 0 ended
    a1 = sm["dx"][np.arange(n) * m].astype(np.float64) * sm["len"][np.arange(n) * m]   # y of piece 0
    x0 = sm["x"][np.arange(n) * m + 1].astype(np.float64)                 # start of piece 1 = y of piece 0 (x started at 0)
    assert np.allclose(a1, x0, atol=2e-4)
    # the (offset, angle) pair of one piece is correlated: Cov(y_0, theta_0) = ds theta0^2 / 2, i.e. corr = sqrt(3)/2;
    # chord 1's direction = theta_0 + (independent offset of piece 1)/ds
    dir1 = sm["dx"][np.arange(n) * m + 1].astype(np.float64)
    cov = np.mean((a1 - a1.mean()) * (dir1 - dir1.mean()))
    assert abs(cov / ((50.0 / m) * th0m ** 2 / 2.0) - 1.0) < 0.06
    # zero density: identical to the magnetic pieces
    vac = dict(atm, overburden=np.zeros(n_nodes, np.float32))
    B = (2.0e-5, -0.5e-5, -4.3e-5)
    sub = {k: v[:200] for k, v in trk.items()}
    r16 = O.substep_tracks(sub, B, 0.01)
    r18 = O.substep_tracks_ms(vac, sub, B, 0.01, 0.0, 36.62)
    assert np.array_equal(r16["offsets"], r18["offsets"])
    for k in ("x", "y", "z", "dx", "dy", "dz", "len", "t0"):
        assert np.allclose(r16["segments"][k], r18["segments"][k], rtol=2e-6, atol=2e-3), k
    # draws depend on (seed, track id, piece): shifting the id base shifts the result
    a = O.substep_tracks_ms(atm, {k: v[5:9] for k, v in trk.items()}, (0, 0, 0), 0.01, 50.0, 36.62, track_id_base=5)
    assert np.array_equal(a["segments"]["dx"], one["segments"]["dx"][5:9])


def _brute_force_ray_3d(atm, A, U, ds=2.0):
    """RK4 on d/ds (n u) = grad n in three dimensions, n(|X - C| - R) from the linearly interpolated
    table, C = (0, 0, -(R + h_obs)), to the plane z = 0; many rays at once (independent numpy code)."""
    eta = atm["refractivity"].astype(np.float64)
    dh, R = atm["dh"], atm["earth_radius"]
    Cc = np.array([0.0, 0.0, -(R + atm["h_obs"])])

    def n_and_grad(p):
        rv = p - Cc
        r = np.linalg.norm(rv, axis=1)
        f = np.clip((r - R) / dh, 0.0, len(eta) - 1.000001)
        i = f.astype(int)
        g = (eta[i + 1] - eta[i]) / dh
        return 1 + eta[i] + (f - i) * (eta[i + 1] - eta[i]), g[:, None] * rv / r[:, None]

    def rhs(y):
        n, g = n_and_grad(y[:, :3])
        return np.concatenate([y[:, 3:6] / n[:, None], g, n[:, None]], axis=1)

    n0, _ = n_and_grad(A)
    y = np.concatenate([A, n0[:, None] * U, np.zeros((len(A), 1))], axis=1)
    out = np.zeros_like(y)
    live = np.ones(len(A), bool)
    while live.any():
        k1 = rhs(y); k2 = rhs(y + 0.5 * ds * k1); k3 = rhs(y + 0.5 * ds * k2); k4 = rhs(y + ds * k3)
        yn = y + ds / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        hit = live & (yn[:, 2] <= 0.0)
        if hit.any():
            f = y[hit, 2] / (y[hit, 2] - yn[hit, 2])
            out[hit] = y[hit] + f[:, None] * (yn[hit] - y[hit])
            live &= ~hit
        y = np.where(live[:, None], yn, y)
    u = out[:, 3:6] / np.linalg.norm(out[:, 3:6], axis=1)[:, None]
    return out[:, :2], u, out[:, 6] / C_LIGHT


def _photons_vs_3d(d_km, az_deg, zen_deg, h, flat, trace, n_ph=10, table=None, return_photons=False, **par):
    """One 1 mm segment (emission point known to 1 mm) at horizontal distance d from the origin; the
    landed photons of the whole oracle run against the 3-D integration of the same rays."""
    cfg = W.make_config(4, n_segments=1)
    cfg["params"].update(trace=trace, trans="weight", lv1=False, lv2=False, write="all", bunch_weight=2e-5, flat_plane=flat, **par)
    cfg["detector"]["tel_xyzr"] = np.zeros((0, 4), np.float32)
    if trace != "table":
        cfg["table"] = None
    elif table is not None:
        cfg["table"] = dict(cfg["table"], **table)
    s = cfg["segments"]
    th, az = math.radians(zen_deg), math.radians(az_deg)
    for k, v in zip(("x", "y", "z", "dx", "dy", "dz"),
                    (d_km * 1e3, 0.0, h, math.sin(th) * math.cos(az), math.sin(th) * math.sin(az), -math.cos(th))):
        s[k][:] = v
    s["len"][:] = 1e-3; s["beta"][:] = 1.0; s["t0"][:] = 0.0; s["charge"][:] = 1.0
    A = np.array([s["x"][0], s["y"][0], s["z"][0]], np.float64)
    ph = O.run(cfg)["photons"]
    ph = ph[ph["status"] == O.ST_LANDED][:n_ph]
    assert len(ph) == n_ph
    if return_photons:
        return ph
    I = np.stack([ph["x_line"], ph["y_line"], np.zeros(len(ph))], 1)
    U = I - A
    U /= np.linalg.norm(U, axis=1)[:, None]
    xy, u, t = _brute_force_ray_3d(cfg["atmosphere"], np.repeat(A[None], len(ph), 0), U)
    dpos = np.hypot(xy[:, 0] - ph["x"], xy[:, 1] - ph["y"]).max()
    ddir = np.arccos(np.clip(u[:, 0] * ph["ux"] + u[:, 1] * ph["uy"] + u[:, 2] * ph["uz"], -1, 1)).max()
    shift = np.hypot(ph["x"] - ph["x_line"], ph["y"] - ph["y_line"]).mean()
    return dpos, np.abs(t - ph["t"]).max(), ddir, shift, np.hypot(I[:, 0], I[:, 1]).mean()


def test_whole_photons_against_3d_ray_integration_flat_plane():
    """R9's application (I' = I + dd e_h, t = t_e + D/c + dt, direction turned in the ray plane) and R19's
    flat observation plane (Fig. 4.10), pinned on whole photons of orc_run: off-centre emission points,
    arbitrary azimuth, against a 3-D ray integration to the plane z = 0.  Near the origin both agree to
    < 1 mm; with flat_plane the agreement stays at the 0.1 mm / 1 ps level out to 25 km from the origin
    (refraction shifts of 1.4-23 m); without it the sag of the sphere under the plane (28 m at 19 km)
    costs centimetres and 0.1 ns - the thesis' reason for tables "relative to a flat observation plane"."""
    for flat in (False, True):
        dpos, dt, ddir, shift, rho = _photons_vs_3d(0.2, 30.0, 20.0, 12000.0, flat, "numeric")
        assert rho > 4000 and 0.3 < shift < 0.6 and dpos < 1e-3 and dt < 1e-3 and ddir < 1e-6
    for case in ((2.0, 200.0, 60.0, 12000.0), (20.0, 90.0, 50.0, 12000.0), (30.0, 180.0, 70.0, 12000.0)):
        dpos, dt, ddir, shift, rho = _photons_vs_3d(*case, True, "numeric")
        assert shift > 2.5 and dpos < 5e-4 and dt < 1e-3 and ddir < 5e-6, (case, dpos, dt, ddir)
    # the table path takes the same step (bilinear error of the 512 x 256 table on top: < 1 cm, 0.01 ns)
    dpos, dt, ddir, shift, rho = _photons_vs_3d(8.0, 170.0, 60.0, 12000.0, True, "table")
    assert rho > 12000 and dpos < 1e-2 and dt < 1e-2 and ddir < 5e-6
    # a dispersive cone angle (R13) does not change the ray: the n(h) table (valid at lambda0) refracts, so the
    # arrival direction still follows the 3-D integration in that medium
    dpos, dt, ddir, shift, rho = _photons_vs_3d(2.0, 200.0, 60.0, 12000.0, True, "numeric", disp_b_nm2=5700.0, disp_lambda0_nm=400.0)
    assert dpos < 5e-4 and dt < 1e-3 and ddir < 5e-6
    # without the flat-plane step the same photons are off by centimetres at 19 km from the origin
    dpos, dt, ddir, shift, rho = _photons_vs_3d(2.0, 200.0, 60.0, 12000.0, False, "numeric")
    assert rho > 18000 and 0.05 < dpos < 0.15 and 0.1 < dt < 0.4


def test_flat_plane_table_of_the_thesis_four_axes():
    """R21 (Fig. 4.10): the table "relative to a flat observation plane" over (height, zenith, polar radius of the
    straight-line point, pointing angle as even / odd part).  Pins: E(rho = 0) is the 2-D table and O(0) = 0; the lookup is
    exact on functions that are trilinear in (h, zenith, rho) and linear in cos(chi); whole photons of orc_run through the
    table land where R19's exact sphere-to-plane step (itself pinned by the 3-D ray integration) puts them, for outward,
    inward and tangential flight (0.3 mm out to 30 km from the origin; the transverse part alone is 6 mm there), and where
    the 3-D integration puts them; the even part grows like rho^2 (sag) and the odd part like rho (tilt of the plane
    against the sphere)."""
    tab = dict(n_h=128, n_zen=128, h_max=20000.0, zen_max_deg=75.0, n_rho=17, rho_max_m=32000.0)
    cfg = W.make_config(4, n_segments=1)
    t = dict(cfg["table"], **tab)
    d2 = O.build_table(cfg["atmosphere"], t)
    d4 = O.build_table_flat(cfg["atmosphere"], t)
    assert d4.shape == (2, 17, 128, 128, 5)
    ok = np.isfinite(d2[..., 0]) & np.isfinite(d4[0, 0, ..., 0])
    # (the refracted ray lands |dd| short of the origin, where the sphere is already dd^2 / 2 Rg below the plane: 5e-5 relative)
    assert ok.mean() > 0.95 and np.allclose(d4[0, 0][ok], d2[ok], rtol=5e-5, atol=1e-5) and np.all(d4[1, 0][ok] == 0)
    # scaling with rho at a node well inside (12 km, 50 deg): even ~ rho^2, odd ~ rho
    a, b = 77, 85
    E, Od = d4[0, :, a, b, 0].astype(np.float64) - d4[0, 0, a, b, 0], d4[1, :, a, b, 0].astype(np.float64)
    assert E[16] / E[8] == pytest.approx(4.0, rel=0.05) and Od[16] / Od[8] == pytest.approx(2.0, rel=0.05)
    assert 0.002 < abs(E[16]) < 0.2 and 0.002 < abs(Od[16]) < 0.2        # millimetres to centimetres at 32 km
    # exactness of the lookup on a function linear in every axis
    lin = np.zeros_like(d4)
    hh, zz, rr = np.meshgrid(np.linspace(0, 20000, 128), np.linspace(0, math.radians(float(np.float32(75.0))), 128), np.linspace(0, 32000, 17), indexing="ij")
    for k in range(5):
        lin[0, ..., k] = np.transpose(1.0 + 2e-4 * hh - 3.0 * zz + 5e-5 * rr + 1e-8 * hh * rr * zz, (2, 0, 1)) * (k + 1)
        lin[1, ..., k] = np.transpose(0.5 - 1e-5 * hh + 2e-5 * rr * zz, (2, 0, 1)) * (k + 1)
    for h, z, r, c in ((1234.5, 0.3, 7777.0, 0.4), (19999.0, 1.2, 31999.0, -1.0), (0.0, 0.0, 0.0, 1.0)):
        bad, v, perp = O.table_flat_lookup(t, d2, lin, h, z, r, c)
        ev, od = (1.0 + 2e-4 * h - 3.0 * z + 5e-5 * r + 1e-8 * h * r * z), (0.5 - 1e-5 * h + 2e-5 * r * z)
        assert not bad and np.allclose(v[:3], (ev + c * od) * np.arange(1, 4), rtol=2e-6)
        assert np.allclose(v[3:], ev * np.arange(4, 6), rtol=2e-6) and perp == pytest.approx(4 * od, rel=2e-6)
    assert O.table_flat_lookup(t, d2, d4, 5000.0, 0.5, 33000.0, 0.0)[0]      # outside the table: TABLE_RANGE
    # whole photons: table (flat_plane = 2) against R19's analytic step (flat_plane = 1) on the same 2-D table, and against
    # the 3-D integration; flight outward (az 0), inward (180), tangential (90), oblique
    worst = 0.0
    for d_km, az, zen in ((15.0, 0.0, 50.0), (25.0, 180.0, 40.0), (20.0, 90.0, 55.0), (12.0, 230.0, 60.0), (0.3, 40.0, 20.0)):
        p1 = _photons_vs_3d(d_km, az, zen, 12000.0, 1, "table", table=tab, return_photons=True)
        p2 = _photons_vs_3d(d_km, az, zen, 12000.0, 2, "table", table=tab, return_photons=True)
        assert np.array_equal(p1["j"], p2["j"])
        dpos = np.hypot(p1["x"] - p2["x"], p1["y"] - p2["y"]).max()
        worst = max(worst, dpos)
        assert dpos < 3e-4 and np.abs(p1["t"] - p2["t"]).max() < 1e-3, (d_km, az, zen, dpos)   # second order in rho/Rg remains
        assert np.abs(p1["ux"] - p2["ux"]).max() < 1e-7 and np.abs(p1["uz"] - p2["uz"]).max() < 1e-7
        dpos3, dt3, ddir3, shift, rho = _photons_vs_3d(d_km, az, zen, 12000.0, 2, "table", table=tab)
        assert dpos3 < 2e-2 and dt3 < 2e-2 and ddir3 < 5e-6, (d_km, az, zen, dpos3, dt3)   # + bilinear error of this coarse table
    print("flat-plane table vs analytic step, worst position difference [m]:", worst)


# ------------------------------------------------------------------ A5 cylindrical atmosphere model (R24, row f1)
def _brute_force_ray_cyl(atm, h_e, zen, psi, ds=2.0):
    """RK4 on d/ds (n u) = grad n with n(h), h = sqrt(x'^2 + z'^2) - R: the medium of coaxial cylinders about the y' axis
    (independent numpy code); from (0, 0, R + h_e) to the cylinder h = h_obs.  Returns position and unit direction."""
    eta = atm["refractivity"].astype(np.float64)
    dh, R, hobs = atm["dh"], atm["earth_radius"], atm["h_obs"]

    def n_and_grad(p):
        r = math.hypot(p[0], p[2])
        f = min(max((r - R) / dh, 0.0), len(eta) - 1.000001)
        i = int(f)
        g = (eta[i + 1] - eta[i]) / dh
        return 1 + eta[i] + (f - i) * (eta[i + 1] - eta[i]), g * np.array([p[0] / r, 0.0, p[2] / r]), r - R

    def rhs(y):
        n, g, _ = n_and_grad(y[:3])
        return np.concatenate([y[3:6] / n, g])

    A = np.array([0.0, 0.0, R + h_e])
    U = np.array([math.sin(zen) * math.cos(psi), math.sin(zen) * math.sin(psi), -math.cos(zen)])
    y = np.concatenate([A, n_and_grad(A)[0] * U])
    while True:
        k1 = rhs(y); k2 = rhs(y + 0.5 * ds * k1); k3 = rhs(y + 0.5 * ds * k2); k4 = rhs(y + ds * k3)
        yn = y + ds / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
        h0, h1 = n_and_grad(y[:3])[2], n_and_grad(yn[:3])[2]
        if h1 <= hobs:
            f = (h0 - hobs) / (h0 - h1)
            out = y + f * (yn - y)
            return out[:3], out[3:6] / np.linalg.norm(out[3:6])
        y = yn


def test_cylindrical_model_tracer_limits_and_brute_force():
    """Reading R24 (thesis sec. 3.3.3): the gradient keeps its rotation angle, only its zenith angle follows the
    position: coaxial cylinders.  Pins of the layered tracer (Eq. 3.15 in three dimensions): flight in the plane of
    curvature is the spherical model's ray, flight along the axis is the planar model's ray, the component of n u along
    the axis is conserved, oblique flight against an independent 3-D RK4 integration in that medium; and the thesis'
    statements: the model agrees with the spherical one near the plane of curvature and loses accuracy with the
    distance travelled across it ("significant impact only for ... several tenths of kilometres")."""
    atm = W.make_config(4, n_segments=1)["atmosphere"]
    hg = atm["h_obs"]
    for h_e, zen in ((12000.0, 0.9), (30000.0, 0.5), (5000.0, 1.2)):
        sph = O.trace(atm, True, h_e, zen, hg)
        bad_c, cyl = O.trace_cyl(atm, h_e, zen, 0.0, hg)
        assert sph is not None and not bad_c
        assert cyl[0] == pytest.approx(sph["disp"], rel=1e-12) and cyl[1] == pytest.approx(sph["S"], rel=1e-13)
        assert cyl[2] == pytest.approx(sph["cT"], rel=1e-13) and cyl[3] == pytest.approx(sph["X"], rel=1e-12) and abs(cyl[5]) < 1e-9
        pla = O.trace(dict(atm, model="planar"), False, h_e, zen, hg)
        bad_c, cyl = O.trace_cyl(atm, h_e, zen, 0.5 * math.pi, hg)
        assert pla is not None and not bad_c and abs(cyl[0]) < 1e-12
        assert cyl[5] == pytest.approx(pla["disp"], rel=1e-12) and cyl[1] == pytest.approx(pla["S"], rel=1e-13) and cyl[2] == pytest.approx(pla["cT"], rel=1e-13)
    Rg = atm["earth_radius"] + hg
    n_e = 1.0 + O.refractivity(atm, 12000.0)
    n_g = 1.0 + O.refractivity(atm, hg)
    for zen, psi in ((0.9, 0.7), (1.05, 2.3), (0.6, -1.1)):
        bad, cyl = O.trace_cyl(atm, 12000.0, zen, psi, hg)
        assert not bad
        assert n_g * cyl[7] == pytest.approx(n_e * math.sin(zen) * math.sin(psi), rel=1e-13)      # n u_axis conserved
        assert np.linalg.norm(cyl[6:9]) == pytest.approx(1.0, abs=1e-13)
        pos, u = _brute_force_ray_cyl(atm, 12000.0, zen, psi)
        got = np.array([Rg * math.sin(cyl[0]), cyl[5], Rg * math.cos(cyl[0])])
        assert np.linalg.norm(got - pos) < 5e-4, (zen, psi, got - pos)
        assert np.arccos(np.clip(u @ np.array(cyl[6:9]), -1, 1)) < 2e-6
    # thesis: agrees with the spherical model near the plane of curvature, degrades with the distance across it.  The same
    # photon (12 km, local zenith 60 deg) flying across the plane of curvature, in both models: the straight line lands
    # 21 km away; the correction along the flight differs by centimetres, in the plane of curvature by nothing
    zen = math.radians(60.0)
    sph = O.trace(atm, True, 12000.0, zen, hg)
    re = atm["earth_radius"] + 12000.0
    dd_sph = Rg * sph["disp"] - Rg * (math.asin(re * math.sin(zen) / Rg) - zen)
    diffs = []
    for psi_deg in (0.0, 10.0, 45.0, 90.0):
        bad, corr = O.cyl_correction(atm, 12000.0, zen, math.radians(psi_deg))
        assert not bad
        diffs.append(abs(corr[0] - dd_sph))
    assert diffs[0] < 1e-9 and diffs[1] < 3e-3 and diffs[2] > 5 * diffs[1] and diffs[3] > diffs[2] > 0.01
    print("cylindrical - spherical, displacement along the flight from 12 km at 60 deg, psi = 0 / 10 / 45 / 90 deg [m]:", diffs)
    # and with the height (= distance travelled): from 3 km the same geometry differs by millimetres
    sph3 = O.trace(atm, True, 3000.0, zen, hg)
    re3 = atm["earth_radius"] + 3000.0
    dd3 = Rg * sph3["disp"] - Rg * (math.asin(re3 * math.sin(zen) / Rg) - zen)
    bad, corr3 = O.cyl_correction(atm, 3000.0, zen, math.radians(90.0))
    assert abs(corr3[0] - dd3) < 5e-3 and diffs[3] > 5 * abs(corr3[0] - dd3)


def test_cylindrical_model_table_and_run():
    """R24: the cylindrical model's table over (height, zenith, cos^2 of the flight azimuth against the plane of curvature):
    nodes are the tracer's corrections, c = 1 is the spherical table and c = 0 the planar one; the lookup is exact on
    multilinear functions; whole runs: table photons against per-photon numerical tracing (interpolation error only),
    and against the spherical model (millimetres near the origin)."""
    cfg = W.make_config(4, n_segments=300)
    cfg["atmosphere"]["model"] = "cylindrical"
    cfg["table"] = dict(n_h=96, n_zen=96, h_max=30000.0, zen_max_deg=60.0, n_c=5)
    cfg["params"].update(write="all")
    atm, t = cfg["atmosphere"], cfg["table"]
    d3 = O.build_table_cyl(atm, t)
    assert d3.shape == (5, 96, 96, 5)
    sph = O.build_table(dict(atm, model="spherical"), t)
    pla = O.build_table(dict(atm, model="planar"), t)
    ok = np.isfinite(sph[..., 0]) & np.isfinite(d3[4, ..., 0])
    assert ok.mean() > 0.99
    for ch in (0, 2, 3):
        assert np.allclose(d3[4, ..., ch][ok], sph[..., ch][ok], rtol=2e-5, atol=2e-6)       # psi = 1e-3 rad inside the end
        assert np.allclose(d3[0, ..., ch][ok], pla[..., ch][ok], rtol=2e-5, atol=2e-6)
    a, b, k = 40, 70, 2
    bad, corr = O.cyl_correction(atm, a * 30000.0 / 95, b * math.radians(float(np.float32(60.0))) / 95, math.acos(math.sqrt(0.5)))
    assert not bad and d3[k, a, b, 0] == pytest.approx(corr[0], rel=1e-6) and d3[k, a, b, 1] == pytest.approx(corr[1] / 0.5, rel=1e-5)
    assert abs(d3[k, a, b, 1]) > 1e-3                                   # the across displacement exists (millimetres)
    gpu_like = O.run(cfg)                                               # trace = table
    num = copy.deepcopy(cfg)
    num["params"]["trace"] = "numeric"
    ref = O.run(num)
    a_, b_ = gpu_like["photons"], ref["photons"]
    both = (a_["status"] == O.ST_LANDED) & (b_["status"] == O.ST_LANDED)
    assert both.sum() > 5e4 and (a_["status"] != b_["status"]).mean() < 2e-4
    d = np.hypot(a_["x"][both] - b_["x"][both], a_["y"][both] - b_["y"][both])
    assert d.max() < 5e-3 and np.abs(a_["t"][both] - b_["t"][both]).max() < 5e-3           # this coarse table's interpolation error
    sphc = copy.deepcopy(cfg)
    sphc["atmosphere"]["model"] = "spherical"
    sphc["table"] = dict(n_h=96, n_zen=96, h_max=30000.0, zen_max_deg=60.0)
    sp = O.run(sphc)["photons"]
    both = (a_["status"] == O.ST_LANDED) & (sp["status"] == O.ST_LANDED)
    d = np.hypot(a_["x"][both] - sp["x"][both], a_["y"][both] - sp["y"][both])
    assert 1e-7 < d.max() < 5e-3                                        # near the origin the two models agree to millimetres


# ------------------------------------------------------------------ sanitizers
def test_oracle_runs_clean_under_address_and_undefined_behaviour_sanitizers():
    """The oracle compiled with -fsanitize=address,undefined (-fno-sanitize-recover) runs small instances of all five
    configs, the optional features, the table builder and the sub-stepping without a report."""
    import subprocess
    import sys
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    if not os.path.isabs(asan) or not os.path.exists(asan):
        pytest.skip("libasan not available")
    code = r"""
import copy, numpy as np
from oracle import c8ph_oracle as O
from paper_2405_04229_b200 import workloads as W
O.build()
tot = 0
for k, n in ((0, 30), (1, 10), (2, 300), (3, 2000), (4, 40)):
    cfg = W.make_config(k, n_segments=n)
    if k == 3:
        cfg["segments"]["edep"][:] *= 400.0
    tot += O.run(cfg, threads=2)["counters"]["emitted"]
cfg = W.make_config(4, n_segments=40)
cfg["params"].update(disp_b_nm2=5700.0, disp_lambda0_nm=400.0, flat_plane=True,
                     eff=np.linspace(0.2, 0.9, 31).astype(np.float32), eff_lambda0_nm=250.0, eff_dlambda_nm=15.0)
cfg["segments"]["x"][3] = np.nan
cfg["segments"]["id"] = np.arange(40, dtype=np.uint64)[::-1].copy()
tot += O.run(cfg, threads=2)["counters"]["emitted"]
trk = {f: v[:16].copy() for f, v in W.make_config(4, n_segments=16)["segments"].items() if f != "edep"}
trk["len"][:] = 300.0
trk["p_GeV"] = np.full(16, 0.05, np.float32)
tot += len(O.substep_tracks(trk, (2e-5, -0.5e-5, -4.3e-5), 0.01)["segments"]["x"])
print("sanitized oracle ok", tot)
"""
    env = dict(os.environ, C8PH_ORACLE_SANITIZE="1", LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0:abort_on_error=0",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1", PYTHONPATH=os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])
    assert "ERROR: AddressSanitizer" not in r.stderr and "runtime error:" not in r.stderr, r.stderr[-4000:]
