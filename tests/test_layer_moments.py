"""The closed form of the planar layered Snell sum that the device uses ("layered sum";
c8ph_init_atmosphere builds the layer moments, k_emit_propagate<.., TRACE_NUMERIC, ..> evaluates the series) against the
oracle's layer-by-layer tracer (Eq. 3.15): the identity behind it, checked in fp64 on the CPU.

For a photon emitted at height h_e with zenith angle z, K = n_e sin z, r_e = 1 / (n_e cos z), nu = n^2 - 1 and
x_l = (nu_l - nu_e) r_e^2, a layer of thickness d_l contributes
    horizontal path   d_l K r_l,      optical path   d_l n_l^2 r_l,      slant depth   dX_l n_l r_l,
with r_l = (n_l^2 - K^2)^(-1/2) = r_e (1 + x_l)^(-1/2).  Expanding in x_l turns the three sums over layers into
polynomials in r_e^2 and nu_e whose coefficients are sums of d_l nu_l^p and dX_l n_l nu_l^p over the layers below the
emission cell: tables over the height grid, built once.
"""
import math
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import c8ph_oracle as O                                    # noqa: E402
from paper_2405_04229_b200 import workloads as W                      # noqa: E402


def _moments(atm):
    """Layer moments up to every node, as c8ph_init_atmosphere builds them (layers, mid-height values)."""
    eta = atm["refractivity"].astype(np.float64)
    xv = atm["overburden"].astype(np.float64)
    n, dh, h0 = len(eta), float(atm["dh"]), float(atm["h0"])
    fg = min(max((atm["h_obs"] - h0) / dh, 0.0), n - 1.0)
    kg = min(int(fg), n - 2)
    frg = fg - kg
    mom = np.zeros((8, n))
    acc = np.zeros(8)
    for k in range(kg + 1, n):
        if k == kg + 1:
            e, th, dx = eta[kg] + 0.5 * (1.0 + frg) * (eta[kg + 1] - eta[kg]), (1.0 - frg) * dh, (1.0 - frg) * (xv[kg] - xv[kg + 1])
        else:
            e, th, dx = 0.5 * (eta[k - 1] + eta[k]), dh, xv[k - 1] - xv[k]
        nu = e * (2.0 + e)
        acc[:4] += th * nu ** np.arange(1, 5)
        acc[4:] += dx * (1.0 + e) * nu ** np.arange(0, 4)
        mom[:, k] = acc
    return mom, fg, kg


def _closed_form(atm, mom, fg, kg, h_e, zen):
    eta = atm["refractivity"].astype(np.float64)
    xv = atm["overburden"].astype(np.float64)
    n, dh, h0 = len(eta), float(atm["dh"]), float(atm["h0"])
    fe = min(max((h_e - h0) / dh, 0.0), n - 1.0)
    ke = min(int(fe), n - 2)
    fre = fe - ke
    assert ke > kg
    eta_e = eta[ke] + fre * (eta[ke + 1] - eta[ke])
    n_e, cz = 1.0 + eta_e, math.cos(zen)
    K, r_e = n_e * math.sin(zen), 1.0 / (n_e * cz)
    re2 = r_e * r_e
    # the partial layer of the emission cell
    e_p = eta[ke] + 0.5 * fre * (eta[ke + 1] - eta[ke])
    nu_p, th_p, g_p = e_p * (2.0 + e_p), fre * dh, fre * (xv[ke] - xv[ke + 1]) * (1.0 + e_p)
    M = [mom[p, ke] + th_p * nu_p ** (p + 1) for p in range(4)]
    G = [mom[4 + p, ke] + g_p * nu_p ** p for p in range(4)]
    H = (fe - fg) * dh
    d = -eta_e * (2.0 + eta_e)
    S1 = re2 * (M[0] + d * H)
    S2 = re2 ** 2 * (M[1] + 2 * d * M[0] + d * d * H)
    S3 = re2 ** 3 * (M[2] + 3 * d * M[1] + 3 * d * d * M[0] + d ** 3 * H)
    S4 = re2 ** 4 * (M[3] + 4 * d * M[2] + 6 * d * d * M[1] + 4 * d ** 3 * M[0] + d ** 4 * H)
    Am = -S1 / 2 + 3 * S2 / 8 - 5 * S3 / 16 + 35 * S4 / 128
    Ap = S1 / 2 - S2 / 8 + S3 / 16 - 5 * S4 / 128
    T1 = re2 * (G[1] + d * G[0])
    T2 = re2 ** 2 * (G[2] + 2 * d * G[1] + d * d * G[0])
    T3 = re2 ** 3 * (G[3] + 3 * d * G[2] + 3 * d * d * G[1] + d ** 3 * G[0])
    x_max = (atm["refractivity"].astype(np.float64).max() * 2.0) * re2
    return dict(dd=K * r_e * Am, dT=H * r_e * n_e * eta_e + Ap * n_e * cz + K * K * r_e * Am,
                X=r_e * (G[0] - T1 / 2 + 3 * T2 / 8 - 5 * T3 / 16), H=H, x_max=x_max)


@pytest.mark.parametrize("scale", [1.0, 6.0])
def test_closed_form_equals_the_layer_loop(scale):
    atm = W.make_atmosphere("planar_exp", h_obs=2000.0, rayleigh=True)
    atm["refractivity"] = (scale * atm["refractivity"].astype(np.float64)).astype(np.float32)
    mom, fg, kg = _moments(atm)
    checked = 0
    for h_e in (2013.0, 2500.0, 4321.0, 9000.0, 18000.0, 40000.0, 99000.0):
        for zen_deg in (0.0, 10.0, 35.0, 60.0, 70.0, 78.0):
            zen = math.radians(zen_deg)
            c = _closed_form(atm, mom, fg, kg, h_e, zen)
            if not c["x_max"] < 0.02:                     # where the device keeps the loop
                continue
            o = O.trace(atm, False, h_e, zen, atm["h_obs"])
            H = c["H"]
            dd_o = o["disp"] - H * math.tan(zen)         # difference to the straight line
            dT_o = o["cT"] - H / math.cos(zen)           # optical path minus the straight length
            # truncation: p = 5 term of the series, 63/256 x^5 against x / 2, times the size of the sum
            assert abs(c["dd"] - dd_o) <= 1e-6 * abs(dd_o) + 1e-9 * H, (h_e, zen_deg, c["dd"], dd_o)
            assert abs(c["dT"] - dT_o) <= 1e-7 * abs(dT_o) + 1e-10 * H, (h_e, zen_deg, c["dT"], dT_o)
            assert abs(c["X"] - o["X"]) <= 2e-7 * o["X"], (h_e, zen_deg, c["X"], o["X"])
            checked += 1
    assert checked >= (30 if scale == 1.0 else 20)
