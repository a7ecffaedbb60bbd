"""Pins of the plane-statistics oracle (oracle/stats.py; Fig. 1) by closed forms."""
import numpy as np

from oracle import stats
from paper_2406_19494_b200 import cases


def test_taylor_green_plane_means_closed_form():
    # u = sin x cos y cos z, v = -cos x sin y cos z, w = 0 on [0, 2 pi]^3: over an (x, z) plane at height y
    #   <u> = <v> = 0,  <uu> = cos^2(y)/4,  <vv> = sin^2(y)/4,  <uv> = 0   (midpoint sums of trigonometric
    #   polynomials on >= 3 uniform points are exact)
    c = cases.tgv(16)
    S = stats.plane_sums(c, c.U0, 1)
    P = stats.profiles(S)
    y = 0.5 * (c.yf[:-1] + c.yf[1:])
    assert np.allclose(S[0], (2 * np.pi) ** 2, rtol=1e-14)                 # plane area
    assert np.max(np.abs(P["u"])) < 1e-15 and np.max(np.abs(P["v"])) < 1e-15 and np.all(P["w"] == 0)
    assert np.allclose(P["u'u'"], np.cos(y) ** 2 / 4, atol=1e-15)
    assert np.allclose(P["v'v'"], np.sin(y) ** 2 / 4, atol=1e-15)
    assert np.max(np.abs(P["u'v'"])) < 1e-15
    # isothermal start: T = 1 everywhere, so T_rms = 0 and <rho> = <p>/R = 1 + (cos 2y)(2)/16 / p0 ... checked via p
    assert np.allclose(P["T"], 1.0, rtol=1e-13) and np.max(P["T_rms"]) < 1e-6
    # planes normal to x: <uu> = sin^2(x)/4
    Px = stats.profiles(stats.plane_sums(c, c.U0, 0))
    x = 0.5 * (c.xf[:-1] + c.xf[1:])
    assert np.allclose(Px["u'u'"], np.sin(x) ** 2 / 4, atol=1e-15)


def test_poiseuille_profile_and_area_weighting():
    # no noise: u = 1.5 (1 - (y-1)^2), v = w = 0, rho = T = 1 on the tanh-stretched channel grid
    c = cases.channel(12, 16, 8, noise=0.0)
    P = stats.profiles(stats.plane_sums(c, c.U0, 1))
    y = 0.5 * (c.yf[:-1] + c.yf[1:])
    assert np.allclose(P["u"], 1.5 * (1 - (y - 1) ** 2), rtol=1e-13)
    assert np.max(np.abs(P["u'u'"])) < 1e-14 and np.allclose(P["rho"], 1.0) and np.allclose(P["T"], 1.0, rtol=1e-13)
    # planes normal to x cut through the stretched y axis: the mean of u must be the AREA-weighted one,
    # (1/2) int_0^2 u dy approximated by the midpoint rule on the stretched cells
    Sx = stats.plane_sums(c, c.U0, 0)
    dy = np.diff(c.yf)
    expect = np.sum(1.5 * (1 - (y - 1) ** 2) * dy) / 2.0
    assert np.allclose(Sx[3] / Sx[0], expect, rtol=1e-13)
    assert np.allclose(Sx[0], 2.0 * (4 * np.pi / 3), rtol=1e-13)           # plane area Ly * Lz
