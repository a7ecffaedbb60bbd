"""Pins for the oracle's scheme-level functions (SURVEY.md §8(c) table "What pins each part").

Every expected value here is a closed form, an invariant or a textbook special case — never the
oracle's own formula retyped.  CPU only.
"""
import itertools

import numpy as np
import pytest

GAMMA = 1.4


def rand_prim(rng, vel=1.0):
    return np.array([rng.uniform(0.2, 3.0), *(vel * rng.uniform(-2, 2, 3)), rng.uniform(0.1, 5.0)])


# ------------------------------------------------------------------ thermodynamics (O1, Eq. 2)
def test_prim_cons_roundtrip_and_energy(ora):
    rng = np.random.default_rng(0)
    for _ in range(50):
        W = rand_prim(rng)
        U = ora.prim_to_cons(GAMMA, W)
        # Eq. 2: E = rho e + 1/2 rho u.u with e = p/((gamma-1) rho)
        assert U[4] == pytest.approx(W[4] / 0.4 + 0.5 * W[0] * np.dot(W[1:4], W[1:4]), rel=1e-15)
        assert np.allclose(U[1:4], W[0] * W[1:4], rtol=1e-15)
        assert np.allclose(ora.cons_to_prim(GAMMA, U), W, rtol=1e-13)


def test_sutherland(ora):
    mu = {"sutherland": 1, "mu_ref": 1.716e-5, "T_ref": 273.15, "S": 110.4}
    assert ora.viscosity(mu, 273.15) == pytest.approx(1.716e-5, rel=1e-15)
    for T in (100.0, 220.0, 300.0, 1500.0):
        r = T / 273.15
        expect = 1.716e-5 * r ** 1.5 * (1 + 110.4 / 273.15) / (r + 110.4 / 273.15)
        assert ora.viscosity(mu, T) == pytest.approx(expect, rel=1e-14)
    # air at 300 K is about 1.846e-5 Pa s (textbook value, 3 digits)
    assert ora.viscosity(mu, 300.0) == pytest.approx(1.846e-5, rel=2e-3)
    mu0 = dict(mu, sutherland=0)
    assert ora.viscosity(mu0, 999.0) == 1.716e-5


# ------------------------------------------------------------------ WENO5-JS (O4)
def test_weno5_candidates_exact_for_parabolas(ora):
    # each candidate p_k interpolates cell averages of any parabola exactly at the face x = 1/2
    rng = np.random.default_rng(1)
    for _ in range(20):
        a, b, c = rng.uniform(-2, 2, 3)
        prim = lambda x: a * x + b * x ** 2 / 2 + c * x ** 3 / 3           # antiderivative
        avg = np.array([prim(i + 0.5) - prim(i - 0.5) for i in range(-2, 3)])  # cells -2..2
        face = a + b * 0.5 + c * 0.25
        _, w, p = ora.weno5_detail(avg)
        assert np.allclose(p, face, rtol=0, atol=1e-13)
        assert w.sum() == pytest.approx(1.0, abs=1e-15)
        assert ora.weno5(avg) == pytest.approx(face, abs=1e-13)


def test_weno5_uniform_data_and_smoothness_zero(ora):
    for c in (1.0, -3.7, 71.428571, 1e-3):
        v = np.full(5, c)
        b, w, _ = ora.weno5_detail(v)
        assert np.all(b <= (4 * np.spacing(abs(c))) ** 2)       # (3c - 4c + c) rounds, not exactly 0
        assert np.allclose(w, [0.1, 0.6, 0.3], rtol=1e-15)
        assert abs(ora.weno5(v) - c) <= 2 * np.spacing(abs(c))


def test_weno5_linear_weight_limit(ora):
    # beta_k << eps => weights -> (1/10, 6/10, 3/10) => 5th-order upwind interpolant
    rng = np.random.default_rng(2)
    for _ in range(20):
        v = 1.0 + 1e-8 * rng.uniform(-1, 1, 5)            # weights deviate by ~beta/eps ~ 1e-10
        lin = (2 * v[0] - 13 * v[1] + 47 * v[2] + 27 * v[3] - 3 * v[4]) / 60.0
        assert ora.weno5(v) == pytest.approx(lin, abs=1e-15)


def test_weno5_smoothness_indicators_are_jiang_shu(ora):
    # beta_k = sum_{l=1,2} int (dx^(2l-1)) (d^l p_k/dx^l)^2 dx over the cell: check by quadrature
    rng = np.random.default_rng(3)
    v = rng.uniform(-1, 1, 5)
    b, _, _ = ora.weno5_detail(v)
    xs, ws = np.polynomial.legendre.leggauss(6)
    xs, ws = 0.5 * xs, 0.5 * ws                                   # cell [-1/2, 1/2] (cell "2")
    for k in range(3):
        cells = np.arange(k - 2, k + 1)                           # cell indices relative to cell 2
        # parabola q(x) with prescribed cell averages over the three cells
        A = np.array([[1.0, c, c * c + 1.0 / 12.0] for c in cells])
        c0, c1, c2 = np.linalg.solve(A, v[k:k + 3])
        d1 = c1 + 2 * c2 * xs
        d2 = 2 * c2 * np.ones_like(xs)
        assert b[k] == pytest.approx(np.sum(ws * (d1 ** 2 + d2 ** 2)), rel=1e-12)


def test_weno5_picks_smooth_stencil_at_a_jump(ora):
    # jump between cells 2|3... stencil 0 (cells 0,1,2) is the only smooth one
    v = np.array([1.0, 1.0, 1.0, 5.0, 5.0])
    _, w, _ = ora.weno5_detail(v)
    assert w[0] > 1 - 1e-9
    assert ora.weno5(v) == pytest.approx(1.0, abs=1e-8)


# ------------------------------------------------------------------ HLLC (O5) and Eq. 3
def eq3_flux(d, W):
    rho, vel, p = W[0], W[1:4], W[4]
    E = p / (GAMMA - 1) + 0.5 * rho * vel.dot(vel)
    F = np.empty(5)
    F[0] = rho * vel[d]
    F[1:4] = rho * vel[d] * vel
    F[1 + d] += p
    F[4] = vel[d] * (E + p)
    return F


@pytest.mark.parametrize("d", [0, 1, 2])
def test_flux_phys_is_eq3(ora, d):
    rng = np.random.default_rng(4)
    for _ in range(20):
        W = rand_prim(rng)
        assert np.allclose(ora.flux_phys(d, GAMMA, W), eq3_flux(d, W), rtol=1e-14)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hllc_consistency(ora, d):
    rng = np.random.default_rng(5)
    for _ in range(200):
        W = rand_prim(rng)
        F, Fe = ora.hllc(d, GAMMA, W, W), eq3_flux(d, W)
        assert np.max(np.abs(F - Fe)) <= 1e-14 * max(1.0, np.max(np.abs(Fe)))


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hllc_mirror_symmetry(ora, d):
    rng = np.random.default_rng(6)
    for _ in range(200):
        WL, WR = rand_prim(rng, 0.5), rand_prim(rng, 0.5)
        ML, MR = WR.copy(), WL.copy()
        ML[1 + d] *= -1
        MR[1 + d] *= -1
        F, G = ora.hllc(d, GAMMA, WL, WR), ora.hllc(d, GAMMA, ML, MR)
        sign = -np.ones(5)
        sign[1 + d] = 1.0
        assert np.max(np.abs(G - sign * F)) <= 4e-15 * max(1.0, np.max(np.abs(F)))


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hllc_supersonic_limits(ora, d):
    rng = np.random.default_rng(7)
    for _ in range(50):
        WL, WR = rand_prim(rng, 0.2), rand_prim(rng, 0.2)
        WL[1 + d], WR[1 + d] = 12.0, 11.0                      # both supersonic to the right
        assert np.array_equal(ora.hllc(d, GAMMA, WL, WR), eq3_flux(d, WL)) or np.allclose(
            ora.hllc(d, GAMMA, WL, WR), eq3_flux(d, WL), rtol=1e-15, atol=0)
        WL[1 + d], WR[1 + d] = -11.0, -12.0
        assert np.allclose(ora.hllc(d, GAMMA, WL, WR), eq3_flux(d, WR), rtol=1e-15, atol=0)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hllc_stationary_contact(ora, d):
    WL = np.array([1.0, 0, 0, 0, 0.7])
    WR = np.array([0.125, 0, 0, 0, 0.7])
    F = ora.hllc(d, GAMMA, WL, WR)
    expect = np.zeros(5)
    expect[1 + d] = 0.7
    assert np.max(np.abs(F - expect)) <= 1e-15


@pytest.mark.parametrize("d", [0, 1, 2])
def test_hllc_moving_contact_is_resolved_exactly(ora, d):
    # isolated contact moving with speed u > 0: exact flux is the upwind (left) physical flux;
    # HLLC restores the contact wave, so it must return it (textbook property, Toro ch. 10).
    WL = np.array([1.0, 0.0, 0.0, 0.0, 1.0])
    WR = np.array([0.3, 0.0, 0.0, 0.0, 1.0])
    WL[1 + d] = WR[1 + d] = 0.4
    WL[1 + (d + 1) % 3], WR[1 + (d + 1) % 3] = 0.2, -0.5      # shear across the contact too
    assert np.allclose(ora.hllc(d, GAMMA, WL, WR), eq3_flux(d, WL), rtol=0, atol=2e-15)
    WL[1 + d] = WR[1 + d] = -0.4
    assert np.allclose(ora.hllc(d, GAMMA, WL, WR), eq3_flux(d, WR), rtol=0, atol=2e-15)


def test_hllc_galilean_tangential_covariance(ora):
    # permuting the roles of axes: hllc(d) on cyclically permuted velocity components gives the
    # cyclically permuted flux
    rng = np.random.default_rng(8)
    for _ in range(30):
        WL, WR = rand_prim(rng, 0.5), rand_prim(rng, 0.5)
        F0 = ora.hllc(0, GAMMA, WL, WR)
        for d in (1, 2):
            perm = lambda W: np.array([W[0], *np.roll(W[1:4], d), W[4]])
            Fd = ora.hllc(d, GAMMA, perm(WL), perm(WR))
            assert np.array_equal(Fd, perm(F0))


# ------------------------------------------------------------------ central stencils (O6)
def test_central_stencils_polynomial_exactness(ora):
    rng = np.random.default_rng(9)
    for _ in range(10):
        c = rng.uniform(-1, 1, 5)
        poly = np.polynomial.Polynomial(c)                       # degree 4, in the index xi
        h = 0.37                                                 # uniform metric X_xi = h
        # centre derivative at xi = 0 from samples at -2..2 (exact to degree 4)
        phi = poly(np.arange(-2, 3, dtype=float))
        assert ora.dc(phi, h) == pytest.approx(poly.deriv()(0.0) / h, rel=1e-13, abs=1e-14)
        # face derivative / interpolation at xi = 1/2 from point samples at -1..2
        phi4 = poly(np.arange(-1, 3, dtype=float))
        c3 = c.copy()
        c3[4] = 0.0
        p3 = np.polynomial.Polynomial(c3)
        assert ora.iface(p3(np.arange(-1, 3, dtype=float))) == pytest.approx(p3(0.5), rel=1e-13, abs=1e-14)
        # D^f is exact for degree <= 4 about the face (odd symmetric stencil)
        assert ora.df(phi4, h) == pytest.approx(poly.deriv()(0.5) / h, rel=1e-12, abs=1e-13)


def test_central_stencils_constant_gives_exact_zero(ora):
    for c in (71.428571428, 1e-5, -3.3):
        assert ora.dc([c] * 5, 0.123) == 0.0
        assert ora.df([c] * 4, 0.123) == 0.0


def test_face_derivative_modified_wavenumber(ora):
    theta = 0.3
    xs = np.arange(-1, 3) - 0.5                                   # centred on the face
    val = ora.df(np.sin(theta * xs), 1.0)                         # d/dxi sin(theta xi) at xi = 0
    expect = (54 * np.sin(theta / 2) - 2 * np.sin(3 * theta / 2)) / 24.0
    assert val == pytest.approx(expect, rel=1e-14)


# ------------------------------------------------------------------ sixth-order central stencils
def test_sixth_order_stencils_polynomial_exactness(ora):
    # the coefficients are fixed by exactness: D^c_6 and D^f_6 differentiate polynomials of degree <= 6 exactly
    # (7 / 6 symmetric points), I^f_6 interpolates degree <= 5 exactly; degree 7 / 7 / 6 is NOT exact (the
    # stencils are sixth order, no more); constants give exactly 0 / the constant
    rng = np.random.default_rng(7)
    h = 0.37
    for deg in range(0, 8):
        co = rng.uniform(-1, 1, deg + 1)
        f = np.polynomial.Polynomial(co)
        df = f.deriv()
        x0 = 0.21
        xs_c = x0 + h * np.arange(-3, 4)
        xs_f = x0 + h * (np.arange(-2, 4) - 0.5)           # cells i-2..i+3 around the face at x0
        scale = np.max(np.abs(co)) * max(1.0, (3.5 * h + abs(x0)) ** deg) * 10
        ec = abs(ora.dc6(f(xs_c), h) - df(x0)) / scale
        ef = abs(ora.df6(f(xs_f), h) - df(x0)) / scale
        ei = abs(ora.iface6(f(xs_f)) - f(x0)) / scale
        if deg <= 6:
            assert ec <= 1e-13 and ef <= 1e-13
        else:
            assert ec > 1e-9 and ef > 1e-9
        if deg <= 5:
            assert ei <= 1e-13
        elif deg == 6:
            assert ei > 1e-9
    assert ora.dc6(np.full(7, 3.3), h) == 0.0 and ora.df6(np.full(6, 3.3), h) == 0.0
    assert ora.iface6(np.full(6, 3.3)) == pytest.approx(3.3, rel=1e-15)


def test_sixth_order_modified_wavenumbers(ora):
    # on exp(i k x): D^c_6 -> i k_c, k_c D = (45 sin t - 9 sin 2t + sin 3t)/30; D^f_6 (cell values -> face):
    # k_f D = 2 (2250 sin(t/2) - 125 sin(3t/2) + 9 sin(5t/2))/1920; I^f_6 -> (150 cos(t/2) - 25 cos(3t/2) + 3 cos(5t/2))/128,
    # with t = k D; and each is within O(t^6) of the exact symbol
    D = 0.1
    for t in (0.05, 0.3, 1.1, 2.4):
        k = t / D
        xc = D * np.arange(-3, 4)
        xf = D * (np.arange(-2, 4) - 0.5)
        kc = ora.dc6(np.sin(k * xc), D)                      # derivative of sin at 0 = k
        kf = ora.df6(np.sin(k * xf), D)
        ci = ora.iface6(np.cos(k * xf))                      # value of cos at 0 = 1
        assert kc * D == pytest.approx((45 * np.sin(t) - 9 * np.sin(2 * t) + np.sin(3 * t)) / 30, rel=1e-13)
        assert kf * D == pytest.approx(2 * (2250 * np.sin(t / 2) - 125 * np.sin(1.5 * t) + 9 * np.sin(2.5 * t)) / 1920, rel=1e-13)
        assert ci == pytest.approx((150 * np.cos(t / 2) - 25 * np.cos(1.5 * t) + 3 * np.cos(2.5 * t)) / 128, rel=1e-13)
    t = 0.05
    k = t / D
    assert abs(ora.dc6(np.sin(k * D * np.arange(-3, 4)), D) / k - 1) < t ** 6 / 100
    assert abs(ora.df6(np.sin(k * D * (np.arange(-2, 4) - 0.5)), D) / k - 1) < t ** 6 / 100
    # and sixth order beats fourth order on the same data
    e4 = abs(ora.df(np.sin(k * D * (np.arange(-1, 3) - 0.5)), D) / k - 1)
    e6 = abs(ora.df6(np.sin(k * D * (np.arange(-2, 4) - 0.5)), D) / k - 1)
    assert e6 < e4 * t ** 2
