"""Pins of the oracle's sixth-order central dissipative flux (the paper's DNS used "6th-order central"
dissipative fluxes; SURVEY.md 8(f) rank 3 — the half of that row the mathematics fixes; TENO6-A's constants are
not in PAPER.md).  Same readings as the fourth-order path (O6): difference form, transverse derivatives = I^f of
D^c, metric-ratio derivatives with X_xi built by the same stencils; only the stencils change.  Stencil-level pins
(polynomial exactness to degree 6 / 5, modified wavenumbers): tests/test_oracle_schemes.py."""
import numpy as np
import pytest

from paper_2406_19494_b200 import cases
from tests.test_oracle_halo_viscous import analytic_case, G, NH, INT
from tests.test_oracle_solver import uniform_case, permute_case


def sixth(c):
    c.visc_order = 6
    return c


def test_viscous_flux_quintic_fields_analytic(ora):
    # u, v, w, T random polynomials of total degree <= 5, analytic halos: every stress / heat-flux component at a
    # face equals the analytic value at the face centre (D^f_6, I^f_6 of D^c_6 and I^f_6 are all exact there).
    # The fourth-order path is NOT exact on this field (checked: it must miss by > 1e-6).
    rng = np.random.default_rng(15)
    n, mu, Pr, Rg = (8, 8, 8), 0.37, 0.72, 1.0
    expo = [(a, b, c) for a in range(6) for b in range(6) for c in range(6) if a + b + c <= 5]

    def make(mean):
        co = rng.uniform(-1, 1, len(expo))
        f = lambda X, Y, Z, co=co: mean + sum(k * X ** a * Y ** b * Z ** c for k, (a, b, c) in zip(co, expo))
        grads = []
        for ax in range(3):
            def g(X, Y, Z, co=co, ax=ax):
                tot = 0.0
                for k, e in zip(co, expo):
                    if e[ax] == 0:
                        continue
                    ee = list(e)
                    ee[ax] -= 1
                    tot = tot + k * e[ax] * X ** ee[0] * Y ** ee[1] * Z ** ee[2]
                return tot
            grads.append(g)
        return f, grads

    (u, du), (v, dv), (w, dw), (T, dT) = make(0.0), make(0.0), make(0.0), make(9.0)
    c, h = analytic_case(n, (u, v, w, T), mu, Rg=Rg, Pr=Pr)
    o6, o4 = ora.Oracle(sixth(c)), None
    U = o6.state()
    vel, dvel = (u, v, w), (du, dv, dw)
    lam = mu * G * Rg / (G - 1) / Pr
    worst4 = 0.0
    c4, _ = analytic_case(n, (u, v, w, T), mu, Rg=Rg, Pr=Pr)
    o4 = ora.Oracle(c4)
    for d in range(3):
        for (i, j, k) in [(-1, 0, 0), (2, 3, 1), (7, 7, 7), (0, 2, 4)]:
            if d != 0 and i == -1:
                continue
            idx = [i, j, k]
            pos = [(idx[a] + 0.5) * h[a] for a in range(3)]
            pos[d] += 0.5 * h[d]
            Gm = np.array([[dvel[a][b](*pos) for b in range(3)] for a in range(3)])
            tau = mu * (Gm[:, d] + Gm[d, :])
            tau[d] -= mu * 2.0 / 3.0 * np.trace(Gm)
            uf = np.array([vel[a](*pos) for a in range(3)])
            expect = np.array([0.0, *tau, uf.dot(tau) + lam * dT[d](*pos)])
            sc = max(1.0, np.max(np.abs(expect)))
            assert np.max(np.abs(o6.viscous_face(U, d, i, j, k) - expect)) <= 2e-12 * sc
            worst4 = max(worst4, np.max(np.abs(o4.viscous_face(U, d, i, j, k) - expect)) / sc)
    assert worst4 > 1e-6


@pytest.mark.parametrize("kind", ["periodic", "walls"])
def test_rhs_equals_naive_path_sixth_order(ora, kind):
    # brute force: the per-cell path with the stencil weights written out as plain tables
    if kind == "periodic":
        c = cases.random_admissible(n=(8, 8, 8), seed=5, stretched=True)
    else:
        bc = cases.periodic_bc()
        bc[0] = cases.FaceBC(cases.BC_ZEROGRAD)
        bc[1] = cases.FaceBC(cases.BC_ZEROGRAD)
        bc[2] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.1, dist={"A": 0.05, "kappa": 2.0, "t1_lo": 0.2, "t1_hi": 0.8})
        bc[3] = cases.FaceBC(cases.BC_WALL_ADIABATIC)
        c = cases.random_admissible(n=(8, 8, 8), seed=6, bc=bc, stretched=True)
        c.mu = {"sutherland": 1, "mu_ref": 0.02, "T_ref": 1.0, "S": 0.4}
    c.body_accel = (0.1, -0.2, 0.05)
    o = ora.Oracle(sixth(c))
    U = o.fill_halo(o.state())
    R, Rn = o.rhs(U), o.rhs(U, naive=True)
    assert np.max(np.abs(R[INT] - Rn[INT])) <= 1e-12 * np.max(np.abs(R[INT]))
    c4 = cases.random_admissible(n=(8, 8, 8), seed=5, stretched=True)
    if kind == "periodic":                                   # and it is a different scheme from the fourth-order one
        o4 = ora.Oracle(c4)
        R4 = o4.rhs(o4.fill_halo(o4.state()))
        assert np.max(np.abs(R4[INT] - R[INT])) > 1e-6 * np.max(np.abs(R[INT]))


@pytest.mark.parametrize("stretched", [False, True])
def test_free_stream_preservation_bit_exact_sixth_order(ora, stretched):
    c = sixth(uniform_case((9, 8, 10), (0.7, -0.4, 0.25), stretched))
    o = ora.Oracle(c)
    R = o.rhs(o.fill_halo(o.state()))
    assert np.max(np.abs(R[INT])) == 0.0


def test_shear_wave_modified_wavenumber_sixth_order(ora):
    # viscous RHS of rho u for u = sin(k y): -mu k_eff^2 sin(k y_j), k_eff^2 = [2 sin(t/2)] [2 (2250 sin(t/2) - 125 sin(3t/2)
    # + 9 sin(5t/2))/1920] / D^2 (the flux-form second difference of D^f_6)
    ny, mu = 16, 0.05
    n = (4, ny, 4)
    h = 1.0 / ny
    k = 2 * np.pi
    u = lambda X, Y, Z: np.sin(k * Y)
    zero = lambda X, Y, Z: 0 * X
    T = lambda X, Y, Z: 1.0 + 0 * X
    c, _ = analytic_case(n, (u, zero, zero, T), mu, h=(h, h, h))
    o = ora.Oracle(sixth(c))
    R = o.rhs(o.state(), parts=(0, 1, 0))
    th = k * h
    keff2 = (2 * np.sin(th / 2)) * (2 * (2250 * np.sin(th / 2) - 125 * np.sin(1.5 * th) + 9 * np.sin(2.5 * th)) / 1920.0) / h ** 2
    yc = (np.arange(ny) + 0.5) * h
    expect = -mu * keff2 * np.sin(k * yc)
    assert np.max(np.abs(R[1][NH:-NH, NH:-NH, NH:-NH] - expect[None, :, None])) <= 1e-13 * mu * keff2
    # the face-derivative factor alone is sixth-order accurate (the outer flux difference of Eq. 6 acts on point values)
    assert abs(2 * (2250 * np.sin(th / 2) - 125 * np.sin(1.5 * th) + 9 * np.sin(2.5 * th)) / 1920.0 / th - 1) < th ** 6 / 100


def test_tgv_dissipation_sixth_order(ora):
    # sum u . R_visc[rho u] dV = -mu 3/4 (2 pi)^3 (<|omega|^2> = 3/4) within 0.2 % at 32^3, as for the fourth-order
    # path: the remaining error is the outer flux difference of Eq. 6 acting on point values (second order in D),
    # common to both orders; the two schemes differ from each other at the level of the fourth-order truncation.
    def work(order):
        c = cases.tgv(32)
        c.visc_order = order
        s = (slice(NH, -NH),) * 3
        u, v, w = (c.U0[q][s] / c.U0[0][s] for q in (1, 2, 3))
        one = np.ones_like(u)
        c.U0 = cases.set_interior_from_prim(cases.empty_state(c.n), c.gamma, one, u, v, w, 71.0 * one)
        o = ora.Oracle(c)
        R = o.rhs(o.fill_halo(o.state()), parts=(0, 1, 0))
        return np.sum(u * R[1][s] + v * R[2][s] + w * R[3][s]) * (2 * np.pi / 32) ** 3, c.mu["mu_ref"]
    w4, mu = work(4)
    w6, _ = work(6)
    exact = -mu * 0.75 * (2 * np.pi) ** 3
    assert w6 == pytest.approx(exact, rel=2e-3)
    assert 1e-8 < abs(w6 / w4 - 1) < 1e-4


def test_axis_permutation_covariance_sixth_order(ora):
    # different sizes per axis + stretched: catches swapped strides / metrics in the sixth-order path
    c = sixth(cases.random_admissible(n=(8, 10, 12), seed=4, stretched=True))
    o = ora.Oracle(c)
    R = o.rhs(o.fill_halo(o.state()))
    c2 = sixth(cases.random_admissible(n=(12, 8, 10), seed=4, stretched=True))
    c2.xf, c2.yf, c2.zf = c.zf, c.xf, c.yf
    c2.U0 = permute_case(c, c.U0)
    o2 = ora.Oracle(c2)
    R2 = o2.rhs(o2.fill_halo(o2.state()))
    assert np.max(np.abs(R2[INT] - permute_case(c, R)[INT])) <= 1e-13 * np.max(np.abs(R[INT]))


def test_linear_field_exact_on_stretched_axis_sixth_order(ora):
    c = cases.random_admissible(n=(8, 12, 8), seed=1, stretched=True)
    o = ora.Oracle(sixth(c))
    _, yc = o.metrics(1)
    a = 0.9
    u = a * yc[None, :, None] * np.ones((c.n[2] + 6, 1, c.n[0] + 6))
    U = np.empty((5,) + u.shape)
    U[0], U[1], U[2], U[3] = 1.0, u, 0.0, 0.0
    U[4] = 1.0 / 0.4 + 0.5 * u * u
    c.mu = {"sutherland": 0, "mu_ref": 0.25, "T_ref": 1.0, "S": 0.0}
    o = ora.Oracle(sixth(c))
    for j in (-1, 0, 5, 11):
        Fd = o.viscous_face(np.ascontiguousarray(U), 1, 3, j, 4)
        assert Fd[1] == pytest.approx(0.25 * a, rel=1e-13)
