"""Pins for the oracle's halo fill (O3, Eq. 8) and dissipative flux (O6,
Eq. 4-5): definitions, the paper's A = 0 statement, closed forms.  CPU only."""
import numpy as np
import pytest

from paper_2406_19494_b200 import cases

NH = 3
INT = (slice(None), slice(NH, -NH), slice(NH, -NH), slice(NH, -NH))
G = 1.4


def prim_of(U, R_gas=1.0):
    rho = U[0]
    with np.errstate(all="ignore"):
        u, v, w = U[1] / rho, U[2] / rho, U[3] / rho
        p = (G - 1) * (U[4] - 0.5 * rho * (u * u + v * v + w * w))
        T = p / (rho * R_gas)
    return rho, u, v, w, p, T


def wall_case(bc_lo, bc_hi, axis=1, seed=2, n=(12, 10, 8)):
    bc = cases.periodic_bc()
    bc[2 * axis], bc[2 * axis + 1] = bc_lo, bc_hi
    return cases.random_admissible(n=n, seed=seed, bc=bc, stretched=True)


# ------------------------------------------------------------------ periodic / zero-gradient
def test_periodic_halo_all_cells_incl_corners(ora):
    c = cases.random_admissible(n=(12, 10, 8), seed=1)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    nx, ny, nz = c.n
    ii = (np.arange(-NH, nx + NH) % nx) + NH
    jj = (np.arange(-NH, ny + NH) % ny) + NH
    kk = (np.arange(-NH, nz + NH) % nz) + NH
    expect = c.U0[:, kk][:, :, jj][:, :, :, ii]
    assert np.array_equal(U, expect)
    assert np.array_equal(o.fill_halo(U.copy()), U)           # fill o fill = fill


def test_zero_gradient_copies_first_interior(ora):
    c = wall_case(cases.FaceBC(cases.BC_ZEROGRAD), cases.FaceBC(cases.BC_ZEROGRAD), axis=0)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    for m in range(1, 4):
        assert np.array_equal(U[:, NH:-NH, NH:-NH, NH - m], U[:, NH:-NH, NH:-NH, NH])
        assert np.array_equal(U[:, NH:-NH, NH:-NH, -NH - 1 + m], U[:, NH:-NH, NH:-NH, -NH - 1])
    # the y pass (periodic) then runs over all padded i: an (x,y) edge cell is the x-ghost of the
    # periodic image
    assert np.array_equal(U[:, NH, NH - 1, NH - 2], U[:, NH, -NH - 1, NH])


def test_dirichlet_sets_prescribed_primitives(ora):
    n = (12, 10, 8)
    rng = np.random.default_rng(3)
    tab = np.empty((5, n[2], n[1]))
    tab[0] = rng.uniform(0.5, 2, tab[0].shape)
    tab[1:4] = rng.uniform(-1, 1, tab[1:4].shape)
    tab[4] = rng.uniform(0.5, 2, tab[0].shape)
    c = wall_case(cases.FaceBC(cases.BC_DIRICHLET, dirichlet=tab), cases.FaceBC(cases.BC_ZEROGRAD), axis=0)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    for m in range(1, 4):
        rho, u, v, w, p, _ = prim_of(U[:, NH:-NH, NH:-NH, NH - m])
        for q, f in enumerate((rho, u, v, w, p)):
            assert np.allclose(f, tab[q], rtol=1e-14)


# ------------------------------------------------------------------ walls
@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("thermal", ["isothermal", "adiabatic"])
def test_wall_mirror_relations(ora, axis, thermal):
    Tw, uw = 1.2, (0.11, -0.07, 0.05)
    t = cases.BC_WALL_ISOTHERMAL if thermal == "isothermal" else cases.BC_WALL_ADIABATIC
    c = wall_case(cases.FaceBC(t, T_wall=Tw, u_wall=uw), cases.FaceBC(t, T_wall=Tw), axis=axis)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    ax = 3 - axis                                              # numpy axis of the array
    N = c.n[axis]
    inner = [slice(None), slice(NH, -NH), slice(NH, -NH), slice(NH, -NH)]
    for side, wall_vel in ((0, uw), (1, (0, 0, 0))):
        for m in range(1, 4):
            g = NH - m if side == 0 else NH + N - 1 + m
            r = NH + m - 1 if side == 0 else NH + N - m
            sg, sr = list(inner), list(inner)
            sg[ax], sr[ax] = g, r
            rg, ug, vg, wg, pg, Tg = prim_of(U[tuple(sg)])
            rr, ur, vr, wr, pr, Tr = prim_of(U[tuple(sr)])
            for a, b, wv in ((ug, ur, wall_vel[0]), (vg, vr, wall_vel[1]), (wg, wr, wall_vel[2])):
                assert np.allclose(0.5 * (a + b), wv, rtol=0, atol=1e-14)
            assert np.allclose(pg, pr, rtol=1e-14)
            if thermal == "isothermal":
                assert np.allclose(0.5 * (Tg + Tr), Tw, rtol=1e-14)
            else:
                assert np.allclose(Tg, Tr, rtol=1e-14)
            assert np.all(rg > 0)


def test_isothermal_wall_temperature_floor(ora):
    # interior so hot that 2 T_w - T_r < 0.05 T_w: ghost temperature is floored at 0.05 T_w
    Tw = 0.1
    c = wall_case(cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=Tw),
                  cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=Tw))
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    _, _, _, _, _, Tg = prim_of(U[:, NH:-NH, NH - 1, NH:-NH])
    assert np.allclose(Tg, 0.05 * Tw, rtol=1e-13)


# ------------------------------------------------------------------ the paper's disturbance wall
def test_disturbance_wall_A0_is_bit_identical_to_plain_wall(ora):
    # zero disturbance velocity "makes the boundary condition exactly the same with
    # a no-slip wall"
    for thermal in (cases.BC_WALL_ISOTHERMAL, cases.BC_WALL_ADIABATIC):
        plain = wall_case(cases.FaceBC(thermal, T_wall=1.1), cases.FaceBC(cases.BC_ZEROGRAD))
        dist = wall_case(cases.FaceBC(thermal, T_wall=1.1,
                                      dist={"A": 0.0, "kappa": 10.0, "t1_lo": 0.2, "t1_hi": 0.7}),
                         cases.FaceBC(cases.BC_ZEROGRAD))
        oa, ob = ora.Oracle(plain), ora.Oracle(dist)
        Ua, Ub = oa.fill_halo(oa.state()), ob.fill_halo(ob.state())
        assert Ua.tobytes() == Ub.tobytes()
        assert oa.rhs(Ua).tobytes() == ob.rhs(Ub).tobytes()


def test_disturbance_wall_velocity_is_eq8(ora):
    A, kappa, lo, hi = 0.01, 10.0, 0.25, 0.75
    c = wall_case(cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.0,
                               dist={"A": A, "kappa": kappa, "t1_lo": lo, "t1_hi": hi}),
                  cases.FaceBC(cases.BC_ZEROGRAD), n=(40, 10, 8))
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    _, xc = o.metrics(0)                                       # padded x centres (incl. halo columns)
    inside = (xc >= lo) & (xc <= hi)
    assert 10 < inside.sum() < 30
    for m in range(1, 4):
        _, ug, vg, wg, _, _ = prim_of(U[:, NH:-NH, NH - m, :])
        _, ur, vr, wr, _, _ = prim_of(U[:, NH:-NH, NH + m - 1, :])
        vw = np.where(inside, A * np.sin(2 * np.pi * kappa * xc), 0.0)   # Eq. 8
        assert np.allclose(0.5 * (vg + vr), vw[None, :], rtol=0, atol=1e-15)
        assert np.allclose(0.5 * (ug + ur), 0.0, atol=1e-15) and np.allclose(0.5 * (wg + wr), 0.0, atol=1e-15)


def test_config3_disturbance_segment_is_one_full_period():
    c = cases.flat_plate(512, 8, 8)                            # x-grid of BASELINE.json configs[3]
    xc = 0.5 * (c.xf[1:] + c.xf[:-1])
    d = c.bc[2].dist
    inside = np.nonzero((xc >= d["t1_lo"]) & (xc <= d["t1_hi"]))[0]
    assert inside[0] == 128 and inside[-1] == 383              # cells 128..383
    vw = d["A"] * np.sin(2 * np.pi * d["kappa"] * xc[inside])
    assert abs(vw.sum()) <= 1e-12 * d["A"] * len(inside)
    assert d["A"] == pytest.approx(0.01 * c.notes["u_inf"]) and d["A"] == pytest.approx(17.84, rel=1e-3)
    # segment ends are zeros of the sine: A sin(2 pi kappa x) = 0 at x = 0.05 and 0.15
    assert abs(np.sin(2 * np.pi * d["kappa"] * 0.05)) < 1e-12 and abs(np.sin(2 * np.pi * d["kappa"] * 0.15)) < 1e-12


# ------------------------------------------------------------------ dissipative flux, closed forms
def analytic_case(n, fields, mu, h=(0.11, 0.13, 0.17), Rg=1.0, Pr=0.72):
    """Whole padded array (halos analytic) from callables u,v,w,T(x,y,z); rho = 1."""
    fs = [cases.uniform_faces(0.0, m * hh, m) for m, hh in zip(n, h)]
    cs = [(np.arange(-NH, m + NH) + 0.5) * hh for m, hh in zip(n, h)]
    Z, Y, X = np.meshgrid(cs[2], cs[1], cs[0], indexing="ij")
    u, v, w, T = (f(X, Y, Z) for f in fields)
    rho = np.ones_like(X)
    p = rho * Rg * T
    U = np.empty((5,) + X.shape)
    U[0], U[1], U[2], U[3] = rho, rho * u, rho * v, rho * w
    U[4] = p / (G - 1) + 0.5 * rho * (u * u + v * v + w * w)
    c = cases.Case(name="analytic", n=n, xf=fs[0], yf=fs[1], zf=fs[2], gamma=G, R_gas=Rg, Pr=Pr,
                   mu={"sutherland": 0, "mu_ref": mu, "T_ref": 1.0, "S": 0.0},
                   bc=cases.periodic_bc(), U0=U)
    return c, h


def test_viscous_flux_cubic_fields_analytic(ora):
    rng = np.random.default_rng(5)
    n, mu, Pr, Rg = (6, 6, 6), 0.37, 0.72, 1.0
    # random polynomials of total degree <= 3 in (x,y,z)
    expo = [(a, b, c) for a in range(4) for b in range(4) for c in range(4) if a + b + c <= 3]

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

    (u, du), (v, dv), (w, dw), (T, dT) = make(0.0), make(0.0), make(0.0), make(5.0)
    c, h = analytic_case(n, (u, v, w, T), mu, Rg=Rg, Pr=Pr)
    o = ora.Oracle(c)
    U = o.state()
    vel, dvel = (u, v, w), (du, dv, dw)
    lam = mu * G * Rg / (G - 1) / Pr
    for d in range(3):
        for (i, j, k) in [(-1, 0, 0), (2, 3, 1), (5, 5, 5), (0, 2, 4)]:
            idx = [i, j, k]
            if idx[d] == -1 or True:
                pos = [(idx[a] + 0.5) * h[a] for a in range(3)]
                pos[d] += 0.5 * h[d]
                if d != 0 and i == -1:
                    continue                                    # transverse index must be interior
                Fd = o.viscous_face(U, d, i, j, k)
                Gm = np.array([[dvel[a][b](*pos) for b in range(3)] for a in range(3)])
                div = np.trace(Gm)
                tau = mu * (Gm[:, d] + Gm[d, :])
                tau[d] -= mu * 2.0 / 3.0 * div                  # Eq. 5
                uf = np.array([vel[a](*pos) for a in range(3)])
                expect = np.array([0.0, *tau, uf.dot(tau) + lam * dT[d](*pos)])   # Eq. 4, q = -lam grad T
                assert np.max(np.abs(Fd - expect)) <= 1e-12 * max(1.0, np.max(np.abs(expect)))


def test_viscous_flux_rigid_motion_gives_zero_stress(ora):
    Om, U0 = np.array([0.3, -0.5, 0.7]), np.array([0.2, 0.1, -0.4])
    u = lambda X, Y, Z: U0[0] + Om[1] * Z - Om[2] * Y
    v = lambda X, Y, Z: U0[1] + Om[2] * X - Om[0] * Z
    w = lambda X, Y, Z: U0[2] + Om[0] * Y - Om[1] * X
    T = lambda X, Y, Z: 2.0 + 0 * X
    c, _ = analytic_case((6, 6, 6), (u, v, w, T), 0.5)
    o = ora.Oracle(c)
    for d in range(3):
        Fd = o.viscous_face(o.state(), d, 2, 3, 1)
        assert np.max(np.abs(Fd)) <= 1e-13


def test_viscous_rhs_shear_wave_modified_wavenumber(ora):
    ny, mu = 16, 0.05
    n = (4, ny, 4)
    h = 1.0 / ny
    k = 2 * np.pi
    u = lambda X, Y, Z: np.sin(k * Y)
    zero = lambda X, Y, Z: 0 * X
    T = lambda X, Y, Z: 1.0 + 0 * X
    c, _ = analytic_case(n, (u, zero, zero, T), mu, h=(h, h, h))
    o = ora.Oracle(c)
    U = o.state()
    R = o.rhs(U, parts=(0, 1, 0))
    th = k * h
    keff2 = (2 * np.sin(th / 2)) * ((54 * np.sin(th / 2) - 2 * np.sin(3 * th / 2)) / 24.0) / h ** 2
    yc = (np.arange(ny) + 0.5) * h
    expect = -mu * keff2 * np.sin(k * yc)
    assert np.max(np.abs(R[1][NH:-NH, NH:-NH, NH:-NH] - expect[None, :, None])) <= 1e-13 * mu * keff2
    assert np.max(np.abs(R[0][INT[1:]])) == 0.0                 # no mass flux in F^d (Eq. 4)


def test_viscous_dissipation_of_tgv(ora):
    c = cases.tgv(32)
    # rho == 1 variant: keep u, v, w of the TGV, uniform density and pressure
    s = (slice(NH, -NH),) * 3
    u, v, w = (c.U0[q][s] / c.U0[0][s] for q in (1, 2, 3))
    one = np.ones_like(u)
    c.U0 = cases.set_interior_from_prim(cases.empty_state(c.n), c.gamma, one, u, v, w, 71.0 * one)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    R = o.rhs(U, parts=(0, 1, 0))
    dV = (2 * np.pi / 32) ** 3
    work = np.sum(u * R[1][s] + v * R[2][s] + w * R[3][s]) * dV
    mu = c.mu["mu_ref"]
    assert work == pytest.approx(-mu * 0.75 * (2 * np.pi) ** 3, rel=2e-3)   # <|omega|^2> = 3/4


def test_derivative_on_stretched_axis_linear_field_exact(ora):
    # phi linear in x on any mesh: metric-ratio derivative is exact => tau_xy = mu * du/dy exactly
    bc = cases.periodic_bc()
    c = cases.random_admissible(n=(8, 12, 8), seed=1, stretched=True, bc=bc)
    o = ora.Oracle(c)
    _, yc = o.metrics(1)
    a = 0.9
    u = a * yc[None, :, None] * np.ones((c.n[2] + 6, 1, c.n[0] + 6))
    U = np.empty((5,) + u.shape)
    U[0], U[1], U[2], U[3] = 1.0, u, 0.0, 0.0
    U[4] = 1.0 / 0.4 + 0.5 * u * u
    c.mu = {"sutherland": 0, "mu_ref": 0.25, "T_ref": 1.0, "S": 0.0}
    o = ora.Oracle(c)
    for j in (-1, 0, 5, 11):
        Fd = o.viscous_face(np.ascontiguousarray(U), 1, 3, j, 4)
        assert Fd[1] == pytest.approx(0.25 * a, rel=1e-13)      # tau_yx = mu du/dy
        assert abs(Fd[2]) <= 1e-15 and abs(Fd[3]) <= 1e-15
