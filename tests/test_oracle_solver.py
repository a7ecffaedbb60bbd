"""Solver-level pins of the oracle: invariants of Eq. 6, exact solutions, closed forms, brute force
(SURVEY.md §8(c)).  CPU only; sized to run in well under a minute."""
import numpy as np
import pytest

from paper_2406_19494_b200 import cases
from tests import exact_riemann

NH = 3
INT = (slice(None), slice(NH, -NH), slice(NH, -NH), slice(NH, -NH))


def uniform_case(n, vel, stretched, viscous=True, rho=1.3, p=2.1):
    c = cases.random_admissible(n=n, seed=0, viscous=viscous, stretched=stretched)
    shp = (n[2], n[1], n[0])
    one = np.ones(shp)
    c.U0 = cases.set_interior_from_prim(cases.empty_state(n), c.gamma, rho * one, vel[0] * one,
                                        vel[1] * one, vel[2] * one, p * one)
    return c


# ------------------------------------------------------------------ free-stream preservation
@pytest.mark.parametrize("stretched", [False, True])
def test_free_stream_preservation_bit_exact(ora, stretched):
    c = uniform_case((9, 8, 10), (0.7, -0.4, 0.25), stretched)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    R = o.rhs(U)
    assert np.max(np.abs(R[INT])) == 0.0
    U1 = o.rk3_step(o.state(), 1e-2)
    assert np.array_equal(U1[INT], c.U0[INT])


# ------------------------------------------------------------------ conservation (telescoping Eq. 6)
@pytest.mark.parametrize("stretched", [False, True])
def test_conservation_periodic(ora, stretched):
    c = cases.random_admissible(n=(12, 10, 8), seed=11, stretched=stretched, amp=0.2)
    o = ora.Oracle(c)
    dlx, dly, dlz = (np.diff(f) for f in (c.xf, c.yf, c.zf))
    vol = dlz[:, None, None] * dly[None, :, None] * dlx[None, None, :]
    import math
    tot0 = [math.fsum((c.U0[q][INT[1:]] * vol).ravel()) for q in range(5)]
    U = o.state()
    for _ in range(5):
        o.rk3_step(U, 2e-3)
    assert not np.array_equal(U[INT], c.U0[INT])
    scale = math.fsum((np.abs(c.U0[4][INT[1:]]) * vol).ravel())
    for q in range(5):
        tot = math.fsum((U[q][INT[1:]] * vol).ravel())
        assert abs(tot - tot0[q]) <= 1e-13 * scale


# ------------------------------------------------------------------ brute force on 8^3
@pytest.mark.parametrize("kind", ["periodic", "walls"])
def test_rhs_equals_naive_path(ora, kind):
    if kind == "periodic":
        c = cases.random_admissible(n=(8, 8, 8), seed=5, stretched=True)
    else:
        bc = cases.periodic_bc()
        bc[0] = cases.FaceBC(cases.BC_ZEROGRAD)
        bc[1] = cases.FaceBC(cases.BC_ZEROGRAD)
        bc[2] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.1,
                             dist={"A": 0.05, "kappa": 2.0, "t1_lo": 0.2, "t1_hi": 0.8})
        bc[3] = cases.FaceBC(cases.BC_WALL_ADIABATIC)
        c = cases.random_admissible(n=(8, 9, 8), seed=6, stretched=True, bc=bc)
        c.body_accel = (0.3, -0.1, 0.2)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    R, Rn = o.rhs(U), o.rhs(U, naive=True)
    # fluxes are O(|F|/dx); the difference of two of them carries ~1e-16 |F|/dx of round-off
    scale = np.max(np.abs(R[INT]))
    assert scale > 1.0
    assert np.max(np.abs(R[INT] - Rn[INT])) <= 1e-13 * scale


# ------------------------------------------------------------------ axis-permutation covariance
def permute_case(c, U):
    """x->y->z->x relabelling: new field V(q', k', j', i') with (i',j',k') = (k,i,j)."""
    Up = np.transpose(U, (0, 2, 3, 1))             # new z = old y, new y = old x, new x = old z
    out = np.empty_like(Up)
    out[0], out[4] = Up[0], Up[4]
    out[1], out[2], out[3] = Up[3], Up[1], Up[2]   # new u = old w, new v = old u, new w = old v
    return np.ascontiguousarray(out)


def test_axis_permutation_covariance(ora):
    c = cases.smooth_periodic(n=(8, 8, 8), seed=3)
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    R = o.rhs(U)
    c2 = cases.smooth_periodic(n=(8, 8, 8), seed=3)
    c2.U0 = permute_case(c, c.U0)
    o2 = ora.Oracle(c2)
    U2 = o2.fill_halo(o2.state())
    R2 = o2.rhs(U2)
    assert np.array_equal(U2, permute_case(c, U))
    assert np.max(np.abs(R2[INT] - permute_case(c, R)[INT])) <= 1e-13 * np.max(np.abs(R[INT]))


def test_axis_permutation_covariance_anisotropic(ora):
    # different sizes per axis + stretched: catches swapped strides / metrics
    c = cases.random_admissible(n=(8, 10, 12), seed=4, stretched=True)
    o = ora.Oracle(c)
    R = o.rhs(o.fill_halo(o.state()))
    c2 = cases.random_admissible(n=(12, 8, 10), seed=4, stretched=True)
    c2.xf, c2.yf, c2.zf = c.zf, c.xf, c.yf
    c2.U0 = permute_case(c, c.U0)
    o2 = ora.Oracle(c2)
    R2 = o2.rhs(o2.fill_halo(o2.state()))
    assert np.max(np.abs(R2[INT] - permute_case(c, R)[INT])) <= 1e-13 * np.max(np.abs(R[INT]))


# ------------------------------------------------------------------ 5th-order convergence
def entropy_wave(N, axis):
    n = [4, 4, 4]
    n[axis] = N
    h = 1.0 / N
    fs = [cases.uniform_faces(0.0, m * h, m) for m in n]
    f = fs[axis]
    avg = 1.0 + 0.2 * (np.cos(2 * np.pi * f[:-1]) - np.cos(2 * np.pi * f[1:])) / (2 * np.pi * h)
    shape = [1, 1, 1]
    shape[2 - axis] = N
    rho = np.broadcast_to(avg.reshape(shape), (n[2], n[1], n[0])).copy()
    vel = [np.zeros_like(rho) for _ in range(3)]
    vel[axis] = np.ones_like(rho)
    U = cases.set_interior_from_prim(cases.empty_state(tuple(n)), 1.4, rho, *vel, np.ones_like(rho))
    return cases.Case(name="entropy", n=tuple(n), xf=fs[0], yf=fs[1], zf=fs[2], gamma=1.4, R_gas=1.0,
                      Pr=0.72, mu={"sutherland": 0, "mu_ref": 0.0, "T_ref": 1.0, "S": 0.0},
                      bc=cases.periodic_bc(), U0=U), avg


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_fifth_order_convergence_entropy_wave(ora, axis):
    errs = []
    for N in (16, 32, 64):
        c, avg = entropy_wave(N, axis)
        o = ora.Oracle(c)
        U = o.state()
        h = 1.0 / N
        T = 0.5
        nsteps = int(np.ceil(T / (0.4 * h ** (5.0 / 3.0))))
        for _ in range(nsteps):
            o.rk3_step(U, T / nsteps)
        f = c.xf if axis == 0 else (c.yf if axis == 1 else c.zf)
        exact = 1.0 + 0.2 * (np.cos(2 * np.pi * (f[:-1] - T)) - np.cos(2 * np.pi * (f[1:] - T))) / (2 * np.pi * h)
        idx = [NH, NH, NH]
        sl = [NH, NH, NH]
        sl[2 - axis] = slice(NH, -NH)
        line = U[0][tuple(sl)]
        errs.append(np.mean(np.abs(line - exact)))
        # velocity and pressure stay uniform (contact-type wave)
        assert np.max(np.abs(U[4][INT[1:]] - (1 / 0.4 + 0.5 * U[0][INT[1:]]))) < 1e-9
    orders = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert errs[1] == pytest.approx(1.39e-5, rel=0.15)      # indicative value, SURVEY §8(c)
    assert np.all(orders > 4.8), (errs, orders)


def test_rk3_is_third_order_in_time(ora):
    # fixed grid, vary dt: the difference to a fine-dt solution scales like dt^3
    c, _ = entropy_wave(32, 0)
    o = ora.Oracle(c)

    def run(nsteps, T=0.2):
        U = o.state()
        for _ in range(nsteps):
            o.rk3_step(U, T / nsteps)
        return U[0][INT[1:]]

    ref = run(256)
    e1, e2 = np.max(np.abs(run(8) - ref)), np.max(np.abs(run(16) - ref))
    assert 2.7 < np.log2(e1 / e2) < 3.3


def test_rk3_exact_for_body_force_quadratic(ora):
    # uniform periodic state + constant acceleration g: m(t) = m0 + rho g t,
    # E(t) = E0 + g m0 t + rho g^2 t^2/2 (a quadratic: any 3rd-order RK reproduces it exactly)
    c = uniform_case((6, 5, 4), (0.3, 0.0, 0.0), False, viscous=True)
    g, dt, rho = 0.7, 0.05, 1.3
    c.body_accel = (g, 0.0, 0.0)
    o = ora.Oracle(c)
    U = o.rk3_step(o.state(), dt)
    m0, E0 = c.U0[1][NH, NH, NH], c.U0[4][NH, NH, NH]
    assert np.allclose(U[1][INT[1:]], m0 + rho * g * dt, rtol=1e-15)
    assert np.allclose(U[4][INT[1:]], E0 + g * m0 * dt + rho * g * g * dt * dt / 2, rtol=1e-15)
    assert np.array_equal(U[0][INT[1:]], c.U0[0][INT[1:]])


# ------------------------------------------------------------------ Sod vs exact Riemann solution
def test_sod_against_exact_riemann(ora):
    c = cases.sod(256)
    U, dts = ora.run_case(c)
    assert sum(dts) == pytest.approx(0.2, abs=1e-14)
    assert 200 <= len(dts) <= 250                           # ~224 steps expected at CFL 0.5
    rho = U[0][INT[1:]]
    # exact cell averages by 8-point sub-sampling
    h = 1.0 / 256
    sub = (np.arange(8) + 0.5) / 8
    xs = (c.xf[:-1, None] + h * sub[None, :]).ravel()
    r_ex, _, _ = exact_riemann.sample((xs - 0.5) / 0.2, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    r_ex = r_ex.reshape(256, 8).mean(axis=1)
    p_s, u_s = exact_riemann.star_state(1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    assert p_s == pytest.approx(0.30313, abs=1e-5) and u_s == pytest.approx(0.92745, abs=1e-5)
    L1 = np.mean(np.abs(rho[0, 0, :] - r_ex))
    assert L1 <= 3e-3
    xc = 0.5 * (c.xf[1:] + c.xf[:-1])                       # centre-sampled exact solution:
    r_c, _, _ = exact_riemann.sample((xc - 0.5) / 0.2, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1)
    assert np.mean(np.abs(rho[0, 0, :] - r_c)) == pytest.approx(1.93e-3, rel=0.02)
    assert len(dts) == 224                                  # 224 steps at CFL 0.5
    assert np.all(U[2][INT[1:]] == 0.0) and np.all(U[3][INT[1:]] == 0.0)
    for q in (0, 1, 4):                                     # identical in all 16 (j,k) lines
        assert np.all(U[q][INT[1:]] == U[q][NH, NH, NH:-NH][None, None, :])
    assert rho.max() - 1.0 <= 1e-3 and rho.min() >= 0.125 - 1e-3


# ------------------------------------------------------------------ CFL closed form
def test_cfl_uniform_state_closed_form(ora):
    vel, rho, p = (0.7, -0.4, 0.25), 1.3, 2.1
    c = uniform_case((6, 5, 4), vel, False, viscous=False, rho=rho, p=p)
    o = ora.Oracle(c)
    st, dt = o.cfl_dt(o.state(), 0.5)
    cs = np.sqrt(1.4 * p / rho)
    d = [c.xf[1] - c.xf[0], c.yf[1] - c.yf[0], c.zf[1] - c.zf[0]]
    expect = 0.5 * min(d[a] / (abs(vel[a]) + cs) for a in range(3))
    assert st == 0 and dt == pytest.approx(expect, rel=1e-15)
    # viscous limits: dt = cfl * min(conv, 3/14 dmin^2 rho/mu, 1/10 dmin^2 rho Pr/mu)
    c2 = uniform_case((6, 5, 4), vel, False, viscous=True, rho=rho, p=p)
    c2.mu = {"sutherland": 0, "mu_ref": 0.5, "T_ref": 1.0, "S": 0.0}
    st, dt = ora.Oracle(c2).cfl_dt(c2.U0.copy(), 0.5)
    dmin = min(d)
    assert dt == pytest.approx(0.5 * min(expect / 0.5, 3 / 14 * dmin ** 2 * rho / 0.5,
                                         0.1 * dmin ** 2 * rho * 0.72 / 0.5), rel=1e-14)


def test_cfl_flags_inadmissible_state(ora):
    c = uniform_case((6, 5, 4), (0.1, 0, 0), False)
    o = ora.Oracle(c)
    U = o.state()
    U[0, NH + 1, NH + 2, NH + 3] = -1.0
    st, dt = o.cfl_dt(U, 0.5)
    assert st == 5 and np.isnan(dt)
    U = o.state()
    U[4, NH, NH, NH] = np.nan
    assert o.cfl_dt(U, 0.5)[0] == 5


@pytest.mark.parametrize("Pr,binding", [(0.72, "heat"), (3.0, "visc")])
def test_cfl_sutherland_two_temperature_field_closed_form(ora, Pr, binding):
    # O9 with Sutherland viscosity: a gas at rest, uniform density, cold everywhere except a few hot cells.
    # mu grows with T, so the hot cells set the diffusive limits: dt = cfl * 3/14 D^2 rho / mu(T_hot)
    # (Pr = 3: the viscous limit binds) or cfl * 1/10 D^2 rho Pr / mu(T_hot) (Pr = 0.72: the heat limit),
    # with T = p/(rho R), R != 1, and mu(T) typed here by hand from Sutherland's law.
    n, rho, R = (6, 5, 4), 1.3, 0.4
    T_cold, T_hot = 0.9, 2.7
    mu_ref, T_ref, S = 0.8, 1.1, 0.35
    c = uniform_case(n, (0.0, 0.0, 0.0), False, viscous=True, rho=rho, p=rho * R * T_cold)
    c.R_gas, c.Pr = R, Pr
    c.mu = {"sutherland": 1, "mu_ref": mu_ref, "T_ref": T_ref, "S": S}
    T = np.full((n[2], n[1], n[0]), T_cold)
    T[1, 2, 3] = T[2, 0, 5] = T_hot
    one = np.ones_like(T)
    c.U0 = cases.set_interior_from_prim(cases.empty_state(n), c.gamma, rho * one, 0 * one, 0 * one, 0 * one, rho * R * T)
    d = min(c.xf[1] - c.xf[0], c.yf[1] - c.yf[0], c.zf[1] - c.zf[0])
    mu_hot = mu_ref * (T_hot / T_ref) ** 1.5 * (T_ref + S) / (T_hot + S)
    mu_cold = mu_ref * (T_cold / T_ref) ** 1.5 * (T_ref + S) / (T_cold + S)
    assert mu_hot > 2 * mu_cold
    visc, heat = 3.0 / 14.0 * d * d * rho / mu_hot, 0.1 * d * d * rho * Pr / mu_hot
    conv = d / np.sqrt(c.gamma * R * T_hot)
    assert (heat < visc) == (binding == "heat") and min(visc, heat) < 0.5 * conv
    st, dt = ora.Oracle(c).cfl_dt(c.U0.copy(), 0.5)
    assert st == 0 and dt == pytest.approx(0.5 * min(visc, heat), rel=1e-14)
    # a constant-viscosity law on the same field gives the mu_ref limit instead
    c.mu = {"sutherland": 0, "mu_ref": mu_ref, "T_ref": T_ref, "S": S}
    st, dt0 = ora.Oracle(c).cfl_dt(c.U0.copy(), 0.5)
    assert dt0 == pytest.approx(0.5 * min(3.0 / 14.0 * d * d * rho / mu_ref, 0.1 * d * d * rho * Pr / mu_ref, conv), rel=1e-14)


# ------------------------------------------------------------------ the arbiter instantiation (x87 long double)
def test_arbiter_is_the_same_scheme_at_higher_precision(ora):
    # "f80" is the oracle's own text on a 64-bit mantissa.  It must (a) agree with the fp64 oracle to fp64
    # round-off on one RHS, (b) be far closer to the truth than fp64: the fp64 oracle with and without FMA
    # contraction are two roundings of the same scheme, so both sit at ~1e-16 of the arbiter while differing
    # from each other by the same amount, (c) keep the exact invariants: free stream -> R == 0 bit-exactly.
    c = cases.random_admissible(n=(10, 9, 8), seed=21, stretched=True)
    o64, o80, ofma = ora.Oracle(c, "f64"), ora.Oracle(c, "f80"), ora.Oracle(c, "f64", variant="fma")
    R64 = o64.rhs(o64.fill_halo(o64.state()))
    R80 = np.asarray(o80.rhs(o80.fill_halo(o80.state())), dtype=np.float64)
    Rf = ofma.rhs(ofma.fill_halo(ofma.state()))
    s = np.max(np.abs(R64[INT]))
    e64, ef, e2 = (np.max(np.abs(a[INT] - b[INT])) / s for a, b in ((R64, R80), (Rf, R80), (R64, Rf)))
    assert 0 < e64 < 1e-13 and 0 < ef < 1e-13
    assert e2 <= e64 + ef and e2 > 0.2 * max(e64, ef)       # the arbiter lies "between" the two roundings
    u = uniform_case((7, 6, 5), (0.7, -0.4, 0.25), True)
    o = ora.Oracle(u, "f80")
    assert np.max(np.abs(o.rhs(o.fill_halo(o.state()))[INT])) == 0.0
    # one quantity known in closed form to all digits: 1/3, 2/3 of the last RK3 stage are formed in long double
    # (a double-rounded 1/3 would leave an error of 1.85e-17 U): U' = 1/3 U + 2/3 (U + dt*0) must return U to 1 ulp80
    U1 = o.rk3_step(o.state(), 1e-2)
    U0 = np.asarray(u.U0, dtype=np.longdouble)
    assert np.max(np.abs(U1[INT] - U0[INT]) / np.abs(U0[INT]).max()) <= 2.0 ** -62
