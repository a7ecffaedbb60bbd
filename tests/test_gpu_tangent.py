"""GPU tests of the tangent solver (JF_F64_TANGENT): the directional derivative of
the hot path with respect to the Disturbance-Wall parameters (A, kappa) of Eq. 8, which the
paper introduces precisely so that they can be differentiated through the solver.

Pins, none of which uses the CUDA path to produce an expected value:
  * the halo seed against the closed form d/dA, d/dkappa of Eq. 8 applied to the oracle's own halo state;
  * the propagated tangent after several RK3 steps against CENTRAL FINITE DIFFERENCES OF THE ORACLE
    (two oracle runs at A +- h, resp. kappa +- h, same fixed dt);
  * the value part of a tangent run against the oracle like any fp64 run, and a zero seed keeps a zero tangent.
"""
import copy

import numpy as np
import pytest

from paper_2406_19494_b200 import cases

pytestmark = pytest.mark.gpu
NH = 3
INT = (slice(None), slice(NH, -NH), slice(NH, -NH), slice(NH, -NH))


@pytest.fixture(scope="module")
def jf():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2406_19494_b200 import binding
    binding.lib()
    return binding


def wall_case(n=(24, 12, 8), A=0.05, kappa=2.0):
    """Seeded random admissible state between a disturbance wall (y-, isothermal, segment 0.2..0.8 in x)
    and an adiabatic moving wall (y+); zero-gradient in x, periodic in z; viscous, stretched axes."""
    bc = cases.periodic_bc()
    bc[0] = cases.FaceBC(cases.BC_ZEROGRAD)
    bc[1] = cases.FaceBC(cases.BC_ZEROGRAD)
    bc[2] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.1, dist={"A": A, "kappa": kappa, "t1_lo": 0.2, "t1_hi": 0.8})
    bc[3] = cases.FaceBC(cases.BC_WALL_ADIABATIC, u_wall=(0.2, 0.0, -0.1))
    return cases.random_admissible(n=n, seed=21, bc=bc, viscous=True, stretched=True)


def with_params(c, A=None, kappa=None):
    c2 = copy.deepcopy(c)
    if A is not None:
        c2.bc[2].dist["A"] = A
    if kappa is not None:
        c2.bc[2].dist["kappa"] = kappa
    return c2


def oracle_run(ora, c, dt, n_steps):
    o = ora.Oracle(c, "f64")
    U = o.state()
    for _ in range(n_steps):
        o.rk3_step(U, dt)
    return np.array(U)


def test_zero_seed_keeps_zero_tangent_and_value_matches_oracle(jf, ora):
    c = wall_case()
    o = ora.Oracle(c, "f64")
    st, dt = o.cfl_dt(o.fill_halo(o.state()), 0.4)
    Uo = oracle_run(ora, c, dt, 5)
    s = jf.Solver(c, "f64t")
    U = s.state()
    for _ in range(5):
        s.jf_rk3_step(U, dt)
    U = U.cpu().numpy()
    assert np.all(U[..., 1] == 0.0)
    val = U[..., 0][INT]
    ref = Uo[INT]
    for q in range(5):
        assert np.max(np.abs(val[q] - ref[q])) <= 1e-10 * max(np.max(np.abs(ref[q])), 1e-3)


@pytest.mark.parametrize("which", ["A", "kappa"])
def test_halo_seed_is_the_derivative_of_eq8(jf, ora, which):
    c = wall_case()
    A, kappa = c.bc[2].dist["A"], c.bc[2].dist["kappa"]
    o = ora.Oracle(c, "f64")
    Uo = o.fill_halo(o.state())
    s = jf.Solver(c, "f64t")
    s.jf_set_tangent_seed(1.0 if which == "A" else 0.0, 1.0 if which == "kappa" else 0.0)
    U = s.jf_fill_halo(s.state()).cpu().numpy()
    assert np.max(np.abs(U[..., 0] - Uo)) <= 1e-13 * np.max(np.abs(Uo))
    xc = 0.5 * (c.xf[:-1] + c.xf[1:])
    inside = (xc >= 0.2) & (xc <= 0.8)
    dvw = np.sin(2 * np.pi * kappa * xc) if which == "A" else A * 2 * np.pi * xc * np.cos(2 * np.pi * kappa * xc)
    dvw = np.where(inside, dvw, 0.0)
    T = U[..., 1]
    for m in (1, 2, 3):                                    # ghost layers of the y- wall, interior i and k
        g = NH - m
        rho_g = Uo[0, NH:-NH, g, NH:-NH]
        v_g = Uo[2, NH:-NH, g, NH:-NH] / rho_g
        dv = 2.0 * dvw[None, :]                            # v_g = 2 v_w - v_r
        assert np.max(np.abs(T[2, NH:-NH, g, NH:-NH] - rho_g * dv)) <= 1e-13
        assert np.max(np.abs(T[4, NH:-NH, g, NH:-NH] - rho_g * v_g * dv)) <= 1e-13
        for q in (0, 1, 3):                                # rho_g, rho u, rho w of the ghost do not depend on v_w
            assert np.all(T[q, NH:-NH, g, NH:-NH] == 0.0)
    assert np.all(T[INT] == 0.0)                           # interior cells carry no tangent yet


@pytest.mark.parametrize("which", ["A", "kappa"])
def test_tangent_matches_central_finite_differences_of_the_oracle(jf, ora, which):
    c = wall_case()
    A, kappa = c.bc[2].dist["A"], c.bc[2].dist["kappa"]
    o = ora.Oracle(c, "f64")
    st, dt = o.cfl_dt(o.fill_halo(o.state()), 0.4)
    n_steps = 6
    h = 1e-5 * (A if which == "A" else kappa)
    if which == "A":
        Up, Um = oracle_run(ora, with_params(c, A=A + h), dt, n_steps), oracle_run(ora, with_params(c, A=A - h), dt, n_steps)
    else:
        Up = oracle_run(ora, with_params(c, kappa=kappa + h), dt, n_steps)
        Um = oracle_run(ora, with_params(c, kappa=kappa - h), dt, n_steps)
    fd = ((Up - Um) / (2 * h))[INT]
    s = jf.Solver(c, "f64t")
    s.jf_set_tangent_seed(1.0 if which == "A" else 0.0, 1.0 if which == "kappa" else 0.0)
    U = s.state()
    for _ in range(n_steps):
        s.jf_rk3_step(U, dt)
    tan = U.cpu().numpy()[..., 1][INT]
    scale = np.max(np.abs(fd))
    assert scale > 0
    err = [float(np.max(np.abs(tan[q] - fd[q])) / scale) for q in range(5)]
    print("tangent d/d" + which, "vs oracle central differences:", err, "scale", scale)
    # FD error: truncation O(h^2) + round-off eps |U| / h ~ 1e-16 / 1e-6: well below 1e-6 of the derivative scale
    assert max(err) <= 1e-6, err


def test_tangent_on_the_mach6_flat_plate_config(jf, ora):
    """Config 3's set-up (Mach-6 plate, disturbance segment x in [0.05, 0.15], kappa = 10 /m, A = 0.01 u_inf;
    PAPER.md:118) at 256 x 32 x 8 cells: dU/dA after 8 steps against central differences of the oracle."""
    c = cases.flat_plate(256, 32, 8, n_steps=8)
    d = c.bc[2].dist
    o = ora.Oracle(c, "f64")
    st, dt = o.cfl_dt(o.fill_halo(o.state()), 0.5)
    h = 1e-5 * d["A"]
    cp, cm = copy.deepcopy(c), copy.deepcopy(c)
    cp.bc[2].dist["A"] = d["A"] + h
    cm.bc[2].dist["A"] = d["A"] - h
    fd = ((oracle_run(ora, cp, dt, 8) - oracle_run(ora, cm, dt, 8)) / (2 * h))[INT]
    s = jf.Solver(c, "f64t")
    s.jf_set_tangent_seed(1.0, 0.0)
    U = s.state()
    for _ in range(8):
        s.jf_rk3_step(U, dt)
    tan = U.cpu().numpy()[..., 1][INT]
    assert np.max(np.abs(fd[1])) > 0
    err = [float(np.max(np.abs(tan[q] - fd[q])) / max(np.max(np.abs(fd[q])), 1e-300)) for q in (0, 1, 2, 4)]
    print("flat plate dU/dA vs oracle central differences (rho, rho u, rho v, E):", err)
    assert max(err) <= 1e-5, err
    # spanwise momentum: no sensitivity in a 2-D flow (only the ~1e-27 round-off seed of rho w itself)
    assert np.max(np.abs(tan[3])) <= 1e-15 * np.max(np.abs(fd[1]))


@pytest.mark.parametrize("which", ["A", "kappa"])
def test_tangent_on_the_papers_own_case(jf, ora, which):
    """The paper's section 3.2 case with its printed A = 0.01, kappa = 10 (tests/golden/paper_section_3_2.txt) on
    the first 150 x 60 cells of its grid: dU/dA and dU/dkappa after 10 steps against central differences of the
    oracle, and the derivative of a scalar objective (the wall-normal momentum in the first cell row: what an
    end-to-end optimisation of the disturbance, would descend on)."""
    c = cases.paper_boundary_layer(nx=150, ny=60, nz=4)
    d = c.bc[2].dist
    o = ora.Oracle(c, "f64")
    st, dt = o.cfl_dt(o.fill_halo(o.state()), 0.5)
    n_steps = 10
    key = "A" if which == "A" else "kappa"
    h = 1e-5 * d[key]
    cp, cm = copy.deepcopy(c), copy.deepcopy(c)
    cp.bc[2].dist[key] = d[key] + h
    cm.bc[2].dist[key] = d[key] - h
    Up, Um = oracle_run(ora, cp, dt, n_steps), oracle_run(ora, cm, dt, n_steps)
    fd = ((Up - Um) / (2 * h))[INT]
    s = jf.Solver(c, "f64t")
    s.jf_set_tangent_seed(1.0 if which == "A" else 0.0, 1.0 if which == "kappa" else 0.0)
    U = s.state()
    for _ in range(n_steps):
        s.jf_rk3_step(U, dt)
    tan = U.cpu().numpy()[..., 1][INT]
    err = [float(np.max(np.abs(tan[q] - fd[q])) / np.max(np.abs(fd[q]))) for q in (0, 1, 2, 4)]
    print("paper case dU/d" + which, "vs oracle central differences (rho, rho u, rho v, E):", err)
    assert max(err) <= 1e-5, err
    J = lambda V: float(np.sum(V[2][:, 0, :] ** 2))           # sum over the first cell row of (rho v)^2
    dJ_fd = (J(Up[INT]) - J(Um[INT])) / (2 * h)
    val = U.cpu().numpy()[..., 0][INT]
    dJ_tan = float(np.sum(2.0 * val[2][:, 0, :] * tan[2][:, 0, :]))
    assert dJ_fd != 0.0 and abs(dJ_tan - dJ_fd) <= 1e-6 * abs(dJ_fd), (dJ_tan, dJ_fd)


def test_seed_rejected_on_plain_solvers(jf):
    c = wall_case()
    s = jf.Solver(c, "f64")
    with pytest.raises(jf.JFError):
        s.jf_set_tangent_seed(1.0, 0.0)


def test_changing_the_seed_on_a_live_solver_takes_effect(jf):
    # the step is replayed from a CUDA graph whose halo kernels carry the face tables by value: a new seed must
    # invalidate the captured steps.  Linear in the seed: the tangent after steps with seed (2, 0) from a zero
    # tangent is twice the one with seed (1, 0), on the same solver and the same state array.
    import torch
    c = wall_case()
    s = jf.Solver(c, "f64t")
    U = s.state()
    U0 = U.clone()
    s.jf_set_tangent_seed(1.0, 0.0)
    for _ in range(2):
        s.jf_rk3_step(U, 1e-3)
    t1 = U[..., 1].clone()
    U.copy_(U0)
    s.jf_set_tangent_seed(2.0, 0.0)
    for _ in range(2):
        s.jf_rk3_step(U, 1e-3)
    torch.cuda.synchronize()
    t2 = U[..., 1]
    scale = float(t1.abs().max())
    assert scale > 0
    assert float((t2 - 2.0 * t1).abs().max()) <= 1e-12 * scale
