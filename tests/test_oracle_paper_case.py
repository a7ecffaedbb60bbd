"""The paper's own section 3.2 case: its printed parameters are the fixture
tests/golden/paper_section_3_2.txt; the oracle's halo fill on exactly that case is pinned to Eq. 8 and to
the paper's "zero disturbance = no-slip wall" statement, and the inflow (compressible Blasius, Eq. 7) to
the textbook recovery-factor estimate of the adiabatic wall temperature.  CPU only."""
import os

import numpy as np
import pytest

from paper_2406_19494_b200 import cases

NH = 3
HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_section_3_2.txt")) as f:
        for ln in f:
            ln = ln.split("#")[0].strip()
            if ln:
                k, v = (t.strip() for t in ln.split("="))
                try:
                    out[k] = float(v)
                except ValueError:
                    out[k] = v
    return out


@pytest.fixture(scope="module")
def paper_case():
    return cases.paper_boundary_layer()


def test_case_is_built_from_the_papers_numbers(paper_case):
    g, c = golden(), paper_case
    assert c.n[:2] == (int(g["nx"]), int(g["ny"])) and c.gamma == g["gamma"] and c.Pr == g["prandtl"]
    assert c.xf[0] == g["x_lo"] and c.xf[-1] == pytest.approx(g["x_hi"], abs=1e-14)
    assert c.yf[0] == g["y_lo"] and c.yf[-1] == pytest.approx(g["y_hi"], abs=1e-14)
    assert np.allclose(np.diff(c.xf), (g["x_hi"] - g["x_lo"]) / g["nx"], rtol=1e-12)        # uniform in x
    dy = np.diff(c.yf)
    assert np.all(np.diff(dy) > 0) and dy[0] < 0.05 * dy[-1]                                  # stretched towards the wall
    assert c.bc[2].type == cases.BC_WALL_ADIABATIC and g["south"] == "adiabatic_noslip"
    assert c.bc[1].type == cases.BC_ZEROGRAD and c.bc[3].type == cases.BC_ZEROGRAD
    assert c.bc[0].type == cases.BC_DIRICHLET
    d = c.bc[2].dist
    assert d["A"] == g["A"] and d["kappa"] == g["kappa"]
    # free stream: rho_e = u_e = T_e = 1, Mach number and unit Reynolds number as printed
    assert 1.0 / np.sqrt(c.gamma * c.R_gas * 1.0) == pytest.approx(g["mach"], rel=1e-14)
    assert 1.0 / c.mu["mu_ref"] == pytest.approx(g["re_unit"], rel=1e-14)


def test_similarity_inflow_adiabatic_wall_temperature(paper_case):
    g, c = golden(), paper_case
    # adiabatic wall: T_w/T_e = 1 + r (gamma-1)/2 M^2 with recovery factor r ~ sqrt(Pr) for a laminar layer
    est = 1.0 + np.sqrt(g["prandtl"]) * 0.5 * (g["gamma"] - 1.0) * g["mach"] ** 2
    assert c.notes["Tw_over_Te"] == pytest.approx(est, rel=0.01)
    assert np.max(np.abs(c.notes["blasius_resid"])) < 1e-10
    # incompressible Blasius has C f''(0) = 0.4696; compressibility (C < 1 near the hot wall) lowers it a little
    assert 0.40 < c.notes["s0"] < 0.4696
    # inflow table: rho T = 1 (p = p_e), u in [0, 1], monotone, free stream reached inside the domain
    rho, u = c.bc[0].dirichlet[0, 0], c.bc[0].dirichlet[1, 0]
    assert np.all(np.diff(u) >= -1e-15) and u[0] < 0.05 and u[-1] == pytest.approx(1.0, abs=1e-9)
    assert 1.0 / rho[0] == pytest.approx(c.notes["Tw_over_Te"], rel=0.02)
    # boundary-layer edge (u = 0.99) at the inlet: delta ~ 5-7 sqrt(2 mu_e x / (rho_e u_e)) << domain height 0.4
    yc = 0.5 * (c.yf[1:] + c.yf[:-1])
    d99 = yc[np.argmax(u >= 0.99)]
    assert 4.0 < d99 / np.sqrt(2.0 * c.mu["mu_ref"] * g["x_lo"]) < 9.0 and d99 < 0.25 * g["y_hi"]


def test_disturbance_wall_on_the_papers_grid_is_eq8(ora, paper_case):
    g, c = golden(), paper_case
    o = ora.Oracle(c)
    U = o.fill_halo(o.state())
    A, kappa = g["A"], g["kappa"]
    xc = 0.5 * (c.xf[1:] + c.xf[:-1])
    vw = A * np.sin(2.0 * np.pi * kappa * xc)                  # Eq. 8 with A, kappa of PAPER.md:118
    I = slice(NH, -NH)
    for m in range(1, 4):
        ghost, mirror = U[:, I, NH - m, I], U[:, I, NH + m - 1, I]
        vg, vr = ghost[2] / ghost[0], mirror[2] / mirror[0]
        assert np.allclose(0.5 * (vg + vr), vw[None, :], rtol=0, atol=1e-16)
        for q in (1, 3):                                       # no slip: tangential wall velocity 0
            assert np.allclose(0.5 * (ghost[q] / ghost[0] + mirror[q] / mirror[0]), 0.0, atol=1e-16)
        # adiabatic: ghost temperature = mirror temperature, pressure even
        pg = (c.gamma - 1) * (ghost[4] - 0.5 * (ghost[1] ** 2 + ghost[2] ** 2 + ghost[3] ** 2) / ghost[0])
        pr = (c.gamma - 1) * (mirror[4] - 0.5 * (mirror[1] ** 2 + mirror[2] ** 2 + mirror[3] ** 2) / mirror[0])
        assert np.allclose(pg, pr, rtol=1e-13) and np.allclose(pg / ghost[0], pr / mirror[0], rtol=1e-13)
    # what the printed numbers imply: kappa (x_hi - x_lo) = 5 full periods over the wall, 60 cells each, so the
    # wall velocity sums to zero, changes sign 9 times inside, and peaks at A cos(pi/60) (cell centres straddle the crest)
    assert kappa * (g["x_hi"] - g["x_lo"]) == pytest.approx(5.0)
    assert abs(vw.sum()) < 1e-14 * len(xc)
    assert np.count_nonzero(np.diff(np.sign(vw)) != 0) == 9
    assert np.max(np.abs(vw)) == pytest.approx(A * np.cos(np.pi / 60.0), rel=1e-12)


def test_zero_disturbance_is_the_no_slip_wall_on_the_papers_case(ora):
    # "First we set the wall disturbance velocity to zero, which makes the boundary condition exactly
    # the same with a no-slip wall."
    a = cases.paper_boundary_layer(nx=60, ny=40, A=0.0)
    b = cases.paper_boundary_layer(nx=60, ny=40, disturbance=False)
    oa, ob = ora.Oracle(a), ora.Oracle(b)
    Ua, Ub = oa.fill_halo(oa.state()), ob.fill_halo(ob.state())
    assert Ua.tobytes() == Ub.tobytes()
    for _ in range(3):
        oa.rk3_step(Ua, 2e-6); ob.rk3_step(Ub, 2e-6)
    assert Ua.tobytes() == Ub.tobytes()


def test_disturbance_drives_a_wall_normal_flow(ora):
    # A > 0 blows and sucks through the wall: after a few steps the wall-adjacent v has the sign pattern of Eq. 8
    c = cases.paper_boundary_layer(nx=120, ny=60, nz=4)
    o = ora.Oracle(c)
    U = o.state()
    for _ in range(20):
        st, dt = o.cfl_dt(U, c.cfl)
        assert st == 0
        o.rk3_step(U, dt)
    xc = 0.5 * (c.xf[1:] + c.xf[:-1])
    v1 = (U[2] / U[0])[NH, NH, NH:-NH]                         # first cell above the wall
    vw = 0.01 * np.sin(2 * np.pi * 10 * xc)
    strong = np.abs(vw) > 0.005
    assert np.all(np.sign(v1[strong]) == np.sign(vw[strong]))
    assert np.isfinite(U[:, NH:-NH, NH:-NH, NH:-NH]).all() and U[0, NH:-NH, NH:-NH, NH:-NH].min() > 0
