"""Long GPU runs that the oracle cannot afford, checked by properties that hold at any length (the parity tests stop at the
step counts BASELINE.json states): exact mass conservation between walls, and the footprint of the paper's Disturbance Wall
(Eq. 8) in the flow above it after a thousand steps."""
import math

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


def test_mass_is_conserved_between_the_walls_over_500_steps(jf):
    # Eq. 6 telescopes, so mass can only change through the non-periodic faces: here two ADIABATIC no-slip walls, whose ghost
    # state is the exact mirror image of the cell next to the wall (u_g = -u_r, p_g = p_r, T_g = T_r, hence rho_g = rho_r):
    # the HLLC mass flux of a mirror-symmetric pair of states is exactly zero (tests/test_oracle_schemes.py:
    # test_hllc_mirror_symmetry), and the dissipative flux carries no mass (Eq. 4).  So the total mass must stay constant to
    # round-off over any number of steps - on the GPU path, 500 CFL steps with the time step formed on the device.
    c = cases.channel(48, 32, 32, n_steps=500)
    for f in (2, 3):
        c.bc[f] = cases.FaceBC(cases.BC_WALL_ADIABATIC)
    s = jf.Solver(c, "f64")
    U = s.state()
    vol = (np.diff(c.zf)[:, None, None] * np.diff(c.yf)[None, :, None] * np.diff(c.xf)[None, None, :])
    m0 = math.fsum((c.U0[0][INT[1:]] * vol).ravel())
    s.jf_dev_time(set_t=0.0)
    for _ in range(500):
        s.jf_cfl_dt_dev(U, c.cfl)
        s.jf_rk3_step_dev(U)
    st, dt, t = s.jf_dev_time()
    assert st == jf.JF_OK and t > 0
    Uh = U.cpu().numpy()
    assert np.isfinite(Uh).all() and Uh[0][INT[1:]].min() > 0
    m1 = math.fsum((Uh[0][INT[1:]] * vol).ravel())
    assert not np.array_equal(Uh[0][INT[1:]], c.U0[0][INT[1:]])
    assert abs(m1 - m0) <= 1e-12 * m0, (m0, m1)


def test_disturbance_wall_prints_its_wavenumber_on_the_flow_after_1000_steps(jf):
    # the paper's own case: v_w = A sin(2 pi kappa x), A = 0.01, kappa = 10 on x in [1, 1.5]: five full
    # periods.  After 1000 CFL steps (the oracle's parity check covers 20) the wall-normal velocity in the first cell row must
    # carry exactly that harmonic (index 5 of the discrete Fourier transform along x dominates, with the phase of a sine), the
    # state must be finite with rho, p > 0, and the same run with A = 0 must stay free of it.
    def run(A):
        c = cases.paper_boundary_layer(n_steps=1000, A=A)
        s = jf.Solver(c, "f64")
        U = s.state()
        s.jf_dev_time(set_t=0.0)
        for _ in range(1000):
            s.jf_cfl_dt_dev(U, c.cfl)
            s.jf_rk3_step_dev(U)
        st, dt, t = s.jf_dev_time()
        assert st == jf.JF_OK
        Uh = U.cpu().numpy()
        assert np.isfinite(Uh).all() and Uh[0][INT[1:]].min() > 0
        v = (Uh[2] / Uh[0])[NH, NH, NH:-NH]                    # first cell row above the wall, first spanwise plane
        return c, v
    c, v = run(0.01)
    nx = c.n[0]
    spec = np.fft.rfft(v - v.mean())
    k = int(np.argmax(np.abs(spec[1:nx // 4]))) + 1
    assert k == 5, (k, np.abs(spec[:12]))
    xc = 0.5 * (c.xf[1:] + c.xf[:-1])
    ref = np.sin(2 * np.pi * 10.0 * xc)
    corr = float(np.dot(v - v.mean(), ref) / (np.linalg.norm(v - v.mean()) * np.linalg.norm(ref)))
    assert corr > 0.9, corr                                   # in phase with Eq. 8: blowing where sin > 0
    assert 0.3 * 0.01 < np.abs(v).max() < 3 * 0.01            # of the size of A in the first cell row
    _, v0 = run(0.0)
    assert np.abs(np.fft.rfft(v0 - v0.mean())[5]) < 1e-3 * np.abs(spec[5])


def test_taylor_green_kinetic_energy_decays_at_the_viscous_rate(jf):
    # low-Mach Taylor-Green vortex (configs[0] / [4] physics, M = 0.1, Re = 1600): while the flow is still laminar the kinetic
    # energy decays at dK/dt = -2 nu * enstrophy = -nu <|omega|^2> = -(3/4) nu = -4.6875e-4 (closed form of the initial field,
    # incompressible limit; SURVEY.md 8(c) lists it as an informational pin).  128^3, 200 steps of dt = 1e-3 on the GPU path.
    c = cases.tgv(128)
    s = jf.Solver(c, "f64")
    U = s.state()

    def K(V):
        W = V[:, NH:-NH, NH:-NH, NH:-NH]
        return float(((W[1] ** 2 + W[2] ** 2 + W[3] ** 2) / W[0]).mean() * 0.5)

    ks = [K(U)]
    for i in range(200):
        s.jf_rk3_step(U, c.dt)
        if (i + 1) % 20 == 0:
            ks.append(K(U))
    assert ks[0] == pytest.approx(0.125, rel=2e-3)            # <1/2 rho |u|^2> of the initial field, rho ~ 1
    slope = np.polyfit(np.arange(len(ks)) * 20 * c.dt, np.array(ks), 1)[0]
    assert slope == pytest.approx(-0.75 * c.mu["mu_ref"], rel=0.01), slope
