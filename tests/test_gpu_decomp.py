"""GPU tests of the block decomposition (include/jf.h "Block
decomposition"): all blocks on ONE device, i.e. the ranks emulated as one launch sequence over all ranks'
data.  Expected values come from the ORACLE on the undivided case (halo fill cell by cell, RK3 steps at
1e-10), and the decomposed run must also reproduce the undivided GPU run cell for cell."""
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


def wall_case(n=(24, 12, 8)):
    bc = cases.periodic_bc()
    bc[0] = cases.FaceBC(cases.BC_ZEROGRAD)
    bc[1] = cases.FaceBC(cases.BC_ZEROGRAD)
    bc[2] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.1, dist={"A": 0.05, "kappa": 2.0, "t1_lo": 0.2, "t1_hi": 0.8})
    bc[3] = cases.FaceBC(cases.BC_WALL_ADIABATIC, u_wall=(0.2, 0.0, -0.1))
    c = cases.random_admissible(n=n, seed=21, bc=bc, viscous=True, stretched=True)
    c.body_accel = (0.3, -0.2, 0.1)
    return c


def channel_sixth():
    c = cases.channel(48, 32, 32, n_steps=3)
    c.visc_order = 6                                          # the sixth-order dissipative flux reads cells -3..2 about a
    return c                                                  # face: the same three exchanged layers suffice


CASES = {
    "periodic": (lambda: cases.random_admissible(n=(24, 16, 12), seed=7, stretched=True), (2, 2, 2)),
    "periodic3x": (lambda: cases.random_admissible(n=(27, 9, 8), seed=8, stretched=True), (3, 1, 2)),
    "walls": (wall_case, (3, 2, 2)),
    "channel": (lambda: cases.channel(48, 32, 32, n_steps=3), (2, 2, 1)),
    "plate": (lambda: cases.flat_plate(256, 32, 8, n_steps=3), (4, 1, 1)),
    "channel_order6": (channel_sixth, (2, 2, 2)),
}


def global_index(case, a, lo, P):
    """Global padded indices of a block's padded cells along axis a (periodic axes wrap into the interior)."""
    g = lo + np.arange(P)
    if case.bc[2 * a].type == cases.BC_PERIODIC:
        N = case.n[a]
        g = (g - NH) % N + NH
    return g


@pytest.mark.parametrize("name", list(CASES))
@pytest.mark.parametrize("transport", ["pull", "pack"])
def test_halo_fill_of_every_block_cell_against_the_oracle(jf, ora, name, transport):
    from paper_2406_19494_b200 import decomp
    make, blocks = CASES[name]
    c = make()
    o = ora.Oracle(c, "f64")
    Ug = o.fill_halo(o.state())                             # undivided, halo-filled, by the oracle
    mb = decomp.MultiBlock(c, blocks, "f64", transport=transport)
    mb.jf_fill_halo()
    scale = np.max(np.abs(Ug))
    for part, U in zip(mb.parts, mb.U):
        U = U.cpu().numpy()
        n = part.case.n
        ix = [global_index(c, a, part.lo[a], n[a] + 2 * NH) for a in range(3)]
        exp = Ug[:, ix[2]][:, :, ix[1]][:, :, :, ix[0]]
        # every padded cell of the block: interior, physical halos, exchanged halos, edges and corners
        assert np.max(np.abs(U - exp)) <= 1e-13 * scale, (name, part.coords)


@pytest.mark.parametrize("name", list(CASES))
def test_decomposed_steps_equal_the_undivided_run(jf, ora, name):
    from paper_2406_19494_b200 import decomp
    make, blocks = CASES[name]
    c = make()
    n_steps = 3
    s = jf.Solver(c, "f64")
    U = s.state()
    mb = decomp.MultiBlock(c, blocks, "f64")
    o = ora.Oracle(c, "f64")
    Uo = o.state()
    for _ in range(n_steps):
        if c.dt is not None:
            dt = dto = c.dt
        else:
            st, dt = s.jf_cfl_dt(U, c.cfl)
            st2, dtm = mb.jf_cfl_dt(c.cfl)
            st3, dto = o.cfl_dt(Uo, c.cfl)
            assert st == 0 and st2 == 0 and dtm == dt        # min over blocks == the undivided reduction, exactly
            assert abs(dt - dto) <= 1e-12 * dto
        s.jf_rk3_step(U, dt)
        mb.jf_rk3_step(dt)
        o.rk3_step(Uo, dto)
    mono = U.cpu().numpy()[INT]
    dec = mb.gather()[INT]
    ref = np.asarray(Uo)[INT]
    bitwise = np.array_equal(mono, dec)
    diff = [float(np.max(np.abs(dec[q] - mono[q])) / max(np.max(np.abs(mono[q])), 1e-300)) for q in range(5)]
    print(name, blocks, "decomposed vs undivided GPU run: bitwise", bitwise, diff)
    assert max(diff) <= 1e-13
    mom = 1e-3 * np.max(np.sqrt(ref[1] ** 2 + ref[2] ** 2 + ref[3] ** 2))
    floor = [0.0, mom, mom, mom, 0.0]
    err = [float(np.max(np.abs(dec[q] - ref[q])) / max(np.max(np.abs(ref[q])), floor[q])) for q in range(5)]
    assert max(err) <= 1e-10, err


def test_tangent_solver_decomposes_too(jf):
    from paper_2406_19494_b200 import decomp
    c = wall_case()
    s = jf.Solver(c, "f64t")
    s.jf_set_tangent_seed(1.0, 0.5)
    U = s.state()
    mb = decomp.MultiBlock(c, (2, 2, 1), "f64t")
    for sb in mb.solvers:
        sb.jf_set_tangent_seed(1.0, 0.5)
    for _ in range(2):
        s.jf_rk3_step(U, 1e-3)
        mb.jf_rk3_step(1e-3)
    mono, dec = U.cpu().numpy()[INT], mb.gather()[INT]
    assert np.max(np.abs(mono[..., 1])) > 0
    assert np.max(np.abs(dec - mono)) <= 1e-13 * np.max(np.abs(mono))
