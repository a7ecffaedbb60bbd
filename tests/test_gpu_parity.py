"""GPU parity tests: the CUDA path (through the C ABI of include/jf.h) against the CPU oracle on the
same seeded inputs.  Metric P: per conserved variable q,
over interior cells, err_q = max|q_gpu - q_ora| / max(max|q_ora|, s_q), s_rho = s_E = 0,
s_mom = 1e-3 max||rho u||_ora in fp64 and max||rho u||_ora in fp32 (a momentum component that is
identically ~0 carries absolute round-off eps32*|rho u|, which no fp32 code can push below 1e-4 of a
1e-3 floor); pass at 1e-10 (fp64) / 1e-4 (fp32, against the fp32 oracle).

Long CFL-driven runs amplify 1-ulp differences (FMA contraction, re-associated divisions) through the
WENO weights: on the Mach-6 plate the fp64 oracle is itself 1.1e-9 away (rho*v, 200 steps) from the
discrete scheme's exact result.  Where GPU-vs-oracle exceeds 1e-10 for that reason the ARBITER decides:
the oracle's own text instantiated on x87 long double (64-bit mantissa, rational constants formed in that
precision: `ora.run_case(..., "f80")`, fed the fp64 oracle's time steps) gives the discrete result ~2000
times more accurately than either side, and the test requires
    |GPU - arbiter| <= max(1e-10, 2 |oracle_fp64 - arbiter|)   per conserved variable
i.e. the GPU must be about as close to the truth as the fp64 oracle is: no free factor.  The 1e-10
bar against the fp64 oracle itself is kept wherever the arithmetic allows it (all other variables / configs)."""
import numpy as np
import pytest

from paper_2406_19494_b200 import cases

pytestmark = pytest.mark.gpu

NH = 3
INT = (slice(None), slice(NH, -NH), slice(NH, -NH), slice(NH, -NH))
TOL = {"f64": 1e-10, "f32": 1e-4}


@pytest.fixture(scope="module")
def jf():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2406_19494_b200 import binding
    binding.lib()
    return binding


def metric_P(Ug, Uo, dtype="f64"):
    Ug, Uo = np.asarray(Ug, dtype=np.float64)[INT], np.asarray(Uo, dtype=np.float64)[INT]
    mom = (1e-3 if dtype == "f64" else 1.0) * np.max(np.sqrt(Uo[1] ** 2 + Uo[2] ** 2 + Uo[3] ** 2))
    floor = [0.0, mom, mom, mom, 0.0]
    return np.array([np.max(np.abs(Ug[q] - Uo[q])) / max(np.max(np.abs(Uo[q])), floor[q]) for q in range(5)])


def metric_R(Rg, Ro):
    Rg, Ro = np.asarray(Rg, dtype=np.float64)[INT], np.asarray(Ro, dtype=np.float64)[INT]
    return np.array([np.max(np.abs(Rg[q] - Ro[q])) / max(np.max(np.abs(Ro[q])), 1e-3 * np.max(np.abs(Ro)))
                     for q in range(5)])


def all_bc_case(n=(12, 10, 8), seed=2, viscous=True, which=0):
    rng = np.random.default_rng(100 + which)
    bc = cases.periodic_bc()
    nx, ny, nz = n
    if which == 0:      # walls in y (isothermal + disturbance | adiabatic moving), zero-grad x, periodic z
        bc[0] = cases.FaceBC(cases.BC_ZEROGRAD)
        bc[1] = cases.FaceBC(cases.BC_ZEROGRAD)
        bc[2] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.1,
                             dist={"A": 0.05, "kappa": 2.0, "t1_lo": 0.2, "t1_hi": 0.8})
        bc[3] = cases.FaceBC(cases.BC_WALL_ADIABATIC, u_wall=(0.2, 0.0, -0.1))
    elif which == 1:    # Dirichlet x-, zero-grad x+, walls in z, periodic y
        tab = np.empty((5, nz, ny))
        tab[0] = rng.uniform(0.8, 1.2, (nz, ny)); tab[4] = rng.uniform(0.8, 1.2, (nz, ny))
        tab[1:4] = rng.uniform(-0.3, 0.3, (3, nz, ny))
        bc[0] = cases.FaceBC(cases.BC_DIRICHLET, dirichlet=tab)
        bc[1] = cases.FaceBC(cases.BC_ZEROGRAD)
        bc[4] = cases.FaceBC(cases.BC_WALL_ADIABATIC, dist={"A": 0.03, "kappa": 1.5, "t1_lo": 0.1, "t1_hi": 0.6})
        bc[5] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=0.9)
    elif which == 2:    # walls in x, Dirichlet on y and z faces (padded-index clamping)
        bc[0] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.05,
                             dist={"A": 0.02, "kappa": 3.0, "t1_lo": 0.0, "t1_hi": 0.5})
        bc[1] = cases.FaceBC(cases.BC_WALL_ADIABATIC)
        for f, shp in ((2, (nz, nx)), (3, (nz, nx)), (4, (ny, nx)), (5, (ny, nx))):
            tab = np.empty((5,) + shp)
            tab[0] = rng.uniform(0.8, 1.2, shp); tab[4] = rng.uniform(0.8, 1.2, shp)
            tab[1:4] = rng.uniform(-0.3, 0.3, (3,) + shp)
            bc[f] = cases.FaceBC(cases.BC_DIRICHLET, dirichlet=tab) if f != 3 else cases.FaceBC(cases.BC_ZEROGRAD)
    return cases.random_admissible(n=n, seed=seed, bc=bc, viscous=viscous, stretched=True)


# ------------------------------------------------------------------ boundary: halo fill cell by cell
@pytest.mark.parametrize("which", [-1, 0, 1, 2])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_halo_fill_every_cell(jf, ora, which, dtype):
    c = cases.random_admissible(n=(12, 10, 8), seed=1, stretched=True) if which < 0 else all_bc_case(which=which)
    o = ora.Oracle(c, dtype)
    Uo = o.fill_halo(o.state())
    s = jf.Solver(c, dtype)
    Ug = s.jf_fill_halo(s.state()).cpu().numpy()
    assert np.array_equal(Ug[INT], Uo[INT])
    tol = 1e-13 if dtype == "f64" else 1e-5
    scale = np.max(np.abs(Uo), axis=(1, 2, 3), keepdims=True)
    assert np.max(np.abs(Ug - Uo) / scale) <= tol
    if which < 0:
        assert np.array_equal(Ug, Uo)                         # pure copies are bit-exact


@pytest.mark.parametrize("which", [-1, 0, 1, 2, 3])
@pytest.mark.parametrize("dtype", ["f64", "f32", "f64t"])
def test_fused_halo_launch_equals_the_three_axis_passes_bitwise(jf, which, dtype):
    # jf_fill_halo is ONE launch that composes the x -> y -> z passes per ghost cell (reading O3);
    # jf_fill_halo_axis runs them one by one: same bits in every padded cell, NaN-poisoned halos on entry
    if which == 3:
        c = cases.flat_plate(nx=64, ny=24, nz=8)
    else:
        c = cases.random_admissible(n=(12, 10, 8), seed=1, stretched=True) if which < 0 else all_bc_case(which=which, n=(37, 21, 13))
    import torch
    s = jf.Solver(c, dtype)
    if dtype == "f64t":
        s.jf_set_tangent_seed(0.7, -0.3)
        rng = np.random.default_rng(5)
        U0 = s.state(dU0=rng.uniform(-0.1, 0.1, np.asarray(c.U0).shape))
    else:
        U0 = s.state()
    poison = torch.full_like(U0, float("nan"))
    poison[INT] = U0[INT]
    Ua, Ub = poison.clone(), poison.clone()
    s.jf_fill_halo(Ua)
    for axis in range(3):
        s.jf_fill_halo_axis(Ub.data_ptr(), axis)
    torch.cuda.synchronize()
    a, b = Ua.cpu().numpy(), Ub.cpu().numpy()
    assert np.isfinite(a).all() and np.isfinite(b).all()
    assert a.tobytes() == b.tobytes()


def test_disturbance_A0_is_plain_wall_on_gpu(jf):
    # PAPER.md:104
    bc = cases.periodic_bc()
    bc[2] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.1)
    bc[3] = cases.FaceBC(cases.BC_ZEROGRAD)
    a = cases.random_admissible(n=(12, 10, 8), seed=2, bc=list(bc), stretched=True)
    bc[2] = cases.FaceBC(cases.BC_WALL_ISOTHERMAL, T_wall=1.1, dist={"A": 0.0, "kappa": 10.0, "t1_lo": 0.2, "t1_hi": 0.7})
    b = cases.random_admissible(n=(12, 10, 8), seed=2, bc=list(bc), stretched=True)
    sa, sb = jf.Solver(a), jf.Solver(b)
    Ua, Ub = sa.jf_fill_halo(sa.state()), sb.jf_fill_halo(sb.state())
    assert np.array_equal(Ua.cpu().numpy(), Ub.cpu().numpy())
    assert np.array_equal(sa.jf_rhs(Ua).cpu().numpy(), sb.jf_rhs(Ub).cpu().numpy())


# ------------------------------------------------------------------ jf_rhs
@pytest.mark.parametrize("name", ["periodic_visc", "periodic_inviscid", "bc0", "bc1", "bc2", "ragged", "tiny", "tgv"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_rhs_parity(jf, ora, name, dtype):
    if name == "periodic_visc":
        c = cases.random_admissible(n=(40, 20, 12), seed=7, stretched=True)
    elif name == "periodic_inviscid":
        c = cases.random_admissible(n=(40, 20, 12), seed=8, stretched=True, viscous=False)
    elif name.startswith("bc"):
        c = all_bc_case(n=(37, 21, 13), which=int(name[2]))
        c.body_accel = (0.3, -0.2, 0.1)
    elif name == "ragged":
        c = cases.random_admissible(n=(70, 35, 67), seed=9, stretched=True)   # several tiles + ragged tails
    elif name == "tiny":
        c = cases.random_admissible(n=(4, 4, 4), seed=10)
    else:
        c = cases.tgv(32)
    o = ora.Oracle(c, dtype)
    Uo = o.fill_halo(o.state())
    Ro = o.rhs(Uo)
    s = jf.Solver(c, dtype)
    U = s.jf_fill_halo(s.state())
    R = s.jf_rhs(U).cpu().numpy()
    err = metric_R(R, Ro)
    if dtype == "f64":
        assert np.all(err <= TOL["f64"]), err
    else:
        # R is a difference of O(|F|/dx) fluxes: in fp32 its round-off floor is eps32*|F|/(dx*|R|)
        # (1e-2 for the M = 0.1 TGV).  Measure that floor as fp32-oracle vs fp64-oracle and require
        # the fp32 GPU result to be as close to the fp32 oracle as the fp32 oracle is to the truth.
        o64 = ora.Oracle(c, "f64")
        R64 = o64.rhs(o64.fill_halo(o64.state()))
        noise = metric_R(Ro, R64)
        assert np.all(err <= 4 * noise + 1e-5), (err, noise)
    assert np.all(R[:, 0] == 0) and np.all(R[:, :, 0] == 0) and np.all(R[..., 0] == 0)   # halo of R untouched


def test_free_stream_preservation_on_gpu(jf):
    c = cases.random_admissible(n=(33, 18, 20), seed=0, stretched=True)
    one = np.ones((20, 18, 33))
    c.U0 = cases.set_interior_from_prim(cases.empty_state(c.n), c.gamma, 1.3 * one, 0.7 * one, -0.4 * one,
                                        0.25 * one, 2.1 * one)
    s = jf.Solver(c)
    U = s.jf_fill_halo(s.state())
    R = s.jf_rhs(U).cpu().numpy()
    assert np.max(np.abs(R)) == 0.0
    U1 = s.jf_rk3_step(s.state(), 1e-2).cpu().numpy()
    assert np.array_equal(U1[INT], c.U0[INT])


# ------------------------------------------------------------------ jf_cfl_dt
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_cfl_dt_parity(jf, ora, dtype):
    for c in (cases.random_admissible(n=(40, 20, 12), seed=7, stretched=True), cases.sod(64),
              cases.channel(24, 16, 16)):
        o = ora.Oracle(c, dtype)
        st_o, dt_o = o.cfl_dt(o.state(), 0.5)
        s = jf.Solver(c, dtype)
        st_g, dt_g = s.jf_cfl_dt(s.state(), 0.5)
        assert st_o == 0 and st_g == 0
        assert abs(dt_g - dt_o) <= (1e-14 if dtype == "f64" else 1e-6) * dt_o


def test_cfl_dt_flags_bad_state(jf):
    c = cases.random_admissible(n=(12, 10, 8), seed=1)
    s = jf.Solver(c)
    U = s.state()
    U[0, NH + 1, NH + 2, NH + 3] = -1.0
    st, dt = s.jf_cfl_dt(U, 0.5)
    assert st == jf.JF_ENOTFINITE and np.isnan(dt)
    U = s.state()
    U[4, NH, NH, NH] = float("nan")
    assert s.jf_cfl_dt(U, 0.5)[0] == jf.JF_ENOTFINITE
    U = s.state()
    U[0, 0, 0, 0] = float("nan")                              # halo cells are not inspected
    assert s.jf_cfl_dt(U, 0.5)[0] == jf.JF_OK


# ------------------------------------------------------------------ jf_rk3_step on the configs
def run_both(jf, ora, c, dtype="f64", n_steps=None, want_dts=False):
    Uo, dts_o = ora.run_case(c, dtype, n_steps=n_steps)
    Ug, dts_g = jf.run_case(c, dtype, n_steps=n_steps)
    assert len(dts_o) == len(dts_g)
    rel = max(abs(a - b) / a for a, b in zip(dts_o, dts_g)) if dts_o else 0.0   # |dt_gpu - dt_ora| / dt, worst step
    err = metric_P(Ug.cpu().numpy(), Uo, dtype)
    print(f"{c.name} {c.n} {dtype} x{len(dts_o)} steps: err {err}  max |dt_gpu-dt_ora|/dt {rel:.2e}")
    if want_dts:
        return err, rel, Ug, Uo, dts_o
    return err, rel, Ug, Uo


def arbiter_check(ora, c, Ug, Uo, dts_o, label):
    """|GPU - arbiter| <= max(1e-10, 2 |oracle_fp64 - arbiter|) per variable (module docstring).  The
    arbiter takes the fp64 oracle's time steps, so the oracle differs from it by rounding alone."""
    Ua, _ = ora.run_case(c, "f80", dts_in=dts_o)
    Ua = np.asarray(Ua, dtype=np.float64)                   # rounding the arbiter to double: 1e-16, irrelevant
    e_gpu, e_ora = metric_P(Ug, Ua), metric_P(Uo, Ua)
    print(f"{label}: |gpu - arbiter| {e_gpu}  |oracle_fp64 - arbiter| {e_ora}")
    assert np.all(e_gpu <= np.maximum(TOL["f64"], 2.0 * e_ora)), (e_gpu, e_ora)
    return e_gpu, e_ora


def test_config0_tgv32_10_steps(jf, ora):
    err, _, _, _ = run_both(jf, ora, cases.tgv(32, n_steps=10))
    assert np.all(err <= TOL["f64"]), err


def test_config0_tgv32_fp32(jf, ora):
    err, _, _, _ = run_both(jf, ora, cases.tgv(32, n_steps=10), "f32")
    assert np.all(err <= TOL["f32"]), err


def test_config1_sod_to_t02(jf, ora):
    err, rel_dt, Ug, Uo = run_both(jf, ora, cases.sod(256))
    assert rel_dt <= 1e-12
    assert np.all(err <= TOL["f64"]), err
    Ug = Ug.cpu().numpy()
    assert np.all(Ug[2][INT[1:]] == 0.0) and np.all(Ug[3][INT[1:]] == 0.0)


@pytest.mark.parametrize("axis", [1, 2])
def test_sod_along_y_and_z(jf, ora, axis):
    err, _, _, _ = run_both(jf, ora, cases.sod(64, axis=axis))
    assert np.all(err <= TOL["f64"]), err


def test_config2_channel_reduced_100_steps(jf, ora):
    err, rel_dt, Ug, _ = run_both(jf, ora, cases.channel(48, 32, 32, n_steps=100))
    assert rel_dt <= 1e-12
    assert np.all(err <= TOL["f64"]), err


def test_config2_channel_full_size_100_steps(jf, ora):
    # BASELINE.json configs[2] as stated: 192 x 128 x 128, 100 RK3 steps at CFL 0.5, element by element
    err, rel_dt, Ug, _ = run_both(jf, ora, cases.channel(192, 128, 128, n_steps=100))
    assert rel_dt <= 1e-12
    assert np.all(err <= TOL["f64"]), err


def test_config3_flat_plate_reduced_200_steps(jf, ora):
    c = cases.flat_plate(128, 64, 8, n_steps=200)
    err, rel_dt, Ug, Uo, dts_o = run_both(jf, ora, c, want_dts=True)
    assert rel_dt <= 1e-12
    assert np.all(err[[0, 1, 4]] <= TOL["f64"]), err         # rho, rho u, E against the fp64 oracle itself
    arbiter_check(ora, c, Ug.cpu().numpy(), Uo, dts_o, "flat plate 128x64x8 x200")   # rho v: who is closer to the truth
    rho = Ug.cpu().numpy()[0][INT[1:]]
    assert rho.min() > 0


def test_config3_flat_plate_full_size_200_steps(jf, ora):
    # BASELINE.json configs[3] as stated: 512 x 192 x 8, 200 RK3 steps at CFL 0.5, element by element.
    # rho, rho u, E: 1e-10 against the fp64 oracle.  rho v: the arbiter (module docstring).  The case is
    # invariant along z (8 identical periodic planes; checked bit for bit on both sides), so the arbiter
    # runs the same case with the minimum of 4 spanwise planes and its plane is compared with every plane.
    c = cases.flat_plate(512, 192, 8, n_steps=200)
    err, rel_dt, Ug, Uo, dts_o = run_both(jf, ora, c, want_dts=True)
    assert rel_dt <= 1e-12
    assert np.all(err[[0, 1, 4]] <= TOL["f64"]), err
    Ug = Ug.cpu().numpy()
    assert Ug[0][INT[1:]].min() > 0
    for U in (Ug, Uo):
        assert all(np.array_equal(U[:, NH + k], U[:, NH]) for k in range(1, 8))
        assert np.all(U[3][INT[1:]] == 0.0)
    if np.all(err <= TOL["f64"]):
        return
    c4 = cases.flat_plate(512, 192, 4, n_steps=200)
    Ua, _ = ora.run_case(c4, "f80", dts_in=dts_o)
    Ua = np.repeat(np.asarray(Ua, dtype=np.float64)[:, NH:NH + 1], 8 + 2 * NH, axis=1)
    e_gpu, e_ora = metric_P(Ug, Ua), metric_P(Uo, Ua)
    print(f"flat plate 512x192x8 x200: |gpu - arbiter| {e_gpu}  |oracle_fp64 - arbiter| {e_ora}")
    assert np.all(e_gpu <= np.maximum(TOL["f64"], 2.0 * e_ora)), (e_gpu, e_ora)


def test_paper_section_3_2_boundary_layer_with_disturbance_wall(jf, ora):
    # the paper's own case (tests/golden/paper_section_3_2.txt): 300 x 200 cells, adiabatic
    # Disturbance Wall A = 0.01, kappa = 10 over the whole south wall, similarity inflow, zero-gradient N/E
    c = cases.paper_boundary_layer(n_steps=20)
    o = ora.Oracle(c)
    s = jf.Solver(c, "f64")
    Ug, Uo = s.jf_fill_halo(s.state()).cpu().numpy(), o.fill_halo(o.state())
    assert np.array_equal(Ug[INT], Uo[INT])
    scale = np.max(np.abs(Uo), axis=(1, 2, 3), keepdims=True)
    scale[1:4] = np.max(scale[1:4])                            # rho v, rho w are ~0 here: scale by the momentum
    assert np.max(np.abs(Ug - Uo) / scale) <= 1e-13             # every halo cell
    err, rel_dt, Ug, Uo, dts_o = run_both(jf, ora, c, want_dts=True)
    assert rel_dt <= 1e-12
    assert np.all(err[[0, 1, 4]] <= TOL["f64"]), err
    arbiter_check(ora, c, Ug.cpu().numpy(), Uo, dts_o, "paper 3.2 case x20")
    # A = 0 is the plain no-slip wall on the GPU path as well, bit for bit after 3 steps
    a = cases.paper_boundary_layer(nx=60, ny=40, A=0.0)
    b = cases.paper_boundary_layer(nx=60, ny=40, disturbance=False)
    Ua, _ = jf.run_case(a, "f64", n_steps=3)
    Ub, _ = jf.run_case(b, "f64", n_steps=3)
    assert np.array_equal(Ua.cpu().numpy(), Ub.cpu().numpy())


def test_config4_tgv64_20_steps(jf, ora):
    err, _, _, _ = run_both(jf, ora, cases.tgv(64, n_steps=20))
    assert np.all(err <= TOL["f64"]), err


def test_config4_tgv128_20_steps_fp64_and_fp32(jf, ora):
    # BASELINE.json configs[4] as stated: 20 RK3 steps, element by element
    err, _, _, _ = run_both(jf, ora, cases.tgv(128, n_steps=20))
    assert np.all(err <= TOL["f64"]), err
    err, _, _, _ = run_both(jf, ora, cases.tgv(128, n_steps=20), "f32")
    assert np.all(err <= TOL["f32"]), err


def test_config4_tgv256_20_steps(jf, ora):
    # the size bench.py times (and north_star's roofline target is quoted at), all 20 steps, element by element
    err, _, _, _ = run_both(jf, ora, cases.tgv(256, n_steps=20))
    assert np.all(err <= TOL["f64"]), err


# ------------------------------------------------------------------ error behaviour of the ABI
# ------------------------------------------------------------------ full size, sampled (bench.py's launch configuration)
def _gather(U, idx):
    """U[:, idx_z][:, :, idx_y][:, :, :, idx_x] of a device state array, as float64 on the host."""
    import torch
    iz, iy, ix = (torch.as_tensor(np.asarray(idx[a]), device=U.device) for a in (2, 1, 0))
    return U.index_select(1, iz).index_select(2, iy).index_select(3, ix).cpu().numpy().astype(np.float64)


def _sub_box_case(c, U, lo, m):
    """Periodic m^3 case cut out of the periodic device state U (full padded array) at interior offset lo."""
    idx = [(np.arange(m) + lo[a]) % c.n[a] + NH for a in range(3)]
    sub = cases.empty_state((m, m, m))
    sub[(slice(None),) + (slice(NH, -NH),) * 3] = _gather(U, idx)
    dx = c.xf[1] - c.xf[0]
    f = cases.uniform_faces(0.0, m * dx, m)
    return cases.Case(name="sub", n=(m, m, m), xf=f, yf=f.copy(), zf=f.copy(), gamma=c.gamma, R_gas=c.R_gas,
                      Pr=c.Pr, mu=c.mu, bc=cases.periodic_bc(), U0=sub, dt=c.dt, n_steps=1)


@pytest.mark.parametrize("n,dtype", [(256, "f32"), (384, "f64"), (512, "f64"), (512, "f32")])
def test_config4_full_size_sampled_against_oracle_sub_boxes(jf, ora, n, dtype):
    """384^3 fp64 and 512^3 fp64 / fp32 (the largest lines of configs[4]; 256^3 fp64 runs all 20 steps against
    the whole-grid oracle above), same kernels / grids / segment lengths as bench.py launches: all 20 RK3
    steps on the GPU, and EVERY step is checked on sampled 16^3 blocks, the oracle being fed the GPU's own
    state before that step.  One RK3 step moves information by at most 3 stages x 3 cells, so the oracle
    stepping a periodic 40^3 cut-out of the GPU's state is exact on the central 16^3 (margin 12 >= 9)
    whatever its (wrong) periodic wrap does at the rim.  Cut-outs are gathered on the device.  dt = 1e-3 is
    above the linear stability limit at these sizes, so a whole-run comparison would measure
    amplified round-off; the per-step check does not accumulate it, and the GPU state must stay finite and
    smooth (kinetic energy within 1 % of its initial value) over the 20 steps."""
    import torch
    c = cases.tgv(n)
    s = jf.Solver(c, dtype)
    U = s.state()
    m, g = 40, 12
    rng = np.random.default_rng(11)
    los = [(0, 0, 0), (n - 6, 3, n // 2 - 7), (100, n - 6, n - 6)] + [tuple(int(v) for v in rng.integers(0, n, 3)) for _ in range(3)]

    def kinetic(V):
        Vi = V[(slice(None),) + (slice(NH, -NH),) * 3].double()
        return float(((Vi[1] ** 2 + Vi[2] ** 2 + Vi[3] ** 2) / Vi[0]).sum())

    ke0 = kinetic(U)
    worst = np.zeros(5)
    for step in range(20):
        subs = [_sub_box_case(c, U, lo, m) for lo in los]          # the GPU state before this step
        s.jf_rk3_step(U, c.dt)
        torch.cuda.synchronize()
        Ud = U.double()
        mom = float(torch.sqrt(Ud[1] ** 2 + Ud[2] ** 2 + Ud[3] ** 2).max())
        scale = [float(Ud[0].abs().max()), mom, mom, mom, float(Ud[4].abs().max())]
        del Ud
        for lo, sc in zip(los, subs):
            o = ora.Oracle(sc, dtype)
            Uo = o.state()
            o.rk3_step(Uo, c.dt)
            Uo = np.asarray(Uo, dtype=np.float64)
            idx = [(np.arange(g, m - g) + lo[a]) % n + NH for a in range(3)]
            got = _gather(U, idx)
            ref = Uo[:, NH + g:NH + m - g, NH + g:NH + m - g, NH + g:NH + m - g]
            for q in range(5):
                worst[q] = max(worst[q], np.max(np.abs(got[q] - ref[q])) / scale[q])
    ke1 = kinetic(U)
    print(f"tgv{n}", dtype, "sampled parity, worst of 20 steps x 6 blocks", worst, "KE ratio", ke1 / ke0)
    assert np.all(worst <= TOL[dtype]), worst
    assert bool(torch.isfinite(U).all()) and abs(ke1 / ke0 - 1.0) < 1e-2


# ------------------------------------------------------------------ out-of-bounds guard (compute-sanitizer is closed on this pool)
@pytest.mark.parametrize("name", ["ragged", "tiny", "bc1"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_no_writes_outside_the_state_arrays(jf, name, dtype):
    """U and R live inside larger buffers filled with a canary; after halo fill, RHS, CFL and an RK3 step
    the guard bands (1 MiB on either side) must be untouched and every interior value finite."""
    import torch
    if name == "ragged":
        c = cases.random_admissible(n=(70, 35, 67), seed=9, stretched=True)
    elif name == "tiny":
        c = cases.random_admissible(n=(4, 4, 4), seed=10)
    else:
        c = all_bc_case(n=(37, 21, 13), which=1)
    s = jf.Solver(c, dtype)
    n = int(np.prod(s.shape))
    guard = (1 << 20) // (8 if dtype == "f64" else 4)
    canary = -12345.678
    bufs = [torch.full((n + 2 * guard,), canary, dtype=s.tdtype, device=s.device) for _ in range(2)]
    U = bufs[0][guard:guard + n].view(s.shape)
    U.copy_(s.state())
    s.jf_fill_halo(U)
    R = bufs[1][guard:guard + n].view(s.shape)
    st = jf.lib().jf_rhs(s.h, s._ptr(U), s._ptr(R))
    assert st == jf.JF_OK
    st, dt = s.jf_cfl_dt(U, 0.4)
    assert st == jf.JF_OK and dt > 0
    s.jf_rk3_step(U, dt)
    torch.cuda.synchronize()
    for b in bufs:
        assert bool((b[:guard] == canary).all()) and bool((b[guard + n:] == canary).all())
    assert bool(torch.isfinite(U[(slice(None),) + (slice(NH, -NH),) * 3]).all())
    Ri = R[(slice(None),) + (slice(NH, -NH),) * 3]
    assert bool(torch.isfinite(Ri).all())
    # jf_rhs leaves the halo cells of R untouched
    mask = torch.ones(s.shape, dtype=torch.bool, device=s.device)
    mask[(slice(None),) + (slice(NH, -NH),) * 3] = False
    assert bool((R[mask] == canary).all())


def test_abi_error_statuses(jf):
    import ctypes as C
    import torch
    c = cases.random_admissible(n=(12, 10, 8), seed=1)
    s = jf.Solver(c)
    L = jf.lib()
    U = s.state()
    assert L.jf_fill_halo(s.h, C.c_void_p(U.data_ptr() + 8)) == jf.JF_EALIGN
    assert L.jf_rhs(s.h, C.c_void_p(U.data_ptr()), C.c_void_p(U.data_ptr())) == jf.JF_EINVAL
    assert L.jf_rk3_step(s.h, None, 0.1) == jf.JF_EINVAL
    assert b"jf_rk3_step" in L.jf_last_error(s.h)
    bad = cases.random_admissible(n=(12, 10, 8), seed=1)
    bad.gamma = 0.9
    with pytest.raises(jf.JFError):
        jf.Solver(bad)
    bad = cases.random_admissible(n=(12, 10, 8), seed=1)
    bad.bc[0] = cases.FaceBC(cases.BC_ZEROGRAD)               # periodic faces must pair
    with pytest.raises(jf.JFError):
        jf.Solver(bad)
    n0 = s.jf_launch_count()
    s.jf_rk3_step(U, 1e-3)
    torch.cuda.synchronize()
    # 3 x (halo, gradient, x, y, z + RK) kernels, replayed from the solver's CUDA graph, plus the one-thread
    # kernel that hands the host's dt to the graph
    assert s.jf_launch_count() - n0 == 3 * (1 + 4) + 1


# ------------------------------------------------------------------ CUDA graph replay and device-resident dt
def _solver_without_graph(jf, c, dtype="f64"):
    import os
    old = os.environ.get("JF_GRAPH")
    os.environ["JF_GRAPH"] = "0"
    try:
        return jf.Solver(c, dtype)
    finally:
        if old is None:
            del os.environ["JF_GRAPH"]
        else:
            os.environ["JF_GRAPH"] = old


@pytest.mark.parametrize("name", ["channel", "walls", "tgv_f32"])
def test_graph_replay_is_bitwise_the_plain_launch_sequence(jf, name):
    import torch
    dtype = "f32" if name == "tgv_f32" else "f64"
    c = {"channel": lambda: cases.channel(24, 16, 16), "walls": lambda: all_bc_case(n=(37, 21, 13), which=0),
         "tgv_f32": lambda: cases.tgv(32)}[name]()
    a, b = jf.Solver(c, dtype), _solver_without_graph(jf, c, dtype)
    Ua, Ub = a.state(), b.state()
    for k in range(4):
        dt = 1e-3 * (1 + 0.1 * k)                            # a different dt every step: same graph
        a.jf_rk3_step(Ua, dt)
        b.jf_rk3_step(Ub, dt)
    torch.cuda.synchronize()
    assert b.jf_launch_count() == 4 * 15 and a.jf_launch_count() == 4 * 16
    assert Ua.cpu().numpy().tobytes() == Ub.cpu().numpy().tobytes()
    # a second state array gets its own graph
    Va, Vb = a.state(), b.state()
    a.jf_rk3_step(Va, 2e-3)
    b.jf_rk3_step(Vb, 2e-3)
    assert Va.cpu().numpy().tobytes() == Vb.cpu().numpy().tobytes()


@pytest.mark.parametrize("variant", ["JF_YZ_PC", "JF_GRAD_TMA", "JF_F32X2"])
@pytest.mark.parametrize("name", ["ragged", "bc0", "bc1", "tiny", "channel"])
def test_selectable_kernel_variants_against_the_oracle(jf, ora, variant, name):
    # the measured variants stay selectable: the producer / consumer form of the marching sweeps
    # (jf_pc.cuh), the TMA-staged gradient pass (jf_tma.cuh; the default on small fields, forced on here) and the fp32
    # marching sweeps with two columns per thread on packed FP32x2 arithmetic (jf_f32x2.cuh; odd extents included: the
    # last thread's second column is a repeat that is not stored).  Same parity bars as the default path.
    import os
    dtype = "f32" if variant == "JF_F32X2" else "f64"
    c = {"ragged": lambda: cases.random_admissible(n=(70, 35, 67), seed=9, stretched=True),
         "bc0": lambda: all_bc_case(n=(38, 21, 13), which=0), "bc1": lambda: all_bc_case(n=(38, 21, 13), which=1),
         "tiny": lambda: cases.random_admissible(n=(4, 4, 4), seed=10), "channel": lambda: cases.channel(48, 32, 32, n_steps=20)}[name]()
    c.body_accel = (0.3, -0.2, 0.1) if name.startswith("bc") else c.body_accel
    os.environ[variant] = "1"
    try:
        s = jf.Solver(c, dtype)
    finally:
        del os.environ[variant]
    o = ora.Oracle(c, dtype)
    Ro = o.rhs(o.fill_halo(o.state()))
    R = s.jf_rhs(s.jf_fill_halo(s.state())).cpu().numpy()
    if dtype == "f64":
        assert np.all(metric_R(R, Ro) <= TOL["f64"])
    else:                                                     # as test_rhs_parity: against the fp32 oracle's own distance from fp64
        o64 = ora.Oracle(c, "f64")
        noise = metric_R(Ro, o64.rhs(o64.fill_halo(o64.state())))
        assert np.all(metric_R(R, Ro) <= 4 * noise + 1e-5)
        d = jf.Solver(c, dtype)                               # and the default (scalar) fp32 kernels give the same to fp32 round-off
        Rd = d.jf_rhs(d.jf_fill_halo(d.state())).cpu().numpy()
        assert np.all(metric_R(R, Rd) <= 4 * noise + 1e-5)
    n_steps = 20 if name == "channel" else 3
    Uo, U = o.state(), s.state()
    for _ in range(n_steps):
        st, dt = o.cfl_dt(Uo, 0.5)
        o.rk3_step(Uo, dt)
        s.jf_rk3_step(U, dt)
    assert np.all(metric_P(U.cpu().numpy(), Uo, dtype) <= TOL[dtype])


@pytest.mark.parametrize("name", ["channel", "sod", "plate"])
def test_device_resident_dt_equals_the_host_loop(jf, ora, name):
    # jf_cfl_dt_dev + jf_rk3_step_dev (the step is formed and consumed on the device, t_end clipping included)
    # against jf_cfl_dt + jf_rk3_step: same dt sequence bit for bit, same state bit for bit; and against the oracle
    c = {"channel": lambda: cases.channel(24, 16, 16, n_steps=12), "sod": lambda: cases.sod(64),
         "plate": lambda: cases.flat_plate(64, 24, 8, n_steps=12)}[name]()
    Uh, dth = jf.run_case(c, "f64")
    Ud, dtd = jf.run_case(c, "f64", device_dt=True)
    assert dth == dtd and len(dth) > 5
    assert Uh.cpu().numpy().tobytes() == Ud.cpu().numpy().tobytes()
    Uo, dto = ora.run_case(c, "f64")
    assert len(dto) == len(dtd) and max(abs(x - y) / x for x, y in zip(dto, dtd)) <= 1e-12
    assert np.all(metric_P(Ud.cpu().numpy(), Uo) <= TOL["f64"])


@pytest.mark.parametrize("dtype", ["f32", "f64t"])
def test_device_resident_dt_other_dtypes(jf, dtype):
    # the same equality (dt sequence and state, bit for bit) for the fp32 and the tangent solver
    c = cases.channel(24, 16, 16, n_steps=8)
    Uh, dth = jf.run_case(c, dtype)
    Ud, dtd = jf.run_case(c, dtype, device_dt=True)
    assert dth == dtd and len(dth) == 8
    assert Uh.cpu().numpy().tobytes() == Ud.cpu().numpy().tobytes()


def test_device_resident_dt_flags_bad_state(jf):
    c = cases.random_admissible(n=(12, 10, 8), seed=1)
    s = jf.Solver(c)
    U = s.state()
    s.jf_cfl_dt_dev(U, 0.5)
    st, dt, t = s.jf_dev_time()
    st_h, dt_h = s.jf_cfl_dt(U, 0.5)
    assert st == jf.JF_OK and dt == dt_h and t == dt
    U[0, NH + 1, NH + 2, NH + 3] = -1.0
    s.jf_cfl_dt_dev(U, 0.5)
    st, dt, t = s.jf_dev_time()
    assert st == jf.JF_ENOTFINITE and np.isnan(dt)
    st, dt, t = s.jf_dev_time(set_t=0.25)                     # reset clears the sticky status
    assert st == jf.JF_OK and t == 0.25 and dt == 0.0
