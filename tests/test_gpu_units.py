"""Unit-level GPU parity: the per-face arithmetic of the sweep kernels (jf_math.cuh, reached through
jf_diag_face_flux of the C ABI) against the oracle's scheme functions on seeded random stencils."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu
G, RG, PR = 1.4, 0.8, 0.72


@pytest.fixture(scope="module")
def jf():
    import torch
    assert torch.cuda.is_available()
    from paper_2406_19494_b200 import binding
    return binding


def stencils(n, seed, jump=False):
    rng = np.random.default_rng(seed)
    W = np.empty((n, 6, 6))
    base = rng.uniform(0.5, 2.0, (n, 1))
    W[:, :, 0] = base + 0.2 * rng.uniform(-1, 1, (n, 6))
    W[:, :, 1:4] = rng.uniform(-1.5, 1.5, (n, 1, 3)) + 0.3 * rng.uniform(-1, 1, (n, 6, 3))
    W[:, :, 4] = rng.uniform(0.5, 3.0, (n, 1)) + 0.2 * rng.uniform(-1, 1, (n, 6))
    if jump:                                   # discontinuity at a random position of the stencil
        k = rng.integers(1, 6, n)
        for f in range(n):
            W[f, k[f]:, 0] *= 4.0
            W[f, k[f]:, 4] *= 7.0
            W[f, k[f]:, 1:4] += 2.0
    W[:, :, 5] = W[:, :, 4] / (W[:, :, 0] * RG)
    return W


def oracle_face(ora, d, W, Gt, Xf, mu):
    n, t1, t2 = d, (d + 1) % 3, (d + 2) % 3
    WL = [ora.weno5(W[0:5, q]) for q in range(5)]
    WR = [ora.weno5(W[5:0:-1, q]) for q in range(5)]
    F = ora.hllc(d, G, WL, WR)
    if mu["mu_ref"] > 0:
        qs = [1 + n, 1 + t1, 1 + t2, 5]
        dn = [ora.df(W[1:5, q], Xf) for q in qs]
        fv = [ora.iface(W[1:5, q]) for q in qs]
        gt = [ora.iface(Gt[:, c]) for c in range(4)]
        m = ora.viscosity(mu, fv[3])
        lam = m * G * RG / (G - 1) / PR
        div = dn[0] + gt[1] + gt[3]
        tnn, tn1, tn2 = m * (2 * dn[0] - 2.0 / 3.0 * div), m * (gt[0] + dn[1]), m * (gt[2] + dn[2])
        F[1 + n] -= tnn
        F[1 + t1] -= tn1
        F[1 + t2] -= tn2
        F[4] -= fv[0] * tnn + fv[1] * tn1 + fv[2] * tn2 + lam * dn[3]
    return F


@pytest.mark.parametrize("d", [0, 1, 2])
@pytest.mark.parametrize("kind", ["smooth", "jump", "viscous"])
def test_face_flux_matches_oracle_functions(jf, ora, d, kind):
    n = 300
    W = stencils(n, seed=10 * d + len(kind), jump=(kind == "jump"))
    rng = np.random.default_rng(5)
    mu = {"sutherland": 1, "mu_ref": 0.05 if kind == "viscous" else 0.0, "T_ref": 1.0, "S": 0.4}
    Gt = rng.uniform(-2, 2, (n, 4, 4))
    Xf = rng.uniform(0.05, 0.2, n)
    F = jf.jf_diag_face_flux("f64", d, G, RG, PR, mu, W, Gt, Xf)
    Fo = np.array([oracle_face(ora, d, W[f], Gt[f], Xf[f], mu) for f in range(n)])
    scale = np.maximum(np.max(np.abs(Fo), axis=1, keepdims=True), 1.0)
    assert np.max(np.abs(F - Fo) / scale) <= 5e-14
    F32 = jf.jf_diag_face_flux("f32", d, G, RG, PR, mu, W, Gt, Xf)
    # fp32 build of the same device code against the fp64 oracle: north_star's fp32 tolerance
    assert np.max(np.abs(F32 - Fo) / scale) <= 1e-4


@pytest.mark.parametrize("d", [0, 1, 2])
def test_fp32_face_flux_in_si_units_with_strong_jumps(jf, ora, d):
    # fp32 with dimensional data: p ~ 1e5 Pa, rho ~ 1 kg/m3, u ~ 300 m/s and jumps of 1e4 .. 1e5 Pa inside the
    # stencil.  Weights formed from products of (beta+eps)^2 overflow here (beta ~ jump^2 => product ~ jump^8);
    # the fp32 kernels form them from reciprocals and must stay finite and within fp32 accuracy of the oracle.
    rng = np.random.default_rng(40 + d)
    n = 400
    W = np.empty((n, 6, 6))
    W[:, :, 0] = rng.uniform(0.8, 1.3, (n, 1)) + 0.05 * rng.uniform(-1, 1, (n, 6))
    W[:, :, 1:4] = rng.uniform(-300, 300, (n, 1, 3)) + 20.0 * rng.uniform(-1, 1, (n, 6, 3))
    W[:, :, 4] = rng.uniform(0.9e5, 1.1e5, (n, 1)) + 500.0 * rng.uniform(-1, 1, (n, 6))
    k = rng.integers(1, 6, n)
    jump = rng.uniform(1e4, 1e5, n) * rng.choice([-0.5, 1.0], n)     # never below ~4e4 Pa
    for f in range(n):
        W[f, k[f]:, 4] += jump[f]
        W[f, k[f]:, 0] *= 1.0 + 0.5 * jump[f] / 1e5
    Rg = 287.058
    W[:, :, 5] = W[:, :, 4] / (W[:, :, 0] * Rg)
    mu = {"sutherland": 0, "mu_ref": 0.0, "T_ref": 1.0, "S": 0.0}
    F32 = jf.jf_diag_face_flux("f32", d, G, Rg, PR, mu, W)
    assert np.isfinite(F32).all()
    Fo = np.array([oracle_face(ora, d, W[f], None, 1.0, mu) for f in range(n)])
    scale = np.max(np.abs(Fo), axis=1, keepdims=True)
    assert np.max(np.abs(F32 - Fo) / scale) <= 1e-4
    F64 = jf.jf_diag_face_flux("f64", d, G, Rg, PR, mu, W)
    assert np.max(np.abs(F64 - Fo) / scale) <= 2e-12       # (jumps of half the pressure: both sides lose digits in the weights)


def test_face_flux_consistency_on_uniform_stencils(jf, ora):
    # F(W,W) = F^c(W) (Eq. 3) to round-off on the GPU as well
    rng = np.random.default_rng(3)
    n = 64
    W = np.repeat(stencils(n, 1)[:, :1, :], 6, axis=1)
    mu = {"sutherland": 0, "mu_ref": 0.0, "T_ref": 1.0, "S": 0.0}
    for d in range(3):
        F = jf.jf_diag_face_flux("f64", d, G, RG, PR, mu, W)
        Fo = np.array([ora.flux_phys(d, G, W[f, 0, :5]) for f in range(n)])
        assert np.max(np.abs(F - Fo) / np.maximum(np.abs(Fo).max(axis=1, keepdims=True), 1)) <= 1e-14


@pytest.mark.parametrize("name", ["stretched_periodic", "channel", "plate", "exchange"])
@pytest.mark.parametrize("dtype", ["f64", "f32"])
def test_geometry_tables_against_the_oracles(jf, ora, name, dtype):
    # reading O2: the library and the oracle each build 1/Delta, the cell centres and the index-space metrics
    # X_xi^c, X_xi^f from the face coordinates (two independent statements of one recipe).  jf_diag_metrics
    # copies back the tables the kernels actually read; compare them entry by entry with the oracle's.
    from paper_2406_19494_b200 import cases, decomp
    if name == "stretched_periodic":
        c = cases.random_admissible(n=(13, 9, 11), seed=4, stretched=True)
        pairs = [(c, c, [slice(None)] * 3)]
    elif name == "channel":
        c = cases.channel(24, 16, 16)
        pairs = [(c, c, [slice(None)] * 3)]
    elif name == "plate":
        c = cases.flat_plate(64, 24, 8)
        pairs = [(c, c, [slice(None)] * 3)]
    else:
        # an exchange-face block must carry the geometry of the undivided grid: compare each block's tables with
        # the slice of the undivided oracle's tables it covers
        c = cases.channel(24, 16, 16)
        pairs = []
        for part in decomp.split_case(c, (2, 2, 1)):
            sl = [slice(part.lo[a], part.lo[a] + part.case.n[a] + 6) for a in range(3)]
            pairs.append((part.case, c, sl))
    tol = 4e-16 if dtype == "f64" else 2e-7
    for blk, whole, sl in pairs:
        s = jf.Solver(blk, dtype)
        o = ora.Oracle(whole, "f64")
        for a in range(3):
            inv_dl, xc, i12Xc, i24Xf = s.jf_diag_metrics(a)
            d, x = (v[sl[a]] for v in o.metrics(a))
            Xc, Xf = (v[sl[a]] for v in o.metrics_index(a))
            n = blk.n[a]
            assert np.max(np.abs(inv_dl * d - 1.0)) <= tol
            assert np.max(np.abs(xc - x)) <= 4e-16 * np.max(np.abs(x))      # centres are kept in fp64 for every dtype
            ci = slice(3, n + 3)                          # X_xi^c: interior cells
            assert np.max(np.abs(i12Xc[ci] * 12.0 * Xc[ci] - 1.0)) <= 4 * tol
            fi = slice(2, n + 3)                          # X_xi^f: faces -1/2 .. n-1/2
            assert np.max(np.abs(i24Xf[fi] * 24.0 * Xf[fi] - 1.0)) <= 4 * tol


def test_bench_line_schema_on_a_small_box(jf):
    # the one JSON line bench.py prints, through the real GPU path on a 48^3 box: the contract's keys and the
    # tier's additions (roofline with both numerators and both clocks, cpu_baseline, e2e with host copies)
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--size", "48", "--steps", "3", "--warmup", "3"],
                         capture_output=True, text=True, timeout=600)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    for k in ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
              "dtype", "data", "config", "clocks", "gpu_launches", "roofline", "roofline_step", "e2e", "cpu_baseline"):
        assert k in d, k
    assert d["unit"] == "cell-updates/s" and d["dtype"] == "f64" and d["steps"] == 3 and d["vs_baseline"] is None
    assert d["gpu_launches"] == 3 * 16 and d["config"]["finite"] is True
    r = d["roofline"]
    assert r["bound"] == "alu" and 0 < r["frac"] < 1 and r["peak"] > 20 and "numerator" in r and "frac_at_run_clock" in r
    assert d["e2e"]["h2d_bytes_per_step"] == d["config"]["state_bytes"] == 5 * 54 ** 3 * 8 and d["e2e"]["value"] < d["value"]
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] > 0
    assert d["value"] == pytest.approx(48 ** 3 * 3 / (d["ms_per_step"] * 3 * 1e-3), rel=1e-9)


def test_decomposition_arm_of_bench_on_one_rank(jf):
    # bench.py --decomp with a single block: the arm's whole code path (RankBlock over torch.distributed, axis-by-axis halo
    # passes, stage calls, max-over-ranks timing, PID of Eq. 9) except the exchange itself, which needs a second GPU
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, MASTER_PORT="29541")
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--decomp", "1,1,1", "--size", "48", "--steps", "4"],
                         capture_output=True, text=True, timeout=600, env=env)
    assert out.returncode == 0, out.stderr[-3000:]
    d = json.loads([ln for ln in out.stdout.splitlines() if ln.startswith("{")][-1])
    assert d["n_gpus"] == 1 and d["scaling"] == "weak" and d["config"]["finite"] is True
    assert d["config"]["exchange_bytes_per_rank_per_step"] == 0
    assert d["gpu_launches"] == 4 * 3 * 7                     # per stage: three axis passes, gradient, x, y, z + RK
    assert d["pid"]["dof_cells"] == pytest.approx(d["ms_per_step"] * 1e-3 / 48 ** 3, rel=1e-9)
    assert d["pid"]["dof_cells_x5"] == pytest.approx(d["pid"]["dof_cells"] / 5, rel=1e-12)
