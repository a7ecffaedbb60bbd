"""the oracle's sources rebuilt with -fsanitize=address,undefined and driven through every call
(halo fill with every BC type, RHS, brute-force RHS, RK3 steps, CFL, the arbiter and fp32 instantiations)
on the 8^3 / 32^3 configs and the small all-BC boxes.  The instrumented library needs libasan loaded first,
so the work runs in a child interpreter with LD_PRELOAD; any report makes the child exit non-zero."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import sys
sys.path.insert(0, %(root)r)
import numpy as np
from oracle import ora
from paper_2406_19494_b200 import cases
sys.path.insert(0, %(root)r + "/tests")

def drive(c, dtype, steps):
    o = ora.Oracle(c, dtype, variant="asan")
    U = o.fill_halo(o.state())
    R = o.rhs(U)
    assert np.isfinite(np.asarray(R, dtype=np.float64)).all()
    for _ in range(steps):
        st, dt = o.cfl_dt(U, 0.4)
        assert st == 0
        o.rk3_step(U, dt if c.dt is None else c.dt)
    return o, U

# 8^3 smooth periodic box: face-loop RHS, brute-force RHS, flop-counting build
c = cases.smooth_periodic(n=(8, 8, 8))
o, U = drive(c, "f64", 2)
o.rhs(o.fill_halo(o.state()), naive=True)
o.count_flops_step(o.state(), 1e-3)
drive(c, "f32", 1)
drive(c, "f80", 1)
# 32^3 Taylor-Green (config 0), one step
drive(cases.tgv(32), "f64", 1)
# the minimum grid and a ragged one
drive(cases.random_admissible(n=(4, 4, 4), seed=10), "f64", 1)
drive(cases.random_admissible(n=(9, 7, 5), seed=3, stretched=True), "f64", 1)
# every BC type on every axis (walls with disturbance segments, Dirichlet tables, zero gradient)
from test_gpu_parity import all_bc_case
for which in (0, 1, 2):
    drive(all_bc_case(which=which), "f64", 1)
# the wall-bounded configs at reduced size, Sod along each axis
drive(cases.channel(12, 8, 8), "f64", 1)
drive(cases.flat_plate(32, 16, 4), "f64", 1)
for axis in range(3):
    drive(cases.sod(16, axis=axis), "f64", 1)
print("SANITIZED-OK")
"""


def test_oracle_under_address_and_undefined_behaviour_sanitizers():
    sys.path.insert(0, os.path.join(ROOT, "oracle"))
    import importlib.util as ilu
    spec = ilu.spec_from_file_location("_ora_build_t", os.path.join(ROOT, "oracle", "build.py"))
    b = ilu.module_from_spec(spec)
    spec.loader.exec_module(b)
    rt = b.asan_runtime()
    if rt is None:
        pytest.skip("no libasan on this box")
    b.build(variant="asan")
    env = dict(os.environ)
    env["LD_PRELOAD"] = rt
    env["ASAN_OPTIONS"] = "detect_leaks=0:abort_on_error=0:exitcode=23"
    env["UBSAN_OPTIONS"] = "halt_on_error=1:print_stacktrace=1"
    env["OMP_NUM_THREADS"] = "4"
    r = subprocess.run([sys.executable, "-c", CHILD % {"root": ROOT}], env=env, capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, (r.returncode, r.stdout[-2000:], r.stderr[-4000:])
    assert "SANITIZED-OK" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
