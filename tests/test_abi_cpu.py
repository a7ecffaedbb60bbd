"""CPU-side checks of the C-ABI library: it builds, loads, exports every symbol include/jf.h declares,
validates arguments, and refuses to compute without a CUDA device (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2406_19494_b200 import binding, build, cases

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    build.build()
    return binding.lib()


def test_exports_every_declared_symbol(L):
    hdr = open(os.path.join(ROOT, "include", "jf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(jf_[a-z0-9_]+)\s*\(", hdr))
    assert {"jf_create", "jf_fill_halo", "jf_rhs", "jf_rk3_step", "jf_cfl_dt"} <= declared
    for name in declared:
        assert hasattr(L, name), name
    assert declared == set(binding.EXPORTS)
    assert b"sm_100a" in L.jf_version()


def test_struct_layouts_match_header_sizes():
    # x86-64 SysV layout of the header's structs
    assert C.sizeof(binding.jf_grid) == 40
    assert C.sizeof(binding.jf_mu_law) == 32
    assert C.sizeof(binding.jf_disturbance) == 40
    assert C.sizeof(binding.jf_bc_face) == 8 + 8 + 24 + 8 + 40 + 24 + 8 + 24   # ..., nb_width[3], nb_has_face (+pad), nb_face[3]
    assert C.sizeof(binding.jf_bc) == 6 * C.sizeof(binding.jf_bc_face)


def _grid(n=(8, 8, 8)):
    keep = []
    c = cases.random_admissible(n=n, seed=1)
    return binding._grid_struct(c, keep), keep


def test_workspace_bytes(L):
    g, keep = _grid((8, 8, 8))
    b64, b32 = L.jf_workspace_bytes(C.byref(g), 0), L.jf_workspace_bytes(C.byref(g), 1)
    vol = 14 ** 3
    assert b64 >= 24 * vol * 8 and b64 < 24 * vol * 8 + 64 * 1024
    assert b32 >= 24 * vol * 4 and b32 < b64
    g.nx = 3
    assert L.jf_workspace_bytes(C.byref(g), 0) == 0
    g, keep = _grid((8, 8, 8))
    keep[0][3] = keep[0][2]                                   # non-monotone faces
    assert L.jf_workspace_bytes(C.byref(g), 0) == 0
    assert L.jf_workspace_bytes(C.byref(g), 7) == 0
    # maximum size: cells of one variable are addressed with 32-bit offsets, (nx+6)(ny+6)(nz+6) < 2^32
    def big(n):                                               # grid description only: no state is allocated
        f = np.linspace(0.0, 1.0, n + 1)
        gg = binding.jf_grid()
        gg.nx = gg.ny = gg.nz = n
        gg.xf = gg.yf = gg.zf = f.ctypes.data_as(C.POINTER(C.c_double))
        return gg, f
    g, keep = big(1618)                                        # 1624^3 = 4 283 098 624 < 2^32: accepted
    assert L.jf_workspace_bytes(C.byref(g), 0) > 24 * 1624 ** 3 * 8
    g, keep = big(1620)                                        # 1626^3 = 4 298 942 376 >= 2^32: refused
    assert L.jf_workspace_bytes(C.byref(g), 0) == 0


def test_create_validates_before_touching_the_device(L):
    g, keep = _grid()
    mu = binding.jf_mu_law(0, 1e-3, 1.0, 0.0)
    bc = binding.jf_bc()
    h = C.c_void_p(123)
    args = lambda **kw: (C.byref(h), kw.get("g", C.byref(g)), kw.get("dt", 0), kw.get("gamma", 1.4), 1.0,
                         kw.get("Pr", 0.72), kw.get("mu", C.byref(mu)), kw.get("bc", C.byref(bc)), None,
                         kw.get("ws", C.c_void_p(256)), kw.get("nb", 1 << 40), None)
    assert L.jf_create(*args(gamma=1.0)) == binding.JF_EINVAL and h.value is None
    assert L.jf_create(*args(Pr=0.0)) == binding.JF_EINVAL
    assert L.jf_create(*args(dt=3)) == binding.JF_EINVAL
    assert L.jf_create(*args(mu=None)) == binding.JF_EINVAL
    bc2 = binding.jf_bc()
    bc2.face[0].type = 1
    assert L.jf_create(*args(bc=C.byref(bc2))) == binding.JF_EINVAL      # unpaired periodic
    bc2.face[1].type = 2
    assert L.jf_create(*args(bc=C.byref(bc2))) == binding.JF_EINVAL      # Dirichlet without table
    bc2.face[1].type = 3
    assert L.jf_create(*args(bc=C.byref(bc2))) == binding.JF_EINVAL      # isothermal wall, T_wall = 0
    assert L.jf_create(*args(ws=C.c_void_p(264))) == binding.JF_EALIGN
    assert L.jf_create(*args(ws=None)) == binding.JF_EWORKSPACE
    assert L.jf_create(*args(nb=1000)) == binding.JF_EWORKSPACE
    assert L.jf_create(None, *args()[1:]) == binding.JF_EINVAL


def test_no_cpu_fallback(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("box has a GPU")
    g, keep = _grid()
    mu = binding.jf_mu_law(0, 1e-3, 1.0, 0.0)
    bc = binding.jf_bc()
    h = C.c_void_p()
    st = L.jf_create(C.byref(h), C.byref(g), 0, 1.4, 1.0, 0.72, C.byref(mu), C.byref(bc), None,
                     C.c_void_p(256), 1 << 40, None)
    assert st == binding.JF_ECUDA and h.value is None
    with pytest.raises(binding.JFError):
        binding.Solver(cases.random_admissible(n=(8, 8, 8), seed=1))
    fl = C.c_double()
    assert L.jf_diag_alu_peak(0, 16, C.byref(fl), None) == binding.JF_ECUDA
    for name in ("jf_fill_halo", "jf_rk3_step", "jf_cfl_dt"):
        assert getattr(L, name)(None, None, *([0.0] if name != "jf_fill_halo" else []),
                                *([None] if name == "jf_cfl_dt" else [])) == binding.JF_EINVAL


def test_product_path_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2406_19494_b200")
    pat = re.compile(r"(^\s*(from|import)\s+oracle\b)|libora|ora_[a-z]+\s*\(|#include\s+\"ora", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h", ".cpp")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), f
