"""ctypes wrapper of the CPU ORACLE (oracle/libora.so).  TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  It shares nothing with paper_2406_19494_b200.binding; both are driven from
the same `cases.Case` input description.
"""
import ctypes as C
import os
import sys

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
import importlib.util as _ilu  # noqa: E402

_spec = _ilu.spec_from_file_location("_ora_build", os.path.join(_HERE, "build.py"))
_build = _ilu.module_from_spec(_spec)
_spec.loader.exec_module(_build)

c_double_p = C.POINTER(C.c_double)


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("xf", c_double_p), ("yf", c_double_p), ("zf", c_double_p)]


class MuLaw(C.Structure):
    _fields_ = [("sutherland", C.c_int), ("mu_ref", C.c_double), ("T_ref", C.c_double), ("S", C.c_double)]


class Disturbance(C.Structure):
    _fields_ = [("enabled", C.c_int), ("A", C.c_double), ("kappa", C.c_double),
                ("t1_lo", C.c_double), ("t1_hi", C.c_double)]


class BCFace(C.Structure):
    _fields_ = [("type", C.c_int), ("T_wall", C.c_double), ("u_wall", C.c_double * 3),
                ("dirichlet", c_double_p), ("dist", Disturbance)]


class BC(C.Structure):
    _fields_ = [("face", BCFace * 6)]


_libs = {}


def lib(variant="ref"):
    """variant "ref": the oracle (-ffp-contract=off).  "fma": same sources with FMA contraction,
    only for measuring the oracle's own round-off sensitivity.  "asan": same sources under
    AddressSanitizer + UBSan (needs libasan preloaded: tests/test_oracle_sanitizers.py)."""
    if variant not in _libs:
        path = _build.build(variant=variant)
        L = C.CDLL(path)
        L.ora_create.restype = C.c_int
        L.ora_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(Grid), C.c_int, C.c_double, C.c_double,
                                 C.c_double, C.POINTER(MuLaw), C.POINTER(BC), c_double_p]
        L.ora_destroy.argtypes = [C.c_void_p]
        L.ora_destroy.restype = None
        L.ora_state_elems.argtypes = [C.c_void_p]
        L.ora_state_elems.restype = C.c_size_t
        for name in ("ora_fill_halo",):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
        for name in ("ora_rhs", "ora_rhs_naive"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.ora_rhs_parts.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int]
        L.ora_rk3_step.argtypes = [C.c_void_p, C.c_void_p, C.c_double]
        L.ora_cfl_dt.argtypes = [C.c_void_p, C.c_void_p, C.c_double, c_double_p]
        L.ora_count_flops_step.argtypes = [C.c_void_p, C.c_void_p, C.c_double, c_double_p]
        L.ora_count_flops_part.argtypes = [C.c_void_p, C.c_void_p, C.c_int, c_double_p]
        L.ora_metrics.argtypes = [C.c_void_p, C.c_int, c_double_p, c_double_p]
        L.ora_metrics_index.argtypes = [C.c_void_p, C.c_int, c_double_p, c_double_p]
        L.ora_weno5.argtypes = [c_double_p]
        L.ora_weno5.restype = C.c_double
        L.ora_weno5_detail.argtypes = [c_double_p] * 4
        L.ora_weno5_detail.restype = None
        L.ora_hllc.argtypes = [C.c_int, C.c_double, c_double_p, c_double_p, c_double_p]
        L.ora_hllc.restype = None
        L.ora_flux_phys.argtypes = [C.c_int, C.c_double, c_double_p, c_double_p]
        L.ora_flux_phys.restype = None
        L.ora_cons_to_prim.argtypes = [C.c_double, c_double_p, c_double_p]
        L.ora_cons_to_prim.restype = None
        L.ora_prim_to_cons.argtypes = [C.c_double, c_double_p, c_double_p]
        L.ora_prim_to_cons.restype = None
        L.ora_viscosity.argtypes = [C.POINTER(MuLaw), C.c_double]
        L.ora_viscosity.restype = C.c_double
        L.ora_dc.argtypes = [c_double_p, C.c_double]
        L.ora_dc.restype = C.c_double
        L.ora_df.argtypes = [c_double_p, C.c_double]
        L.ora_df.restype = C.c_double
        L.ora_if.argtypes = [c_double_p]
        L.ora_if.restype = C.c_double
        L.ora_set_visc_order.argtypes = [C.c_void_p, C.c_int]
        L.ora_dc6.argtypes = [c_double_p, C.c_double]
        L.ora_dc6.restype = C.c_double
        L.ora_df6.argtypes = [c_double_p, C.c_double]
        L.ora_df6.restype = C.c_double
        L.ora_if6.argtypes = [c_double_p]
        L.ora_if6.restype = C.c_double
        L.ora_viscous_face.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int, c_double_p]
        _libs[variant] = L
    return _libs[variant]


def _dp(a):
    return a.ctypes.data_as(c_double_p)


def _arr(x, n=None):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    if n is not None:
        assert a.size == n
    return a


class Oracle:
    """The five calls of the oracle on host numpy arrays, built from a cases.Case."""

    def __init__(self, case, dtype="f64", variant="ref"):
        self.case = case
        self.L = lib(variant)
        self.np_dtype = {"f64": np.float64, "f32": np.float32, "f80": np.longdouble}[dtype]
        if dtype == "f80":
            assert np.finfo(np.longdouble).nmant == 63 and np.dtype(np.longdouble).itemsize == 16
        self._keep = []
        nx, ny, nz = case.n
        xf, yf, zf = _arr(case.xf, nx + 1), _arr(case.yf, ny + 1), _arr(case.zf, nz + 1)
        self._keep += [xf, yf, zf]
        g = Grid(nx, ny, nz, _dp(xf), _dp(yf), _dp(zf))
        mu = MuLaw(int(case.mu["sutherland"]), case.mu["mu_ref"], case.mu["T_ref"], case.mu["S"])
        bc = BC()
        for f, fb in enumerate(case.bc):
            b = bc.face[f]
            b.type = int(fb.type)
            b.T_wall = float(fb.T_wall)
            for d in range(3):
                b.u_wall[d] = float(fb.u_wall[d])
            if fb.dirichlet is not None:
                t = _arr(fb.dirichlet)
                self._keep.append(t)
                b.dirichlet = _dp(t)
            if fb.dist is not None:
                b.dist = Disturbance(1, fb.dist["A"], fb.dist["kappa"], fb.dist["t1_lo"], fb.dist["t1_hi"])
        ga = _arr(case.body_accel, 3)
        h = C.c_void_p()
        st = self.L.ora_create(C.byref(h), C.byref(g), {"f64": 0, "f32": 1, "f80": 2}[dtype], case.gamma, case.R_gas,
                              case.Pr, C.byref(mu), C.byref(bc), _dp(ga))
        if st != 0:
            raise ValueError(f"ora_create failed with status {st}")
        self.h = h
        if getattr(case, "visc_order", 4) != 4:
            assert self.L.ora_set_visc_order(h, int(case.visc_order)) == 0
        self.shape = (5, nz + 6, ny + 6, nx + 6)

    def __del__(self):
        if getattr(self, "h", None) and getattr(self, "L", None) is not None:
            self.L.ora_destroy(self.h)
            self.h = None

    def state(self, U0=None):
        U = np.array(self.case.U0 if U0 is None else U0, dtype=self.np_dtype, order="C")
        assert U.shape == self.shape
        return U

    def _chk(self, U):
        assert U.dtype == self.np_dtype and U.flags.c_contiguous and U.shape == self.shape

    def fill_halo(self, U):
        self._chk(U)
        assert self.L.ora_fill_halo(self.h, U.ctypes.data) == 0
        return U

    def rhs(self, U, naive=False, parts=None):
        self._chk(U)
        R = np.zeros_like(U)
        if naive:
            st = self.L.ora_rhs_naive(self.h, U.ctypes.data, R.ctypes.data)
        elif parts is not None:
            st = self.L.ora_rhs_parts(self.h, U.ctypes.data, R.ctypes.data, *[int(p) for p in parts])
        else:
            st = self.L.ora_rhs(self.h, U.ctypes.data, R.ctypes.data)
        assert st == 0
        return R

    def rk3_step(self, U, dt):
        self._chk(U)
        assert self.L.ora_rk3_step(self.h, U.ctypes.data, float(dt)) == 0
        return U

    def cfl_dt(self, U, cfl):
        self._chk(U)
        dt = C.c_double()
        st = self.L.ora_cfl_dt(self.h, U.ctypes.data, float(cfl), C.byref(dt))
        return st, dt.value

    def count_flops_step(self, U, dt):
        self._chk(U)
        out = np.zeros(4)
        assert self.L.ora_count_flops_step(self.h, U.ctypes.data, float(dt), _dp(out)) == 0
        return out

    def count_flops_part(self, U, what):
        self._chk(U)
        out = np.zeros(4)
        assert self.L.ora_count_flops_part(self.h, U.ctypes.data, int(what), _dp(out)) == 0
        return out

    def metrics(self, axis):
        n = self.case.n[axis] + 6
        d, c = np.zeros(n), np.zeros(n)
        assert self.L.ora_metrics(self.h, axis, _dp(d), _dp(c)) == 0
        return d, c

    def metrics_index(self, axis):
        n = self.case.n[axis] + 6
        Xc, Xf = np.zeros(n), np.zeros(n)
        assert self.L.ora_metrics_index(self.h, axis, _dp(Xc), _dp(Xf)) == 0
        return Xc, Xf

    def viscous_face(self, U, d, i, j, k):
        self._chk(U)
        F = np.zeros(5)
        assert self.L.ora_viscous_face(self.h, U.ctypes.data, d, i, j, k, _dp(F)) == 0
        return F


def run_case(case, dtype="f64", n_steps=None, log=None, variant="ref", dts_in=None):
    """Advance a case with the oracle exactly as the drivers do: fixed dt x n_steps, or CFL steps
    (clipped to t_end when given).  Returns (U, list of dt).  dts_in: take these time steps instead
    (the arbiter run "f80" is fed the fp64 oracle's own sequence, so that the two differ by the
    rounding of the scheme's arithmetic only)."""
    o = Oracle(case, dtype, variant)
    if dts_in is not None:
        U = o.state()
        for step, dt in enumerate(dts_in):
            o.rk3_step(U, dt)
            if log:
                log(step + 1, None, dt)
        return U, list(dts_in)
    U = o.state()
    dts, t = [], 0.0
    n = n_steps if n_steps is not None else case.n_steps
    step = 0
    while True:
        if n is not None and step >= n:
            break
        if case.t_end is not None and t >= case.t_end * (1 - 1e-14):
            break
        if case.dt is not None:
            dt = case.dt
        else:
            st, dt = o.cfl_dt(U, case.cfl)
            assert st == 0, f"oracle cfl_dt status {st} at step {step}"
            if case.t_end is not None:
                dt = min(dt, case.t_end - t)
        o.rk3_step(U, dt)
        t += dt
        dts.append(dt)
        step += 1
        if log:
            log(step, t, dt)
    return U, dts


# ---- unit-level helpers for the pins
def weno5(v):
    v = _arr(v, 5)
    return lib().ora_weno5(_dp(v))


def weno5_detail(v):
    v = _arr(v, 5)
    b, w, p = np.zeros(3), np.zeros(3), np.zeros(3)
    lib().ora_weno5_detail(_dp(v), _dp(b), _dp(w), _dp(p))
    return b, w, p


def hllc(d, gamma, WL, WR):
    WL, WR, F = _arr(WL, 5), _arr(WR, 5), np.zeros(5)
    lib().ora_hllc(d, gamma, _dp(WL), _dp(WR), _dp(F))
    return F


def flux_phys(d, gamma, W):
    W, F = _arr(W, 5), np.zeros(5)
    lib().ora_flux_phys(d, gamma, _dp(W), _dp(F))
    return F


def cons_to_prim(gamma, U):
    U, W = _arr(U, 5), np.zeros(5)
    lib().ora_cons_to_prim(gamma, _dp(U), _dp(W))
    return W


def prim_to_cons(gamma, W):
    W, U = _arr(W, 5), np.zeros(5)
    lib().ora_prim_to_cons(gamma, _dp(W), _dp(U))
    return U


def viscosity(mu, T):
    m = MuLaw(int(mu["sutherland"]), mu["mu_ref"], mu["T_ref"], mu["S"])
    return lib().ora_viscosity(C.byref(m), float(T))


def dc(phi, Xc):
    return lib().ora_dc(_dp(_arr(phi, 5)), float(Xc))


def df(phi, Xf):
    return lib().ora_df(_dp(_arr(phi, 4)), float(Xf))


def iface(phi):
    return lib().ora_if(_dp(_arr(phi, 4)))


def dc6(phi, Xc):
    return lib().ora_dc6(_dp(_arr(phi, 7)), float(Xc))


def df6(phi, Xf):
    return lib().ora_df6(_dp(_arr(phi, 6)), float(Xf))


def iface6(phi):
    return lib().ora_if6(_dp(_arr(phi, 6)))
