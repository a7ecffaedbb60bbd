"""Thin ctypes binding of libjf.so (include/jf.h): same names, argument marshalling only.

PyTorch is used for device memory and streams; every step of the path runs in the CUDA
kernels.  There is no CPU fallback: if libjf.so is missing or no CUDA device is present the
calls fail loudly.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# JF_LIB: load another build of the same library (e.g. one compiled with different tuning macros)
LIB_PATH = os.environ.get("JF_LIB") or os.path.join(_HERE, "libjf.so")

JF_OK, JF_EINVAL, JF_EALIGN, JF_EWORKSPACE, JF_ECUDA, JF_ENOTFINITE = range(6)
JF_F64, JF_F32, JF_F64_TANGENT = 0, 1, 2
_DTYPES = {"f64": JF_F64, "f32": JF_F32, "f64t": JF_F64_TANGENT}
_STATUS = {0: "JF_OK", 1: "JF_EINVAL", 2: "JF_EALIGN", 3: "JF_EWORKSPACE", 4: "JF_ECUDA", 5: "JF_ENOTFINITE"}

c_double_p = C.POINTER(C.c_double)


class jf_grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("xf", c_double_p), ("yf", c_double_p), ("zf", c_double_p)]


class jf_mu_law(C.Structure):
    _fields_ = [("sutherland", C.c_int), ("mu_ref", C.c_double), ("T_ref", C.c_double), ("S", C.c_double)]


class jf_disturbance(C.Structure):
    _fields_ = [("enabled", C.c_int), ("A", C.c_double), ("kappa", C.c_double),
                ("t1_lo", C.c_double), ("t1_hi", C.c_double)]


class jf_bc_face(C.Structure):
    _fields_ = [("type", C.c_int), ("T_wall", C.c_double), ("u_wall", C.c_double * 3),
                ("dirichlet", c_double_p), ("dist", jf_disturbance), ("nb_width", C.c_double * 3),
                ("nb_has_face", C.c_int), ("nb_face", C.c_double * 3)]


class jf_bc(C.Structure):
    _fields_ = [("face", jf_bc_face * 6)]


EXPORTS = ["jf_workspace_bytes", "jf_create", "jf_destroy", "jf_state_elems", "jf_fill_halo", "jf_rhs",
           "jf_rk3_step", "jf_cfl_dt", "jf_cfl_dt_dev", "jf_rk3_step_dev", "jf_dev_time", "jf_set_visc_order", "jf_set_tangent_seed", "jf_fill_halo_axis", "jf_face_elems", "jf_pack_face",
           "jf_unpack_face", "jf_pull_face", "jf_rk3_stage_input", "jf_rk3_stage_advance", "jf_plane_sums", "jf_plane_sums_static", "jf_plane_sums_static_max_planes", "jf_last_error", "jf_launch_count", "jf_diag_alu_peak", "jf_diag_timing",
           "jf_diag_kernel_times", "jf_diag_kernel_name", "jf_diag_face_flux", "jf_diag_metrics", "jf_version"]

_lib = None


class JFError(RuntimeError):
    def __init__(self, status, msg=""):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


def lib():
    """Load libjf.so (raises if it has not been built: no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(f"{LIB_PATH} not built; run `python -m paper_2406_19494_b200.build`")
        L = C.CDLL(LIB_PATH)
        L.jf_workspace_bytes.restype = C.c_size_t
        L.jf_workspace_bytes.argtypes = [C.POINTER(jf_grid), C.c_int]
        L.jf_create.restype = C.c_int
        L.jf_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(jf_grid), C.c_int, C.c_double, C.c_double,
                                C.c_double, C.POINTER(jf_mu_law), C.POINTER(jf_bc), c_double_p, C.c_void_p,
                                C.c_size_t, C.c_void_p]
        L.jf_destroy.restype = C.c_int
        L.jf_destroy.argtypes = [C.c_void_p]
        L.jf_state_elems.restype = C.c_size_t
        L.jf_state_elems.argtypes = [C.c_void_p]
        L.jf_fill_halo.restype = C.c_int
        L.jf_fill_halo.argtypes = [C.c_void_p, C.c_void_p]
        L.jf_rhs.restype = C.c_int
        L.jf_rhs.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.jf_fill_halo_axis.restype = C.c_int
        L.jf_fill_halo_axis.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.jf_face_elems.restype = C.c_size_t
        L.jf_face_elems.argtypes = [C.c_void_p, C.c_int]
        L.jf_pack_face.restype = C.c_int
        L.jf_pack_face.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.jf_unpack_face.restype = C.c_int
        L.jf_unpack_face.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.jf_pull_face.restype = C.c_int
        L.jf_pull_face.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.POINTER(C.c_int)]
        L.jf_rk3_stage_input.restype = C.c_void_p
        L.jf_rk3_stage_input.argtypes = [C.c_void_p, C.c_void_p, C.c_int]
        L.jf_rk3_stage_advance.restype = C.c_int
        L.jf_rk3_stage_advance.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_double]
        L.jf_plane_sums.restype = C.c_int
        L.jf_plane_sums.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.jf_plane_sums_static.restype = C.c_int
        L.jf_plane_sums_static.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]
        L.jf_plane_sums_static_max_planes.restype = C.c_int
        L.jf_plane_sums_static_max_planes.argtypes = []
        L.jf_set_tangent_seed.restype = C.c_int
        L.jf_set_tangent_seed.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.jf_rk3_step.restype = C.c_int
        L.jf_rk3_step.argtypes = [C.c_void_p, C.c_void_p, C.c_double]
        L.jf_cfl_dt.restype = C.c_int
        L.jf_cfl_dt.argtypes = [C.c_void_p, C.c_void_p, C.c_double, c_double_p]
        L.jf_cfl_dt_dev.restype = C.c_int
        L.jf_cfl_dt_dev.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double]
        L.jf_rk3_step_dev.restype = C.c_int
        L.jf_rk3_step_dev.argtypes = [C.c_void_p, C.c_void_p]
        L.jf_dev_time.restype = C.c_int
        L.jf_dev_time.argtypes = [C.c_void_p, C.c_int, c_double_p, c_double_p]
        L.jf_set_visc_order.restype = C.c_int
        L.jf_set_visc_order.argtypes = [C.c_void_p, C.c_int]
        L.jf_last_error.restype = C.c_char_p
        L.jf_last_error.argtypes = [C.c_void_p]
        L.jf_launch_count.restype = C.c_ulonglong
        L.jf_launch_count.argtypes = [C.c_void_p]
        L.jf_diag_alu_peak.restype = C.c_int
        L.jf_diag_alu_peak.argtypes = [C.c_int, C.c_int, c_double_p, c_double_p]
        L.jf_diag_timing.restype = C.c_int
        L.jf_diag_timing.argtypes = [C.c_void_p, C.c_int]
        L.jf_diag_kernel_times.restype = C.c_int
        L.jf_diag_kernel_times.argtypes = [C.c_void_p, c_double_p, C.POINTER(C.c_ulonglong)]
        L.jf_diag_kernel_name.restype = C.c_char_p
        L.jf_diag_kernel_name.argtypes = [C.c_int]
        L.jf_diag_face_flux.restype = C.c_int
        L.jf_diag_face_flux.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.POINTER(jf_mu_law),
                                        C.c_int, c_double_p, c_double_p, c_double_p, c_double_p]
        L.jf_diag_metrics.restype = C.c_int
        L.jf_diag_metrics.argtypes = [C.c_void_p, C.c_int, c_double_p, c_double_p, c_double_p, c_double_p]
        L.jf_version.restype = C.c_char_p
        L.jf_version.argtypes = []
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(c_double_p)


def _grid_struct(case, keep):
    nx, ny, nz = case.n
    arrs = [np.ascontiguousarray(np.asarray(f, dtype=np.float64)) for f in (case.xf, case.yf, case.zf)]
    keep += arrs
    return jf_grid(nx, ny, nz, _dp(arrs[0]), _dp(arrs[1]), _dp(arrs[2]))


def jf_version():
    return lib().jf_version().decode()


def jf_diag_alu_peak(dtype="f64", iters=4096):
    fl, ms = C.c_double(), C.c_double()
    st = lib().jf_diag_alu_peak(JF_F64 if dtype == "f64" else JF_F32, iters, C.byref(fl), C.byref(ms))
    if st != JF_OK:
        raise JFError(st, "jf_diag_alu_peak")
    return fl.value, ms.value


def jf_diag_face_flux(dtype, d, gamma, R_gas, Pr, mu, W, Gt=None, Xf=None):
    """F[n,5] = total face flux of n faces from W[n,6,6], Gt[n,4,4], Xf[n] (host numpy arrays)."""
    W = np.ascontiguousarray(W, dtype=np.float64)
    n = W.shape[0]
    assert W.shape == (n, 6, 6)
    Gt = None if Gt is None else np.ascontiguousarray(Gt, dtype=np.float64)
    Xf = None if Xf is None else np.ascontiguousarray(Xf, dtype=np.float64)
    F = np.zeros((n, 5))
    m = jf_mu_law(int(mu["sutherland"]), mu["mu_ref"], mu["T_ref"], mu["S"])
    st = lib().jf_diag_face_flux(JF_F64 if dtype == "f64" else JF_F32, d, gamma, R_gas, Pr, C.byref(m), n, _dp(W),
                                 None if Gt is None else _dp(Gt), None if Xf is None else _dp(Xf), _dp(F))
    if st != JF_OK:
        raise JFError(st, "jf_diag_face_flux")
    return F


class Solver:
    """jf_solver handle + its device workspace, built from a cases.Case description.

    Methods carry the names of the C calls; tensors are torch CUDA tensors of the solver dtype
    and shape [5, nz+6, ny+6, nx+6]; dtype "f64t" (JF_F64_TANGENT) adds a trailing axis of 2:
    [..., 0] value, [..., 1] tangent."""

    def __init__(self, case, dtype="f64", device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise JFError(JF_ECUDA, "no CUDA device: libjf has no CPU fallback")
        self.torch = torch
        self.case = case
        self.device = torch.device(device)
        self.dtype = dtype
        self.tdtype = torch.float32 if dtype == "f32" else torch.float64
        self._keep = []
        L = lib()
        g = _grid_struct(case, self._keep)
        dt = _DTYPES[dtype]
        nbytes = L.jf_workspace_bytes(C.byref(g), dt)
        if nbytes == 0:
            raise JFError(JF_EINVAL, "jf_workspace_bytes")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        ws_ptr = (base + 255) // 256 * 256
        mu = jf_mu_law(int(case.mu["sutherland"]), case.mu["mu_ref"], case.mu["T_ref"], case.mu["S"])
        bc = jf_bc()
        for f, fb in enumerate(case.bc):
            b = bc.face[f]
            b.type = int(fb.type)
            b.T_wall = float(fb.T_wall)
            for d in range(3):
                b.u_wall[d] = float(fb.u_wall[d])
            if fb.dirichlet is not None:
                t = np.ascontiguousarray(np.asarray(fb.dirichlet, dtype=np.float64))
                self._keep.append(t)
                b.dirichlet = _dp(t)
            if fb.dist is not None:
                b.dist = jf_disturbance(1, fb.dist["A"], fb.dist["kappa"], fb.dist["t1_lo"], fb.dist["t1_hi"])
            if getattr(fb, "nb_width", None) is not None:
                for d in range(3):
                    b.nb_width[d] = float(fb.nb_width[d])
            if getattr(fb, "nb_face", None) is not None:
                b.nb_has_face = 1
                for d in range(3):
                    b.nb_face[d] = float(fb.nb_face[d])
        ga = np.asarray(case.body_accel, dtype=np.float64)
        self._keep.append(ga)
        self.stream = stream
        sptr = C.c_void_p(stream.cuda_stream) if stream is not None else C.c_void_p(
            torch.cuda.current_stream(self.device).cuda_stream)
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            st = L.jf_create(C.byref(h), C.byref(g), dt, case.gamma, case.R_gas, case.Pr, C.byref(mu),
                             C.byref(bc), _dp(ga), C.c_void_p(ws_ptr), nbytes, sptr)
        if st != JF_OK:
            raise JFError(st, "jf_create")
        self.h = h
        if getattr(case, "visc_order", 4) != 4:
            self._check(L.jf_set_visc_order(h, int(case.visc_order)))
        nx, ny, nz = case.n
        self.shape = (5, nz + 6, ny + 6, nx + 6)
        assert L.jf_state_elems(h) == int(np.prod(self.shape))
        if dtype == "f64t":
            self.shape = self.shape + (2,)

    def close(self):
        if getattr(self, "h", None):
            lib().jf_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st):
        if st != JF_OK:
            raise JFError(st, lib().jf_last_error(self.h).decode())

    def _ptr(self, t):
        assert t.is_cuda and t.dtype == self.tdtype and t.is_contiguous() and tuple(t.shape) == self.shape
        return C.c_void_p(t.data_ptr())

    def state(self, U0=None, dU0=None):
        """Device copy of a host state array (case.U0 by default); tangent solvers interleave
        (value, tangent) with the tangent dU0 (zero by default)."""
        U = np.asarray(self.case.U0 if U0 is None else U0)
        if self.dtype == "f64t":
            dU = np.zeros_like(U) if dU0 is None else np.asarray(dU0)
            U = np.stack([U, dU], axis=-1)
        return self.torch.as_tensor(U, dtype=self.tdtype).contiguous().to(self.device)

    # ---- block decomposition (include/jf.h "Block decomposition"); pointers are raw device addresses
    def jf_fill_halo_axis(self, U_ptr, axis):
        self._check(lib().jf_fill_halo_axis(self.h, C.c_void_p(U_ptr), int(axis)))

    def jf_face_elems(self, face):
        return int(lib().jf_face_elems(self.h, int(face)))

    def jf_pack_face(self, U_ptr, face, buf):
        self._check(lib().jf_pack_face(self.h, C.c_void_p(U_ptr), int(face), C.c_void_p(buf.data_ptr())))

    def jf_unpack_face(self, U_ptr, face, buf):
        self._check(lib().jf_unpack_face(self.h, C.c_void_p(U_ptr), int(face), C.c_void_p(buf.data_ptr())))

    def jf_pull_face(self, U_ptr, face, peer_ptr, n_peer):
        n = (C.c_int * 3)(*[int(v) for v in n_peer])
        self._check(lib().jf_pull_face(self.h, C.c_void_p(U_ptr), int(face), C.c_void_p(peer_ptr), n))

    def jf_rk3_stage_input(self, U, stage):
        p = lib().jf_rk3_stage_input(self.h, self._ptr(U), int(stage))
        if not p:
            raise JFError(JF_EINVAL, "jf_rk3_stage_input")
        return int(p)

    def jf_rk3_stage_advance(self, U, stage, dt):
        self._check(lib().jf_rk3_stage_advance(self.h, self._ptr(U), int(stage), float(dt)))

    def jf_plane_sums(self, U, axis):
        """[JF_NSTATS = 14][n_axis] float64 device tensor of the area-weighted plane sums (include/jf.h)."""
        out = self.torch.empty((14, self.case.n[axis]), dtype=self.torch.float64, device=self.device)
        self._check(lib().jf_plane_sums(self.h, self._ptr(U), int(axis), C.c_void_p(out.data_ptr())))
        return out

    def jf_plane_sums_static(self, U, axis, out=None):
        """jf_plane_sums through the library's static scratch array (allocation-free entry point, include/jf.h);
        `out`: a preallocated [14, n_axis] float64 device tensor (allocated here if None)."""
        if out is None:
            out = self.torch.empty((14, self.case.n[axis]), dtype=self.torch.float64, device=self.device)
        self._check(lib().jf_plane_sums_static(self.h, self._ptr(U), int(axis), C.c_void_p(out.data_ptr())))
        return out

    def jf_set_visc_order(self, order):
        self._check(lib().jf_set_visc_order(self.h, int(order)))

    def jf_set_tangent_seed(self, dA, dkappa):
        self._check(lib().jf_set_tangent_seed(self.h, float(dA), float(dkappa)))

    def jf_fill_halo(self, U):
        self._check(lib().jf_fill_halo(self.h, self._ptr(U)))
        return U

    def jf_rhs(self, U, R=None):
        if R is None:
            R = self.torch.zeros_like(U)
        self._check(lib().jf_rhs(self.h, self._ptr(U), self._ptr(R)))
        return R

    def jf_rk3_step(self, U, dt):
        self._check(lib().jf_rk3_step(self.h, self._ptr(U), float(dt)))
        return U

    def jf_cfl_dt(self, U, cfl):
        dt = C.c_double()
        st = lib().jf_cfl_dt(self.h, self._ptr(U), float(cfl), C.byref(dt))
        return st, dt.value

    def jf_cfl_dt_dev(self, U, cfl, t_end=None):
        self._check(lib().jf_cfl_dt_dev(self.h, self._ptr(U), float(cfl), float("nan") if t_end is None else float(t_end)))

    def jf_rk3_step_dev(self, U):
        self._check(lib().jf_rk3_step_dev(self.h, self._ptr(U)))
        return U

    def jf_dev_time(self, set_t=None):
        """(status, dt, t) of the device-side clock (synchronises); set_t: reset the clock to that time first."""
        dt, t = C.c_double(), C.c_double()
        if set_t is not None:
            t.value = float(set_t)
            self._check(lib().jf_dev_time(self.h, 1, None, C.byref(t)))
        st = lib().jf_dev_time(self.h, 0, C.byref(dt), C.byref(t))
        return st, dt.value, t.value

    def jf_diag_timing(self, enable):
        self._check(lib().jf_diag_timing(self.h, int(bool(enable))))

    def jf_diag_kernel_times(self):
        """{kernel class name: (total ms, launches)} since the previous call (synchronises)."""
        ms = (C.c_double * 6)()
        n = (C.c_ulonglong * 6)()
        self._check(lib().jf_diag_kernel_times(self.h, ms, n))
        return {lib().jf_diag_kernel_name(k).decode(): (ms[k], int(n[k])) for k in range(6)}

    def jf_diag_metrics(self, axis):
        """(1/Delta, centre, 1/(12 X_xi^c), 1/(24 X_xi^f)) of one axis as the kernels read them (padded arrays)."""
        out = [np.zeros(self.case.n[axis] + 6) for _ in range(4)]
        self._check(lib().jf_diag_metrics(self.h, int(axis), *[_dp(a) for a in out]))
        return out

    def jf_launch_count(self):
        return int(lib().jf_launch_count(self.h))


def run_case(case, dtype="f64", n_steps=None, device="cuda:0", solver=None, device_dt=False):
    """Advance a case on the GPU the way the drivers do (mirror of the oracle-side driver in
    tests): fixed dt x n_steps, or CFL steps clipped to t_end.  Returns (U tensor, list of dt).
    device_dt: CFL-driven cases take jf_cfl_dt_dev + jf_rk3_step_dev (the step never leaves the device);
    dt is read back after each step only to report it and to detect t_end."""
    s = solver or Solver(case, dtype, device)
    U = s.state()
    dts, t, step = [], 0.0, 0
    n = n_steps if n_steps is not None else case.n_steps
    if device_dt and case.dt is None:
        s.jf_dev_time(set_t=0.0)
        while True:
            if n is not None and step >= n:
                break
            if case.t_end is not None and t >= case.t_end * (1 - 1e-14):
                break
            s.jf_cfl_dt_dev(U, case.cfl, case.t_end)
            s.jf_rk3_step_dev(U)
            st, dt, t = s.jf_dev_time()
            if st != JF_OK:
                raise JFError(st, f"jf_cfl_dt_dev at step {step}")
            dts.append(dt)
            step += 1
        return U, dts
    while True:
        if n is not None and step >= n:
            break
        if case.t_end is not None and t >= case.t_end * (1 - 1e-14):
            break
        if case.dt is not None:
            dt = case.dt
        else:
            st, dt = s.jf_cfl_dt(U, case.cfl)
            if st != JF_OK:
                raise JFError(st, f"jf_cfl_dt at step {step}")
            if case.t_end is not None:
                dt = min(dt, case.t_end - t)
        s.jf_rk3_step(U, dt)
        t += dt
        dts.append(dt)
        step += 1
    return U, dts
