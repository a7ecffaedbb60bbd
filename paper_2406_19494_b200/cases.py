"""Seeded synthetic inputs for the five BASELINE.json configs (and the parity/edge cases).

This module serves BOTH the CPU oracle (oracle/) and the CUDA library: it only builds input
arrays (grids, boundary tables, initial conservative fields) with numpy and holds none of the
method's arithmetic (no reconstruction, flux, halo fill, time stepping).  Recipes follow
SURVEY.md §8(d); each one is restated in DESIGN.md.  Nothing here reads /root/reference.

Layout of every state array: U[5][nz+6][ny+6][nx+6] (Nh = 3), float64, halos 0.
"""
from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

NH = 3
BC_PERIODIC, BC_ZEROGRAD, BC_DIRICHLET, BC_WALL_ISOTHERMAL, BC_WALL_ADIABATIC, BC_EXCHANGE = range(6)


@dataclass
class FaceBC:
    type: int = BC_PERIODIC
    T_wall: float = 0.0
    u_wall: tuple = (0.0, 0.0, 0.0)
    dirichlet: Optional[np.ndarray] = None   # prim[5][n_t2][n_t1] (rho,u,v,w,p)
    dist: Optional[dict] = None              # {"A","kappa","t1_lo","t1_hi"}  (Eq. 8)
    nb_width: Optional[tuple] = None         # BC_EXCHANGE: widths of the neighbour block's 3 nearest cells
    nb_face: Optional[tuple] = None          # BC_EXCHANGE across an interior cut: the neighbour's 3 faces beyond this one


@dataclass
class Case:
    name: str
    n: tuple                                  # (nx, ny, nz)
    xf: np.ndarray
    yf: np.ndarray
    zf: np.ndarray
    gamma: float
    R_gas: float
    Pr: float
    mu: dict                                  # {"sutherland","mu_ref","T_ref","S"}
    bc: List[FaceBC]                          # x-, x+, y-, y+, z-, z+
    U0: np.ndarray                            # [5, nz+6, ny+6, nx+6] float64
    body_accel: tuple = (0.0, 0.0, 0.0)
    dt: Optional[float] = None                # fixed dt, or
    cfl: Optional[float] = None               # CFL number (jf_cfl_dt each step)
    n_steps: Optional[int] = None
    t_end: Optional[float] = None
    notes: dict = field(default_factory=dict)
    visc_order: int = 4                       # central dissipative-flux stencils: 4 (north_star) or 6

    @property
    def cells(self):
        return self.n[0] * self.n[1] * self.n[2]


def uniform_faces(lo, hi, n):
    return lo + (hi - lo) * np.arange(n + 1, dtype=np.float64) / n


def centres(f):
    return 0.5 * (f[:-1] + f[1:])


def empty_state(n):
    nx, ny, nz = n
    return np.zeros((5, nz + 2 * NH, ny + 2 * NH, nx + 2 * NH), dtype=np.float64)


def set_interior_from_prim(U, gamma, rho, u, v, w, p):
    """Write interior cells of U from primitive fields shaped [nz, ny, nx] (input preparation:
    Eq. 2)."""
    s = (slice(NH, -NH),) * 3
    U[0][s] = rho
    U[1][s] = rho * u
    U[2][s] = rho * v
    U[3][s] = rho * w
    U[4][s] = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return U


def periodic_bc():
    return [FaceBC(BC_PERIODIC) for _ in range(6)]


# ------------------------------------------------------------------ config 0 / 4: Taylor-Green
def tgv(n=32, dt=1e-3, n_steps=10, faces=None):
    """Taylor-Green vortex, periodic [0,2pi]^3, gamma=1.4, Pr=0.71, M=0.1, Re=1600, constant mu
    (BASELINE.json configs[0], configs[4]).  faces = (xf, yf, zf): the same field on another
    box (the field has period 2 pi along every axis: a block of a [0, 2 pi S]^3 box for the decomposition bench)."""
    gamma, M, Re = 1.4, 0.1, 1600.0
    p0 = 1.0 / (gamma * M * M)
    R = p0                       # rho0 = T0 = 1
    if faces is not None:
        fx, fy, fz = (np.asarray(a, dtype=np.float64) for a in faces)
        nn = (len(fx) - 1, len(fy) - 1, len(fz) - 1)
        Z, Y, X = np.meshgrid(centres(fz), centres(fy), centres(fx), indexing="ij")
        u = np.sin(X) * np.cos(Y) * np.cos(Z)
        v = -np.cos(X) * np.sin(Y) * np.cos(Z)
        p = p0 + (1.0 / 16.0) * (np.cos(2 * X) + np.cos(2 * Y)) * (np.cos(2 * Z) + 2.0)
        U = set_interior_from_prim(empty_state(nn), gamma, p / R, u, v, np.zeros_like(u), p)
        return Case(name=f"tgv{nn[0]}x{nn[1]}x{nn[2]}", n=nn, xf=fx, yf=fy, zf=fz, gamma=gamma, R_gas=R,
                    Pr=0.71, mu={"sutherland": 0, "mu_ref": 1.0 / Re, "T_ref": 1.0, "S": 0.0},
                    bc=periodic_bc(), U0=U, dt=dt, n_steps=n_steps)
    f = uniform_faces(0.0, 2.0 * np.pi, n)
    c = centres(f)
    Z, Y, X = np.meshgrid(c, c, c, indexing="ij")
    u = np.sin(X) * np.cos(Y) * np.cos(Z)
    v = -np.cos(X) * np.sin(Y) * np.cos(Z)
    w = np.zeros_like(u)
    p = p0 + (1.0 / 16.0) * (np.cos(2 * X) + np.cos(2 * Y)) * (np.cos(2 * Z) + 2.0)
    rho = p / (R * 1.0)
    U = set_interior_from_prim(empty_state((n, n, n)), gamma, rho, u, v, w, p)
    return Case(name=f"tgv{n}", n=(n, n, n), xf=f, yf=f.copy(), zf=f.copy(), gamma=gamma, R_gas=R,
                Pr=0.71, mu={"sutherland": 0, "mu_ref": 1.0 / Re, "T_ref": 1.0, "S": 0.0},
                bc=periodic_bc(), U0=U, dt=dt, n_steps=n_steps)


# ------------------------------------------------------------------ config 1: Sod
def sod(nx=256, ny=4, nz=4, axis=0):
    """Sod shock tube as a 3-D grid nx x 4 x 4, x in [0,1], cubic cells, inviscid, zero-gradient
    in x, periodic in y/z, CFL 0.5 to t = 0.2 (BASELINE.json configs[1]).  axis != 0 rotates the
    tube onto y or z (for the axis tests)."""
    gamma = 1.4
    n = [ny, ny, ny]
    n[axis] = nx
    if axis == 0:
        n = [nx, ny, nz]
    h = 1.0 / nx
    faces = [uniform_faces(0.0, n[a] * h, n[a]) for a in range(3)]
    cs = [centres(f) for f in faces]
    Z, Y, X = np.meshgrid(cs[2], cs[1], cs[0], indexing="ij")
    s = (X, Y, Z)[axis]
    left = s < 0.5
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    zero = np.zeros_like(rho)
    U = set_interior_from_prim(empty_state(tuple(n)), gamma, rho, zero, zero, zero, p)
    bc = periodic_bc()
    bc[2 * axis] = FaceBC(BC_ZEROGRAD)
    bc[2 * axis + 1] = FaceBC(BC_ZEROGRAD)
    return Case(name=f"sod{nx}", n=tuple(n), xf=faces[0], yf=faces[1], zf=faces[2], gamma=gamma,
                R_gas=1.0, Pr=0.72, mu={"sutherland": 0, "mu_ref": 0.0, "T_ref": 1.0, "S": 0.0},
                bc=bc, U0=U, cfl=0.5, t_end=0.2)


# ------------------------------------------------------------------ seeded noise (counter based)
def splitmix64(x):
    """splitmix64 finaliser on uint64 counters (vectorised)."""
    x = (x + np.uint64(0x9E3779B97F4A7C15)).astype(np.uint64)
    z = x
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def uniform_pm1(seed, counters):
    """i.i.d. uniform in [-1, 1) from splitmix64(seed xor counter)."""
    with np.errstate(over="ignore"):
        z = splitmix64(np.uint64(seed) ^ counters.astype(np.uint64))
    return (z >> np.uint64(11)).astype(np.float64) * (2.0 ** -53) * 2.0 - 1.0


def tanh_faces_two_sided(n, beta, L=2.0):
    """y_f = L/2 * (1 + tanh(beta (2j/n - 1))/tanh(beta)): clustered at both walls."""
    j = np.arange(n + 1, dtype=np.float64)
    f = 0.5 * L * (1.0 + np.tanh(beta * (2.0 * j / n - 1.0)) / np.tanh(beta))
    f[0], f[-1] = 0.0, L
    return f


def tanh_faces_one_sided(n, beta, L):
    """y_f = L (1 + tanh(beta (j/n - 1))/tanh(beta)): clustered at y = 0."""
    j = np.arange(n + 1, dtype=np.float64)
    f = L * (1.0 + np.tanh(beta * (j / n - 1.0)) / np.tanh(beta))
    f[0], f[-1] = 0.0, L
    return f


# ------------------------------------------------------------------ config 2: channel
def channel(nx=192, ny=128, nz=128, seed=20240619, cfl=0.5, n_steps=100, noise=0.1):
    """Compressible channel, 4pi x 2 x 4pi/3, tanh wall-normal stretching beta = 2.0, M_b = 1.5,
    Re_b = 3000, isothermal no-slip walls T_w = 1, Sutherland, gamma = 1.4, Pr = 0.72, laminar
    Poiseuille + seeded uniform noise of 10 % U_b, constant body force (BASELINE.json configs[2];
    stands in for the paper's channel DNS set-up)."""
    gamma, Mb, Reb = 1.4, 1.5, 3000.0
    R = 1.0 / (gamma * Mb * Mb)
    xf = uniform_faces(0.0, 4.0 * np.pi, nx)
    yf = tanh_faces_two_sided(ny, 2.0, 2.0)
    zf = uniform_faces(0.0, 4.0 * np.pi / 3.0, nz)
    yc = centres(yf)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    lin = ((k * ny + j) * nx + i).astype(np.uint64)
    r1 = uniform_pm1(seed, np.uint64(3) * lin + np.uint64(0))
    r2 = uniform_pm1(seed, np.uint64(3) * lin + np.uint64(1))
    r3 = uniform_pm1(seed, np.uint64(3) * lin + np.uint64(2))
    Y = yc[None, :, None]
    u = 1.5 * (1.0 - (Y - 1.0) ** 2) + noise * r1
    v = noise * r2
    w = noise * r3
    rho = np.ones_like(u)
    p = np.full_like(u, R)      # T = 1
    U = set_interior_from_prim(empty_state((nx, ny, nz)), gamma, rho, u, v, w, p)
    mu_w = 1.0 / Reb
    bc = periodic_bc()
    bc[2] = FaceBC(BC_WALL_ISOTHERMAL, T_wall=1.0)
    bc[3] = FaceBC(BC_WALL_ISOTHERMAL, T_wall=1.0)
    return Case(name=f"channel{nx}x{ny}x{nz}", n=(nx, ny, nz), xf=xf, yf=yf, zf=zf, gamma=gamma,
                R_gas=R, Pr=0.72, mu={"sutherland": 1, "mu_ref": mu_w, "T_ref": 1.0, "S": 0.4},
                bc=bc, U0=U, body_accel=(3.0 * mu_w, 0.0, 0.0), cfl=cfl, n_steps=n_steps)


# ------------------------------------------------------------------ config 3: Mach-6 flat plate
def _sutherland(T, mu_ref, T_ref, S):
    return mu_ref * (T / T_ref) ** 1.5 * (T_ref + S) / (T + S)


def blasius_compressible(M, Pr, gamma, T_inf, Tw_over_Tinf, mu_law, eta_max=8.0, n_eta=1601):
    """Compressible Blasius similarity solve (Eq. 7): (C f'')' + f f'' = 0,
    (C g'/Pr)' + f g' + C (gamma-1) M^2 f''^2 = 0, C = rho mu/(rho_e mu_e), f(0)=f'(0)=0,
    g(0)=T_w/T_inf (isothermal wall) or, with Tw_over_Tinf=None, g'(0)=0 (adiabatic wall, g(0) found),
    f'(inf)=g(inf)=1; RK4 + damped-Newton shooting.  Input generation only."""
    adiabatic = Tw_over_Tinf is None
    mu_e = _sutherland(T_inf, **mu_law)

    def Cfun(g):
        return _sutherland(g * T_inf, **mu_law) / mu_e / g

    def deriv(y):
        f, fp, s, g, h = y
        C = Cfun(g)
        return np.array([fp, s / C, -f * s / C, Pr * h / C,
                         -f * Pr * h / C - (gamma - 1.0) * M * M * s * s / C])

    eta = np.linspace(0.0, eta_max, n_eta)
    d = eta[1] - eta[0]

    def integrate(a, b):
        # unknowns: a = C f''(0) and b = (C/Pr) g'(0) (isothermal) or b = g(0) (adiabatic)
        y = np.array([0.0, 0.0, a, b, 0.0]) if adiabatic else np.array([0.0, 0.0, a, Tw_over_Tinf, b])
        out = np.empty((n_eta, 5))
        out[0] = y
        for n in range(1, n_eta):
            k1 = deriv(y); k2 = deriv(y + 0.5 * d * k1); k3 = deriv(y + 0.5 * d * k2); k4 = deriv(y + d * k3)
            y = y + d / 6.0 * (k1 + 2 * k2 + 2 * k3 + k4)
            out[n] = y
        return out

    def resid(a, b):
        o = integrate(a, b)
        return np.array([o[-1, 1] - 1.0, o[-1, 3] - 1.0])

    x = np.array([0.5, 1.0 + 0.5 * np.sqrt(Pr) * (gamma - 1.0) * M * M]) if adiabatic else np.array([0.5, 4.0])
    r = resid(*x)
    for _ in range(60):
        if np.max(np.abs(r)) < 1e-11:
            break
        J = np.empty((2, 2))
        for c in range(2):
            e = np.zeros(2); e[c] = 1e-6 * max(1.0, abs(x[c]))
            J[:, c] = (resid(*(x + e)) - r) / e[c]
        step = np.linalg.solve(J, -r)
        lam = 1.0
        while lam > 1e-4:
            xn = x + lam * step
            with np.errstate(all="ignore"):
                rn = resid(*xn) if xn[0] > 0 and (not adiabatic or xn[1] > 0) else np.array([np.inf, np.inf])
            if np.all(np.isfinite(rn)) and np.linalg.norm(rn) < np.linalg.norm(r):
                break
            lam *= 0.5
        x, r = xn, rn
    o = integrate(*x)
    return {"eta": eta, "fp": o[:, 1], "g": o[:, 3], "s0": x[0], "h0": x[1], "resid": r}


def flat_plate(nx=512, ny=192, nz=8, cfl=0.5, n_steps=200, A_frac=0.01, disturbance=True):
    """Mach-6 laminar flat-plate boundary layer with the paper's disturbance ("porous") wall on
    x in [0.05, 0.15] (Eq. 8), isothermal wall elsewhere, Blasius-type
    supersonic inflow, zero-gradient outflow/top, spanwise periodic (BASELINE.json configs[3])."""
    gamma, Rg, Pr = 1.4, 287.058, 0.72
    mu_law = {"mu_ref": 1.716e-5, "T_ref": 273.15, "S": 110.4}
    T_inf, M, Re_unit, T_w = 220.0, 6.0, 1.0e7, 300.0
    u_inf = M * np.sqrt(gamma * Rg * T_inf)
    mu_e = _sutherland(T_inf, **mu_law)
    rho_inf = Re_unit * mu_e / u_inf
    p_inf = rho_inf * Rg * T_inf
    Lx, Ly = 0.2, 0.02
    xf = uniform_faces(0.0, Lx * nx / 512.0, nx)      # dx fixed at 0.2/512 for reduced sizes
    yf = tanh_faces_one_sided(ny, 2.2, Ly)
    dx = xf[1] - xf[0]
    zf = uniform_faces(0.0, nz * dx, nz)
    sim = blasius_compressible(M, Pr, gamma, T_inf, T_w / T_inf, mu_law)
    x_s = 0.02
    yeta = np.sqrt(2.0 * mu_e * x_s / (rho_inf * u_inf)) * np.concatenate(
        ([0.0], np.cumsum(0.5 * (sim["g"][1:] + sim["g"][:-1]) * np.diff(sim["eta"]))))
    yc = centres(yf)
    u_prof = u_inf * np.interp(yc, yeta, sim["fp"], right=1.0)
    T_prof = T_inf * np.interp(yc, yeta, sim["g"], right=1.0)
    rho_prof = p_inf / (Rg * T_prof)
    shp = (nz, ny, nx)
    u = np.broadcast_to(u_prof[None, :, None], shp).copy()
    rho = np.broadcast_to(rho_prof[None, :, None], shp).copy()
    zero = np.zeros(shp)
    p = np.full(shp, p_inf)
    U = set_interior_from_prim(empty_state((nx, ny, nz)), gamma, rho, u, zero, zero, p)
    inflow = np.empty((5, nz, ny))                    # x-face: t1 = y, t2 = z -> [5][nz][ny]
    inflow[0] = rho_prof[None, :]
    inflow[1] = u_prof[None, :]
    inflow[2] = 0.0
    inflow[3] = 0.0
    inflow[4] = p_inf
    bc = periodic_bc()
    bc[0] = FaceBC(BC_DIRICHLET, dirichlet=inflow)
    bc[1] = FaceBC(BC_ZEROGRAD)
    dist = {"A": A_frac * u_inf, "kappa": 10.0, "t1_lo": 0.05, "t1_hi": 0.15} if disturbance else None
    bc[2] = FaceBC(BC_WALL_ISOTHERMAL, T_wall=T_w, dist=dist)
    bc[3] = FaceBC(BC_ZEROGRAD)
    return Case(name=f"plate{nx}x{ny}x{nz}", n=(nx, ny, nz), xf=xf, yf=yf, zf=zf, gamma=gamma,
                R_gas=Rg, Pr=Pr, mu=dict(sutherland=1, **mu_law), bc=bc, U0=U, cfl=cfl,
                n_steps=n_steps,
                notes={"u_inf": u_inf, "rho_inf": rho_inf, "p_inf": p_inf, "s0": sim["s0"],
                       "h0": sim["h0"], "blasius_resid": sim["resid"]})


# ------------------------------------------------------------------ parity / edge-case inputs
def paper_boundary_layer(nx=300, ny=200, nz=4, cfl=0.5, n_steps=20, A=0.01, kappa=10.0, disturbance=True):
    """The paper's own section 3.2 case (parameters in tests/golden/paper_section_3_2.txt):
    laminar compressible boundary layer, M = 2.25, Pr = 0.72, unit Reynolds number 1e4, (x, y) in
    [1, 1.5] x [0, 0.4] on 300 x 200 cells, uniform in x, stretched in y (beta = 2.2), no-slip ADIABATIC south
    wall carrying the Disturbance Wall v = A sin(2 pi kappa x) (Eq. 8, A = 0.01, kappa = 10) over its whole
    length, zero-gradient north and east, self-similar (compressible Blasius, Eq. 7) profile at the west inlet.
    Units: rho_e = u_e = T_e = 1, x measured from the leading edge (so that Re_x = 1e4 x).  Readings where the
    paper is silent: R = 1/(gamma M^2); Sutherland with T_ref = T_e, mu_ref = mu_e = 1e-4, S = 110.4/273.15 T_e;
    one-sided tanh map; nz spanwise cells of width dx, periodic; the local similarity profile at every x as the
    initial field (v = w = 0)."""
    gamma, M, Pr, Re_unit = 1.4, 2.25, 0.72, 1.0e4
    Rg = 1.0 / (gamma * M * M)
    mu_law = {"mu_ref": 1.0 / Re_unit, "T_ref": 1.0, "S": 110.4 / 273.15}
    xf = uniform_faces(1.0, 1.0 + 0.5 * nx / 300.0, nx)            # dx fixed at 0.5/300 for reduced sizes
    yf = tanh_faces_one_sided(ny, 2.2, 0.4)
    dx = xf[1] - xf[0]
    zf = uniform_faces(0.0, nz * dx, nz)
    sim = blasius_compressible(M, Pr, gamma, 1.0, None, mu_law)
    Ieta = np.concatenate(([0.0], np.cumsum(0.5 * (sim["g"][1:] + sim["g"][:-1]) * np.diff(sim["eta"]))))
    xc, yc = centres(xf), centres(yf)

    def profile(x):                                                 # Eq. 7 inverted: y(eta) at distance x
        yeta = np.sqrt(2.0 * mu_law["mu_ref"] * x) * Ieta
        return np.interp(yc, yeta, sim["fp"], right=1.0), np.interp(yc, yeta, sim["g"], right=1.0)

    shp = (nz, ny, nx)
    u, T = np.empty(shp), np.empty(shp)
    for i, x in enumerate(xc):
        up, Tp = profile(x)
        u[:, :, i], T[:, :, i] = up[None, :], Tp[None, :]
    p = np.full(shp, Rg)                                            # p_e = rho_e R T_e
    zero = np.zeros(shp)
    U = set_interior_from_prim(empty_state((nx, ny, nz)), gamma, p / (Rg * T), u, zero, zero, p)
    u_in, T_in = profile(xf[0])
    inflow = np.empty((5, nz, ny))
    inflow[0] = (1.0 / T_in)[None, :]
    inflow[1] = u_in[None, :]
    inflow[2] = 0.0
    inflow[3] = 0.0
    inflow[4] = Rg
    bc = periodic_bc()
    bc[0] = FaceBC(BC_DIRICHLET, dirichlet=inflow)
    bc[1] = FaceBC(BC_ZEROGRAD)
    dist = {"A": A, "kappa": kappa, "t1_lo": xf[0], "t1_hi": xf[-1]} if disturbance else None
    bc[2] = FaceBC(BC_WALL_ADIABATIC, dist=dist)
    bc[3] = FaceBC(BC_ZEROGRAD)
    return Case(name=f"paperbl{nx}x{ny}x{nz}", n=(nx, ny, nz), xf=xf, yf=yf, zf=zf, gamma=gamma, R_gas=Rg, Pr=Pr,
                mu=dict(sutherland=1, **mu_law), bc=bc, U0=U, cfl=cfl, n_steps=n_steps,
                notes={"M": M, "Tw_over_Te": sim["h0"], "s0": sim["s0"], "blasius_resid": sim["resid"]})


def random_admissible(n=(12, 10, 8), seed=1, bc=None, viscous=True, stretched=False, amp=0.3):
    """Seeded random admissible state (rho > 0, p > 0) with distinct per-cell values."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = n
    shp = (nz, ny, nx)
    rho = 1.0 + amp * rng.uniform(-1, 1, shp)
    u, v, w = (0.5 * rng.uniform(-1, 1, shp) for _ in range(3))
    p = 1.0 + amp * rng.uniform(-1, 1, shp)
    gamma = 1.4
    U = set_interior_from_prim(empty_state(n), gamma, rho, u, v, w, p)

    def faces(m, L):
        f = uniform_faces(0.0, L, m)
        if stretched:
            f = f + 0.15 * L / m * np.sin(2 * np.pi * np.arange(m + 1) / m)
        return f

    return Case(name=f"rand{nx}x{ny}x{nz}s{seed}", n=n, xf=faces(nx, 1.0), yf=faces(ny, 0.9),
                zf=faces(nz, 0.8), gamma=gamma, R_gas=1.0, Pr=0.72,
                mu={"sutherland": 1 if viscous else 0, "mu_ref": 2e-3 if viscous else 0.0,
                    "T_ref": 1.0, "S": 0.4},
                bc=bc if bc is not None else periodic_bc(), U0=U, dt=1e-3, n_steps=3)


def smooth_periodic(n=(8, 8, 8), seed=3, viscous=True, L=1.0):
    """Random smooth (few Fourier modes) admissible periodic field on a uniform cubic grid."""
    rng = np.random.default_rng(seed)
    nx, ny, nz = n
    fs = [uniform_faces(0.0, L * m / max(n), m) for m in n]
    cs = [centres(f) for f in fs]
    Z, Y, X = np.meshgrid(cs[2], cs[1], cs[0], indexing="ij")
    per = [fs[0][-1], fs[1][-1], fs[2][-1]]

    def field(mean, amp):
        out = np.full(X.shape, mean)
        for _ in range(4):
            kx, ky, kz = rng.integers(0, 2, 3)
            ph = rng.uniform(0, 2 * np.pi)
            out = out + amp * rng.uniform(-1, 1) * np.sin(
                2 * np.pi * (kx * X / per[0] + ky * Y / per[1] + kz * Z / per[2]) + ph)
        return out

    rho, p = field(1.0, 0.05), field(1.0, 0.05)
    u, v, w = field(0.3, 0.1), field(-0.2, 0.1), field(0.1, 0.1)
    gamma = 1.4
    U = set_interior_from_prim(empty_state(n), gamma, rho, u, v, w, p)
    return Case(name="smooth", n=n, xf=fs[0], yf=fs[1], zf=fs[2], gamma=gamma, R_gas=1.0, Pr=0.72,
                mu={"sutherland": 1 if viscous else 0, "mu_ref": 5e-3 if viscous else 0.0,
                    "T_ref": 1.0, "S": 0.4},
                bc=periodic_bc(), U0=U, dt=1e-3, n_steps=2)
