"""ORACLE (test infrastructure, not the product): plane statistics, written out as their definition.

PAPER.md:92-96 / Fig. 1 validate the channel DNS with profiles averaged over the two homogeneous directions:
mean density, temperature, streamwise velocity, Reynolds stresses (and r.m.s. of density and temperature).  For a
plane p of `axis` the area-weighted sum of a quantity phi over the plane's interior cells is
    S_phi(p) = sum_{t1,t2} phi dA,   dA = Delta_t1 * Delta_t2,
the plane mean is <phi> = S_phi / S_1, and the Reynolds stress <u_i' u_j'> = <u_i u_j> - <u_i><u_j>
(Reynolds averaging; the paper does not say Reynolds or Favre - DESIGN.md reading).  Plain numpy, fp64, no
blocking.  Pinned in tests/test_oracle_stats.py by closed forms (Taylor-Green, Poiseuille).
"""
import numpy as np

NH = 3
NAMES = ["1", "rho", "T", "u", "v", "w", "uu", "vv", "ww", "uv", "uw", "vw", "rho2", "T2"]


def plane_sums(case, U, axis):
    """sums[14][n_axis] of the quantities NAMES for the padded conservative state U[5, nz+6, ny+6, nx+6]."""
    U = np.asarray(U, dtype=np.float64)[:, NH:-NH, NH:-NH, NH:-NH]          # interior, indexed [q, k, j, i]
    rho = U[0]
    u, v, w = U[1] / rho, U[2] / rho, U[3] / rho                          # Eq. 2
    p = (case.gamma - 1.0) * (U[4] - 0.5 * rho * (u * u + v * v + w * w))
    T = p / (rho * case.R_gas)
    d = [np.diff(np.asarray(f, dtype=np.float64)) for f in (case.xf, case.yf, case.zf)]
    dx, dy, dz = d[0][None, None, :], d[1][None, :, None], d[2][:, None, None]
    dA = [dy * dz, dx * dz, dx * dy][axis] * np.ones_like(rho)
    other = [(0, 1), (0, 2), (1, 2)][axis]                                 # numpy axes summed over ([k, j, i] order)
    phis = [np.ones_like(rho), rho, T, u, v, w, u * u, v * v, w * w, u * v, u * w, v * w, rho * rho, T * T]
    return np.stack([np.sum(phi * dA, axis=other) for phi in phis])


def profiles(sums):
    """Means and Reynolds stresses from the sums: dict of arrays over the planes."""
    m = {n: sums[i] / sums[0] for i, n in enumerate(NAMES) if i > 0}
    out = {"rho": m["rho"], "T": m["T"], "u": m["u"], "v": m["v"], "w": m["w"]}
    for a, b in (("u", "u"), ("v", "v"), ("w", "w"), ("u", "v"), ("u", "w"), ("v", "w")):
        out[a + "'" + b + "'"] = m[a + b] - m[a] * m[b]
    out["rho_rms"] = np.sqrt(np.maximum(m["rho2"] - m["rho"] ** 2, 0.0))
    out["T_rms"] = np.sqrt(np.maximum(m["T2"] - m["T"] ** 2, 0.0))
    return out
