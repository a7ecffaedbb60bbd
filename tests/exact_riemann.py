"""Exact solution of the 1-D Riemann problem for an ideal gas (textbook: pressure function of
two shocks/rarefactions solved by Newton, then wave sampling).  Independent of oracle/ and of the
CUDA path; used to pin the inviscid path on the Sod tube (BASELINE.json configs[1])."""
import numpy as np


def _fK(p, rhoK, pK, g):
    cK = np.sqrt(g * pK / rhoK)
    if p > pK:  # shock
        A, B = 2.0 / ((g + 1) * rhoK), (g - 1) / (g + 1) * pK
        f = (p - pK) * np.sqrt(A / (p + B))
        df = np.sqrt(A / (p + B)) * (1 - (p - pK) / (2 * (B + p)))
    else:       # rarefaction
        f = 2 * cK / (g - 1) * ((p / pK) ** ((g - 1) / (2 * g)) - 1)
        df = 1.0 / (rhoK * cK) * (p / pK) ** (-(g + 1) / (2 * g))
    return f, df


def star_state(rhoL, uL, pL, rhoR, uR, pR, g=1.4):
    p = 0.5 * (pL + pR)
    for _ in range(100):
        fL, dL = _fK(p, rhoL, pL, g)
        fR, dR = _fK(p, rhoR, pR, g)
        dp = (fL + fR + uR - uL) / (dL + dR)
        p = max(p - dp, 1e-12)
        if abs(dp) < 1e-15 * p:
            break
    fL, _ = _fK(p, rhoL, pL, g)
    fR, _ = _fK(p, rhoR, pR, g)
    u = 0.5 * (uL + uR) + 0.5 * (fR - fL)
    return p, u


def sample(xi, rhoL, uL, pL, rhoR, uR, pR, g=1.4):
    """(rho, u, p) at similarity coordinate xi = (x - x0)/t, vectorised over xi."""
    ps, us = star_state(rhoL, uL, pL, rhoR, uR, pR, g)
    xi = np.asarray(xi, dtype=np.float64)
    rho, u, p = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    cL, cR = np.sqrt(g * pL / rhoL), np.sqrt(g * pR / rhoR)
    gm, gp = g - 1, g + 1
    for n, s in enumerate(xi.flat):
        if s <= us:   # left of contact
            if ps > pL:
                SL = uL - cL * np.sqrt(gp / (2 * g) * ps / pL + gm / (2 * g))
                if s < SL:
                    r, v, q = rhoL, uL, pL
                else:
                    r = rhoL * ((ps / pL + gm / gp) / (gm / gp * ps / pL + 1))
                    v, q = us, ps
            else:
                cs = cL * (ps / pL) ** (gm / (2 * g))
                if s < uL - cL:
                    r, v, q = rhoL, uL, pL
                elif s > us - cs:
                    r, v, q = rhoL * (ps / pL) ** (1 / g), us, ps
                else:
                    c = 2 / gp * (cL + gm / 2 * (uL - s))
                    v = 2 / gp * (cL + gm / 2 * uL + s)
                    r = rhoL * (c / cL) ** (2 / gm)
                    q = pL * (c / cL) ** (2 * g / gm)
        else:
            if ps > pR:
                SR = uR + cR * np.sqrt(gp / (2 * g) * ps / pR + gm / (2 * g))
                if s > SR:
                    r, v, q = rhoR, uR, pR
                else:
                    r = rhoR * ((ps / pR + gm / gp) / (gm / gp * ps / pR + 1))
                    v, q = us, ps
            else:
                cs = cR * (ps / pR) ** (gm / (2 * g))
                if s > uR + cR:
                    r, v, q = rhoR, uR, pR
                elif s < us + cs:
                    r, v, q = rhoR * (ps / pR) ** (1 / g), us, ps
                else:
                    c = 2 / gp * (cR - gm / 2 * (uR - s))
                    v = 2 / gp * (-cR + gm / 2 * uR + s)
                    r = rhoR * (c / cR) ** (2 / gm)
                    q = pR * (c / cR) ** (2 * g / gm)
        rho.flat[n], u.flat[n], p.flat[n] = r, v, q
    return rho, u, p
