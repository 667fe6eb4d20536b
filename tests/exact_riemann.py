"""Exact solution of the 1D Riemann problem for the ideal-gas Euler equations.

Textbook construction (pressure function of the two nonlinear waves, Newton iteration for the
star pressure, then sampling of the self-similar solution in xi = x/t); written here from the
Rankine-Hugoniot and isentropic relations, independent of the oracle and of the CUDA path.
Used as pin P2 (Sod convergence).
"""
import math

import numpy as np


def _f_and_df(p, rho_k, p_k, c_k, g):
    if p > p_k:                                   # shock
        A = 2.0 / ((g + 1.0) * rho_k)
        B = (g - 1.0) / (g + 1.0) * p_k
        s = math.sqrt(A / (p + B))
        return (p - p_k) * s, s * (1.0 - 0.5 * (p - p_k) / (p + B))
    pr = p / p_k                                  # rarefaction
    f = 2.0 * c_k / (g - 1.0) * (pr ** ((g - 1.0) / (2.0 * g)) - 1.0)
    df = 1.0 / (rho_k * c_k) * pr ** (-(g + 1.0) / (2.0 * g))
    return f, df


def star_state(rhoL, uL, pL, rhoR, uR, pR, g):
    cL, cR = math.sqrt(g * pL / rhoL), math.sqrt(g * pR / rhoR)
    p = max(1e-12, 0.5 * (pL + pR))
    for _ in range(200):
        fL, dL = _f_and_df(p, rhoL, pL, cL, g)
        fR, dR = _f_and_df(p, rhoR, pR, cR, g)
        pn = p - (fL + fR + (uR - uL)) / (dL + dR)
        pn = max(pn, 1e-14)
        if abs(pn - p) <= 1e-15 * (pn + p):
            p = pn
            break
        p = pn
    fL, _ = _f_and_df(p, rhoL, pL, cL, g)
    fR, _ = _f_and_df(p, rhoR, pR, cR, g)
    u = 0.5 * (uL + uR) + 0.5 * (fR - fL)
    return p, u


def sample(xi, rhoL, uL, pL, rhoR, uR, pR, g):
    """(rho, u, p) at similarity coordinate(s) xi = (x - x0)/t."""
    xi = np.atleast_1d(np.asarray(xi, dtype=np.float64))
    ps, us = star_state(rhoL, uL, pL, rhoR, uR, pR, g)
    cL, cR = math.sqrt(g * pL / rhoL), math.sqrt(g * pR / rhoR)
    gm, gp = g - 1.0, g + 1.0
    rho = np.empty_like(xi); u = np.empty_like(xi); p = np.empty_like(xi)
    for n, s in enumerate(xi):
        if s <= us:                               # left of the contact
            if ps > pL:                           # left shock
                SL = uL - cL * math.sqrt(gp / (2 * g) * ps / pL + gm / (2 * g))
                if s <= SL:
                    r, v, q = rhoL, uL, pL
                else:
                    r = rhoL * (ps / pL + gm / gp) / (gm / gp * ps / pL + 1.0)
                    v, q = us, ps
            else:                                 # left rarefaction
                cs = cL * (ps / pL) ** (gm / (2 * g))
                if s <= uL - cL:
                    r, v, q = rhoL, uL, pL
                elif s >= us - cs:
                    r, v, q = rhoL * (ps / pL) ** (1.0 / g), us, ps
                else:
                    v = 2.0 / gp * (cL + gm / 2.0 * uL + s)
                    c = 2.0 / gp * (cL + gm / 2.0 * (uL - s))
                    r = rhoL * (c / cL) ** (2.0 / gm)
                    q = pL * (c / cL) ** (2.0 * g / gm)
        else:
            if ps > pR:                           # right shock
                SR = uR + cR * math.sqrt(gp / (2 * g) * ps / pR + gm / (2 * g))
                if s >= SR:
                    r, v, q = rhoR, uR, pR
                else:
                    r = rhoR * (ps / pR + gm / gp) / (gm / gp * ps / pR + 1.0)
                    v, q = us, ps
            else:                                 # right rarefaction
                cs = cR * (ps / pR) ** (gm / (2 * g))
                if s >= uR + cR:
                    r, v, q = rhoR, uR, pR
                elif s <= us + cs:
                    r, v, q = rhoR * (ps / pR) ** (1.0 / g), us, ps
                else:
                    v = 2.0 / gp * (-cR + gm / 2.0 * uR + s)
                    c = 2.0 / gp * (cR - gm / 2.0 * (uR - s))
                    r = rhoR * (c / cR) ** (2.0 / gm)
                    q = pR * (c / cR) ** (2.0 * g / gm)
        rho[n], u[n], p[n] = r, v, q
    return rho, u, p
