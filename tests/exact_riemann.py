"""Exact Riemann solver for the 1D ideal-gas Euler equations (Newton iteration on the pressure
function; the textbook construction: shock branch from Rankine-Hugoniot, rarefaction branch from the
Riemann invariants).  Written for the tests only — it is the independent reference the oracle's HLLC
flux and 1D shock-tube results are pinned against.  Shares nothing with oracle/ or the CUDA path."""
import numpy as np


def _fK(p, rhoK, pK, g):
    cK = np.sqrt(g * pK / rhoK)
    if p > pK:  # shock
        A = 2.0 / ((g + 1.0) * rhoK)
        B = (g - 1.0) / (g + 1.0) * pK
        f = (p - pK) * np.sqrt(A / (p + B))
        df = np.sqrt(A / (p + B)) * (1.0 - 0.5 * (p - pK) / (p + B))
    else:  # rarefaction
        f = 2.0 * cK / (g - 1.0) * ((p / pK) ** ((g - 1.0) / (2.0 * g)) - 1.0)
        df = 1.0 / (rhoK * cK) * (p / pK) ** (-(g + 1.0) / (2.0 * g))
    return f, df


def star_state(rhoL, uL, pL, rhoR, uR, pR, g):
    """(p*, u*) of the exact solution."""
    p = max(1e-14, 0.5 * (pL + pR))
    for _ in range(200):
        fL, dL = _fK(p, rhoL, pL, g)
        fR, dR = _fK(p, rhoR, pR, g)
        pn = p - (fL + fR + (uR - uL)) / (dL + dR)
        if pn <= 0.0:
            pn = 0.5 * p
        if abs(pn - p) <= 1e-15 * max(p, pn):
            p = pn
            break
        p = pn
    fL, _ = _fK(p, rhoL, pL, g)
    fR, _ = _fK(p, rhoR, pR, g)
    return p, 0.5 * (uL + uR) + 0.5 * (fR - fL)


def sample(xi, rhoL, uL, pL, rhoR, uR, pR, g):
    """(rho, u, p) of the exact solution on the ray x/t = xi (scalar)."""
    ps, us = star_state(rhoL, uL, pL, rhoR, uR, pR, g)
    gm, gp = g - 1.0, g + 1.0
    if xi <= us:  # left of the contact
        cL = np.sqrt(g * pL / rhoL)
        if ps > pL:  # left shock
            SL = uL - cL * np.sqrt(gp / (2 * g) * ps / pL + gm / (2 * g))
            if xi <= SL:
                return rhoL, uL, pL
            return rhoL * ((ps / pL + gm / gp) / (gm / gp * ps / pL + 1.0)), us, ps
        sHL = uL - cL
        if xi <= sHL:
            return rhoL, uL, pL
        cs = cL * (ps / pL) ** (gm / (2 * g))
        sTL = us - cs
        if xi >= sTL:
            return rhoL * (ps / pL) ** (1.0 / g), us, ps
        c = 2.0 / gp * (cL + gm / 2.0 * (uL - xi))
        return rhoL * (c / cL) ** (2.0 / gm), 2.0 / gp * (cL + gm / 2.0 * uL + xi), pL * (c / cL) ** (2.0 * g / gm)
    cR = np.sqrt(g * pR / rhoR)
    if ps > pR:  # right shock
        SR = uR + cR * np.sqrt(gp / (2 * g) * ps / pR + gm / (2 * g))
        if xi >= SR:
            return rhoR, uR, pR
        return rhoR * ((ps / pR + gm / gp) / (gm / gp * ps / pR + 1.0)), us, ps
    sHR = uR + cR
    if xi >= sHR:
        return rhoR, uR, pR
    cs = cR * (ps / pR) ** (gm / (2 * g))
    sTR = us + cs
    if xi <= sTR:
        return rhoR * (ps / pR) ** (1.0 / g), us, ps
    c = 2.0 / gp * (cR - gm / 2.0 * (uR - xi))
    return rhoR * (c / cR) ** (2.0 / gm), 2.0 / gp * (-cR + gm / 2.0 * uR + xi), pR * (c / cR) ** (2.0 * g / gm)


def godunov_flux(WL, WR, g):
    """Exact (Godunov) flux through x/t = 0 for 1D states W = (rho, u, vt1, vt2, p); passive
    transverse velocities are taken from the upwind side of the contact."""
    rho, u, p = sample(0.0, WL[0], WL[1], WL[4], WR[0], WR[1], WR[4], g)
    _, us = star_state(WL[0], WL[1], WL[4], WR[0], WR[1], WR[4], g)
    vt = (WL[2], WL[3]) if us >= 0.0 else (WR[2], WR[3])
    E = p / (g - 1.0) + 0.5 * rho * (u * u + vt[0] ** 2 + vt[1] ** 2)
    return np.array([rho * u, rho * u * u + p, rho * u * vt[0], rho * u * vt[1], u * (E + p)])
