"""ORACLE — test infrastructure only.

Self-gravity as a source term of the hydro step (§6; the force-class form of PAPER.md:88-107), plain numpy,
fp64: the potential of Eq. 27 (L phi = 4 pi G rho, mean of rho removed on the torus: reading A23) from oracle/poisson.py, the
acceleration g = -grad phi by "the usual finite-difference gradient" (reading A27: second-order central differences
on the periodic grid), and the operator-split update of the force class printed in PAPER.md:88-107:
    s_g = (0, rho g, m . g);   u <- u + s_g dt        (momentum source rho g, energy source m . g, both from the incoming u).
A self-gravitating step (reading A27) = potential of the incoming density, hydro step (oracle.step), then the kick with that potential.
The VJPs are the hand-written transposes of these linear-in-(phi) / bilinear maps; tests pin them with finite differences and
the dot-product identity.  Only tests/ may import this module; the product never does.

Arrays are [nz, ny, nx] (phi) and [5, nz, ny, nx] (state), x fastest; dx = (dx, dy, dz).
"""
from __future__ import annotations

import numpy as np

from . import oracle as _o
from . import poisson as _p


def acceleration(phi, dx):
    """g_a = -(phi_{i+1} - phi_{i-1}) / (2 dx_a), a = x, y, z (periodic).  Returns [3, nz, ny, nx]."""
    phi = np.asarray(phi, dtype=np.float64)
    return np.stack([-(np.roll(phi, -1, axis=2 - a) - np.roll(phi, 1, axis=2 - a)) / (2.0 * dx[a]) for a in range(3)])


def source(U, phi, dt, dx):
    """u + s_g dt with s_g = (0, rho g, m . g)."""
    U = np.asarray(U, dtype=np.float64)
    g = acceleration(phi, dx)
    out = U.copy()
    for a in range(3):
        out[1 + a] += dt * U[0] * g[a]
        out[4] += dt * U[1 + a] * g[a]
    return out


def source_vjp(U, phi, dt, dx, g_out):
    """(dL/dU, dL/dphi) of source() given dL/d(out)."""
    U = np.asarray(U, dtype=np.float64)
    g_out = np.asarray(g_out, dtype=np.float64)
    g = acceleration(phi, dx)
    gU = g_out.copy()
    gphi = np.zeros_like(np.asarray(phi, dtype=np.float64))
    for a in range(3):
        gU[0] += dt * g[a] * g_out[1 + a]
        gU[1 + a] += dt * g[a] * g_out[4]
        gbar = dt * (U[0] * g_out[1 + a] + U[1 + a] * g_out[4])          # cotangent of g_a
        gphi += (np.roll(gbar, -1, axis=2 - a) - np.roll(gbar, 1, axis=2 - a)) / (2.0 * dx[a])   # transpose of the central difference
    return gU, gphi


def potential(rho, four_pi_g, h, ncycles=12, **kw):
    """phi of Eq. 27 by multigrid cycles on the zero-mean part of 4 pi G rho (poisson.solve)."""
    return _p.solve(four_pi_g * np.asarray(rho, dtype=np.float64), h, ncycles=ncycles, **kw)[0]


def step(U, dt, p, four_pi_g, h, ncycles=12, **kw):
    """Self-gravitating step: phi from the incoming density, the hydro step, then the kick with that phi."""
    U = np.asarray(U, dtype=np.float64)
    phi = potential(U[0], four_pi_g, h, ncycles, **kw)
    U1 = _o.step(U, dt, p)
    return source(U1, phi, dt, (p.dx[0], p.dx[1], p.dx[2]))


def step_vjp(U, dt, g_out, p, four_pi_g, h, ncycles=12, **kw):
    """Transpose of step(): through the kick (at the post-hydro state), the Poisson solve (another solve, Eqs. 46-48) and
    the hydro step; dt held constant."""
    U = np.asarray(U, dtype=np.float64)
    dx = (p.dx[0], p.dx[1], p.dx[2])
    phi = potential(U[0], four_pi_g, h, ncycles, **kw)
    U1 = _o.step(U, dt, p)
    gU1, gphi = source_vjp(U1, phi, dt, dx, g_out)
    gF = _p.solve_vjp(gphi, h, ncycles=ncycles, **kw)
    gF = gF[0] if isinstance(gF, tuple) else gF
    gU = _o.step_vjp(U, dt, gU1, p)
    gU[0] += four_pi_g * (gF - gF.mean())                              # F = 4 pi G (rho - mean rho): transpose of the mean removal
    return gU
