"""CPU oracle of the periodic multigrid Poisson solver of arxiv/paper_2512_13403 §6.2 and Appendix C — TEST
INFRASTRUCTURE ONLY (plain numpy, fp64, one array operation per printed formula; no blocking, no fusion).  Only
tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference legs may import it; it shares no code with
the CUDA path.

Arrays are [nz, ny, nx] (x fastest), cubic cells of size h, periodic in every direction.

What follows the paper line by line:
  laplacian   Eq. 38   seven-point Laplacian A
  jacobi      Eq. 39   phi <- phi + omega D^-1 (F - A phi), D = -6/h^2, omega = 2/3
  residual    Eq. 41   r = F - A phi
  restrict    Eq. 42   mean of the 2x2x2 children (cell-centred full weighting)
  prolong     Eq. 44   trilinear, weights from the offset of the fine cell centre in the coarse cell
  cycle       Fig. 9, Eqs. 43-45, Appendix C: V-cycle (one recursive call) / W-cycle (two)
  solve       repeated cycles from phi = 0;  solve_vjp: Eqs. 46-48: g_F = A^-1 g_phi, the same solve
  exact_solve the plain definition the converged solve reaches: A^+ F by the discrete eigenvalues of Eq. 38 (FFT)

Readings (A21-A23):
  A21  Eq. 40 as printed has (1-omega)/6 in front of phi, which contradicts Eq. 39; Eq. 39 is followed:
       phi_new = (1-omega) phi + (omega/6) (sum of the six neighbours - h^2 F).
  A22  "direct solver on the coarse grid" (Fig. 9): A is singular on the torus.  Levels coarsen by 2 while every
       extent is even and > 2; the coarsest level is solved by `nu_coarse` Jacobi sweeps from zero (default 64;
       2^3 for power-of-two grids, where the slowest mode contracts by 0.56 per sweep).
  A23  F must have zero mean for A phi = F to be solvable: solve() removes the mean of F and returns the zero-mean phi.
"""
from __future__ import annotations

import numpy as np

OMEGA = 2.0 / 3.0


def _nbr_sum(phi):
    return (np.roll(phi, 1, 0) + np.roll(phi, -1, 0) + np.roll(phi, 1, 1) + np.roll(phi, -1, 1)
            + np.roll(phi, 1, 2) + np.roll(phi, -1, 2))


def laplacian(phi, h):
    """Eq. 38."""
    phi = np.asarray(phi, dtype=np.float64)
    return (_nbr_sum(phi) - 6.0 * phi) / (h * h)


def jacobi(phi, F, h, sweeps=1, omega=OMEGA):
    """Eq. 39 (reading A21)."""
    phi = np.asarray(phi, dtype=np.float64)
    for _ in range(sweeps):
        phi = (1.0 - omega) * phi + (omega / 6.0) * (_nbr_sum(phi) - h * h * F)
    return phi


def residual(phi, F, h):
    """Eq. 41."""
    return F - laplacian(phi, h)


def restrict(r):
    """Eq. 42: r2h[K, J, I] = 1/8 sum of r[2K+k, 2J+j, 2I+i], i, j, k in {0, 1}."""
    nz, ny, nx = r.shape
    return r.reshape(nz // 2, 2, ny // 2, 2, nx // 2, 2).mean(axis=(1, 3, 5))


def _prolong_axis(e, axis):
    # fine cell 2I sits at 1/4 of a coarse cell below the centre of coarse cell I: 3/4 e[I] + 1/4 e[I-1];
    # fine cell 2I+1 at 1/4 above it: 3/4 e[I] + 1/4 e[I+1]
    lo = 0.75 * e + 0.25 * np.roll(e, 1, axis)
    hi = 0.75 * e + 0.25 * np.roll(e, -1, axis)
    out = np.stack([lo, hi], axis=axis + 1)
    shape = list(e.shape)
    shape[axis] *= 2
    return out.reshape(shape)


def prolong(e):
    """Eq. 44: trilinear interpolation from coarse cell centres to fine cell centres (tensor product of the 1D rule)."""
    for axis in range(3):
        e = _prolong_axis(e, axis)
    return e


def can_coarsen(shape):
    return all(n % 2 == 0 and n > 2 for n in shape)


def cycle(phi, F, h, nu1=2, nu2=2, gamma=1, nu_coarse=64, omega=OMEGA):
    """One multigrid cycle for A phi = F starting from phi (Fig. 9; gamma = 1: V-cycle, 2: W-cycle, Eq. C12)."""
    if not can_coarsen(phi.shape):
        return jacobi(phi, F, h, nu_coarse, omega)            # coarsest level (reading A22)
    phi = jacobi(phi, F, h, nu1, omega)                       # pre-smoothing
    r2 = restrict(residual(phi, F, h))                        # Eqs. 41-42
    e2 = np.zeros_like(r2)
    for _ in range(gamma):                                    # A^2h e^2h = r^2h (Eq. 43), one or two recursive visits
        e2 = cycle(e2, r2, 2.0 * h, nu1, nu2, gamma, nu_coarse, omega)
    phi = phi + prolong(e2)                                   # Eqs. 44-45
    return jacobi(phi, F, h, nu2, omega)                      # post-smoothing


def solve(F, h, ncycles=10, **kw):
    """ncycles cycles from phi = 0 on the zero-mean part of F (reading A23).  Returns (phi, |r| / |F|)."""
    F = np.asarray(F, dtype=np.float64)
    F0 = F - F.mean()
    phi = np.zeros_like(F0)
    for _ in range(ncycles):
        phi = cycle(phi, F0, h, **kw)
    phi = phi - phi.mean()
    nF = np.sqrt(np.sum(F0 * F0))
    return phi, float(np.sqrt(np.sum(residual(phi, F0, h) ** 2)) / nF) if nF > 0 else 0.0


def solve_vjp(g_phi, h, ncycles=10, **kw):
    """Eqs. 46-48: the cotangent of F is another Poisson solve with the incoming cotangent as right-hand side."""
    return solve(g_phi, h, ncycles, **kw)


def exact_solve(F, h):
    """A^+ F on the torus from the eigenvalues of Eq. 38: lambda(k) = -(4/h^2) sum_a sin^2(pi k_a / n_a); zero mode -> 0."""
    F = np.asarray(F, dtype=np.float64)
    lam = np.zeros(F.shape)
    for axis, n in enumerate(F.shape):
        s = np.sin(np.pi * np.arange(n) / n) ** 2
        lam = lam + s.reshape([-1 if a == axis else 1 for a in range(3)])
    lam = -4.0 / (h * h) * lam
    Fh = np.fft.fftn(F)
    with np.errstate(divide="ignore", invalid="ignore"):
        ph = np.where(lam != 0.0, Fh / lam, 0.0)
    return np.real(np.fft.ifftn(ph))
