"""Pins for oracle/gravity.py (self-gravity as a source of the hydro step; readings A23, A27):
the central-difference acceleration of a sine against its closed form along each axis; a constant potential is no force
(bitwise); a gas at rest gains momentum rho g dt and no energy; self-gravity with the potential of the discrete Poisson
problem conserves total momentum to rounding (antisymmetric gradient x symmetric inverse Laplacian); a plane-wave density
perturbation against the closed form built from the discrete eigenvalues; the VJPs against central finite differences and
the dot-product identity (the source is linear in phi and bilinear in (U, phi): differences are exact to rounding); the
VJP of the whole self-gravitating step against finite differences."""
import numpy as np
import pytest

import oracle
from oracle import gravity, poisson


def _state(shape, seed, g=5 / 3, mach=0.4):
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.6, 1.8, shape)
    v = rng.normal(0, mach, (3,) + shape)
    P = rng.uniform(0.6, 1.8, shape)
    return np.stack([rho, rho * v[0], rho * v[1], rho * v[2], P / (g - 1) + 0.5 * rho * (v ** 2).sum(0)])


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_acceleration_of_a_sine_closed_form(axis):
    shape, dx = (12, 10, 16), (1 / 16, 1 / 10, 1 / 12)       # [nz, ny, nx]
    n = shape[2 - axis]
    m, A = 2, 0.7
    x = (np.arange(n) + 0.5) * dx[axis]
    L = n * dx[axis]
    prof = A * np.sin(2 * np.pi * m * x / L)
    phi = np.broadcast_to(prof.reshape([-1 if a == 2 - axis else 1 for a in range(3)]), shape).copy()
    g = gravity.acceleration(phi, dx)
    want = -A * np.sin(2 * np.pi * m * dx[axis] / L) / dx[axis] * np.cos(2 * np.pi * m * x / L)
    got = np.moveaxis(g[axis], 2 - axis, -1)
    assert np.abs(got - want).max() <= 1e-12
    for other in range(3):
        if other != axis:
            assert np.array_equal(g[other], np.zeros(shape))


def test_constant_potential_is_no_force_and_rest_gas_gains_rho_g_dt():
    shape, dx = (6, 7, 8), (0.1, 0.2, 0.3)
    U = _state(shape, 1)
    assert np.array_equal(gravity.source(U, np.full(shape, 3.7), 0.2, dx), U)
    rng = np.random.default_rng(2)
    phi = rng.normal(size=shape)
    R = U.copy()
    R[1:4] = 0.0
    out = gravity.source(R, phi, 0.2, dx)
    g = gravity.acceleration(phi, dx)
    assert np.array_equal(out[0], R[0]) and np.array_equal(out[4], R[4])      # no work on a gas at rest
    assert np.allclose(out[1:4], 0.2 * R[0] * g, rtol=1e-15, atol=0)


def test_self_gravity_conserves_total_momentum():
    shape, h = (16, 16, 16), 1 / 16
    U = _state(shape, 3)
    phi = poisson.exact_solve(4 * np.pi * (U[0] - U[0].mean()), h)
    out = gravity.source(U, phi, 0.05, (h, h, h))
    for a in range(3):
        kick = (out[1 + a] - U[1 + a]).sum()
        assert abs(kick) <= 1e-12 * np.abs(out[1 + a] - U[1 + a]).sum()
    assert np.abs(out[1:4] - U[1:4]).max() > 1e-4                              # and the force is not trivially zero


def test_plane_wave_perturbation_closed_form():
    n, h = 32, 1 / 32
    m, eps, rho0, fpg = 3, 1e-2, 1.3, 7.0
    x = (np.arange(n) + 0.5) * h
    k = 2 * np.pi * m
    rho = rho0 * (1 + eps * np.cos(k * x))
    U = np.zeros((5, n, n, n))
    U[0] = rho[None, None, :]
    U[4] = 1.0
    phi = poisson.exact_solve(fpg * (U[0] - U[0].mean()), h)
    lam = -(4 / h ** 2) * np.sin(np.pi * m / n) ** 2                           # eigenvalue of Eq. 38 for this mode
    gx = (fpg * rho0 * eps / lam) * np.sin(2 * np.pi * m / n) / h * np.sin(k * x)     # -(phi_{i+1} - phi_{i-1}) / 2h of phi = (F/lam) cos
    out = gravity.source(U, phi, 0.1, (h, h, h))
    assert np.abs(out[1][5, 7] - 0.1 * rho * gx).max() <= 1e-12
    assert np.abs(out[2]).max() <= 1e-13 and np.abs(out[3]).max() <= 1e-13


def test_source_vjp_finite_differences_and_dot_product():
    shape, dx = (6, 7, 8), (0.11, 0.13, 0.17)
    rng = np.random.default_rng(5)
    U, phi = _state(shape, 4), rng.normal(size=shape)
    gout = rng.normal(size=U.shape)
    gU, gphi = gravity.source_vjp(U, phi, 0.3, dx, gout)
    for _ in range(3):
        vU, vphi = rng.normal(size=U.shape), rng.normal(size=shape)
        eps = 1e-3                                                             # bilinear: the central difference is exact
        Jv = (gravity.source(U + eps * vU, phi + eps * vphi, 0.3, dx) - gravity.source(U - eps * vU, phi - eps * vphi, 0.3, dx)) / (2 * eps)
        lhs, rhs = float((gout * Jv).sum()), float((gU * vU).sum() + (gphi * vphi).sum())
        assert abs(lhs - rhs) <= 1e-11 * (abs(lhs) + abs(rhs))
    e = np.zeros(shape)
    e[2, 3, 4] = 1.0
    fd = float((gout * (gravity.source(U, phi + e, 0.3, dx) - gravity.source(U, phi - e, 0.3, dx))).sum() / 2)
    assert abs(fd - gphi[2, 3, 4]) <= 1e-12 * max(1.0, abs(fd))


@pytest.mark.parametrize("kw", [dict(), dict(limiter="vanleer"), dict(cooling=True, lambda0=0.5)], ids=["minmod", "vanleer", "cooling"])
def test_self_gravitating_step_vjp_finite_differences(kw):
    shape, h = (8, 8, 8), 1 / 8
    U = _state(shape, 6)
    p = oracle.params(shape=shape, **kw)
    dt = oracle.cfl_dt(U, p)[0]
    rng = np.random.default_rng(7)
    g = rng.normal(size=U.shape)
    fpg, nc = 20.0, 26                                                          # 26 V-cycles: converged to ~1e-13
    gin = gravity.step_vjp(U, dt, g, p, fpg, h, ncycles=nc)
    base = oracle.step_vjp(U, dt, g, p)
    assert np.abs(gin - base).max() > 1e-3 * np.abs(base).max()                # gravity matters in this gradient
    eps = 1e-6
    for _ in range(3):
        v = rng.normal(size=U.shape)
        fd = (gravity.step(U + eps * v, dt, p, fpg, h, ncycles=nc) - gravity.step(U - eps * v, dt, p, fpg, h, ncycles=nc)) / (2 * eps)
        lhs, rhs = float((g * fd).sum()), float((gin * v).sum())
        assert abs(lhs - rhs) <= 2e-6 * abs(rhs), (lhs, rhs)
