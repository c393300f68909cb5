"""Pins for the oracle's whole step: exact Riemann solution (Sod) along each axis, smooth-wave
convergence order, uniform-state preservation, conservation, translation equivariance, isotropy,
Sedov-Taylor radius law.  (SURVEY.md §8(c) "What pins each part".)"""
import math

import numpy as np
import pytest

import oracle
from exact_riemann import sample


def _cons(rho, v, P, g):
    return np.stack([rho, rho * v[0], rho * v[1], rho * v[2], P / (g - 1) + 0.5 * rho * (v[0] ** 2 + v[1] ** 2 + v[2] ** 2)])


def _line_shape(n, ax):
    shp = [4, 4, 4]          # (nz, ny, nx)
    shp[2 - ax] = n
    return tuple(shp)


def _along(ax, arr1d, shape):
    """broadcast a 1D profile along axis ax (0=x,1=y,2=z) of a (nz,ny,nx) grid"""
    idx = [None, None, None]
    idx[2 - ax] = slice(None)
    return np.broadcast_to(arr1d[tuple(idx)], shape).copy()


def _run(U, p, t_end, cfl=0.4):
    t = 0.0
    while t < t_end * (1 - 1e-14):
        dt, _ = oracle.cfl_dt(U, p, cfl)
        dt = min(dt, t_end - t)
        U = oracle.step(U, dt, p)
        t += dt
    return U


def _sod_l1(n, ax):
    g, t_end = 1.4, 0.1
    shape = _line_shape(n, ax)
    x = (np.arange(n) + 0.5) / n
    hi = (x >= 0.25) & (x < 0.75)
    rho = _along(ax, np.where(hi, 1.0, 0.125), shape)
    P = _along(ax, np.where(hi, 1.0, 0.1), shape)
    z = np.zeros(shape)
    dx = [1.0, 1.0, 1.0]
    dx[ax] = 1.0 / n
    p = oracle.params(gamma=g, dx=dx)
    U = _run(_cons(rho, [z, z, z], P, g), p, t_end)
    # exact solution: two independent Riemann problems (the fans do not meet by t = 0.1)
    ex = np.empty(n)
    for i, xi in enumerate(x):
        if xi >= 0.5:
            ex[i] = sample((xi - 0.75) / t_end, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, g)[0]
        else:
            ex[i] = sample((xi - 0.25) / t_end, 0.125, 0.0, 0.1, 1.0, 0.0, 1.0, g)[0]
    rho_num = np.moveaxis(U[0], 2 - ax, -1)
    assert np.abs(rho_num - rho_num[0, 0]).max() < 1e-13          # stays 1D
    mom_t = [U[1 + a] for a in range(3) if a != ax]
    assert max(np.abs(m).max() for m in mom_t) == 0.0             # no transverse momentum
    return np.abs(rho_num[0, 0] - ex).mean()


@pytest.mark.parametrize("ax", [0, 1, 2])
def test_sod_tube_against_exact_solution(ax):
    e128, e256 = _sod_l1(128, ax), _sod_l1(256, ax)
    assert e256 < 1e-2
    rate = math.log2(e128 / e256)
    assert 0.6 < rate < 1.1, rate


def test_smooth_advected_wave_is_second_order():
    """rho = 1 + 0.2 sin(2 pi x), v = 1, P = 1 advected once around the box: L1 order >= 1.5."""
    g = 1.4
    errs = []
    for n in (32, 64):
        shape = _line_shape(n, 0)
        x = (np.arange(n) + 0.5) / n
        rho = _along(0, 1 + 0.2 * np.sin(2 * np.pi * x), shape)
        one = np.ones(shape)
        p = oracle.params(gamma=g, dx=(1.0 / n, 1.0, 1.0), limiter="vanleer")
        U = _run(_cons(rho, [one, 0 * one, 0 * one], one, g), p, 1.0)
        errs.append(np.abs(U[0] - rho).mean())
    assert math.log2(errs[0] / errs[1]) > 1.5, errs


@pytest.mark.parametrize("integrator", ["vl2", "heun", "ssprk3"])
def test_uniform_state_is_preserved_bitwise(integrator):
    g = 5 / 3
    shape = (6, 5, 7)
    one = np.ones(shape)
    for v in ((0, 0, 0), (0.3, -1.7, 2.2)):
        U = _cons(1.3 * one, [v[0] * one, v[1] * one, v[2] * one], 0.7 * one, g)
        out = oracle.step(U, 0.01, oracle.params(gamma=g, shape=shape, integrator=integrator))
        assert np.array_equal(out, U)


def _random_state(n, seed, g=5 / 3, shape=None):
    rng = np.random.default_rng(seed)
    shape = shape or (n, n, n)
    rho = rng.uniform(0.5, 2.0, shape)
    v = rng.normal(0, 0.5, (3,) + shape)
    P = rng.uniform(0.5, 2.0, shape)
    return _cons(rho, v, P, g)


@pytest.mark.parametrize("cooling", [False, True])
def test_conservation_to_rounding(cooling):
    """sum rho, sum rho v, sum E unchanged by a periodic step (relative 1e-13); with cooling on, mass
    and momentum still are."""
    U = _random_state(12, 4)
    p = oracle.params(shape=U.shape, cooling=cooling)
    dt = oracle.cfl_dt(U, p)[0]
    out = oracle.step(U, dt, p)
    for f in range(4 if cooling else 5):
        before, after = math.fsum(U[f].ravel()), math.fsum(out[f].ravel())
        scale = math.fsum(np.abs(U[f]).ravel())
        assert abs(after - before) <= 1e-13 * scale
    if cooling:
        assert out[4].sum() < U[4].sum()


def test_translation_equivariance_bitwise():
    U = _random_state(10, 5, shape=(8, 9, 10))
    p = oracle.params(shape=U.shape)
    dt = oracle.cfl_dt(U, p)[0]
    ref = oracle.step(U, dt, p)
    for shift in ((1, 0, 0), (0, 3, 0), (0, 0, -2), (5, 4, 7)):
        out = oracle.step(np.roll(U, shift, axis=(1, 2, 3)), dt, p)
        assert np.array_equal(out, np.roll(ref, shift, axis=(1, 2, 3)))


def test_axis_permutation_and_mirror_symmetry():
    U = _random_state(8, 6, shape=(8, 8, 8))
    p = oracle.params(shape=U.shape)
    dt = 0.5 * oracle.cfl_dt(U, p)[0]
    ref = oracle.step(U, dt, p)
    scale = np.abs(ref).max()
    # swap x <-> y: transpose the last two array axes and swap the momentum components
    perm = lambda A: np.stack([A[0], A[2], A[1], A[3], A[4]]).transpose(0, 1, 3, 2)
    assert np.abs(oracle.step(perm(U), dt, p) - perm(ref)).max() <= 1e-14 * scale
    # swap x <-> z
    perm = lambda A: np.stack([A[0], A[3], A[2], A[1], A[4]]).transpose(0, 3, 2, 1)
    assert np.abs(oracle.step(perm(U), dt, p) - perm(ref)).max() <= 1e-14 * scale
    # mirror x
    mir = lambda A: np.stack([A[0], -A[1], A[2], A[3], A[4]])[..., ::-1]
    assert np.abs(oracle.step(mir(U), dt, p) - mir(ref)).max() <= 1e-14 * scale


def test_two_stage_form_matches_its_definition_with_numpy():
    """U^{n+1} = U^n - dt D(U^n - dt/2 D(U^n))  (Eqs. A6-A7 unsplit) and Heun, assembled in numpy from
    the oracle's D()."""
    U = _random_state(6, 8, shape=(6, 6, 6))
    p = oracle.params(shape=U.shape)
    dt = 0.01
    Us = U - 0.5 * dt * oracle.flux_divergence(U, p)
    assert np.allclose(oracle.step(U, dt, p), U - dt * oracle.flux_divergence(Us, p), rtol=0, atol=1e-15)
    ph = oracle.params(shape=U.shape, integrator="heun")
    U1 = U - dt * oracle.flux_divergence(U, ph)
    want = 0.5 * (U + U1 - dt * oracle.flux_divergence(U1, ph))
    assert np.allclose(oracle.step(U, dt, ph), want, rtol=0, atol=1e-15)
    p3 = oracle.params(shape=U.shape, integrator="ssprk3")
    U1 = U - dt * oracle.flux_divergence(U, p3)
    U2 = 0.75 * U + 0.25 * (U1 - dt * oracle.flux_divergence(U1, p3))
    want = U / 3 + (2 / 3) * (U2 - dt * oracle.flux_divergence(U2, p3))
    assert np.allclose(oracle.step(U, dt, p3), want, rtol=0, atol=1e-15)


@pytest.mark.parametrize("integrator,order", [("vl2", 2), ("heun", 2), ("ssprk3", 3)])
def test_temporal_order_of_the_integrators(integrator, order):
    """PAPER.md:843-845 ("second-order RK2 (Heun's method), third-order SSPRK3"): with the spatial operator frozen
    (first-order reconstruction on a smooth supersonic flow, where D is a smooth function of U) the error of one step
    against a finely sub-stepped solution falls as dt^(order+1): halving dt divides it by 2^(order+1).  A wrong stage
    weight lowers the order and fails this."""
    n, g = 8, 5 / 3
    x = (np.arange(n) + 0.5) / n
    Z, Y, X = np.meshgrid(x, x, x, indexing="ij")
    rho = 1.0 + 0.1 * np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Y)
    v = [3.0 + 0.1 * np.sin(2 * np.pi * Z), 2.5 + 0.1 * np.cos(2 * np.pi * X), 2.8 + 0.1 * np.sin(2 * np.pi * Y)]
    P = 0.6 + 0.05 * np.cos(2 * np.pi * (X + Z))
    U = _cons(rho, v, P, g)
    p = oracle.params(gamma=g, shape=U.shape, limiter="constant", integrator=integrator)
    T = 0.2 * oracle.cfl_dt(U, p)[0]

    def run(k):
        V = U.copy()
        for _ in range(k):
            V = oracle.step(V, T / k, p)
        return V

    ref = run(64)
    e1, e2 = np.abs(run(1) - ref).max(), np.abs(run(2) - ref).max()
    # global error over the fixed interval T: e(dt) ~ dt^order
    rate = math.log2(e1 / e2)
    assert abs(rate - order) < 0.25, (e1, e2, rate)


def test_flux_divergence_of_1d_profile_by_hand():
    """D(U) on a 1D piecewise profile equals (F_{i+1/2} - F_{i-1/2})/dx assembled from the oracle's own
    reconstruct() and riemann() pieces along each axis (checks indexing, roll direction A5, dx)."""
    g = 1.4
    n = 12
    rng = np.random.default_rng(12)
    W = np.stack([rng.uniform(0.5, 2, n), *rng.normal(0, 0.5, (3, n)), rng.uniform(0.5, 2, n)])
    for ax in range(3):
        shape = _line_shape(n, ax)
        dx = [0.3, 0.7, 1.1]
        p = oracle.params(gamma=g, dx=dx)
        U = _cons(_along(ax, W[0], shape), [_along(ax, W[1 + c], shape) for c in range(3)], _along(ax, W[4], shape), g)
        D = np.moveaxis(oracle.flux_divergence(U, p), 3 - ax, -1)[:, 0, 0, :]
        WL, WR = oracle.reconstruct(W, p)
        F = oracle.riemann(WL, WR, ax, p)
        want = (F - np.roll(F, 1, axis=1)) / dx[ax]
        assert np.allclose(D, want, rtol=0, atol=1e-13)


@pytest.mark.slow
def test_sedov_taylor_radius_law():
    """Config 2 at reduced size (48^3, fp64 oracle): R_s(t_end) within 7% of 1.15 (E t^2/rho)^(1/5) = 0.3,
    log-log slope of R_s(t) = 0.4 +- 0.04, energy conserved, octant symmetry kept."""
    import torch
    from paper_2512_13403_b200 import workloads
    n = 48
    wl = workloads.sedov(n, dtype=torch.float64)
    U = wl.U.numpy()
    p = oracle.params(gamma=wl.gamma, shape=U.shape)
    x = (np.arange(n) + 0.5) / n
    r = np.sqrt((x[None, None, :] - 0.5) ** 2 + (x[None, :, None] - 0.5) ** 2 + (x[:, None, None] - 0.5) ** 2)
    bins = np.arange(0, 0.5, 1.0 / n)

    def radius(U):
        which = np.digitize(r.ravel(), bins) - 1
        prof = np.bincount(which, U[0].ravel(), len(bins)) / np.maximum(np.bincount(which, minlength=len(bins)), 1)
        half = 0.5 * (prof.max() + 1.0)
        k = np.nonzero(prof >= half)[0].max()           # outermost shell above half height
        # linear interpolation of the crossing between shell k and k+1
        rc = 0.5 * (bins[:-1] + bins[1:])
        rc = np.append(rc, bins[-1] + 0.5 / n)
        return rc[k] + (prof[k] - half) / (prof[k] - prof[k + 1]) * (rc[k + 1] - rc[k])

    E0 = math.fsum(U[4].ravel())
    t, ts, rs = 0.0, [], []
    checkpoints = [wl.t_end / 4, wl.t_end / 2, wl.t_end]
    for tc in checkpoints:
        while t < tc * (1 - 1e-13):
            dt = min(oracle.cfl_dt(U, p, 0.4)[0], tc - t)
            U = oracle.step(U, dt, p)
            t += dt
        ts.append(t)
        rs.append(radius(U))
    assert abs(rs[-1] - 0.3) / 0.3 <= 0.07, rs
    slope = np.polyfit(np.log(ts), np.log(rs), 1)[0]
    assert abs(slope - 0.4) <= 0.04, slope
    assert abs(math.fsum(U[4].ravel()) - E0) <= 1e-12 * E0
    assert np.abs(U[0] - U[0][::-1]).max() < 1e-9 and np.abs(U[0] - U[0].transpose(2, 1, 0)).max() < 1e-9
