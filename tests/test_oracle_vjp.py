"""Pins for the oracle's reverse mode (SURVEY.md §8(c) row "VJP"): central finite differences on 8^3,
exact dual-number JVP dot-product identity, the closed form that conservation implies, linearity, and
structure (reach of the cotangent stencil)."""
import numpy as np
import pytest

import oracle


def _state(shape, seed, g=5 / 3, amp=0.3):
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.6, 1.8, shape)
    v = rng.normal(0, amp, (3,) + shape)
    P = rng.uniform(0.6, 1.8, shape)
    return np.stack([rho, rho * v[0], rho * v[1], rho * v[2], P / (g - 1) + 0.5 * rho * (v ** 2).sum(0)])


CASES = [
    dict(),
    dict(cooling=True, lambda0=0.5),
    dict(limiter="vanleer"),
    dict(limiter="mc"),
    dict(riemann="hll"),
    dict(riemann="rusanov"),
    dict(integrator="heun"),
    dict(integrator="heun", cooling=True, lambda0=0.5),
    dict(integrator="ssprk3"),
    dict(integrator="ssprk3", cooling=True, lambda0=0.5),
    dict(cooling=True, lambda0=0.5, cool_nsub=4),
    dict(cooling=True, lambda0=0.5, cool_mode="trapezoid"),
]


@pytest.mark.parametrize("kw", CASES, ids=lambda k: "-".join(f"{a}={b}" for a, b in k.items()) or "default")
def test_vjp_equals_transposed_dual_number_jvp(kw):
    """<g, J v> = <J^T g, v> to rounding, J v from one-slot dual numbers pushed through the whole step."""
    shape = (8, 8, 8)
    U = _state(shape, 21)
    p = oracle.params(shape=shape, **kw)
    dt = oracle.cfl_dt(U, p)[0]
    rng = np.random.default_rng(22)
    g = rng.normal(size=U.shape)
    gin = oracle.step_vjp(U, dt, g, p)
    for _ in range(3):
        v = rng.normal(size=U.shape)
        out, Jv = oracle.step_jvp(U, v, dt, p)
        assert np.array_equal(out, oracle.step(U, dt, p))
        lhs, rhs = float((g * Jv).sum()), float((gin * v).sum())
        assert abs(lhs - rhs) <= 1e-13 * (np.abs(g * Jv).sum() + np.abs(gin * v).sum())


@pytest.mark.parametrize("kw", [dict(), dict(cooling=True, lambda0=0.5), dict(integrator="heun"), dict(integrator="ssprk3"),
                                dict(cooling=True, lambda0=0.5, cool_nsub=4), dict(cooling=True, lambda0=0.5, cool_mode="trapezoid")],
                         ids=["hydro", "cooling", "heun", "ssprk3", "cooling-nsub4", "cooling-trapezoid"])
def test_vjp_against_central_finite_differences(kw):
    """BASELINE requirement: 8^3 fp64, <g, (H(U+eps v) - H(U-eps v)) / 2 eps> vs <J^T g, v>.
    The scheme is piecewise smooth (limiter / HLLC / floor switches); eps is small enough that for these
    seeds no switch is crossed, which the tight agreement itself demonstrates."""
    shape = (8, 8, 8)
    U = _state(shape, 31)
    p = oracle.params(shape=shape, **kw)
    dt = oracle.cfl_dt(U, p)[0]
    rng = np.random.default_rng(32)
    g = rng.normal(size=U.shape)
    gin = oracle.step_vjp(U, dt, g, p)
    eps = 1e-7
    for _ in range(4):
        v = rng.normal(size=U.shape)
        fd = (oracle.step(U + eps * v, dt, p) - oracle.step(U - eps * v, dt, p)) / (2 * eps)
        lhs, rhs = float((g * fd).sum()), float((gin * v).sum())
        assert abs(lhs - rhs) <= 1e-6 * abs(rhs), (lhs, rhs)


def test_vjp_fd_single_components():
    """Entry by entry: perturb single cells/fields and compare with that entry of J^T g.  (A generic
    random state is used on purpose: grid-symmetric analytic profiles sit exactly on the limiter's
    ties |a| = |b| and a b = 0, where the one-sided derivative of reading A7 and a central difference
    legitimately differ.)"""
    shape = (8, 8, 8)
    g0 = 5 / 3
    U = _state(shape, 34)
    p = oracle.params(shape=shape, gamma=g0)
    dt = oracle.cfl_dt(U, p)[0]
    rng = np.random.default_rng(33)
    g = rng.normal(size=U.shape)
    gin = oracle.step_vjp(U, dt, g, p)
    eps = 1e-7
    for f, k, j, i in [(0, 1, 2, 3), (1, 0, 0, 0), (2, 7, 7, 7), (3, 4, 0, 6), (4, 3, 5, 1)]:
        e = np.zeros_like(U)
        e[f, k, j, i] = 1.0
        fd = float((g * (oracle.step(U + eps * e, dt, p) - oracle.step(U - eps * e, dt, p))).sum() / (2 * eps))
        assert abs(fd - gin[f, k, j, i]) <= 2e-7 * max(1.0, abs(fd)), (f, k, j, i, fd, gin[f, k, j, i])


@pytest.mark.parametrize("integrator", ["vl2", "heun", "ssprk3"])
def test_vjp_of_constant_cotangent_is_itself(integrator):
    """sum_i U_f is invariant under the step (no cooling) => J^T 1_f = 1_f exactly up to rounding."""
    shape = (6, 7, 8)
    U = _state(shape, 41)
    p = oracle.params(shape=shape, integrator=integrator)
    dt = oracle.cfl_dt(U, p)[0]
    for f in range(5):
        g = np.zeros_like(U)
        g[f] = 1.0
        gin = oracle.step_vjp(U, dt, g, p)
        assert np.abs(gin - g).max() <= 1e-13


def test_vjp_is_linear_in_the_cotangent():
    shape = (6, 6, 6)
    U = _state(shape, 51)
    p = oracle.params(shape=shape)
    dt = oracle.cfl_dt(U, p)[0]
    rng = np.random.default_rng(52)
    g1, g2 = rng.normal(size=U.shape), rng.normal(size=U.shape)
    a = oracle.step_vjp(U, dt, 2.0 * g1 - 3.0 * g2, p)
    b = 2.0 * oracle.step_vjp(U, dt, g1, p) - 3.0 * oracle.step_vjp(U, dt, g2, p)
    assert np.abs(a - b).max() <= 1e-13 * np.abs(a).max()


def test_vjp_stencil_reach_and_window():
    """A delta cotangent at one cell reaches at most +-4 cells per axis (two stages x halo 2), and the
    windowed VJP reproduces the full-grid one on the window interior."""
    shape = (20, 20, 20)
    U = _state(shape, 61)
    p = oracle.params(shape=shape)
    dt = oracle.cfl_dt(U, p)[0]
    g = np.zeros_like(U)
    g[4, 10, 10, 10] = 1.0
    gin = oracle.step_vjp(U, dt, g, p)
    nz = np.nonzero(np.abs(gin).sum(0))
    for a in range(3):
        assert nz[a].min() >= 6 and nz[a].max() <= 14        # never beyond +-4
        assert nz[a].min() <= 8 and nz[a].max() >= 12        # minmod drops one of (a, b): reach can be 3
    rng = np.random.default_rng(62)
    g = rng.normal(size=U.shape)
    full = oracle.step_vjp(U, dt, g, p)
    win = oracle.window_step_vjp(U, dt, g, p, lo=(17, 0, 9), size=(5, 4, 6))
    idx = [np.arange(lo, lo + s) % 20 for lo, s in zip((17, 0, 9), (5, 4, 6))]
    want = full[:, idx[0][:, None, None], idx[1][None, :, None], idx[2][None, None, :]]
    # scatter-add order differs between the window and the full grid: equal to rounding, not bitwise
    assert np.abs(win - want).max() <= 1e-14 * np.abs(want).max()
    fwin = oracle.window_step(U, dt, p, lo=(17, 0, 9), size=(5, 4, 6))
    fwant = oracle.step(U, dt, p)[:, idx[0][:, None, None], idx[1][None, :, None], idx[2][None, None, :]]
    assert np.array_equal(fwin, fwant)


def test_stage_vjp_matches_dense_jacobian_on_tiny_grid():
    """Brute force: build the full Jacobian of V = -tau D(U) column by column with the dual-number JVP of
    a full step is not available per stage, so use central differences of D() on a 4x4x4 grid and compare
    J^T g with the scatter-form stage VJP."""
    shape = (4, 4, 4)
    U = _state(shape, 71, amp=0.2)
    p = oracle.params(shape=shape)
    tau = 0.003
    rng = np.random.default_rng(72)
    g = rng.normal(size=U.shape)
    got = oracle.stage_vjp(U, tau, g, p)
    eps = 1e-6
    want = np.zeros_like(U)
    flat = want.reshape(-1)
    for m in range(flat.size):
        e = np.zeros(flat.size)
        e[m] = eps
        e = e.reshape(U.shape)
        dD = (oracle.flux_divergence(U + e, p) - oracle.flux_divergence(U - e, p)) / (2 * eps)
        flat[m] = -tau * float((g * dD).sum())
    assert np.abs(got - want).max() <= 5e-8 * max(1.0, np.abs(want).max())


def test_multistep_adjoint_against_finite_differences():
    """oracle.adjoint (composition of step_vjp with the dt sequence frozen) against central finite
    differences of L(U_0) = <g, H_dt3(H_dt2(H_dt1(U_0)))> along random directions, 6^3 fp64."""
    rng = np.random.default_rng(77)
    shape = (6, 6, 6)
    rho = rng.uniform(0.8, 1.5, shape)
    v = rng.normal(0, 0.3, (3,) + shape)
    P = rng.uniform(0.8, 1.5, shape)
    gamma = 1.4
    U0 = np.stack([rho, rho * v[0], rho * v[1], rho * v[2], P / (gamma - 1) + 0.5 * rho * (v ** 2).sum(0)])
    p = oracle.params(gamma=gamma, shape=U0.shape)
    g = rng.normal(size=U0.shape)
    Un, g0, dts = oracle.adjoint(U0, 3, g, p)
    assert len(dts) == 3 and all(d > 0 for d in dts)

    def run(U):
        for d in dts:                                      # dt sequence held constant
            U = oracle.step(U, d, p)
        return U

    assert np.array_equal(run(U0), Un)
    for _ in range(3):
        w = rng.normal(size=U0.shape)
        eps = 1e-6
        fd = float(((run(U0 + eps * w) - run(U0 - eps * w)) * g).sum() / (2 * eps))
        an = float((g0 * w).sum())
        assert abs(fd - an) <= 2e-6 * max(abs(fd), abs(an), 1e-3), (fd, an)
