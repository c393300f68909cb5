"""Pins for oracle.decision_margins / cooling_margins and the stencil composition of tests/vjp_margins.py (the
instrument behind the fp32 VJP parity check).  None of them retypes a margin formula:

* along a line U(t) = U + t V the oracle's VJP is piecewise smooth in t; the first jump is located by bisection on the
  VJP itself.  At the jump (i) every entry that changes must be flagged (margin ~ 0 in its stencil): a compare the
  margins forgot, or a stencil drawn too small, leaves a changed entry unflagged; (ii) only a bounded neighbourhood may
  be flagged: margins that cry wolf everywhere fail.  Repeated over limiters, Riemann solvers, integrators, cooling
  and Mach numbers so that every kind of compare produces first jumps;
* constructed ties of the limiter (|a| = |b|, a = 0) at a known cell: the margin there is the constructed offset;
* a perturbation of fp32 size changes no well-conditioned entry by more than a smooth amount, while it does flip
  ill-conditioned ones (the situation of the GPU parity tests, reproduced on the CPU).
"""
import numpy as np
import pytest

import oracle
from vjp_margins import FP32_BOUND, plus_min, stage_condition, vjp_condition


def _state(shape, seed, g=5 / 3, mach=0.5):
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.6, 1.8, shape)
    v = rng.normal(0, mach, (3,) + shape)
    P = rng.uniform(0.6, 1.8, shape)
    return np.stack([rho, rho * v[0], rho * v[1], rho * v[2], P / (g - 1) + 0.5 * rho * (v ** 2).sum(0)])


def _from_prims(W, g):
    rho, vx, vy, vz, P = W
    return np.stack([rho, rho * vx, rho * vy, rho * vz, P / (g - 1) + 0.5 * rho * (vx ** 2 + vy ** 2 + vz ** 2)])


LINE_CASES = [
    dict(), dict(mach=1.5), dict(mach=0.05),
    dict(limiter="vanleer"), dict(limiter="mc"),
    dict(riemann="hll", mach=1.2), dict(riemann="rusanov"), dict(riemann="rusanov", mach=1.5),
    dict(integrator="heun"), dict(integrator="ssprk3"),
    dict(cooling=True, lambda0=40.0, t_floor=0.6), dict(cooling=True, lambda0=40.0, t_floor=0.6, cool_nsub=3),
    dict(cooling=True, lambda0=40.0, t_floor=0.6, cool_mode="trapezoid"),
    dict(twobranch=True), dict(twobranch=True, cool_mode="masked", cool_nsub=3, f_sub=0.3),
]


@pytest.mark.parametrize("kw", LINE_CASES, ids=lambda k: "-".join(f"{a}={b}" for a, b in k.items()) or "default")
def test_every_jump_of_the_vjp_along_a_line_is_flagged_and_only_its_neighbourhood(kw):
    kw = dict(kw)
    mach = kw.pop("mach", 0.5)
    shape = (6, 7, 8)
    if kw.pop("twobranch", False):                       # Eqs. 17-19: switch temperature and table nodes inside the gas' range
        from paper_2512_13403_b200 import workloads
        logT0, dlogT, vals = workloads.cooling_table(log10_t_lo=-0.13, log10_t_hi=0.6, n=5)   # t_switch inside the first interval
        kw.update(cooling=True, cool_law="twobranch", t_switch=1.0, lambda1=8.0, alpha1=2.0, lambda2=4.0, alpha2=0.5, gamma0=3.0,
                  table=(logT0, dlogT, vals.numpy() + 2.3), t_floor=0.3)
    p = oracle.params(shape=shape, **kw)
    found = 0
    for seed in range(6):
        U = _state(shape, 1000 + seed, mach=mach)
        rng = np.random.default_rng(2000 + seed)
        V = rng.normal(size=U.shape) * np.abs(U).mean(axis=(1, 2, 3), keepdims=True)
        g = rng.normal(size=U.shape)
        dt = oracle.cfl_dt(U, p)[0]
        vjp = lambda t: oracle.step_vjp(U + t * V, dt, g, p)
        start, T = 0.0, 2e-3
        for _ in range(8):                               # walk from jump to jump along the line
            g0 = vjp(start)
            rms = float(np.sqrt(np.mean(g0 ** 2)))
            jumped = lambda t: float(np.abs(vjp(t) - g0).max()) > 0.05 * rms
            hi = min(T, start + 5e-4)
            if not jumped(hi):
                start = hi
                if start >= T:
                    break
                continue
            lo = start
            while hi - lo > 1e-13:
                mid = 0.5 * (lo + hi)
                if jumped(mid):
                    hi = mid
                else:
                    lo = mid
            start = hi + 1e-12
            ga, gb = vjp(lo), vjp(hi)
            changed = (np.abs(ga - gb) > 1e-6 * rms).any(axis=0)
            if not changed.any():                        # steep but continuous (e.g. van Leer near a = b = 0): not a jump
                continue
            cond = np.minimum(vjp_condition(U + lo * V, dt, p), vjp_condition(U + hi * V, dt, p))
            flagged = cond <= 1e-9
            assert not (changed & ~flagged).any(), (seed, int((changed & ~flagged).sum()), float(cond[changed].max()))
            assert flagged.mean() <= (0.9 if p.integrator == 2 else 0.7), (seed, float(flagged.mean()))
            found += 1
    assert found >= 10, found


@pytest.mark.parametrize("axis", [0, 1, 2])
@pytest.mark.parametrize("field", [0, 2, 4])
def test_constructed_limiter_ties_have_the_constructed_margin(axis, field):
    """|a| = |b| (1 + delta) and a = delta on one primitive at one cell: the margin of that cell and axis is the offset
    divided by the scale, every other compare of a random state is far from its tie."""
    g = 5 / 3
    shape = (6, 7, 8)
    p = oracle.params(shape=shape, gamma=g)
    W0 = oracle.prims(_state(shape, 77, g), p)
    c = [3, 2, 4]                                        # (k, j, i)
    ax = 2 - axis                                        # numpy axis of the direction
    up, dn = list(c), list(c)
    up[ax] += 1
    dn[ax] -= 1
    for kind, delta in (("compare", 1e-7), ("sign", 1e-8)):
        W = W0.copy()
        b = W[(field,) + tuple(c)] - W[(field,) + tuple(dn)]
        if kind == "compare":
            W[(field,) + tuple(up)] = W[(field,) + tuple(c)] + b * (1 + delta)
            offset = abs(b) * delta
        else:
            W[(field,) + tuple(up)] = W[(field,) + tuple(c)] + np.sign(b) * delta
            offset = delta
        M = oracle.decision_margins(_from_prims(W, g), p)
        got = M[(axis,) + tuple(c)]
        assert 0.05 * offset <= got <= 20 * offset, (kind, got, offset)
        rest = M[:3].copy()
        rest[(axis,) + tuple(c)] = 1.0
        if kind == "sign":                               # the tiny difference is also the b of the next cell's limiter call
            assert 0.05 * offset <= rest[(axis,) + tuple(up)] <= 20 * offset
            rest[(axis,) + tuple(up)] = 1.0
        assert rest.min() > 100 * got


def test_uniform_data_is_not_a_tie_and_floors_are_seen():
    shape = (6, 6, 6)
    g = 5 / 3
    one = np.ones(shape)
    U = _from_prims(np.stack([1.3 * one, 0.2 * one, -0.1 * one, 0.4 * one, 0.9 * one]), g)
    p = oracle.params(shape=shape, gamma=g)
    M = oracle.decision_margins(U, p)
    assert M[:3].min() > 0.05    # a = b = 0 and L = R exactly: identical operands everywhere
    assert M[3].min() > 0.5
    U2 = U.copy()
    U2[4, 2, 3, 4] = 0.5 * 1.3 * (0.04 + 0.01 + 0.16) + 1e-10 / (g - 1) * (1 + 1e-6)   # pressure at the floor (+1e-6)
    M2 = oracle.decision_margins(U2, p)
    assert M2[3, 2, 3, 4] < 1e-5 and np.delete(M2[3].ravel(), (2 * 6 + 3) * 6 + 4).min() > 0.5


def test_cooling_margin_is_the_distance_to_the_floor():
    shape = (4, 4, 4)
    g = 5 / 3
    rng = np.random.default_rng(5)
    rho = rng.uniform(0.5, 2, shape)
    T = rng.uniform(0.5, 2, shape)
    U = _from_prims(np.stack([rho, 0 * rho, 0 * rho, 0 * rho, rho * T]), g)
    p = oracle.params(shape=shape, gamma=g, cooling=True, lambda0=1.0, alpha=0.5, t_floor=0.3)
    dt = 0.2
    out = oracle.cooling(U, dt, p)
    Tn = (g - 1) * out[4] / rho
    free = T - (g - 1) * rho * np.sqrt(T) * dt            # the closed form of test_oracle_pieces (gas at rest, alpha = 1/2)
    M = oracle.cooling_margins(U, dt, p)
    expect = np.abs(free - 0.3) / T                       # |E_th' - E_floor| / E_th
    assert np.allclose(M, np.minimum(expect, 1.0), rtol=1e-12)
    assert ((Tn == 0.3) == (free < 0.3)).all() or np.allclose(Tn[free < 0.3], 0.3)


def test_masked_integrator_choice_has_the_distance_to_its_criterion_as_margin():
    """A cell whose dt |Edot| equals f_sub |E_th| (found by bisection on the oracle's own rate) has margin ~ 0; moved
    away from it by a relative d the margin is ~ d."""
    g = 5 / 3
    p = oracle.params(shape=(1, 1, 1), dx=(1, 1, 1), gamma=g, cooling=True, lambda0=2.0, alpha=0.5, t_floor=1e-3,
                      cool_mode="masked", cool_nsub=4, f_sub=0.2)
    rho, dt = 1.4, 0.3
    crit = lambda E: dt * abs(oracle.cool_rate(E, rho, p)) - 0.2 * E
    lo, hi = 1e-3, 1e3                                    # rate ~ sqrt(E): rapid (crit > 0) at small E, slow at large E
    assert crit(lo) > 0 > crit(hi)
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if crit(mid) > 0 else (lo, mid)
    E0 = 0.5 * (lo + hi)
    for d in (0.0, 1e-6, 1e-3):
        U = np.array([rho, 0.0, 0.0, 0.0, E0 * (1 + d)]).reshape(5, 1, 1, 1)
        m = float(oracle.cooling_margins(U, dt, p)[0, 0, 0])
        assert (m <= 1e-12) if d == 0.0 else (0.2 * d <= m <= 5 * d), (d, m)


@pytest.mark.parametrize("case", ["random", "turbulence"])
def test_fp32_sized_perturbation_moves_only_flagged_entries(case):
    """The GPU parity situation on the CPU: the oracle at U (1 + 2^-24 xi) against the oracle at U.  Entries whose
    stencil margin is above FP32_BOUND move smoothly (<= 2e-5 of the rms); on the smooth turbulence recipe (neighbouring
    differences nearly equal) a few percent of the entries are flagged and some of those do jump."""
    import torch
    from paper_2512_13403_b200 import workloads
    g = 5 / 3
    rng = np.random.default_rng(11)
    if case == "random":
        shape = (16, 16, 16)
        U = _state(shape, 12, g)
        p = oracle.params(shape=shape, gamma=g)
    else:
        U = workloads.turbulence(24, seed=3, mach=1.0, dtype=torch.float64).U.numpy()
        shape = U.shape[1:]
        p = oracle.params(shape=shape, gamma=g)
        for _ in range(2):                                # leave the exactly uniform initial pressure behind
            U = oracle.step(U, oracle.cfl_dt(U, p)[0], p)
    dt = oracle.cfl_dt(U, p)[0]
    gg = rng.normal(size=U.shape)
    ref = oracle.step_vjp(U, dt, gg, p)
    cond = vjp_condition(U, dt, p)
    well = cond >= FP32_BOUND
    rms = np.sqrt(np.mean(ref ** 2))
    worst_well, worst_ill = 0.0, 0.0
    for trial in range(6):
        Up = U * (1 + 2.0 ** -24 * rng.uniform(-1, 1, U.shape))
        e = np.abs(oracle.step_vjp(Up, dt, gg, p) - ref) / rms
        worst_well = max(worst_well, float(e[:, well].max()))
        if (~well).any():
            worst_ill = max(worst_ill, float(e[:, ~well].max()))
    assert worst_well <= 2e-5, worst_well
    assert well.mean() > 0.9, float(well.mean())
    if case == "turbulence":
        assert well.mean() < 0.999 and worst_ill > 1e-3, (float(well.mean()), worst_ill)
