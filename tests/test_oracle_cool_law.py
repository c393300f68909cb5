"""Pins for the two-branch heating / cooling law (Eqs. 17-19; reading A25), the masked choice of the
integrator (reading A26) and the gradient with respect to the table:

* the tabulated branch: exact at the nodes, geometric-mean property at interval midpoints and equal log-log slopes inside an
  interval (what "linear interpolation in log T - log Lambda" means), end values held outside;
* a table that samples a power law reproduces the power-law law of reading A10 (index, weights and units of the lookup);
* the lower branch: Eq. 18 + uniform heating: thermal equilibrium where Gamma_0 = n Lambda_KI(T_eq) (gas neither heats nor
  cools, the rate changes sign across it), reduction to the power law when the second term and the heating vanish;
* the switch: with the recipe's table (first node matched to Eq. 18) Lambda is continuous at t_switch and Edot jumps by
  exactly the heating term rho Gamma_0;
* masked integrator = the trapezoid where dt |Edot| <= f_sub |E_th|, the sub-cycled update elsewhere;
* VJP of the step with respect to the state: dual-number transpose identity and finite differences; with respect to the
  table nodes: finite differences, and the sum rule (raising every node by d log Lambda scales Lambda everywhere).
"""
import numpy as np
import pytest

import oracle
from paper_2512_13403_b200 import workloads

G = 5 / 3


def _kw(**over):
    logT0, dlogT, vals = workloads.cooling_table()
    lam1, a1, lam2, a2 = 2.0e-2, 2.0, 1.0e-2, 0.5
    kw = dict(cooling=True, cool_law="twobranch", t_switch=1.0, lambda1=lam1, alpha1=a1, lambda2=lam2, alpha2=a2,
              gamma0=8.0e-3, table=(logT0, dlogT, vals.numpy()), t_floor=0.05)
    kw.update(over)
    return kw


def _state(shape, seed, mach=0.5, tlo=0.2, thi=8.0):
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.5, 2.0, shape)
    v = rng.normal(0, mach, (3,) + shape)
    T = np.exp(rng.uniform(np.log(tlo), np.log(thi), shape))         # both branches of Eq. 17 populated
    return np.stack([rho, rho * v[0], rho * v[1], rho * v[2], rho * T / (G - 1) + 0.5 * rho * (v ** 2).sum(0)])


def test_table_is_exact_at_nodes_loglinear_between_and_held_outside():
    p = oracle.params(shape=(4, 4, 4), **_kw())
    logT0, dlogT, vals = workloads.cooling_table()
    vals = vals.numpy()
    for k in range(len(vals)):
        assert np.isclose(oracle.lambda_table(10 ** (logT0 + k * dlogT), p), 10 ** vals[k], rtol=1e-12)
    for k in (0, 5, len(vals) - 2):
        Ta, Tb = 10 ** (logT0 + k * dlogT), 10 ** (logT0 + (k + 1) * dlogT)
        mid = oracle.lambda_table(np.sqrt(Ta * Tb), p)
        assert np.isclose(mid, np.sqrt(10 ** vals[k] * 10 ** vals[k + 1]), rtol=1e-12)       # geometric mean at the midpoint
        ts = Ta * (Tb / Ta) ** np.array([0.1, 0.35, 0.8])
        ls = np.log([oracle.lambda_table(t, p) for t in ts])
        s1 = (ls[1] - ls[0]) / np.log(ts[1] / ts[0])
        s2 = (ls[2] - ls[1]) / np.log(ts[2] / ts[1])
        assert abs(s1 - s2) <= 1e-10 * max(1.0, abs(s1))                                      # one slope per interval
        assert abs(s1 - (vals[k + 1] - vals[k]) / dlogT) <= 1e-10 * max(1.0, abs(s1))
    Tlast = 10 ** (logT0 + (len(vals) - 1) * dlogT)
    assert np.isclose(oracle.lambda_table(30 * Tlast, p), 10 ** vals[-1], rtol=1e-12)
    assert np.isclose(oracle.lambda_table(10 ** (logT0 - 1), p), 10 ** vals[0], rtol=1e-12)


def test_power_law_table_reproduces_the_power_law_law():
    """log10 Lambda = log10 lambda0 + alpha log10 T sampled at the nodes is linear in log T, so the interpolant IS the power
    law: with t_switch below every temperature the two laws must give the same update."""
    shape = (6, 5, 4)
    U = _state(shape, 3)
    lam0, alpha = 0.7, 0.5
    logT0, dlogT, n = -2.0, 0.25, 24
    tab = np.log10(lam0) + alpha * (logT0 + dlogT * np.arange(n))
    pa = oracle.params(shape=shape, cooling=True, lambda0=lam0, alpha=alpha, t_floor=0.05)
    pb = oracle.params(shape=shape, **_kw(t_switch=1e-30, table=(logT0, dlogT, tab)))
    for mode in (dict(), dict(cool_nsub=4), dict(cool_mode="trapezoid")):
        pa2 = oracle.params(shape=shape, cooling=True, lambda0=lam0, alpha=alpha, t_floor=0.05, **mode)
        pb2 = oracle.params(shape=shape, **_kw(t_switch=1e-30, table=(logT0, dlogT, tab), **mode))
        a, b = oracle.cooling(U, 0.3, pa2), oracle.cooling(U, 0.3, pb2)
        assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()
    assert pa.cool_law == 0 and pb.cool_law == 1


def test_lower_branch_equilibrium_and_reduction_to_the_power_law():
    kw = _kw()
    p = oracle.params(shape=(4, 4, 4), **kw)
    rho = 1.3
    # thermal equilibrium of Eq. 15 on the lower branch: Gamma_0 = rho Lambda_KI(T_eq); bisection on the oracle's own rate
    lo, hi = 1e-3, 0.999
    rate = lambda T: oracle.cool_rate(rho * T / (G - 1), rho, p)
    assert rate(lo) > 0 > rate(hi)                                    # heating wins when cold, cooling when warm
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        lo, hi = (mid, hi) if rate(mid) > 0 else (lo, mid)
    Teq = 0.5 * (lo + hi)
    assert np.isclose(kw["gamma0"], rho * (kw["lambda1"] * Teq ** kw["alpha1"] + kw["lambda2"] * Teq ** kw["alpha2"]), rtol=1e-10)   # Eq. 18
    U = np.zeros((5, 1, 1, 1))
    U[0], U[4] = rho, rho * Teq / (G - 1)
    pe = oracle.params(shape=(1, 1, 1), dx=(1, 1, 1), **kw)
    assert np.isclose(oracle.cooling(U, 5.0, pe)[4, 0, 0, 0], U[4, 0, 0, 0], rtol=1e-9)
    # second term and heating off, switch at infinity: the power law of reading A10
    shape = (5, 4, 6)
    Us = _state(shape, 8)
    pa = oracle.params(shape=shape, cooling=True, lambda0=0.4, alpha=1.5, t_floor=0.05)
    pb = oracle.params(shape=shape, **_kw(t_switch=1e30, lambda1=0.4, alpha1=1.5, lambda2=0.0, gamma0=0.0))
    a, b = oracle.cooling(Us, 0.2, pa), oracle.cooling(Us, 0.2, pb)
    assert np.abs(a - b).max() <= 1e-14 * np.abs(a).max()


def test_switch_temperature_lambda_continuous_rate_jumps_by_the_heating_term():
    kw = _kw()
    lam_sw = kw["lambda1"] + kw["lambda2"]                             # Eq. 18 at T = t_switch = 1
    logT0, dlogT, vals = workloads.cooling_table(lambda_lo=lam_sw)
    kw["table"] = (logT0, dlogT, vals.numpy())
    p = oracle.params(shape=(4, 4, 4), **kw)
    rho = 0.8
    below = oracle.cool_rate(rho * (1 - 1e-12) / (G - 1), rho, p)
    above = oracle.cool_rate(rho * (1 + 1e-12) / (G - 1), rho, p)
    assert np.isclose(below - above, rho * kw["gamma0"], rtol=1e-8)
    assert np.isclose(above, -rho * rho * lam_sw, rtol=1e-9)


@pytest.mark.parametrize("f_sub", [0.05, 0.3])
def test_masked_integrator_is_the_trapezoid_or_the_subcycled_update_per_cell(f_sub):
    shape = (6, 6, 6)
    U = _state(shape, 21)
    dt = 0.8
    kw = _kw(lambda1=0.3, lambda2=0.2, gamma0=0.05, cool_nsub=4)
    pm = oracle.params(shape=shape, cool_mode="masked", f_sub=f_sub, **kw)
    pt = oracle.params(shape=shape, cool_mode="trapezoid", **kw)
    ps = oracle.params(shape=shape, cool_mode="euler", **kw)
    rho = U[0]
    Eth = U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / rho
    rate = np.vectorize(lambda e, r: oracle.cool_rate(e, r, pm))(Eth, rho)
    rapid = dt * np.abs(rate) > f_sub * np.abs(Eth)
    assert 0.1 < rapid.mean() < 0.9                                   # both paths taken
    out = oracle.cooling(U, dt, pm)
    want = np.where(rapid, oracle.cooling(U, dt, ps)[4], oracle.cooling(U, dt, pt)[4])
    assert np.array_equal(out[4], want) and np.array_equal(out[:4], U[:4])


STEP_CASES = [dict(), dict(cool_nsub=3), dict(cool_mode="trapezoid"), dict(cool_mode="masked", cool_nsub=3, f_sub=0.02),
              dict(cool_mode="masked", cool_nsub=2, f_sub=0.02, integrator="ssprk3")]


@pytest.mark.parametrize("case", STEP_CASES, ids=lambda k: "-".join(f"{a}={b}" for a, b in k.items()) or "euler")
def test_step_vjp_with_the_two_branch_law(case):
    """<g, J v> = <J^T g, v> with J v by dual numbers through the whole step, and central finite differences."""
    shape = (8, 8, 8)
    U = _state(shape, 31, mach=0.3)
    p = oracle.params(shape=shape, **_kw(lambda1=0.3, lambda2=0.2, gamma0=0.05, **case))
    dt = oracle.cfl_dt(U, p)[0]
    rng = np.random.default_rng(32)
    g = rng.normal(size=U.shape)
    gin = oracle.step_vjp(U, dt, g, p)
    assert np.abs(oracle.step(U, dt, p)[4] - oracle.step_nocool(U, dt, p)[4]).max() > 1e-4     # the source really acts
    for _ in range(3):
        v = rng.normal(size=U.shape)
        out, Jv = oracle.step_jvp(U, v, dt, p)
        lhs, rhs = float((g * Jv).sum()), float((gin * v).sum())
        assert abs(lhs - rhs) <= 1e-12 * (np.abs(g * Jv).sum() + np.abs(gin * v).sum())
    eps = 1e-7
    v = rng.normal(size=U.shape)
    fd = (oracle.step(U + eps * v, dt, p) - oracle.step(U - eps * v, dt, p)) / (2 * eps)
    lhs, rhs = float((g * fd).sum()), float((gin * v).sum())
    assert abs(lhs - rhs) <= 2e-6 * abs(rhs), (lhs, rhs)


@pytest.mark.parametrize("mode", [dict(), dict(cool_nsub=3), dict(cool_mode="trapezoid")], ids=["euler", "nsub3", "trapezoid"])
def test_gradient_with_respect_to_the_table(mode):
    shape = (6, 6, 6)
    U1 = _state(shape, 41, tlo=0.5, thi=60.0)
    kw = _kw(**mode)
    p = oracle.params(shape=shape, **kw)
    dt = 0.5
    rng = np.random.default_rng(42)
    g = rng.normal(size=U1.shape)
    gt = oracle.cooling_table_vjp(U1, dt, g, p)
    assert np.count_nonzero(gt) >= 10                                  # the gas samples most of the table
    logT0, dlogT, vals = kw["table"]
    L = lambda tab: float((g[4] * oracle.cooling(U1, dt, oracle.params(shape=shape, **dict(kw, table=(logT0, dlogT, tab))))[4]).sum())
    eps = 1e-6
    for k in (1, 4, 9, len(vals) - 2):
        e = np.zeros_like(vals)
        e[k] = eps
        fd = (L(vals + e) - L(vals - e)) / (2 * eps)
        assert abs(fd - gt[k]) <= 2e-4 * abs(fd) + 1e-6 * np.abs(gt).max(), (k, fd, gt[k])   # (cells at a floor kink limit the FD)
    # raising every node by d multiplies Lambda_CIE by 10^d wherever the table is used: d L = sum_k gt[k] d
    d = 1e-6
    assert np.isclose((L(vals + d) - L(vals - d)) / (2 * d), gt.sum(), rtol=2e-4)
