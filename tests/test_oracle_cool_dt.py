"""Pins for the oracle's cooling-time limit on dt, Eqs. 20-21 (reading A24).

None of them retypes the formula of t_cool: they tie it to the cooling ODE whose solution the paper's source term has
(already the pin of oracle.cooling), to the oracle's own Euler update, and to invariances."""
import numpy as np
import pytest

import oracle

G = 5.0 / 3.0


def _uniform(rho, v, T, shape=(2, 3, 4), g=G):
    U = np.empty((5,) + shape)
    U[0] = rho
    for c in range(3):
        U[1 + c] = rho * v[c]
    U[4] = rho * T / (g - 1) + 0.5 * rho * sum(x * x for x in v)
    return U


def _random_state(seed, n=(5, 6, 7), dtype=np.float64):
    rng = np.random.default_rng(seed)
    rho = np.exp(rng.normal(0, 0.5, n))
    v = rng.normal(0, 1, (3,) + n)
    T = rng.uniform(0.2, 3, n)
    return np.stack([rho, *(rho * v), rho * T / (G - 1) + 0.5 * rho * (v ** 2).sum(0)]).astype(dtype)


def test_tcool_is_half_the_time_to_zero_temperature_for_alpha_half():
    """alpha = 1/2: sqrt(T(t)) = sqrt(T0) - (gamma-1) lambda0 rho t / 2 reaches 0 at t0 = 2 sqrt(T0) / ((gamma-1) lambda0 rho);
    the initial slope -T0 / t_cool of T(t) gives t_cool = t0 / 2."""
    rho, T0, lam = 2.0, 1.44, 0.05
    p = oracle.params(gamma=G, dx=(1, 1, 1), cooling=True, lambda0=lam, alpha=0.5, t_floor=1e-6)
    tmin, _ = oracle.cool_dt(_uniform(rho, (0.3, -0.4, 0.2), T0), p, 1.0)
    t0 = 2 * 1.2 / ((G - 1) * lam * rho)      # = 36
    assert tmin == pytest.approx(t0 / 2, rel=1e-14)
    assert tmin == pytest.approx(18.0, rel=1e-14)


def test_tcool_is_the_e_folding_time_for_alpha_one():
    """alpha = 1: Edot = -E_th / t_cool exactly, so sub-cycled cooling over t_cool divides E_th by e (error ~ 1/(2 N_sub))."""
    rho, T0, lam, nsub = 1.7, 2.0, 0.03, 64
    p = oracle.params(gamma=G, dx=(1, 1, 1), cooling=True, lambda0=lam, alpha=1.0, t_floor=1e-9, cool_nsub=nsub)
    U = _uniform(rho, (0, 0, 0), T0)
    tmin, _ = oracle.cool_dt(U, p, 1.0)
    reps = 16                                  # 16 x 64 substeps over one t_cool
    V = U
    for _ in range(reps):
        V = oracle.cooling(V, tmin / reps, p)
    ratio = V[4, 0, 0, 0] / U[4, 0, 0, 0]
    n = reps * nsub
    assert ratio == pytest.approx((1 - 1 / n) ** n, rel=1e-12)    # the Euler recurrence for a linear ODE
    assert ratio == pytest.approx(np.exp(-1), rel=1e-3)


@pytest.mark.parametrize("alpha", [0.5, 0.7, 1.3])
def test_euler_update_changes_eth_by_at_most_ccool_with_equality_at_the_argmin(alpha):
    """With dt = c_cool min t_cool, Eq. 23 (N_sub = 1, floor out of reach) lowers E_th by a fraction <= c_cool in every
    cell and by exactly c_cool in the cell that sets the minimum: |dt Edot| / E_th = dt / t_cool."""
    U = _random_state(3)
    c_cool = 0.1
    p = oracle.params(gamma=G, shape=U.shape, cooling=True, lambda0=0.2, alpha=alpha, t_floor=1e-8)
    tmin, dt = oracle.cool_dt(U, p, 1e30, c_cool=c_cool)
    assert dt == c_cool * tmin
    out = oracle.cooling(U, dt, p)
    Ek = 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0]
    frac = (U[4] - out[4]) / (U[4] - Ek)
    assert frac.max() == pytest.approx(c_cool, rel=1e-12)
    assert (frac > 0).all()
    # and the per-cell fractions give every t_cool back: brute-force minimum over the cells
    assert dt / frac.max() == pytest.approx(tmin, rel=1e-12)


def test_tcool_invariances():
    U = _random_state(5)
    p = oracle.params(gamma=G, shape=U.shape, cooling=True, lambda0=0.2, alpha=0.7)
    t1, _ = oracle.cool_dt(U, p, 1.0)
    # proportional to 1 / lambda0
    p2 = oracle.params(gamma=G, shape=U.shape, cooling=True, lambda0=0.8, alpha=0.7)
    assert oracle.cool_dt(U, p2, 1.0)[0] == pytest.approx(t1 / 4, rel=1e-14)
    # Galilean boost: only the thermal energy enters (not E)
    rho = U[0]
    v = U[1:4] / rho
    w = v + np.array([3.0, -2.0, 1.0])[:, None, None, None]
    Ub = np.stack([rho, *(rho * w), U[4] - 0.5 * rho * (v ** 2).sum(0) + 0.5 * rho * (w ** 2).sum(0)])
    assert oracle.cool_dt(Ub, p, 1.0)[0] == pytest.approx(t1, rel=1e-12)
    # axis permutation and cell order do not matter; the minimum over a sub-block is never smaller
    assert oracle.cool_dt(np.ascontiguousarray(U.transpose(0, 3, 1, 2)), p, 1.0)[0] == t1
    assert oracle.cool_dt(np.ascontiguousarray(U[:, :3]), p, 1.0)[0] >= t1
    # at fixed temperature t_cool ~ 1 / rho: doubling every conserved field halves it
    assert oracle.cool_dt(2 * U, p, 1.0)[0] == pytest.approx(t1 / 2, rel=1e-14)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_eq21_takes_the_smallest_of_the_three(dtype):
    U = _random_state(7, dtype=dtype)
    p = oracle.params(gamma=G, shape=U.shape, cooling=True, lambda0=0.2, alpha=0.5)
    dth, _ = oracle.cfl_dt(U, p, cfl=0.4)
    tmin, dt = oracle.cool_dt(U, p, dth)                       # both candidates off
    assert dt == dth
    assert oracle.cool_dt(U, p, dth, c_cool=1e9)[1] == dth      # hydro limited: the very same bits
    assert oracle.cool_dt(U, p, dth, c_cool=1e9, dt_max=10.0)[1] == dth
    c = 0.5 * dth / tmin
    want = dtype(c * tmin)
    assert oracle.cool_dt(U, p, dth, c_cool=c, dt_max=10.0)[1] == float(want)       # cooling limited, rounded to T once
    assert oracle.cool_dt(U, p, dth, c_cool=c, dt_max=dth / 4)[1] == float(dtype(dth / 4))   # dt_max limited
    assert float(want) < dth


def test_zero_rate_cells_do_not_decide_and_all_zero_gives_inf():
    U = _uniform(1.0, (0, 0, 0), 1.0)
    p = oracle.params(gamma=G, dx=(1, 1, 1), cooling=True, lambda0=0.1, alpha=0.5)
    t1, _ = oracle.cool_dt(U, p, 1.0)
    V = U.copy()
    V[4, 0, 0, 0] = -1.0          # negative thermal energy: T <= 0, rate 0 (cool_rate clips T at 0)
    assert oracle.cool_dt(V, p, 1.0)[0] == t1
    V[4] = -1.0
    tmin, dt = oracle.cool_dt(V, p, 0.25, c_cool=0.1)
    assert np.isinf(tmin) and dt == 0.25
