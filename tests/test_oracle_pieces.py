"""Pins for the oracle's pointwise pieces: Riemann flux, limiter/reconstruction, primitives, cooling, CFL.
Each pin is something the paper or the mathematics fixes independently of the oracle's own code
(SURVEY.md §8(c) "What pins each part")."""
import os

import numpy as np
import pytest

import oracle
from exact_riemann import godunov_flux, sample, star_state

G = 1.4


def _P(**kw):
    kw.setdefault("gamma", G)
    kw.setdefault("dx", (1.0, 1.0, 1.0))
    return oracle.params(**kw)


def _phys_flux(W, ax, g):
    """Euler flux written straight from Eq. 2 for W = (rho, vx, vy, vz, P)."""
    rho, v, P = W[0], np.array(W[1:4]), W[4]
    E = P / (g - 1.0) + 0.5 * rho * (v @ v)
    F = np.array([rho * v[ax], rho * v[ax] * v[0], rho * v[ax] * v[1], rho * v[ax] * v[2], v[ax] * (E + P)])
    F[1 + ax] += P
    return F


# ------------------------------------------------------------------------------- exact solver sanity
def test_exact_solver_matches_textbook_sod_star_values():
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "sod_star_values.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                vals[k] = float(v)
    ps, us = star_state(1.0, 0.0, 1.0, 0.125, 0.0, 0.1, G)
    assert abs(ps - vals["p_star"]) < 6e-6
    assert abs(us - vals["u_star"]) < 6e-6
    assert abs(sample(us - 1e-9, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, G)[0] - vals["rho_star_left"]) < 6e-6
    assert abs(sample(us + 1e-9, 1.0, 0.0, 1.0, 0.125, 0.0, 0.1, G)[0] - vals["rho_star_right"]) < 6e-6


# ------------------------------------------------------------------------------------- Riemann flux
@pytest.mark.parametrize("riemann", ["hllc", "hll", "rusanov"])
@pytest.mark.parametrize("ax", [0, 1, 2])
def test_flux_consistency(riemann, ax):
    """F(W, W) = F_phys(W) for any state (sub- and supersonic, both signs)."""
    rng = np.random.default_rng(3)
    p = _P(riemann=riemann)
    for _ in range(40):
        W = np.array([rng.uniform(0.1, 3), *rng.normal(0, 2.0, 3), rng.uniform(0.1, 3)])
        F = oracle.riemann(W[:, None], W[:, None], ax, p)[:, 0]
        ref = _phys_flux(W, ax, G)
        assert np.allclose(F, ref, rtol=0, atol=8e-15 * max(1.0, np.abs(ref).max()))


@pytest.mark.parametrize("ax", [0, 1, 2])
def test_hllc_supersonic_upwinding_is_exact(ax):
    """S_L > 0 => F = F_L bitwise; S_R < 0 => F = F_R bitwise."""
    p = _P()
    WL = np.array([1.0, 0.3, -0.2, 0.1, 1.0])
    WR = np.array([0.7, 0.1, 0.4, -0.3, 0.8])
    for sgn, pick in ((+1, 0), (-1, 1)):
        L, R = WL.copy(), WR.copy()
        L[1 + ax] = sgn * 5.0
        R[1 + ax] = sgn * 6.0
        F = oracle.riemann(L[:, None], R[:, None], ax, p)[:, 0]
        ref = _phys_flux((L, R)[pick], ax, G)
        # F_L as the oracle forms it: rho*u*v (+P); allow 1 ulp of association difference
        assert np.allclose(F, ref, rtol=4e-16, atol=0)


@pytest.mark.parametrize("ax", [0, 1, 2])
def test_hllc_preserves_isolated_stationary_contact(ax):
    """u = 0, equal P, rho_L != rho_R: mass and energy flux vanish, momentum flux = P (PAPER.md:898:
    this is what HLLC buys over HLL)."""
    L = np.array([1.0, 0.0, 0.0, 0.0, 0.7])
    R = np.array([0.1, 0.0, 0.0, 0.0, 0.7])
    F = oracle.riemann(L[:, None], R[:, None], ax, _P())[:, 0]
    ref = np.zeros(5)
    ref[1 + ax] = 0.7
    assert np.abs(F - ref).max() < 1e-15
    Fhll = oracle.riemann(L[:, None], R[:, None], ax, _P(riemann="hll"))[:, 0]
    assert abs(Fhll[0]) > 0.1  # HLL smears it


def test_hllc_moving_contact_and_transverse_advection():
    """A contact moving at speed u>0 (equal u, P) must give the upwind flux exactly-ish, including
    the passively advected transverse velocities."""
    L = np.array([1.0, 0.4, 0.3, -0.2, 1.0])
    R = np.array([0.25, 0.4, -0.5, 0.6, 1.0])
    F = oracle.riemann(L[:, None], R[:, None], 0, _P())[:, 0]
    assert np.allclose(F, _phys_flux(L, 0, G), rtol=0, atol=5e-15)
    L[1] = R[1] = -0.4
    F = oracle.riemann(L[:, None], R[:, None], 0, _P())[:, 0]
    assert np.allclose(F, _phys_flux(R, 0, G), rtol=0, atol=5e-15)


def test_hllc_converges_to_exact_flux_faster_than_the_jump():
    """Brute force on random states against the exact Riemann solver: |HLLC - Godunov| = O(jump^2)."""
    rng = np.random.default_rng(7)
    p = _P()
    worst = []
    for _ in range(25):
        W0 = np.array([rng.uniform(0.5, 2), *rng.normal(0, 0.4, 3), rng.uniform(0.5, 2)])
        dW = rng.normal(0, 1, 5) * np.array([1, 1, 1, 1, 1.0])
        errs = []
        for eps in (1e-1, 1e-2, 1e-3):
            L, R = W0 - 0.5 * eps * dW, W0 + 0.5 * eps * dW
            F = oracle.riemann(L[:, None], R[:, None], 0, p)[:, 0]
            errs.append(np.abs(F - godunov_flux(L, R, G)).max())
        # error / jump must fall with the jump (second order or better)
        assert errs[1] < 0.2 * errs[0] * 1.0 + 1e-13 and errs[2] < 0.2 * errs[1] + 1e-13, errs
        worst.append(errs[2] / 1e-3)
    assert max(worst) < 2e-2


def test_riemann_mirror_symmetry():
    """Mirroring the problem (swap L/R, negate normal velocity) negates mass/energy/transverse fluxes and
    keeps the normal momentum flux."""
    rng = np.random.default_rng(11)
    p = _P()
    L = np.array([rng.uniform(0.2, 2, 200), *rng.normal(0, 1, (3, 200)), rng.uniform(0.2, 2, 200)])
    R = np.array([rng.uniform(0.2, 2, 200), *rng.normal(0, 1, (3, 200)), rng.uniform(0.2, 2, 200)])
    for ax in range(3):
        F = oracle.riemann(L, R, ax, p)
        Lm, Rm = R.copy(), L.copy()
        Lm[1 + ax] *= -1
        Rm[1 + ax] *= -1
        Fm = oracle.riemann(Lm, Rm, ax, p)
        sign = -np.ones(5)
        sign[1 + ax] = 1.0
        assert np.allclose(Fm, sign[:, None] * F, rtol=1e-13, atol=1e-13)


# ------------------------------------------------------------------------- limiter / reconstruction
def test_minmod_definition_brute_force():
    """minmod(a,b) = median(a, b, 0) (textbook identity), ties -> a (A7)."""
    rng = np.random.default_rng(0)
    for a, b in rng.normal(0, 1, (500, 2)):
        assert oracle.limiter(a, b) == float(np.median([a, b, 0.0]))
    assert oracle.limiter(0.0, 1.0) == 0.0 and oracle.limiter(-1.0, 2.0) == 0.0
    assert oracle.limiter(2.0, 2.0) == 2.0 and oracle.limiter(-3.0, -1.0) == -1.0


@pytest.mark.parametrize("kind", ["vanleer", "mc"])
def test_other_limiters_are_symmetric_tvd_and_second_order(kind):
    rng = np.random.default_rng(1)
    for a, b in rng.normal(0, 1, (300, 2)):
        s = oracle.limiter(a, b, kind)
        assert s == pytest.approx(oracle.limiter(b, a, kind), abs=1e-15)
        if a * b <= 0:
            assert s == 0.0
        else:
            assert abs(s) <= 2 * min(abs(a), abs(b)) + 1e-15 and s * a > 0
            assert abs(s) >= min(abs(a), abs(b)) - 1e-15  # at least minmod
    assert oracle.limiter(0.7, 0.7, kind) == pytest.approx(0.7, abs=1e-15)


@pytest.mark.parametrize("kind", ["minmod", "vanleer", "mc"])
def test_reconstruction_reproduces_linear_profile_and_clips_extrema(kind):
    n = 16
    p = _P(limiter=kind)
    x = np.arange(n, dtype=float)
    W = np.stack([2.0 + 0.25 * x, 0.5 * x, -0.125 * x, 1.0 + 0 * x, 3.0 + 0.5 * x])
    WL, WR = oracle.reconstruct(W, p)
    # away from the periodic jump (cells 2..n-4) face values are the exact linear interpolant
    for i in range(2, n - 3):
        exact = 0.5 * (W[:, i] + W[:, i + 1])
        assert np.array_equal(WL[:, i], exact) and np.array_equal(WR[:, i], exact)
    # an extremum gets zero slope: face values equal the cell value
    W2 = np.ones((5, 8))
    W2[:, 3] = 2.0
    WL, WR = oracle.reconstruct(W2, p)
    assert np.array_equal(WL[:, 3], W2[:, 3]) and np.array_equal(WR[:, 2], W2[:, 3])


def test_minmod_face_states_bounded_by_neighbours():
    rng = np.random.default_rng(5)
    W = rng.uniform(0.1, 2.0, (5, 64))
    WL, WR = oracle.reconstruct(W, _P())
    Wp = np.roll(W, -1, axis=1)
    lo, hi = np.minimum(W, Wp), np.maximum(W, Wp)
    assert (WL >= lo - 1e-15).all() and (WL <= hi + 1e-15).all()
    assert (WR >= lo - 1e-15).all() and (WR <= hi + 1e-15).all()


# ---------------------------------------------------------------------------------------- primitives
def test_prims_roundtrip_and_floors():
    rng = np.random.default_rng(2)
    rho = rng.uniform(0.1, 2, (2, 3, 4))
    v = rng.normal(0, 1, (3, 2, 3, 4))
    P = rng.uniform(0.1, 2, (2, 3, 4))
    U = np.stack([rho, rho * v[0], rho * v[1], rho * v[2], P / (G - 1) + 0.5 * rho * (v ** 2).sum(0)])
    W = oracle.prims(U, _P())
    assert np.allclose(W, np.stack([rho, *v, P]), rtol=1e-13, atol=1e-14)
    U[4, 0, 0, 0] = 0.0          # negative pressure -> floored
    U[0, 1, 1, 1] = -1.0         # negative density -> floored
    W = oracle.prims(U, _P(p_floor=1e-7, rho_floor=1e-3))
    assert W[4, 0, 0, 0] == 1e-7 and W[0, 1, 1, 1] == 1e-3


# ------------------------------------------------------------------------------------------- cooling
def _uniform(rho, v, P, shape=(1, 1, 4), g=5.0 / 3.0):
    U = np.empty((5,) + shape)
    U[0] = rho
    for c in range(3):
        U[1 + c] = rho * v[c]
    U[4] = P / (g - 1) + 0.5 * rho * sum(x * x for x in v)
    return U


def test_cooling_one_euler_step_closed_form():
    """alpha = 1/2, gas at rest: T1 = T0 - (gamma-1) rho lambda0 sqrt(T0) dt."""
    g, rho, T0, lam, dt = 5.0 / 3.0, 1.7, 2.3, 1e-3, 0.37
    p = oracle.params(gamma=g, dx=(1, 1, 1), cooling=True, lambda0=lam, alpha=0.5, t_floor=0.01)
    U = _uniform(rho, (0.3, -0.2, 0.1), rho * T0)
    out = oracle.cooling(U, dt, p)
    assert np.array_equal(out[:4], U[:4])  # rho and momentum untouched bitwise
    T1 = (g - 1) * (out[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0]) / rho
    assert np.allclose(T1, T0 - (g - 1) * rho * lam * np.sqrt(T0) * dt, rtol=1e-14)


def test_cooling_converges_first_order_to_ode_solution():
    """sqrt(T(t)) = sqrt(T0) - (gamma-1) lambda0 rho t / 2."""
    g, rho, T0, lam, t = 5.0 / 3.0, 2.0, 1.0, 0.05, 4.0
    p = oracle.params(gamma=g, dx=(1, 1, 1), cooling=True, lambda0=lam, alpha=0.5, t_floor=1e-6)
    exact = (np.sqrt(T0) - 0.5 * (g - 1) * lam * rho * t) ** 2
    errs = []
    for n in (20, 40, 80):
        U = _uniform(rho, (0, 0, 0), rho * T0)
        for _ in range(n):
            U = oracle.cooling(U, t / n, p)
        errs.append(abs((g - 1) * U[4, 0, 0, 0] / rho - exact))
    assert 1.8 < errs[0] / errs[1] < 2.2 and 1.8 < errs[1] / errs[2] < 2.2


def test_cooling_floor_engages_exactly():
    g, rho = 5.0 / 3.0, 1.5
    p = oracle.params(gamma=g, dx=(1, 1, 1), cooling=True, lambda0=10.0, alpha=0.5, t_floor=0.01)
    out = oracle.cooling(_uniform(rho, (0, 0, 0), rho * 0.5), 100.0, p)
    assert np.array_equal(out[4], np.full_like(out[4], rho * 0.01 / (g - 1)))
    # literal max(): gas below the floor is raised to it (reading A9)
    out = oracle.cooling(_uniform(rho, (0, 0, 0), rho * 0.001), 1e-9, p)
    assert np.allclose(out[4], rho * 0.01 / (g - 1), rtol=1e-15)


def _T_of(U, g):
    return (g - 1) * (U[4] - 0.5 * (U[1] ** 2 + U[2] ** 2 + U[3] ** 2) / U[0]) / U[0]


@pytest.mark.parametrize("nsub", [1, 3, 8])
def test_cooling_subcycled_is_the_numpy_recurrence(nsub):
    """Eq. 23 retyped in numpy for moving gas and a general alpha: N_sub Euler substeps of
    dt / N_sub with T re-evaluated each substep and the floor of Eq. 24 applied each substep; a dropped
    re-evaluation (rate frozen at T^n) or a floor applied only at the end changes the result."""
    g, lam, al, tf, dt = 1.4, 0.8, 0.7, 0.4, 0.9
    rng = np.random.default_rng(12)
    rho, T0 = rng.uniform(0.5, 2.0, 16), rng.uniform(0.3, 3.0, 16)   # some cells reach the floor mid-way
    v = rng.normal(0, 0.5, (3, 16))
    U = np.stack([rho, rho * v[0], rho * v[1], rho * v[2], rho * T0 / (g - 1) + 0.5 * rho * (v ** 2).sum(0)]).reshape(5, 1, 1, 16)
    p = oracle.params(gamma=g, dx=(1, 1, 1), cooling=True, lambda0=lam, alpha=al, t_floor=tf, cool_nsub=nsub)
    out = oracle.cooling(U, dt, p)
    assert np.array_equal(out[:4], U[:4])
    Eth = rho * T0 / (g - 1)
    hit_midway = False
    for k in range(nsub):
        T = (g - 1) * Eth / rho
        new = Eth - rho * rho * lam * np.maximum(T, 0.0) ** al * (dt / nsub)
        hit_midway |= bool(np.any(new < rho * tf / (g - 1))) and k < nsub - 1
        Eth = np.maximum(rho * tf / (g - 1), new)
    assert np.allclose(_T_of(out, g).ravel(), (g - 1) * Eth / rho, rtol=1e-13)
    if nsub > 1:
        assert hit_midway
        frozen = np.maximum(rho * tf / (g - 1), rho * T0 / (g - 1) - rho * rho * lam * T0 ** al * dt)
        assert not np.allclose((g - 1) * frozen / rho, (g - 1) * Eth / rho, rtol=1e-3)


def test_cooling_subcycling_error_falls_as_one_over_nsub():
    """One step of size t against the ODE solution sqrt(T(t)) = sqrt(T0) - (gamma-1) lambda0 rho t / 2 (alpha = 1/2):
    the sub-cycled Euler update is first order in dt / N_sub."""
    g, rho, T0, lam, t = 5.0 / 3.0, 2.0, 1.0, 0.05, 4.0
    exact = (np.sqrt(T0) - 0.5 * (g - 1) * lam * rho * t) ** 2
    errs = []
    for n in (16, 32, 64):
        p = oracle.params(gamma=g, dx=(1, 1, 1), cooling=True, lambda0=lam, alpha=0.5, t_floor=1e-6, cool_nsub=n)
        out = oracle.cooling(_uniform(rho, (0.2, 0, -0.1), rho * T0), t, p)
        errs.append(abs(_T_of(out, g)[0, 0, 0] - exact))
    assert 1.8 < errs[0] / errs[1] < 2.2 and 1.8 < errs[1] / errs[2] < 2.2


def test_cooling_trapezoid_closed_form_and_second_order():
    """Eq. 22 with reading A20 (T^pred = temperature of the Euler-predicted energy): one step retyped in
    numpy; repeated steps converge to the ODE solution at second order (error ratio 4 per halving of dt), which a
    missing factor 1/2 or a predictor evaluated at T^n would not."""
    g, rho, T0, lam = 5.0 / 3.0, 1.7, 2.3, 0.05
    p = oracle.params(gamma=g, dx=(1, 1, 1), cooling=True, lambda0=lam, alpha=0.5, t_floor=1e-6, cool_mode="trapezoid")
    dt = 0.37
    out = oracle.cooling(_uniform(rho, (0.3, -0.2, 0.1), rho * T0), dt, p)
    k = (g - 1) * rho * lam
    Tp = T0 - k * np.sqrt(T0) * dt
    assert np.allclose(_T_of(out, g), T0 - 0.5 * dt * k * (np.sqrt(T0) + np.sqrt(Tp)), rtol=1e-14)
    t = 4.0
    exact = (np.sqrt(T0) - 0.5 * k * t) ** 2
    errs = []
    for n in (10, 20, 40):
        U = _uniform(rho, (0, 0, 0), rho * T0)
        for _ in range(n):
            U = oracle.cooling(U, t / n, p)
        errs.append(abs(_T_of(U, g)[0, 0, 0] - exact))
    assert 3.6 < errs[0] / errs[1] < 4.4 and 3.6 < errs[1] / errs[2] < 4.4


def test_cooling_trapezoid_floor():
    g, rho = 5.0 / 3.0, 1.5
    p = oracle.params(gamma=g, dx=(1, 1, 1), cooling=True, lambda0=10.0, alpha=0.5, t_floor=0.01, cool_mode="trapezoid")
    out = oracle.cooling(_uniform(rho, (0, 0, 0), rho * 0.5), 100.0, p)
    assert np.array_equal(out[4], np.full_like(out[4], rho * 0.01 / (g - 1)))


# ----------------------------------------------------------------------------------------------- CFL
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_cfl_closed_form_uniform_state(dtype):
    """Eq. A8 on a uniform state: dt = C min_a dx_a / (|v_a| + sqrt(gamma P / rho))."""
    g, rho, v, P = 1.4, 1.3, (0.5, -1.25, 0.25), 0.9
    U = _uniform(rho, v, P, shape=(6, 5, 8), g=g).astype(dtype)
    p = oracle.params(gamma=g, dx=(0.1, 0.2, 0.05))
    dt, smax = oracle.cfl_dt(U, p, cfl=0.4)
    cs = np.sqrt(g * P / rho)
    want = 0.4 * min(0.1 / (0.5 + cs), 0.2 / (1.25 + cs), 0.05 / (0.25 + cs))
    assert dt == pytest.approx(want, rel=1e-14 if dtype == np.float64 else 3e-7)
    assert np.allclose(smax, [abs(x) + cs for x in v], rtol=1e-14 if dtype == np.float64 else 3e-7)
    if dtype == np.float32:
        assert dt == float(np.float32(dt))  # dt is a T value widened exactly


def test_cfl_scaling_and_thread_independence():
    rng = np.random.default_rng(9)
    n = 24
    rho = rng.uniform(0.5, 2, (n, n, n))
    v = rng.normal(0, 1, (3, n, n, n))
    U = np.stack([rho, *(rho * v), 1.5 + 0.5 * rho * (v ** 2).sum(0)]).astype(np.float32)
    p = oracle.params(gamma=5 / 3, shape=U.shape)
    nt = oracle.num_threads()
    dts = []
    for t in (1, 2, nt):
        oracle.set_num_threads(t)
        dts.append(oracle.cfl_dt(U, p)[0])
    oracle.set_num_threads(nt)
    assert dts[0] == dts[1] == dts[2]  # bit-identical
    # brute force in numpy float32 following the same recipe (max over cells is order independent)
    f = np.float32
    rt = np.maximum(U[0], f(1e-10))
    q = ((U[1] * U[1]) + (U[2] * U[2])) + (U[3] * U[3])
    P = np.maximum(f(5 / 3 - 1.0) * (U[4] - f(0.5) * (q / rt)), f(1e-10))
    cs = np.sqrt((f(5 / 3) * P) / rt)
    s = [np.max(np.abs(U[1 + a] / rt) + cs) for a in range(3)]
    want = f(0.4) * min(f(1.0 / n) / s[a] for a in range(3))
    assert dts[0] == float(want)
    # doubling all velocities and sound speed (E x4 at fixed rho) halves dt up to rounding
    U2 = U.copy()
    U2[1:4] *= 2
    U2[4] *= 4
    assert oracle.cfl_dt(U2, p)[0] == pytest.approx(dts[0] / 2, rel=1e-6)


def test_cfl_rejects_nonfinite():
    U = _uniform(1.0, (0, 0, 0), 1.0, shape=(4, 4, 4))
    U[4, 1, 2, 3] = np.nan
    with pytest.raises(FloatingPointError):
        oracle.cfl_dt(U, oracle.params(shape=U.shape))
