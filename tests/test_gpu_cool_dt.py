"""GPU parity of the cooling-time limit on dt, Eqs. 20-21 (reading A24), through the C ABI against
oracle.cool_dt on the same seeded inputs.

Bars: dt_hydro bit-identical (Eq. A8 recipe); min_x t_cool, formed in fp64 on both sides, to 1e-14 relative (the two
power functions differ by at most a few ulp); the limited dt bit-identical when the hydro or dt_max candidate decides, and
within one ulp of T (fp32) / 1e-14 (fp64) when the cooling candidate decides."""
import numpy as np
import pytest
import torch

import oracle
from test_gpu_parity import _solver, max_rel_err, oracle_params, random_state

pytestmark = pytest.mark.gpu

SHAPES = [(20, 30, 132), (7, 9, 33), (5, 5, 7)]      # vector path, ragged tail, scalar path (N odd)


def _lognormal_state(shape, seed, gamma, dtype, mach=1.0):
    """rho lognormal (sigma_ln = 0.5), T spread over two decades: the shape of configs[3]'s cooling turbulence."""
    rng = np.random.default_rng(seed)
    rho = np.exp(rng.normal(0, 0.5, shape))
    v = rng.normal(0, mach, (3,) + tuple(shape))
    T = 10 ** rng.uniform(-1.5, 0.5, shape)
    U = np.stack([rho, rho * v[0], rho * v[1], rho * v[2], rho * T / (gamma - 1) + 0.5 * rho * (v ** 2).sum(0)])
    return torch.from_numpy(U).to(dtype)


@pytest.mark.parametrize("alpha", [0.5, 0.7, 1.0])
@pytest.mark.parametrize("shape", SHAPES)
@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_tcool_min_and_dt_hydro(dtype, shape, alpha):
    gamma = 5 / 3
    U = _lognormal_state(shape, 700 + shape[0], gamma, dtype)
    p = oracle_params(U, gamma, cooling=True, lambda0=0.3, alpha=alpha)
    s = _solver(U, gamma, lambda0=0.3, alpha=alpha)          # DH_OPT_COOLING need not be on for dh_cool_tmin
    t_gpu, dth_gpu = s.cool_tmin(U.cuda())
    dth_ora, _ = oracle.cfl_dt(U.numpy(), p)
    t_ora, _ = oracle.cool_dt(U.numpy(), p, dth_ora)
    assert dth_gpu == dth_ora
    assert t_gpu == pytest.approx(t_ora, rel=1e-14)
    # cooling off and no dt_max: the device dt stayed the hydro one
    assert s.cfl_dt(U.cuda()) == dth_ora


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_eq21_three_regimes(dtype):
    gamma = 5 / 3
    U = _lognormal_state((12, 16, 36), 711, gamma, dtype)
    Ud = U.cuda()
    p = oracle_params(U, gamma, cooling=True, lambda0=0.3, alpha=0.5)
    dth, _ = oracle.cfl_dt(U.numpy(), p)
    tmin, _ = oracle.cool_dt(U.numpy(), p, dth)
    s = _solver(U, gamma, cooling=1, lambda0=0.3)
    assert s.cfl_dt(Ud) == dth                                  # c_cool = 0: off
    s.set_options(c_cool=1e9)
    assert s.cfl_dt(Ud) == dth                                  # hydro limited: the same bits
    c = 0.37 * dth / tmin
    s.set_options(c_cool=c)
    _, want = oracle.cool_dt(U.numpy(), p, dth, c_cool=c)
    got = s.cfl_dt(Ud)
    assert want < dth
    ulp = 1.2e-7 if dtype == torch.float32 else 1e-14
    assert got == pytest.approx(want, rel=ulp)
    if dtype == torch.float32:
        assert got == float(np.float32(got))                    # a T value widened exactly
    s.set_options(dt_max=dth / 8)
    assert s.cfl_dt(Ud) == oracle.cool_dt(U.numpy(), p, dth, c_cool=c, dt_max=dth / 8)[1]   # dt_max limited: exact
    s.set_options(cooling=0, dt_max=dth / 8)                    # dt_max applies without cooling, c_cool does not
    assert s.cfl_dt(Ud) == float(np.asarray(dth / 8, dtype=U.numpy().dtype))
    s.set_options(dt_max=0)
    assert s.cfl_dt(Ud) == dth


def test_zero_rate_cells_and_all_zero():
    gamma = 5 / 3
    U = _lognormal_state((4, 6, 16), 721, gamma, torch.float64)
    p = oracle_params(U, gamma, cooling=True, lambda0=0.3, alpha=0.5)
    t0, _ = oracle.cool_dt(U.numpy(), p, 1.0)
    V = U.clone()
    V[4, 1, 2, 3] = 0.0                 # E < kinetic energy: T < 0, rate 0, never the minimum
    s = _solver(U, gamma, lambda0=0.3)
    t_ora, _ = oracle.cool_dt(V.numpy(), p, 1.0)
    t_gpu, _ = s.cool_tmin(V.cuda())
    assert t_gpu == pytest.approx(t_ora, rel=1e-14) and np.isfinite(t_gpu)
    V[4] = 0.0
    V[1:4] = 0.0                        # E_th = 0 everywhere: no cell cools
    t_gpu, _ = s.cool_tmin(V.cuda())
    assert np.isinf(t_gpu) and np.isinf(oracle.cool_dt(V.numpy(), p, 1.0)[0])
    # the slot is re-armed: the next pass is unaffected
    assert s.cool_tmin(U.cuda())[0] == pytest.approx(t0, rel=1e-14)


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_advance_with_the_cooling_limit_follows_the_oracle_loop(dtype):
    """dh_advance with c_cool > 0 (full reduction with the t_cool branch every step, device-resident dt) against the
    oracle's loop of cfl_dt, cool_dt and step; cooling-limited from the first step (strong cooling), and bit for bit the
    host-driven loop of dh_cfl_dt + dh_step."""
    gamma = 5 / 3
    f64 = dtype == torch.float64
    U = _lognormal_state((10, 12, 36), 731, gamma, dtype)
    kw = dict(cooling=True, lambda0=20.0, alpha=0.5, t_floor=0.01)
    p = oracle_params(U, gamma, **kw)
    s = _solver(U, gamma, cooling=1, lambda0=20.0, t_floor=0.01, c_cool=0.1)
    a, b = U.cuda(), U.cuda()
    dts = []
    for _ in range(3):
        dts.append(s.cfl_dt(b))
        s.step(b, dts[-1])
    dt_last = s.advance(a, 3)
    assert dt_last == dts[-1] and torch.equal(a, b)
    assert s.cfl_stats()["candidate_passes"] == 0               # the candidate list is not used with the limit
    ref = U.numpy().astype(np.float64)
    nlim = 0
    cur = U.numpy().copy()
    for k in range(3):
        dth, _ = oracle.cfl_dt(cur, p)
        _, dt = oracle.cool_dt(cur, p, dth, c_cool=0.1)
        nlim += dt < dth
        if k == 0:
            assert dts[0] == pytest.approx(dt, rel=1e-14 if f64 else 1.2e-7)
        ref = oracle.step(ref, dt, p)
        cur = ref.astype(cur.dtype)
    assert nlim >= 1
    assert max_rel_err(a.cpu().numpy(), ref) <= (5e-12 if f64 else 1e-4)


@pytest.mark.parametrize("alpha", [0.5, 1.0, 2.5])
@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_fp32_screen_never_drops_the_minimum(dtype, alpha):
    """The kernel screens cells with an fp32 estimate before the fp64 evaluation (dh_cfl.cu, tcool_may_decide); the minimum
    must stay the exact one where that screen is weakest: (a) near-ties, every cell within 1e-6 (fp64) / a few ulp (fp32) of
    the minimum; (b) Mach 30 gas, E_th a 1e-3 part of E (ill-conditioned in fp32); (c) values far outside the fp32 range
    (fp64 arrays only); (d) the minimum in the last, partly filled warp iteration."""
    gamma = 5 / 3
    np_t = np.float32 if dtype == torch.float32 else np.float64
    rng = np.random.default_rng(751)
    shape = (6, 10, 36)
    cases = []
    # (a) near ties
    rho = np.full(shape, 1.3)
    T = 0.8 * (1 + 1e-6 * rng.uniform(-1, 1, shape))
    v = np.zeros((3,) + shape)
    cases.append(np.stack([rho, *(rho * v), rho * T / (gamma - 1)]))
    # (b) kinetic-energy dominated
    rho = np.exp(rng.normal(0, 0.5, shape))
    T = rng.uniform(0.5, 2, shape)
    v = rng.normal(0, 30 * np.sqrt(gamma), (3,) + shape)
    cases.append(np.stack([rho, *(rho * v), rho * T / (gamma - 1) + 0.5 * rho * (v ** 2).sum(0)]))
    # (d) one cold dense cell at the very end of the array
    U = _lognormal_state(shape, 752, gamma, torch.float64).numpy()
    U[:, -1, -1, -1] = [50.0, 0, 0, 0, 50.0 * 3.0 / (gamma - 1)]
    cases.append(U)
    if dtype == torch.float64:      # (c)
        cases.append(cases[1] * 1e-60)
        cases.append(cases[1] * 1e60)
    for k, U in enumerate(cases):
        U = np.ascontiguousarray(U.astype(np_t))
        p = oracle_params(torch.from_numpy(U), gamma, cooling=True, lambda0=0.3, alpha=alpha)
        s = _solver(torch.from_numpy(U), gamma, lambda0=0.3, alpha=alpha)
        t_ora, _ = oracle.cool_dt(U, p, 1.0)
        t_gpu, dth_gpu = s.cool_tmin(torch.from_numpy(U).cuda())
        assert np.isfinite(t_ora) and t_gpu == pytest.approx(t_ora, rel=1e-14), (k, t_gpu, t_ora)
        # the same sweep screens the wave-speed recipe in fp32 too (speeds_may_decide): dt_hydro keeps its bits
        assert dth_gpu == oracle.cfl_dt(U, p)[0], k


def test_adjoint_holds_the_limited_dt_constant():
    """dh_adjoint with c_cool > 0: the forward sweep's dt sequence is the limited one (Eq. 21), and the reverse sweep is the
    chain of step VJPs at those dt held constant, checked against the oracle's step VJP chained over the
    oracle's own limited-dt loop."""
    gamma = 5 / 3
    U = _lognormal_state((9, 10, 36), 761, gamma, torch.float64)
    kw = dict(cooling=True, lambda0=20.0, alpha=0.5, t_floor=0.01)
    p = oracle_params(U, gamma, **kw)
    s = _solver(U, gamma, cooling=1, lambda0=20.0, t_floor=0.01, c_cool=0.1)
    g = np.random.default_rng(762).normal(size=tuple(U.shape))
    Ud, gd = U.cuda(), torch.from_numpy(g).cuda()
    dts = s.adjoint(Ud, gd, 3, 2)
    states, dts_ref, cur = [], [], U.numpy().copy()
    for _ in range(3):
        dth, _ = oracle.cfl_dt(cur, p)
        _, dt = oracle.cool_dt(cur, p, dth, c_cool=0.1)
        assert dt < dth
        states.append(cur)
        dts_ref.append(dt)
        cur = oracle.step(cur, dt, p)
    assert np.allclose(dts, dts_ref, rtol=1e-13, atol=0)
    assert max_rel_err(Ud.cpu().numpy(), cur) <= 5e-12
    gref = g
    for k in (2, 1, 0):
        gref = oracle.step_vjp(states[k], dts_ref[k], gref, p)
    err = np.abs(gd.cpu().numpy() - gref) / np.sqrt(np.mean(gref ** 2))
    assert err.max() <= 1e-11, float(err.max())


def test_option_errors_and_defaults():
    from paper_2512_13403_b200 import dh
    U = random_state((4, 4, 4), 741, 1.4, torch.float32)
    s = _solver(U, 1.4)
    assert s.get_option("c_cool") == 0 and s.get_option("dt_max") == 0
    for key, bad in (("c_cool", -1.0), ("c_cool", float("inf")), ("dt_max", -1e-3), ("dt_max", float("nan"))):
        with pytest.raises(dh.DhError):
            s.set_options(**{key: bad})
    U[0, 1, 1, 1] = float("nan")
    with pytest.raises(dh.DhError) as e:
        s.cool_tmin(U.cuda())
    assert e.value.code == dh.DH_ERR_NONFINITE
