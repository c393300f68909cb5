"""GPU parity for the two-branch heating / cooling law (DH_OPT_COOL_LAW = 1; Eqs. 17-19), the masked
choice of the integrator (DH_OPT_COOL_MODE = 2) and the gradient with respect to the table
(dh_cool_table_vjp): against oracle/ on the same seeded states and the same synthetic table (workloads.cooling_table)."""
import numpy as np
import pytest
import torch

import oracle
import vjp_margins
from paper_2512_13403_b200 import workloads
from test_gpu_parity import TOL, _solver, max_rel_err

pytestmark = pytest.mark.gpu
G = 5 / 3


def _law(**over):
    logT0, dlogT, vals = workloads.cooling_table(lambda_lo=0.5)
    kw = dict(t_switch=1.0, lambda1=0.3, alpha1=2.0, lambda2=0.2, alpha2=0.5, gamma0=0.5, t_floor=0.05)
    kw.update(over)
    table = (logT0, dlogT, vals.numpy())
    okw = dict(cooling=True, cool_law="twobranch", table=table, **kw)
    skw = dict(cooling=1, cool_law="twobranch", table=(logT0, dlogT, list(vals.numpy())), **kw)
    return okw, skw


def _state(shape, seed, dtype, mach=0.5, tlo=0.2, thi=30.0):
    rng = np.random.default_rng(seed)
    rho = rng.uniform(0.5, 2.0, shape)
    v = rng.normal(0, mach, (3,) + tuple(shape))
    T = np.exp(rng.uniform(np.log(tlo), np.log(thi), shape))          # both branches of Eq. 17
    U = np.stack([rho, rho * v[0], rho * v[1], rho * v[2], rho * T / (G - 1) + 0.5 * rho * (v ** 2).sum(0)])
    return torch.from_numpy(U).to(dtype)


MODES = [dict(), dict(cool_nsub=4), dict(cool_mode="trapezoid"), dict(cool_mode="masked", cool_nsub=3, f_sub=0.05)]
_id = lambda v: "-".join(f"{a}={b}" for a, b in v.items()) or "euler"


@pytest.mark.parametrize("kernel", ["fused", "gather"])
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("mode", MODES, ids=_id)
def test_step_parity_two_branch_law(mode, dtype, kernel):
    okw, skw = _law(**mode)
    U = _state((9, 12, 34), 701, dtype)
    p = oracle.params(gamma=G, shape=tuple(U.shape), **okw)
    s = _solver(U, G, kernel=kernel, **skw)
    Ud = U.cuda()
    dt = s.cfl_dt(Ud)
    assert dt == oracle.cfl_dt(U.numpy(), p)[0]
    s.step(Ud, dt)
    ref = oracle.step(U.numpy(), dt, p)
    assert max_rel_err(Ud.cpu().numpy(), ref) <= TOL[dtype]
    base = oracle.step_nocool(U.numpy(), dt, p)
    d = ref[4] - base[4]
    assert (d > 1e-6).any() and (d < -1e-6).any()                      # heating below the equilibrium, cooling above it


@pytest.mark.parametrize("integrator", ["vl2", "ssprk3"])
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("mode", MODES, ids=_id)
def test_vjp_parity_two_branch_law(mode, dtype, integrator):
    okw, skw = _law(**mode)
    U = _state((8, 10, 14), 711, dtype)
    p = oracle.params(gamma=G, shape=tuple(U.shape), integrator=integrator, **okw)
    s = _solver(U, G, integrator=integrator, **skw)
    Ud = U.cuda()
    dt = s.cfl_dt(Ud)
    g = torch.from_numpy(np.random.default_rng(712).normal(size=tuple(U.shape))).to(dtype)
    gin = s.step_vjp(Ud, dt, g.cuda()).cpu().numpy()
    ref = oracle.step_vjp(U.numpy(), dt, g.numpy(), p)
    if dtype == torch.float64:
        assert np.abs(gin - ref).max() <= 1e-11 * np.sqrt(np.mean(ref ** 2))
    else:
        cond = vjp_margins.vjp_condition(U.numpy(), dt, p)
        vjp_margins.check_vjp(gin, ref, cond, 2e-5, max_excluded=0.3, label=f"two-branch {mode} {integrator}")


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("mode", MODES[:3], ids=_id)
def test_table_gradient(mode, dtype):
    """dh_cool_table_vjp against the oracle's dual-number gradient at the oracle's pre-cooling state."""
    okw, skw = _law(**mode)
    U = _state((8, 10, 14), 721, dtype, tlo=0.5, thi=80.0)
    p = oracle.params(gamma=G, shape=tuple(U.shape), **okw)
    s = _solver(U, G, **skw)
    Ud = U.cuda()
    dt = s.cfl_dt(Ud)
    g = torch.from_numpy(np.random.default_rng(722).normal(size=tuple(U.shape))).to(dtype)
    got = np.array(s.cool_table_vjp(Ud, dt, g.cuda()))
    U1 = oracle.step_nocool(U.numpy(), dt, p)
    ref = oracle.cooling_table_vjp(U1, dt, g.numpy(), p)
    scale = np.abs(ref).max()
    assert scale > 0 and np.count_nonzero(ref) >= 8
    assert np.abs(got - ref).max() <= (1e-10 if dtype == torch.float64 else 2e-4) * scale, (got, ref)


def test_cooling_time_limit_follows_the_law():
    """Eqs. 20-21 with the two-branch law: min t_cool to 1e-12 of the oracle's, dt limited by it."""
    from paper_2512_13403_b200 import dh
    okw, skw = _law(lambda1=300.0, lambda2=200.0, gamma0=20.0)
    for dtype in (torch.float64, torch.float32):
        U = _state((9, 12, 34), 731, dtype)
        p = oracle.params(gamma=G, shape=tuple(U.shape), **okw)
        s = _solver(U, G, c_cool=0.1, **skw)
        Ud = U.cuda()
        dt = s.cfl_dt(Ud)
        dt_h = oracle.cfl_dt(U.numpy(), p)[0]
        tmin, dt_ref = oracle.cool_dt(U.numpy(), p, dt_h, c_cool=0.1)
        assert dt < dt_h and abs(dt - dt_ref) <= (1e-12 if dtype == torch.float64 else 2e-7) * dt_ref


def test_option_errors():
    from paper_2512_13403_b200 import dh
    U = _state((4, 4, 4), 741, torch.float32)
    s = _solver(U, G)
    with pytest.raises(dh.DhError):
        s.set_options(cool_law=1)                                      # no table yet
    with pytest.raises(dh.DhError):
        s.set_cooling_table(0.0, 0.1, [1.0])
    with pytest.raises(dh.DhError):
        s.set_cooling_table(0.0, -0.1, [1.0, 2.0])
    with pytest.raises(dh.DhError):
        s.set_cooling_table(0.0, 0.1, [1.0, float("nan")])
    s.set_cooling_table(0.0, 0.1, [1.0, 2.0, 1.5])
    s.set_options(cool_law="twobranch", cool_mode="masked", f_sub=0.2)
    assert s.get_option("cool_law") == 1 and s.get_option("cool_mode") == 2
    for key, bad in (("f_sub", 0.0), ("t_switch", -1.0), ("lambda1", -1.0), ("gamma0", -1.0), ("cool_mode", 3)):
        with pytest.raises(dh.DhError):
            s.set_options(**{key: bad})
