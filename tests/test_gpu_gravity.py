"""GPU parity for self-gravity as a source of the hydro step (dh_gravity_source*, dh_step_gravity*)
against oracle/gravity.py on the same seeded states."""
import numpy as np
import pytest
import torch

import oracle
import vjp_margins
from oracle import gravity
from test_gpu_parity import TOL, _solver, max_rel_err, random_state

pytestmark = pytest.mark.gpu


def _mg(shape, h, dtype, **kw):
    from paper_2512_13403_b200 import dh
    nz, ny, nx = shape
    return dh.Multigrid(nx, ny, nz, h, dtype=dtype, **kw)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_source_and_its_vjp(dtype):
    shape = (9, 12, 34)
    U = random_state(shape, 801, 5 / 3, dtype)
    rng = np.random.default_rng(802)
    phi = torch.from_numpy(rng.normal(size=shape)).to(dtype)
    L = (1.7, 0.9, 1.2)
    dx = (L[0] / 34, L[1] / 12, L[2] / 9)
    s = _solver(U, 5 / 3, lx=L[0], ly=L[1], lz=L[2])
    Ud = U.cuda()
    s.gravity_source(Ud, phi.cuda(), 0.3)
    ref = gravity.source(U.numpy(), phi.numpy(), 0.3, dx)
    tol = 1e-13 if dtype == torch.float64 else 2e-6
    assert max_rel_err(Ud.cpu().numpy(), ref) <= tol
    g = torch.from_numpy(rng.normal(size=tuple(U.shape))).to(dtype)
    gin, gphi = s.gravity_source_vjp(U.cuda(), phi.cuda(), 0.3, g.cuda())
    rU, rphi = gravity.source_vjp(U.numpy(), phi.numpy(), 0.3, dx, g.numpy())
    assert np.abs(gin.cpu().numpy() - rU).max() <= tol * np.abs(rU).max()
    assert np.abs(gphi.cpu().numpy() - rphi).max() <= tol * np.abs(rphi).max()


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("kw", [dict(), dict(limiter="vanleer"), dict(cooling=True, lambda0=0.5)], ids=["minmod", "vanleer", "cooling"])
def test_self_gravitating_step_and_vjp(kw, dtype):
    shape, h = (16, 16, 32), 1 / 16                       # cubic cells (the multigrid solver needs them), non-cubic box
    U = random_state(shape, 811, 5 / 3, dtype)
    okw = dict(kw)
    skw = dict(kw)
    if "cooling" in skw:
        skw["cooling"] = 1
    p = oracle.params(gamma=5 / 3, dx=(h, h, h), **okw)
    s = _solver(U, 5 / 3, lx=32 * h, ly=16 * h, lz=16 * h, **skw)
    mg = _mg(shape, h, dtype)
    Ud = U.cuda()
    dt = s.cfl_dt(Ud)
    assert dt == oracle.cfl_dt(U.numpy(), p)[0]
    fpg, nc = 25.0, 14
    g = torch.from_numpy(np.random.default_rng(812).normal(size=tuple(U.shape))).to(dtype)
    gin = s.step_gravity_vjp(mg, Ud, dt, fpg, g.cuda(), ncycles=nc).cpu().numpy()
    assert torch.equal(Ud.cpu(), U)
    s.step_gravity(mg, Ud, dt, fpg, ncycles=nc)
    ref = gravity.step(U.numpy(), dt, p, fpg, h, ncycles=nc)
    plain = oracle.step(U.numpy(), dt, p)
    assert np.abs(ref[1:4] - plain[1:4]).max() > 1e-4                       # the kick is visible
    assert max_rel_err(Ud.cpu().numpy(), ref) <= TOL[dtype]
    gref = gravity.step_vjp(U.numpy(), dt, g.numpy(), p, fpg, h, ncycles=nc)
    if dtype == torch.float64:
        assert np.abs(gin - gref).max() <= 1e-10 * np.sqrt(np.mean(gref ** 2))
    else:
        cond = vjp_margins.vjp_condition(U.numpy(), dt, p)
        sens = vjp_margins.vjp_sensitivity(U.numpy(), dt, p)
        vjp_margins.check_vjp(gin, gref, cond, 2e-5, max_excluded=0.3, label=f"self-gravitating step {kw}", sens=sens)


def test_argument_errors():
    from paper_2512_13403_b200 import dh
    U = random_state((8, 8, 8), 821, 5 / 3, torch.float32).cuda()
    s = _solver(U, 5 / 3)
    mg = _mg((8, 8, 8), 1 / 8, torch.float32)
    with pytest.raises(dh.DhError):
        s.step_gravity(mg, U, -1.0, 1.0)
    with pytest.raises(dh.DhError):
        s.step_gravity(mg, U, 0.1, 1.0, ncycles=0)
    with pytest.raises(ValueError):
        s.gravity_source(U, U[0].double(), 0.1)
