"""GPU parity of the multigrid Poisson path (dh_mg_* of include/dh.h) against oracle/poisson.py, element by element on
the same seeded inputs.  Tolerances: everything is a short chain of linear stencil operations, so fp64 agrees to
1e-12 of the field's maximum and fp32 to 2e-5 (the bar of the hydro path); converged solves are compared with the FFT
definition of A^+ at the accuracy the cycle count reaches."""
import numpy as np
import pytest
import torch

from oracle import poisson as mg

pytestmark = pytest.mark.gpu

TOL = {torch.float64: 1e-12, torch.float32: 2e-5}


def _solver(shape, h, dtype, **opts):
    from paper_2512_13403_b200 import dh
    nz, ny, nx = shape
    return dh.Multigrid(nx, ny, nz, h, dtype=dtype, **opts)


def _rand(shape, seed, dtype, zero_mean=True):
    a = np.random.default_rng(seed).normal(size=shape)
    if zero_mean:
        a -= a.mean()
    return torch.from_numpy(a).to(dtype)


def _err(got, ref):
    ref = np.asarray(ref, dtype=np.float64)
    return float(np.abs(np.asarray(got, dtype=np.float64) - ref).max() / np.abs(ref).max())


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape", [(4, 4, 4), (4, 8, 12), (6, 4, 20)], ids=lambda s: "x".join(map(str, s)))
def test_jacobi_sweeps_alone(shape, dtype):
    """nu_coarse = 0 on a grid whose first coarse level is the coarsest: the correction is zero and the cycle is exactly
    nu1 + nu2 sweeps of Eq. 39 (both the 4-wide and the scalar kernel: nx = 4, 12, 20)."""
    h = 0.25
    F, phi = _rand(shape, 1, dtype), _rand(shape, 2, dtype, zero_mean=False)
    for nu1, nu2 in ((1, 0), (2, 1)):
        s = _solver(shape, h, dtype, nu1=nu1, nu2=nu2, nu_coarse=0)
        assert s.levels == 2
        got = phi.cuda()
        s.cycle(got, F.cuda())
        ref = mg.jacobi(phi.numpy().astype(np.float64), F.numpy().astype(np.float64), h, nu1 + nu2)
        assert _err(got.cpu().numpy(), ref) <= TOL[dtype]


@pytest.mark.parametrize("cycle", ["V", "W"])
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape", [(16, 16, 16), (12, 24, 48), (8, 8, 20), (32, 16, 64), (9, 12, 16), (3, 5, 7)],
                         ids=lambda s: "x".join(map(str, s)))
def test_cycle_parity(shape, dtype, cycle):
    """One and two cycles from a random iterate: power-of-two, 3 x 2^k (3-cell coarsest level), an nx that stops being a
    multiple of 4 on a coarse level, non-cubic, and grids that cannot be coarsened at all (single level: <= 1024 cells in
    the one-block kernel, more through per-sweep launches)."""
    h = 1.0 / shape[2]
    F, phi = _rand(shape, 11, dtype), _rand(shape, 12, dtype, zero_mean=False)
    s = _solver(shape, h, dtype, cycle=cycle)
    got = phi.cuda()
    Fd = F.cuda()
    ref = phi.numpy().astype(np.float64)
    for _ in range(2):
        s.cycle(got, Fd)
        ref = mg.cycle(ref, F.numpy().astype(np.float64), h, gamma={"V": 1, "W": 2}[cycle])
        assert _err(got.cpu().numpy(), ref) <= TOL[dtype] * (1 if dtype == torch.float64 else 4)
    assert torch.equal(Fd.cpu(), F)                      # right-hand side untouched


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_cycle_options_and_graph_replay(dtype):
    """nu1 / nu2 / nu_coarse / omega are honoured; the CUDA-graph replay is bitwise the plain launch sequence, also after
    an option change (re-capture) and with an odd total sweep count (iterate copied back from the scratch buffer)."""
    shape, h = (16, 8, 24), 0.1
    F, phi = _rand(shape, 21, dtype), _rand(shape, 22, dtype, zero_mean=False)
    kw = dict(nu1=3, nu2=2, nu_coarse=17, omega=0.8)
    a, b = phi.cuda(), phi.cuda()
    sa, sb = _solver(shape, h, dtype, graph=1, cycle="W", **kw), _solver(shape, h, dtype, graph=0, cycle="W", **kw)
    Fd = F.cuda()
    for _ in range(3):
        sa.cycle(a, Fd)
        sb.cycle(b, Fd)
    assert torch.equal(a, b)
    ref = phi.numpy().astype(np.float64)
    for _ in range(3):
        ref = mg.cycle(ref, F.numpy().astype(np.float64), h, gamma=2, **kw)
    assert _err(a.cpu().numpy(), ref) <= TOL[dtype] * (1 if dtype == torch.float64 else 4)
    sa.set_options(nu2=1)
    sb.set_options(nu2=1)
    sa.cycle(a, Fd)
    sb.cycle(b, Fd)
    assert torch.equal(a, b)
    assert sa.launches == sb.launches > 0


@pytest.mark.parametrize("cycle", ["V", "W"])
@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape", [(64, 64, 64), (16, 16, 16), (32, 16, 64), (24, 48, 96), (16, 8, 24), (64, 8, 8)],
                         ids=lambda s: "x".join(map(str, s)))
def test_coarse_levels_in_one_block_equal_the_launch_sequence(shape, dtype, cycle):
    """DH_MG_SUBTREE: a level of <= 4096 cells and everything below it as ONE kernel (levels in shared memory, the one-warp
    coarsest grid swept by warp 0 alone) against one launch per operator: the same operators in the same order of
    operations, so the results agree to rounding of differently contracted expressions (1e-14 / 2e-6 of the maximum), with
    far fewer launches; and both agree with the oracle (64^3: two levels of launches above the 16^3 subtree)."""
    h = 1.0 / shape[2]
    kw = dict(nu1=2, nu2=3, nu_coarse=9)                   # odd sweep counts: the iterate changes buffers inside the block
    F, phi = _rand(shape, 41, dtype), _rand(shape, 42, dtype, zero_mean=False)
    sa, sb = _solver(shape, h, dtype, cycle=cycle, subtree=1, **kw), _solver(shape, h, dtype, cycle=cycle, subtree=0, **kw)
    a, b, Fd = phi.cuda(), phi.cuda(), F.cuda()
    ref = phi.numpy().astype(np.float64)
    for _ in range(2):
        sa.cycle(a, Fd)
        sb.cycle(b, Fd)
        ref = mg.cycle(ref, F.numpy().astype(np.float64), h, gamma={"V": 1, "W": 2}[cycle], **kw)
    assert _err(a.cpu().numpy(), b.cpu().numpy()) <= (1e-14 if dtype == torch.float64 else 2e-6)
    assert _err(a.cpu().numpy(), ref) <= TOL[dtype] * (1 if dtype == torch.float64 else 4)
    assert sa.launches < sb.launches
    if shape == (64, 64, 64) and cycle == "W":
        # levels 64^3, 32^3 by launches: (1 + 2) x (5 sweeps + restrict + prolong) + 4 visits of the 16^3 subtree
        assert sa.launches == 2 * (3 * 7 + 4)


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
@pytest.mark.parametrize("shape", [(32, 32, 32), (12, 24, 48)], ids=lambda s: "x".join(map(str, s)))
def test_solve_matches_oracle_and_the_fft_definition(shape, dtype):
    """dh_mg_solve: same cycle count as the oracle's solve -> same iterate; enough cycles -> A^+ F of the FFT definition
    (fp64 to 1e-8, fp32 to the 1e-5 its rounding allows); F with a non-zero mean is handled by reading A23."""
    h = 1.0 / shape[2]
    F = _rand(shape, 31, dtype, zero_mean=False) + 0.3
    s = _solver(shape, h, dtype, cycle="W")
    phi, rel = s.solve(F.cuda(), 6)
    ref, rel_ref = mg.solve(F.numpy().astype(np.float64), h, 6, gamma=2)
    assert _err(phi.cpu().numpy(), ref) <= (1e-11 if dtype == torch.float64 else 2e-5)
    assert abs(rel - rel_ref) <= (1e-6 if dtype == torch.float64 else 2e-2) * rel_ref + 1e-7
    phi, rel = s.solve(F.cuda(), 24)
    exact = mg.exact_solve(F.numpy().astype(np.float64), h)
    assert _err(phi.cpu().numpy(), exact) <= (1e-8 if dtype == torch.float64 else 2e-5)
    assert rel <= (1e-9 if dtype == torch.float64 else 5e-6), rel
    assert abs(float(phi.double().mean())) <= 1e-6 * float(phi.abs().max())


@pytest.mark.parametrize("dtype", [torch.float64, torch.float32])
def test_solve_vjp_is_the_transposed_solve(dtype):
    """Eqs. 46-48: g_F = A^+ g_phi.  Against the FFT definition, and as the transpose of the forward solve:
    <g, solve(F)> = <solve_vjp(g), F> to the accuracy of the converged solves."""
    shape, h = (24, 16, 32), 1.0 / 32
    F, g = _rand(shape, 41, dtype), _rand(shape, 42, dtype)
    s = _solver(shape, h, dtype, cycle="W")
    phi, _ = s.solve(F.cuda(), 24)
    gF, _ = s.solve_vjp(g.cuda(), 24)
    exact = mg.exact_solve(g.numpy().astype(np.float64), h)
    assert _err(gF.cpu().numpy(), exact) <= (1e-8 if dtype == torch.float64 else 2e-5)
    lhs = float((g.double() * phi.cpu().double()).sum())
    rhs = float((gF.cpu().double() * F.double()).sum())
    assert abs(lhs - rhs) <= (1e-8 if dtype == torch.float64 else 1e-4) * (abs(lhs) + abs(rhs))


def test_multigrid_error_codes():
    from paper_2512_13403_b200 import dh
    with pytest.raises(dh.DhError):
        dh.dh_mg_create(1, 8, 8, 0.1, dh.DH_F32)
    with pytest.raises(dh.DhError):
        dh.dh_mg_create(8, 8, 8, 0.0, dh.DH_F32)
    s = _solver((8, 8, 8), 0.1, torch.float32)
    assert s.levels == 3                                  # 8 -> 4 -> 2
    for key, bad in (("gamma", 3), ("nu1", -1), ("nu2", 2.5), ("omega", 0.0), ("nu_coarse", 5000)):
        with pytest.raises(dh.DhError):
            s.set_options(**{key: bad})
    a = torch.zeros((8, 8, 8), device="cuda")
    with pytest.raises(dh.DhError):
        dh.dh_mg_cycle(s.ctx, a.data_ptr(), a.data_ptr())
    with pytest.raises(ValueError):
        s.cycle(a.double(), a.double())
