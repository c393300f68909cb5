"""Pins of the multigrid Poisson oracle (oracle/poisson.py; §6.2, Appendix C) against what the mathematics
fixes: discrete eigenmodes of Eq. 38, the smoothing factor of Eq. 39, exactness of the transfer operators on constants
and linear functions, the textbook convergence factor of the cycle, and the FFT definition of A^+."""
import numpy as np
import pytest

from oracle import poisson as mg


def _mode(shape, k):
    z, y, x = np.meshgrid(*[np.arange(n) for n in shape], indexing="ij")
    return np.cos(2 * np.pi * (k[0] * z / shape[0] + k[1] * y / shape[1] + k[2] * x / shape[2]) + 0.3)


def _theta(shape, k):
    return [2 * np.pi * k[a] / shape[a] for a in range(3)]


def test_laplacian_eigenmodes_closed_form():
    """A cos(k.x) = -(4/h^2) sum_a sin^2(theta_a / 2) cos(k.x): pins the stencil weights, the sign and the 1/h^2."""
    shape, h = (8, 12, 16), 0.37
    for k in ((1, 0, 0), (0, 2, 0), (0, 0, 3), (2, 5, 7)):
        u = _mode(shape, k)
        lam = -4.0 / h ** 2 * sum(np.sin(t / 2) ** 2 for t in _theta(shape, k))
        assert np.allclose(mg.laplacian(u, h), lam * u, rtol=0, atol=1e-12 * abs(lam) + 1e-13)


def test_jacobi_smoothing_factor_and_fixed_point():
    """Eq. 39 on the error of one eigenmode: e <- (1 - omega + omega/3 sum_a cos theta_a) e; with omega = 2/3 the
    highest mode (theta = pi in all three) gets -1/3 (Eq. 40's printed (1-omega)/6 would give a different factor: A21).
    The exact solution is a fixed point."""
    shape, h = (8, 8, 16), 0.5
    rng = np.random.default_rng(1)
    phi_star = rng.normal(size=shape)
    F = mg.laplacian(phi_star, h)
    assert np.allclose(mg.jacobi(phi_star, F, h, 3), phi_star, atol=1e-13)
    for k in ((1, 0, 0), (4, 4, 8), (2, 3, 5)):
        e = _mode(shape, k)
        out = mg.jacobi(phi_star + e, F, h, 1) - phi_star
        fac = 1 - mg.OMEGA + mg.OMEGA / 3 * sum(np.cos(t) for t in _theta(shape, k))
        assert np.allclose(out, fac * e, atol=1e-13)
    assert abs(1 - mg.OMEGA + mg.OMEGA / 3 * (-3) + 1 / 3) < 1e-15


def test_transfer_operators_on_constants_and_linear_functions():
    """Restriction (Eq. 42) preserves the mean and averages exactly the 8 children; prolongation (Eq. 44) reproduces
    constants and, away from the periodic seam, linear functions of the cell-centre coordinate exactly: this pins the
    3/4-1/4 weights and which neighbour each parity of fine cell takes."""
    rng = np.random.default_rng(2)
    r = rng.normal(size=(8, 12, 16))
    rc = mg.restrict(r)
    assert rc.shape == (4, 6, 8) and abs(rc.mean() - r.mean()) < 1e-15
    assert np.isclose(rc[1, 2, 3], r[2:4, 4:6, 6:8].mean())
    assert np.array_equal(mg.prolong(np.full((4, 4, 4), 2.5)), np.full((8, 8, 8), 2.5))
    nc = 8
    Z, Y, X = np.meshgrid(*[(np.arange(nc) + 0.5) * 2.0] * 3, indexing="ij")       # coarse centres, H = 2
    e = 0.3 * X - 1.1 * Y + 0.7 * Z + 0.2
    zf, yf, xf = np.meshgrid(*[(np.arange(2 * nc) + 0.5) * 1.0] * 3, indexing="ij")  # fine centres, h = 1
    want = 0.3 * xf - 1.1 * yf + 0.7 * zf + 0.2
    got = mg.prolong(e)
    assert np.allclose(got[1:-1, 1:-1, 1:-1], want[1:-1, 1:-1, 1:-1], atol=1e-13)
    # adjointness up to the volume factor fails for trilinear vs 8-cell mean (P != 8 R^T): the cycle is not symmetric,
    # which is why the VJP is a converged solve (Eq. 48) and not a transposed cycle
    u, v = rng.normal(size=(4, 4, 4)), rng.normal(size=(8, 8, 8))
    assert abs((mg.prolong(u) * v).sum() - 8 * (u * mg.restrict(v)).sum()) > 1e-3


@pytest.mark.parametrize("gamma", [1, 2])
def test_cycle_convergence_factor_is_grid_independent(gamma):
    """Textbook multigrid behaviour: the residual falls by a fixed factor per cycle, about the same
    at 16^3 and 32^3, and the W-cycle's factor is not worse than the V-cycle's."""
    facs = {}
    for n in (16, 32):
        rng = np.random.default_rng(n)
        F = rng.normal(size=(n, n, n))
        F -= F.mean()
        h = 1.0 / n
        phi = np.zeros_like(F)
        res = [np.linalg.norm(mg.residual(phi, F, h))]
        for _ in range(5):
            phi = mg.cycle(phi, F, h, gamma=gamma)
            res.append(np.linalg.norm(mg.residual(phi, F, h)))
        facs[n] = (res[5] / res[1]) ** 0.25
    assert all(f < 0.35 for f in facs.values()), facs
    assert abs(facs[16] - facs[32]) < 0.1, facs
    test_cycle_convergence_factor_is_grid_independent.seen = getattr(test_cycle_convergence_factor_is_grid_independent, "seen", {})
    test_cycle_convergence_factor_is_grid_independent.seen[gamma] = facs[32]
    seen = test_cycle_convergence_factor_is_grid_independent.seen
    if 1 in seen and 2 in seen:
        assert seen[2] <= seen[1] + 1e-3, seen


def test_exact_solve_is_the_pseudo_inverse_and_solve_converges_to_it():
    """exact_solve: A phi = F - mean(F), zero-mean phi, symmetric (<g, A^+ F> = <A^+ g, F>, Eq. 46).  The cycled solve
    converges to it, non-cubic grid with a 3-cell coarsest level included."""
    rng = np.random.default_rng(5)
    for shape in ((16, 16, 16), (12, 24, 48)):
        h = 1.0 / shape[2]
        F, g = rng.normal(size=shape), rng.normal(size=shape)
        phi = mg.exact_solve(F, h)
        assert abs(phi.mean()) < 1e-15 * np.abs(phi).max() + 1e-18
        assert np.allclose(mg.laplacian(phi, h), F - F.mean(), atol=1e-9 * np.abs(F).max())
        lhs, rhs = (g * phi).sum(), (mg.exact_solve(g, h) * F).sum()
        assert abs(lhs - rhs) <= 1e-12 * (abs(lhs) + abs(rhs))
        got, rel = mg.solve(F, h, ncycles=20, gamma=2)
        assert rel < 1e-8, rel
        assert np.abs(got - phi).max() <= 1e-7 * np.abs(phi).max()
        gF, _ = mg.solve_vjp(g, h, ncycles=20, gamma=2)
        assert np.abs(gF - mg.exact_solve(g, h)).max() <= 1e-7 * np.abs(gF).max()


def test_point_mass_potential_matches_continuum_far_field_shape():
    """A smooth zero-mean source with a known continuum solution: F = -(2 pi)^2 |k|^2 cos(2 pi k.x) has phi = cos(2 pi
    k.x); the discrete solution converges to it at second order in h (pins h^2 scaling end to end)."""
    errs = []
    for n in (16, 32):
        h = 1.0 / n
        c = (np.arange(n) + 0.5) * h
        z, y, x = np.meshgrid(c, c, c, indexing="ij")
        phi_c = np.cos(2 * np.pi * (x + 2 * y - z))
        F = -(2 * np.pi) ** 2 * 6 * phi_c
        got, _ = mg.solve(F, h, ncycles=12)
        errs.append(np.abs(got - phi_c).max())
    assert 3.5 < errs[0] / errs[1] < 4.5, errs
