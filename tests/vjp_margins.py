"""Element-by-element validity of a VJP computed in another precision (test helper; calls only oracle/).

The step is piecewise smooth ("non-smooth operators"; readings A7 / A17 in DESIGN.md): its a.e. derivative
follows the branch every compare takes.  An fp32 evaluation takes the same branches as the fp64 oracle except where the
compared quantities agree to within fp32 rounding; there both one-sided derivatives are valid and the entries whose
stencil contains such a compare may differ by O(1).  Everything else is unique up to rounding and is held to the stated
per-cell tolerance.

`vjp_condition` returns, for every cell, the smallest decision margin (oracle.decision_margins: distance from the tie
relative to the rounding scale of the operands) over all compares its gradient entry depends on:

  one reversed stage  [J_D(X)^T g]_i  uses, per axis, the limiter calls of cells i-2..i+2 and the Riemann compares of
  faces i-2..i+1 on the line through i, the floors of prim() at i, and g on the "plus" stencil i +- 2 along each axis;

  the step chains its stages backwards (oracle step_vjp): cond_k = min(stage_k, plus_min(cond_{k+1})),
  with the compares of the cooling update at the last stage (they act on g_out pointwise).

FP32_BOUND: the margin below which an fp32 evaluation may decide differently.  Primitives carry <= 3 ulp (MUFU
reciprocal + multiply, or the subtraction in P), the second stage starts from a state that is itself rounded and carries
the rounded fluxes of the first (<= 3 ulp more), a difference of two such values doubles it: 12 ulp = 12 x 2^-24 of the
scale; 16 x 2^-24 ~ 9.5e-7 is used.
"""
import numpy as np

import oracle

FP32_BOUND = 16.0 * 2.0 ** -24


def _line_min(m, a, r=2):
    """min over cells i-r..i+r along axis a (0 = x = last array axis), periodic."""
    ax = m.ndim - 1 - a
    out = m.copy()
    for s in range(1, r + 1):
        np.minimum(out, np.roll(m, s, axis=ax), out=out)
        np.minimum(out, np.roll(m, -s, axis=ax), out=out)
    return out


def plus_min(c):
    out = _line_min(c, 0)
    for a in (1, 2):
        np.minimum(out, _line_min(c, a), out=out)
    return out


def stage_condition(X, p):
    """Per cell: smallest margin of the compares [J_D(X)^T g]_i depends on."""
    M = oracle.decision_margins(X, p)
    c = M[3].copy()
    for a in range(3):
        np.minimum(c, _line_min(M[a], a), out=c)
    return c


def _line_max(m, a, r=2):
    ax = m.ndim - 1 - a
    out = m.copy()
    for s in range(1, r + 1):
        np.maximum(out, np.roll(m, s, axis=ax), out=out)
        np.maximum(out, np.roll(m, -s, axis=ax), out=out)
    return out


def plus_max(c):
    out = _line_max(c, 0)
    for a in (1, 2):
        np.maximum(out, _line_max(c, a), out=out)
    return out


def vjp_sensitivity(U, dt, p):
    """[nz, ny, nx]: the largest limiter conditioning number (oracle.limiter_conditioning) over the slopes a cell's step-VJP entries
    depend on (same stencil chain as vjp_condition).  Zero unless the limiter is van Leer, whose derivative 2 b^2 / (a + b)^2 is
    smooth but moves by ~ 12 eps s / (|a| + |b|) when the differences are rounded to eps s; check_vjp widens the tolerance of an
    entry by SENS_ULPS x 2^-24 x this number."""
    if p.limiter != 1:
        return None
    states, _ = stage_states(U, dt, p)
    sens = None
    for X in reversed(states):
        C = oracle.limiter_conditioning(X, p)
        c = np.zeros(C.shape[1:])
        for a in range(3):
            np.maximum(c, _line_max(C[a], a), out=c)
        if sens is not None:
            np.maximum(c, plus_max(sens), out=c)
        sens = c
    return sens


SENS_ULPS = 2.0


def stage_states(U, dt, p):
    """The states at which D() is evaluated, in forward order, and the pre-cooling result (oracle step(), Eqs. A6-A7 /
    reading A18), assembled from oracle.flux_divergence."""
    U = np.asarray(U, dtype=np.float64)
    D = oracle.flux_divergence
    if p.integrator == 0:
        Us = U - 0.5 * dt * D(U, p)
        return [U, Us], U - dt * D(Us, p)
    if p.integrator == 1:
        Ua = U - dt * D(U, p)
        return [U, Ua], 0.5 * (U + (Ua - dt * D(Ua, p)))
    Ua = U - dt * D(U, p)
    Ub = 0.75 * U + 0.25 * (Ua - dt * D(Ua, p))
    return [U, Ua, Ub], U / 3.0 + (2.0 / 3.0) * (Ub - dt * D(Ub, p))


def vjp_condition(U, dt, p):
    """[nz, ny, nx]: for every cell the smallest decision margin its five step-VJP entries depend on."""
    states, U1 = stage_states(U, dt, p)
    cool = oracle.cooling_margins(U1, dt, p) if p.cooling else None
    cond = None
    for X in reversed(states):
        c = stage_condition(X, p)
        if cond is None:
            if cool is not None:
                np.minimum(c, plus_min(cool), out=c)
        else:
            np.minimum(c, plus_min(cond), out=c)
        cond = c
    if cool is not None:
        np.minimum(cond, cool, out=cond)
    return cond


def gradient_scales(ref):
    """s_f of reading A15 for a gradient: grid rms of the field, the three momentum components pooled."""
    rms = lambda a: float(np.sqrt(np.mean(np.square(a, dtype=np.float64))))
    sm = float(np.sqrt(np.mean(ref[1] ** 2 + ref[2] ** 2 + ref[3] ** 2)))
    return np.array([rms(ref[0]), sm, sm, sm, rms(ref[4])]).reshape(5, 1, 1, 1)


def check_vjp(got, ref, cond, tol, bound=FP32_BOUND, max_excluded=1.0, scales=None, label="", sens=None):
    """Every entry whose stencil margin is >= bound within `tol` (per-cell relative error, A15 normalisation); the
    others (either one-sided derivative is valid there) finite and of the gradient's magnitude.  Returns (worst
    well-conditioned error, excluded fraction)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    s = gradient_scales(ref) if scales is None else scales
    e = np.abs(got - ref) / np.maximum(np.abs(ref), s)
    if sens is not None:                                 # van Leer: per-entry tolerance tol + SENS_ULPS 2^-24 sens; e is rescaled to `tol`
        e = e * (tol / (tol + SENS_ULPS * 2.0 ** -24 * np.minimum(sens, 1e6)))
    well = np.broadcast_to(cond >= bound, e.shape)
    excluded = 1.0 - float(well[0].mean())
    worst = float(e[well].max()) if well.any() else 0.0
    print(f"vjp check {label}: worst well-conditioned rel err {worst:.3e} (tol {tol:.1e}), "
          f"excluded {100 * excluded:.3f} % of the cells (margin < {bound:.2e})")
    assert np.isfinite(got).all(), label
    assert worst <= tol, (label, worst)
    assert excluded <= max_excluded, (label, excluded)
    if (~well).any():
        loose = float((np.abs(got - ref) / s)[~well].max())
        assert loose <= 1e3, (label, loose)
    return worst, excluded
