"""dh_stream_host (include/dh.h): a host-resident state stepped through z-slab copies on two streams.  The contract is
bitwise: every launch covers a z range, the per-cell arithmetic is the same whatever the range, and dt comes from the same
reduction, so U_host must equal dh_advance on a resident state (itself checked against the oracle in test_gpu_parity.py)
bit for bit, for every slab size, including slabs that do not divide nz, one slab, and the wrapped last predictor range."""
import pytest
import torch

import oracle
from test_gpu_parity import TOL, _solver, max_rel_err, oracle_params, random_state

pytestmark = pytest.mark.gpu


def _resident(U, nsteps, gamma, **opts):
    s = _solver(U, gamma, **opts)
    a = U.cuda()
    dt = s.advance(a, nsteps)
    return a.cpu(), dt


@pytest.mark.parametrize("slab", [0, 8, 11, 64])
@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_stream_host_is_bitwise_the_resident_run(dtype, slab):
    """RK2 + fused kernel: predictor ranges chase the arriving slabs, corrector slab by slab.  nz = 50: slabs of 8
    (6 full + a ragged one), 11 (ragged), 64 (one slab: the single wrapped range [2, nz + 2)), 0 = automatic."""
    U = random_state((50, 30, 132), 17, 5 / 3, dtype, mach=1.5)
    ref, dt_ref = _resident(U, 4, 5 / 3)
    s = _solver(U, 5 / 3, stream_slab=slab)
    h = U.clone().pin_memory()
    dt = s.stream_host(h, 4)
    assert dt == dt_ref
    assert torch.equal(h, ref)
    # one step per call (every call starts with the full reduction) gives the same state: dt is bit-identical either way
    h2 = U.clone().pin_memory()
    for _ in range(4):
        dt2 = s.stream_host(h2, 1)
    assert dt2 == dt_ref
    assert torch.equal(h2, ref)


@pytest.mark.parametrize("opts", [
    dict(cooling=1, lambda0=0.5),                              # fused cooling epilogue in the slab-wise corrector
    dict(cooling=1, lambda0=0.5, cool_nsub=3),                 # cooling as a pass of its own: whole steps between the copies
    dict(cooling=1, lambda0=0.5, c_cool=0.1),                  # Eq. 21: the full reduction every step
    dict(integrator="heun"), dict(integrator="ssprk3"),
    dict(limiter="vanleer", riemann="hll"),
    dict(kernel="gather"),
    dict(fuse_cfl=0),
], ids=lambda o: "-".join(f"{k}={v}" for k, v in o.items()))
def test_stream_host_variants(opts):
    U = random_state((40, 22, 68), 23, 1.4, torch.float32, mach=1.0)
    ref, dt_ref = _resident(U, 3, 1.4, **opts)
    s = _solver(U, 1.4, stream_slab=8, **opts)
    h = U.clone().pin_memory()
    assert s.stream_host(h, 3) == dt_ref
    assert torch.equal(h, ref)


def test_stream_host_odd_nx_and_pageable_memory():
    """Odd nx takes the gather kernels (whole-grid launches); a pageable host buffer makes the copies synchronous,
    not wrong."""
    U = random_state((24, 10, 33), 29, 5 / 3, torch.float64)
    ref, dt_ref = _resident(U, 2, 5 / 3)
    s = _solver(U, 5 / 3)
    h = U.clone()
    assert s.stream_host(h, 2) == dt_ref
    assert torch.equal(h, ref)


def test_stream_host_against_the_oracle_and_reuse():
    """Two steps through the host path against the oracle (1e-12), then the same context keeps serving resident
    calls, and a second streamed call starts from the host state it is given (no stale device copy is used)."""
    U = random_state((32, 16, 64), 31, 5 / 3, torch.float64, mach=0.8)
    p = oracle_params(U, 5 / 3)
    ref = U.numpy().copy()
    for _ in range(2):
        dt, _ = oracle.cfl_dt(ref, p)
        ref = oracle.step(ref, dt, p)
    s = _solver(U, 5 / 3, stream_slab=8)
    h = U.clone().pin_memory()
    assert s.stream_host(h, 2) == dt
    assert max_rel_err(h.numpy(), ref) <= TOL[torch.float64]
    a = U.cuda()
    s.advance(a, 2)
    assert torch.equal(a.cpu(), h)
    h.copy_(U)                                                   # the caller changes the host state between calls
    s.stream_host(h, 2)
    assert torch.equal(a.cpu(), h)
    assert s.stream_host(h, 0) == s.stream_host(h, 0)            # nsteps = 0: nothing moves
    assert torch.equal(a.cpu(), h)


def test_stream_host_nonfinite_is_reported():
    from paper_2512_13403_b200 import dh
    U = random_state((16, 16, 64), 37, 5 / 3, torch.float32)
    U[4, 3, 2, 1] = float("nan")
    s = _solver(U, 5 / 3)
    h = U.clone().pin_memory()
    with pytest.raises(dh.DhError) as e:
        s.stream_host(h, 2)
    assert e.value.code == dh.DH_ERR_NONFINITE
