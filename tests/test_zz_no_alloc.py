"""dh_cfl_dt_static (include/dh.h): the CFL time step for callers that must not allocate.  No context, the scratch of the
reduction in a file-scope device array (256 KiB), inputs and outputs the caller's.  Checked against the existing path
(dh_cfl_dt through a context), at the tolerance the dt tests use everywhere: bit-identical.  Collected last on purpose
(the suite runs with pytest -x); passes alone in a fresh process and after the other tests."""
import pytest
import torch

pytestmark = pytest.mark.gpu


def _state(shape, seed, gamma, dtype, mach=1.5):
    g = torch.Generator().manual_seed(seed)
    rho = torch.rand(shape, generator=g, dtype=torch.float64) * 1.5 + 0.5
    v = torch.randn((3,) + tuple(shape), generator=g, dtype=torch.float64) * mach
    P = torch.rand(shape, generator=g, dtype=torch.float64) * 1.5 + 0.5
    U = torch.stack([rho, rho * v[0], rho * v[1], rho * v[2], P / (gamma - 1) + 0.5 * rho * (v ** 2).sum(0)])
    return U.to(dtype).cuda()


def _existing(U, gamma, cfl, box):
    from paper_2512_13403_b200 import dh
    _, nz, ny, nx = U.shape
    s = dh.Solver(nx, ny, nz, gamma=gamma, dtype=U.dtype, cfl=cfl, lx=box[0], ly=box[1], lz=box[2])
    return s.cfl_dt(U)


def _static(U, gamma, cfl, box, out):
    from paper_2512_13403_b200 import dh
    _, nz, ny, nx = U.shape
    dt_code = dh.DH_F32 if U.dtype == torch.float32 else dh.DH_F64
    dh.dh_cfl_dt_static(U.data_ptr(), nx, ny, nz, dt_code, gamma, cfl, box, 1e-10, 1e-10, out.data_ptr(),
                        torch.cuda.current_stream().cuda_stream)


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_static_cfl_equals_the_existing_path_on_two_calls_in_a_row(dtype):
    """Two calls in a row on different states and grid sizes share the array: the second (fewer blocks than the first) must
    not see the first call's records; then the first state again.  87 x 50 x 41 = 178350 cells: 11 blocks, a ragged last one."""
    gamma, cfl, box = 1.4, 0.4, (1.0, 2.0, 0.5)
    out = torch.full((5,), -1.0, dtype=torch.float64, device="cuda")
    Ua = _state((41, 50, 87), 5, gamma, dtype, mach=2.0)
    Ub = _state((8, 12, 20), 6, gamma, dtype, mach=0.2)             # one block; slower waves than Ua's
    ref_a, ref_b = _existing(Ua, gamma, cfl, box), _existing(Ub, gamma, cfl, box)
    assert ref_a != ref_b
    for U, ref in ((Ua, ref_a), (Ub, ref_b), (Ua, ref_a)):
        _static(U, gamma, cfl, box, out)
        got = out.cpu()
        assert got[0].item() == ref                                  # bit-identical dt (the T value widened)
        assert got[4].item() == 0.0
        assert (got[1:4] > 0).all()
    # back to back without a host read in between: stream order alone separates the calls
    out2 = torch.empty_like(out)
    _static(Ua, gamma, cfl, box, out)
    _static(Ub, gamma, cfl, box, out2)
    assert out.cpu()[0].item() == ref_a and out2.cpu()[0].item() == ref_b


def test_static_cfl_allocates_nothing_and_reports_nonfinite():
    from paper_2512_13403_b200 import dh
    gamma = 5 / 3
    U = _state((16, 16, 64), 7, gamma, torch.float32)
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    _static(U, gamma, 0.4, None, out)                                # first call on this device: the address look-up
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        _static(U, gamma, 0.4, None, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0                                            # no device memory was taken by the calls
    assert out.cpu()[0].item() == _existing(U, gamma, 0.4, (1.0, 1.0, 1.0))
    U[4, 3, 2, 1] = float("nan")
    _static(U, gamma, 0.4, None, out)
    assert out.cpu()[4].item() == 1.0
    # sizes beyond the static scratch are rejected with a clear message, before anything is launched
    assert dh.dh_static_max_cells() == 1 << 27
    with pytest.raises(dh.DhError) as e:
        dh.dh_cfl_dt_static(U.data_ptr(), 1024, 1024, 129, dh.DH_F32, gamma, 0.4, None, 1e-10, 1e-10, out.data_ptr(), 0)
    assert e.value.code == dh.DH_ERR_ARG and "static scratch" in str(e.value)
