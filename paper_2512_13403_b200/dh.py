"""Thin ctypes binding over the C-ABI library (include/dh.h): argument marshalling only.

Every step of the path (CFL reduction, both RK2 stages, cooling, the reverse-mode stages) runs in the CUDA
kernels of ``libdh.so``; PyTorch is used for device memory and streams.  There is no CPU fallback: if the
library cannot be built/loaded, or no CUDA device is present, calls raise.

The module-level functions carry the C names (``dh_create`` ... ``dh_destroy``); ``Solver`` wraps a context.
"""
from __future__ import annotations

import ctypes
import os

import torch

from . import build as _build

DH_F32, DH_F64 = 0, 1
DH_OK, DH_ERR_ARG, DH_ERR_CUDA, DH_ERR_ALLOC, DH_ERR_NONFINITE = 0, -1, -2, -3, -4
OPTIONS = {
    "cfl": 0, "lx": 1, "ly": 2, "lz": 3, "cooling": 4, "lambda0": 5, "alpha": 6, "t_floor": 7,
    "rho_floor": 8, "p_floor": 9, "kernel": 10, "limiter": 11, "rev_slab": 12, "integrator": 13, "fuse_cfl": 14,
    "riemann": 15, "cool_mode": 16, "cool_nsub": 17, "c_cool": 18, "dt_max": 19, "cool_law": 20, "t_switch": 21,
    "lambda1": 22, "alpha1": 23, "lambda2": 24, "alpha2": 25, "gamma0": 26, "f_sub": 27, "stream_slab": 28,
}
LIMITERS = {"minmod": 0, "vanleer": 1, "mc": 2}
RIEMANN = {"hllc": 0, "hll": 1, "rusanov": 2}       # DH_OPT_RIEMANN
COOL_MODES = {"euler": 0, "trapezoid": 1, "masked": 2}   # DH_OPT_COOL_MODE
COOL_LAWS = {"powerlaw": 0, "twobranch": 1}         # DH_OPT_COOL_LAW
INTEGRATORS = {"vl2": 0, "heun": 1, "ssprk3": 2}    # DH_OPT_INTEGRATOR
KERNELS = {"fused": 0, "gather": 1}

# every symbol include/dh.h declares (checked by tests/test_abi.py)
SYMBOLS = [
    "dh_create", "dh_destroy", "dh_set_stream", "dh_set_option", "dh_get_option", "dh_cfl_dt", "dh_step",
    "dh_step_devdt", "dh_cfl_dt_async", "dh_poll_status", "dh_step_vjp", "dh_run_host", "dh_stream_host", "dh_step_vjp_host",
    "dh_advance", "dh_adjoint", "dh_launch_count", "dh_last_error", "dh_version", "dh_profile_enable", "dh_profile_read",
    "dh_cfl_stats", "dh_cool_tmin", "dh_set_cooling_table", "dh_cool_table_vjp",
    "dh_cfl_dt_static", "dh_static_max_cells", "dh_gravity_source", "dh_gravity_source_vjp", "dh_step_gravity", "dh_step_gravity_vjp",
    "dh_mg_create", "dh_mg_destroy", "dh_mg_set_stream", "dh_mg_set_option", "dh_mg_levels", "dh_mg_launches",
    "dh_mg_cycle", "dh_mg_solve", "dh_mg_solve_vjp", "dh_issue_probe", "dh_issue_probe_name",
]
MG_OPTIONS = {"nu1": 0, "nu2": 1, "gamma": 2, "nu_coarse": 3, "omega": 4, "graph": 5, "subtree": 6}
MG_CYCLES = {"V": 1, "W": 2}
KERNEL_KINDS = ["cfl_reduce", "cfl_finish", "stage1", "stage2", "rev2", "rev1", "cool_vjp", "lincomb", "cool", "cfl_cand"]

_lib = None


class DhError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"dh error {code}: {msg}")
        self.code = code


def load(rebuild: bool = False):
    """Load libdh.so (building it in-tree with nvcc if it is missing or stale).  Raises on failure."""
    global _lib
    if _lib is not None and not rebuild:
        return _lib
    path = _build.build(force=rebuild)
    lib = ctypes.CDLL(path)
    vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
    pd = ctypes.POINTER(ctypes.c_double)
    lib.dh_create.restype = vp
    lib.dh_create.argtypes = [ci, ci, ci, cd, ci]
    lib.dh_destroy.restype = None
    lib.dh_destroy.argtypes = [vp]
    lib.dh_set_stream.argtypes = [vp, vp]
    lib.dh_set_option.argtypes = [vp, ci, cd]
    lib.dh_get_option.argtypes = [vp, ci, pd]
    lib.dh_cfl_dt.argtypes = [vp, vp, pd]
    lib.dh_cfl_dt_async.argtypes = [vp, vp]
    lib.dh_poll_status.argtypes = [vp, pd]
    lib.dh_step.argtypes = [vp, vp, cd]
    lib.dh_step_devdt.argtypes = [vp, vp]
    lib.dh_step_vjp.argtypes = [vp, vp, cd, vp, vp]
    lib.dh_run_host.argtypes = [vp, vp, ci, pd]
    lib.dh_stream_host.argtypes = [vp, vp, ci, pd]
    lib.dh_cfl_dt_static.argtypes = [vp, ci, ci, ci, ci, cd, cd, pd, cd, cd, vp, vp]
    lib.dh_cfl_dt_static.restype = ci
    lib.dh_static_max_cells.argtypes = []
    lib.dh_static_max_cells.restype = ctypes.c_size_t
    lib.dh_issue_probe.argtypes = [ci, ci, ci, pd, ctypes.POINTER(ci)]
    lib.dh_issue_probe.restype = ci
    lib.dh_issue_probe_name.argtypes = [ci]
    lib.dh_issue_probe_name.restype = ctypes.c_char_p
    lib.dh_stream_host.restype = ci
    lib.dh_advance.argtypes = [vp, vp, ci, pd]
    lib.dh_adjoint.argtypes = [vp, vp, vp, ci, ci, pd]
    lib.dh_step_vjp_host.argtypes = [vp, vp, cd, vp, vp]
    lib.dh_launch_count.restype = ctypes.c_ulonglong
    lib.dh_launch_count.argtypes = [vp]
    lib.dh_profile_enable.argtypes = [vp, ci]
    lib.dh_profile_read.argtypes = [vp, pd, ctypes.POINTER(ctypes.c_ulonglong)]
    lib.dh_cfl_stats.argtypes = [vp, ctypes.POINTER(ctypes.c_ulonglong)]
    lib.dh_cfl_stats.restype = ci
    lib.dh_cool_tmin.argtypes = [vp, vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
    lib.dh_cool_tmin.restype = ci
    lib.dh_set_cooling_table.argtypes = [vp, pd, ci, cd, cd]
    lib.dh_set_cooling_table.restype = ci
    lib.dh_cool_table_vjp.argtypes = [vp, vp, cd, vp, pd]
    lib.dh_cool_table_vjp.restype = ci
    lib.dh_gravity_source.argtypes = [vp, vp, vp, cd]
    lib.dh_gravity_source_vjp.argtypes = [vp, vp, vp, cd, vp, vp, vp]
    lib.dh_step_gravity.argtypes = [vp, vp, vp, cd, cd, ci]
    lib.dh_step_gravity_vjp.argtypes = [vp, vp, vp, cd, cd, ci, vp, vp]
    for fn in ("dh_gravity_source", "dh_gravity_source_vjp", "dh_step_gravity", "dh_step_gravity_vjp"):
        getattr(lib, fn).restype = ci
    lib.dh_last_error.restype = ctypes.c_char_p
    lib.dh_version.restype = ctypes.c_char_p
    for fn in ("dh_set_stream", "dh_set_option", "dh_get_option", "dh_cfl_dt", "dh_cfl_dt_async", "dh_poll_status",
               "dh_step", "dh_step_devdt", "dh_step_vjp", "dh_run_host", "dh_advance", "dh_adjoint", "dh_step_vjp_host", "dh_profile_enable",
               "dh_profile_read"):
        getattr(lib, fn).restype = ci
    lib.dh_mg_create.restype = vp
    lib.dh_mg_create.argtypes = [ci, ci, ci, cd, ci]
    lib.dh_mg_destroy.restype = None
    lib.dh_mg_destroy.argtypes = [vp]
    lib.dh_mg_set_stream.argtypes = [vp, vp]
    lib.dh_mg_set_option.argtypes = [vp, ci, cd]
    lib.dh_mg_levels.argtypes = [vp]
    lib.dh_mg_launches.argtypes = [vp]
    lib.dh_mg_launches.restype = ctypes.c_longlong
    lib.dh_mg_cycle.argtypes = [vp, vp, vp]
    lib.dh_mg_solve.argtypes = [vp, vp, vp, ci, pd]
    lib.dh_mg_solve_vjp.argtypes = [vp, vp, vp, ci, pd]
    for fn in ("dh_mg_set_stream", "dh_mg_set_option", "dh_mg_levels", "dh_mg_cycle", "dh_mg_solve", "dh_mg_solve_vjp"):
        getattr(lib, fn).restype = ci
    _lib = lib
    return lib


def library_path() -> str:
    return _build.LIB


def _check(rc: int):
    if rc != DH_OK:
        raise DhError(rc, load().dh_last_error().decode())


# ------------------------------------------------------------------------------------ C-named functions
def dh_version() -> str:
    return load().dh_version().decode()


def dh_last_error() -> str:
    return load().dh_last_error().decode()


def dh_create(nx: int, ny: int, nz: int, gamma: float, dtype: int):
    h = load().dh_create(int(nx), int(ny), int(nz), float(gamma), int(dtype))
    if not h:
        raise DhError(DH_ERR_ARG, dh_last_error())
    return h


def dh_destroy(ctx) -> None:
    load().dh_destroy(ctx)


def dh_set_stream(ctx, cuda_stream: int) -> None:
    _check(load().dh_set_stream(ctx, ctypes.c_void_p(cuda_stream)))


def dh_set_option(ctx, key: int, value: float) -> None:
    _check(load().dh_set_option(ctx, int(key), float(value)))


def dh_get_option(ctx, key: int) -> float:
    out = ctypes.c_double()
    _check(load().dh_get_option(ctx, int(key), ctypes.byref(out)))
    return out.value


def dh_cfl_dt(ctx, U_ptr: int) -> float:
    out = ctypes.c_double()
    _check(load().dh_cfl_dt(ctx, ctypes.c_void_p(U_ptr), ctypes.byref(out)))
    return out.value


def dh_cfl_dt_static(U_ptr: int, nx: int, ny: int, nz: int, dtype: int, gamma: float, cfl: float, box, rho_floor: float,
                     p_floor: float, out5_ptr: int, stream_ptr: int = 0) -> None:
    """No context, no allocation (include/dh.h): out5_ptr is a DEVICE array of 5 doubles the caller owns."""
    b = (ctypes.c_double * 3)(*[float(v) for v in box]) if box is not None else None
    _check(load().dh_cfl_dt_static(ctypes.c_void_p(U_ptr), int(nx), int(ny), int(nz), int(dtype), float(gamma), float(cfl), b,
                                   float(rho_floor), float(p_floor), ctypes.c_void_p(out5_ptr), ctypes.c_void_p(stream_ptr)))


def dh_static_max_cells() -> int:
    return int(load().dh_static_max_cells())


ISSUE_PROBE_MIXES = 24


def issue_probe(warps_per_scheduler: int = 4, iters: int = 4000) -> list[dict]:
    """dh_issue_probe for every mix: SM cycles per instruction group per scheduler (a measurement)."""
    lib = load()
    out = []
    for mix in range(ISSUE_PROBE_MIXES):
        cyc, n = ctypes.c_double(0.0), ctypes.c_int(0)
        _check(lib.dh_issue_probe(mix, int(warps_per_scheduler), int(iters), ctypes.byref(cyc), ctypes.byref(n)))
        out.append({"mix": lib.dh_issue_probe_name(mix).decode(), "instructions": n.value, "cycles_per_group": cyc.value})
    return out


def dh_cfl_dt_async(ctx, U_ptr: int) -> None:
    _check(load().dh_cfl_dt_async(ctx, ctypes.c_void_p(U_ptr)))


def dh_poll_status(ctx) -> float:
    out = ctypes.c_double()
    _check(load().dh_poll_status(ctx, ctypes.byref(out)))
    return out.value


def dh_step(ctx, U_ptr: int, dt: float) -> None:
    _check(load().dh_step(ctx, ctypes.c_void_p(U_ptr), float(dt)))


def dh_step_devdt(ctx, U_ptr: int) -> None:
    _check(load().dh_step_devdt(ctx, ctypes.c_void_p(U_ptr)))


def dh_step_vjp(ctx, U_ptr: int, dt: float, gout_ptr: int, gin_ptr: int) -> None:
    _check(load().dh_step_vjp(ctx, ctypes.c_void_p(U_ptr), float(dt), ctypes.c_void_p(gout_ptr), ctypes.c_void_p(gin_ptr)))


def dh_advance(ctx, U_ptr: int, nsteps: int, sync: bool = True):
    """nsteps x (CFL dt + RK2 step) on the device; returns the last dt if `sync`, else None (asynchronous)."""
    if sync:
        out = ctypes.c_double()
        _check(load().dh_advance(ctx, ctypes.c_void_p(U_ptr), int(nsteps), ctypes.byref(out)))
        return out.value
    _check(load().dh_advance(ctx, ctypes.c_void_p(U_ptr), int(nsteps), None))
    return None


def dh_adjoint(ctx, U_ptr: int, gU_ptr: int, nsteps: int, every: int) -> list:
    """Adjoint of nsteps steps with checkpoints every `every` steps; returns the dt sequence."""
    dts = (ctypes.c_double * max(nsteps, 1))()
    _check(load().dh_adjoint(ctx, ctypes.c_void_p(U_ptr), ctypes.c_void_p(gU_ptr), int(nsteps), int(every), dts))
    return [dts[i] for i in range(nsteps)]


def dh_run_host(ctx, U_host_ptr: int, nsteps: int) -> float:
    out = ctypes.c_double()
    _check(load().dh_run_host(ctx, ctypes.c_void_p(U_host_ptr), int(nsteps), ctypes.byref(out)))
    return out.value


def dh_stream_host(ctx, U_host_ptr: int, nsteps: int) -> float:
    out = ctypes.c_double()
    _check(load().dh_stream_host(ctx, ctypes.c_void_p(U_host_ptr), int(nsteps), ctypes.byref(out)))
    return out.value


def dh_step_vjp_host(ctx, U_host_ptr: int, dt: float, gout_host_ptr: int, gin_host_ptr: int) -> None:
    _check(load().dh_step_vjp_host(ctx, ctypes.c_void_p(U_host_ptr), float(dt), ctypes.c_void_p(gout_host_ptr),
                                   ctypes.c_void_p(gin_host_ptr)))


def dh_launch_count(ctx) -> int:
    return int(load().dh_launch_count(ctx))


def dh_profile_enable(ctx, on: bool) -> None:
    _check(load().dh_profile_enable(ctx, 1 if on else 0))


def dh_cool_tmin(ctx, U_ptr: int):
    """(min_x t_cool(x) of Eq. 20, dt_hydro of Eq. A8) from one pass of the CFL reduction (include/dh.h)."""
    t, d = ctypes.c_double(), ctypes.c_double()
    _check(load().dh_cool_tmin(ctx, ctypes.c_void_p(U_ptr), ctypes.byref(t), ctypes.byref(d)))
    return t.value, d.value


def dh_set_cooling_table(ctx, log10_lambda, log10_t0: float, dlog10_t: float) -> None:
    """The table of Eq. 19 for DH_OPT_COOL_LAW = 1 (include/dh.h): log10 Lambda at equally spaced log10 T nodes."""
    vals = [float(v) for v in log10_lambda]
    arr = (ctypes.c_double * len(vals))(*vals)
    _check(load().dh_set_cooling_table(ctx, arr, len(vals), float(log10_t0), float(dlog10_t)))


def dh_cool_table_vjp(ctx, U: int, dt: float, g_out: int, n: int) -> list:
    """dL / d log10_lambda[k] for the step at this dt and the cotangent g_out (device pointers), include/dh.h."""
    out = (ctypes.c_double * n)()
    _check(load().dh_cool_table_vjp(ctx, U, float(dt), g_out, out))
    return [float(v) for v in out]


def dh_cfl_stats(ctx) -> dict:
    """Counters of the CFL candidate path of dh_advance (include/dh.h)."""
    out = (ctypes.c_ulonglong * 3)()
    _check(load().dh_cfl_stats(ctx, out))
    return {"candidate_passes": int(out[0]), "fallbacks": int(out[1]), "packs": int(out[2])}


def dh_profile_read(ctx) -> dict:
    """{kernel kind: (milliseconds, launches)} recorded since the last read."""
    n = len(KERNEL_KINDS)
    ms = (ctypes.c_double * n)()
    cnt = (ctypes.c_ulonglong * n)()
    _check(load().dh_profile_read(ctx, ms, cnt))
    return {k: (ms[i], int(cnt[i])) for i, k in enumerate(KERNEL_KINDS)}


# ------------------------------------------------------------------------------------------- convenience
class Solver:
    """A dh context bound to a grid; states are torch CUDA tensors [5, nz, ny, nx]."""

    def __init__(self, nx: int, ny: int, nz: int, gamma: float = 5.0 / 3.0, dtype=torch.float32, stream=None, **options):
        if dtype not in (torch.float32, torch.float64):
            raise TypeError("dtype must be torch.float32 or torch.float64")
        if not torch.cuda.is_available():
            raise RuntimeError("dh needs a CUDA device; there is no CPU fallback")
        self.shape = (5, int(nz), int(ny), int(nx))
        self.dtype = dtype
        self.ctx = dh_create(nx, ny, nz, gamma, DH_F32 if dtype == torch.float32 else DH_F64)
        stream = stream if stream is not None else torch.cuda.current_stream()
        dh_set_stream(self.ctx, stream.cuda_stream)
        self.stream = stream
        table = options.pop("table", None)            # (log10_t0, dlog10_t, values): must precede cool_law = 1
        if table is not None:
            self.set_cooling_table(*table)
        self.set_options(**options)

    def set_options(self, **options):
        for k, v in options.items():
            if k == "limiter" and isinstance(v, str):
                v = LIMITERS[v]
            if k == "cool_mode" and isinstance(v, str):
                v = COOL_MODES[v]
            if k == "cool_law" and isinstance(v, str):
                v = COOL_LAWS[v]
            if k == "riemann" and isinstance(v, str):
                v = RIEMANN[v]
            if k == "integrator" and isinstance(v, str):
                v = INTEGRATORS[v]
            if k == "kernel" and isinstance(v, str):
                v = KERNELS[v]
            dh_set_option(self.ctx, OPTIONS[k], float(v))

    def get_option(self, name: str) -> float:
        return dh_get_option(self.ctx, OPTIONS[name])

    def _dev(self, t: torch.Tensor, name: str) -> int:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == self.dtype and tuple(t.shape) == self.shape):
            raise ValueError(f"{name} must be a contiguous CUDA tensor of shape {self.shape} and dtype {self.dtype}")
        return t.data_ptr()

    def _host(self, t: torch.Tensor, name: str) -> int:
        if not (isinstance(t, torch.Tensor) and not t.is_cuda and t.is_contiguous() and t.dtype == self.dtype and tuple(t.shape) == self.shape):
            raise ValueError(f"{name} must be a contiguous host tensor of shape {self.shape} and dtype {self.dtype}")
        return t.data_ptr()

    def cfl_dt(self, U) -> float:
        return dh_cfl_dt(self.ctx, self._dev(U, "U"))

    def cfl_dt_async(self, U) -> None:
        dh_cfl_dt_async(self.ctx, self._dev(U, "U"))

    def poll(self) -> float:
        return dh_poll_status(self.ctx)

    def step(self, U, dt: float) -> None:
        dh_step(self.ctx, self._dev(U, "U"), dt)

    def advance(self, U, nsteps: int, sync: bool = True):
        return dh_advance(self.ctx, self._dev(U, "U"), nsteps, sync)

    def adjoint(self, U, gU, nsteps: int, every: int) -> list:
        """U: U_0 -> U_n in place; gU: dL/dU_n -> dL/dU_0 in place; returns the dt sequence."""
        return dh_adjoint(self.ctx, self._dev(U, "U"), self._dev(gU, "gU"), nsteps, every)

    def step_devdt(self, U) -> None:
        dh_step_devdt(self.ctx, self._dev(U, "U"))

    def step_vjp(self, U, dt: float, g_out, g_in=None):
        if g_in is None:
            g_in = torch.empty_like(U)
        dh_step_vjp(self.ctx, self._dev(U, "U"), dt, self._dev(g_out, "g_out"), self._dev(g_in, "g_in"))
        return g_in

    def set_cooling_table(self, log10_t0: float, dlog10_t: float, log10_lambda) -> None:
        self._ntab = len(log10_lambda)
        dh_set_cooling_table(self.ctx, log10_lambda, log10_t0, dlog10_t)

    def cool_table_vjp(self, U, dt: float, g_out) -> list:
        return dh_cool_table_vjp(self.ctx, self._dev(U, "U"), dt, self._dev(g_out, "g_out"), self._ntab)

    def _field(self, t: torch.Tensor, name: str) -> int:
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous() and t.dtype == self.dtype and tuple(t.shape) == self.shape[1:]):
            raise ValueError(f"{name} must be a contiguous CUDA tensor of shape {self.shape[1:]} and dtype {self.dtype}")
        return t.data_ptr()

    def gravity_source(self, U, phi, dt: float) -> None:
        _check(load().dh_gravity_source(self.ctx, self._dev(U, "U"), self._field(phi, "phi"), float(dt)))

    def gravity_source_vjp(self, U, phi, dt: float, g_out):
        g_in, g_phi = torch.empty_like(U), torch.empty_like(phi)
        _check(load().dh_gravity_source_vjp(self.ctx, self._dev(U, "U"), self._field(phi, "phi"), float(dt), self._dev(g_out, "g_out"),
                                            self._dev(g_in, "g_in"), self._field(g_phi, "g_phi")))
        return g_in, g_phi

    def step_gravity(self, mg, U, dt: float, four_pi_g: float, ncycles: int = 12) -> None:
        _check(load().dh_step_gravity(self.ctx, mg.ctx, self._dev(U, "U"), float(dt), float(four_pi_g), int(ncycles)))

    def step_gravity_vjp(self, mg, U, dt: float, four_pi_g: float, g_out, ncycles: int = 12):
        g_in = torch.empty_like(U)
        _check(load().dh_step_gravity_vjp(self.ctx, mg.ctx, self._dev(U, "U"), float(dt), float(four_pi_g), int(ncycles),
                                          self._dev(g_out, "g_out"), self._dev(g_in, "g_in")))
        return g_in

    def run_host(self, U_host, nsteps: int) -> float:
        return dh_run_host(self.ctx, self._host(U_host, "U_host"), nsteps)

    def stream_host(self, U_host, nsteps: int) -> float:
        return dh_stream_host(self.ctx, self._host(U_host, "U_host"), nsteps)

    def step_vjp_host(self, U_host, dt: float, g_out_host, g_in_host) -> None:
        dh_step_vjp_host(self.ctx, self._host(U_host, "U_host"), dt, self._host(g_out_host, "g_out_host"),
                         self._host(g_in_host, "g_in_host"))

    def profile(self, on: bool) -> None:
        dh_profile_enable(self.ctx, on)

    def profile_read(self) -> dict:
        return dh_profile_read(self.ctx)

    def cfl_stats(self) -> dict:
        return dh_cfl_stats(self.ctx)

    def cool_tmin(self, U):
        return dh_cool_tmin(self.ctx, self._dev(U, "U"))

    @property
    def launch_count(self) -> int:
        return dh_launch_count(self.ctx)

    def close(self):
        if getattr(self, "ctx", None):
            dh_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ------------------------------------------------------------------ multigrid Poisson solver (§6.2)
def dh_mg_create(nx: int, ny: int, nz: int, h: float, dtype: int):
    p = load().dh_mg_create(int(nx), int(ny), int(nz), float(h), int(dtype))
    if not p:
        raise DhError(DH_ERR_ARG, dh_last_error())
    return p


def dh_mg_destroy(ctx) -> None:
    load().dh_mg_destroy(ctx)


def dh_mg_set_stream(ctx, cuda_stream: int) -> None:
    _check(load().dh_mg_set_stream(ctx, ctypes.c_void_p(cuda_stream)))


def dh_mg_set_option(ctx, key: int, value: float) -> None:
    _check(load().dh_mg_set_option(ctx, int(key), float(value)))


def dh_mg_levels(ctx) -> int:
    return int(load().dh_mg_levels(ctx))


def dh_mg_launches(ctx) -> int:
    return int(load().dh_mg_launches(ctx))


def dh_mg_cycle(ctx, phi_ptr: int, F_ptr: int) -> None:
    _check(load().dh_mg_cycle(ctx, ctypes.c_void_p(phi_ptr), ctypes.c_void_p(F_ptr)))


def dh_mg_solve(ctx, F_ptr: int, phi_ptr: int, ncycles: int, want_residual: bool = True):
    r = ctypes.c_double(0.0)
    _check(load().dh_mg_solve(ctx, ctypes.c_void_p(F_ptr), ctypes.c_void_p(phi_ptr), int(ncycles), ctypes.byref(r) if want_residual else None))
    return r.value if want_residual else None


def dh_mg_solve_vjp(ctx, g_phi_ptr: int, g_F_ptr: int, ncycles: int, want_residual: bool = True):
    r = ctypes.c_double(0.0)
    _check(load().dh_mg_solve_vjp(ctx, ctypes.c_void_p(g_phi_ptr), ctypes.c_void_p(g_F_ptr), int(ncycles), ctypes.byref(r) if want_residual else None))
    return r.value if want_residual else None


class Multigrid:
    """Thin owner of a dh_mg context for [nz, ny, nx] torch CUDA tensors (argument marshalling only)."""

    def __init__(self, nx: int, ny: int, nz: int, h: float, dtype=None, stream=None, **options):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("dh.Multigrid needs a CUDA device: the path has no CPU fallback")
        dtype = dtype or torch.float32
        self.shape, self.dtype, self.h = (nz, ny, nx), dtype, float(h)
        self.ctx = dh_mg_create(nx, ny, nz, h, DH_F32 if dtype == torch.float32 else DH_F64)
        stream = stream if stream is not None else torch.cuda.current_stream()
        dh_mg_set_stream(self.ctx, stream.cuda_stream)
        self.set_options(**options)

    def set_options(self, **options):
        for k, v in options.items():
            if k == "cycle":
                k, v = "gamma", MG_CYCLES[v]
            dh_mg_set_option(self.ctx, MG_OPTIONS[k], float(v))

    def _chk(self, *ts):
        for t in ts:
            if not (t.is_cuda and t.is_contiguous() and t.dtype == self.dtype and tuple(t.shape) == self.shape):
                raise ValueError(f"expected a contiguous CUDA {self.dtype} tensor of shape {self.shape}")

    @property
    def levels(self) -> int:
        return dh_mg_levels(self.ctx)

    @property
    def launches(self) -> int:
        return dh_mg_launches(self.ctx)

    def cycle(self, phi, F) -> None:
        self._chk(phi, F)
        dh_mg_cycle(self.ctx, phi.data_ptr(), F.data_ptr())

    def solve(self, F, ncycles: int = 10, want_residual: bool = True):
        import torch

        self._chk(F)
        phi = torch.empty_like(F)
        rel = dh_mg_solve(self.ctx, F.data_ptr(), phi.data_ptr(), ncycles, want_residual)
        return phi, rel

    def solve_vjp(self, g_phi, ncycles: int = 10, want_residual: bool = True):
        import torch

        self._chk(g_phi)
        g_F = torch.empty_like(g_phi)
        rel = dh_mg_solve_vjp(self.ctx, g_phi.data_ptr(), g_F.data_ptr(), ncycles, want_residual)
        return g_F, rel

    def close(self):
        if getattr(self, "ctx", None):
            dh_mg_destroy(self.ctx)
            self.ctx = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

