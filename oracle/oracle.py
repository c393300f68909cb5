"""ORACLE — test infrastructure only.

ctypes wrapper around ``oracle/dh_oracle.{hpp,cpp}``: the plain CPU implementation of the hot path
of arxiv/paper_2512_13403 (one periodic 3D Euler finite-volume step, its CFL dt, cooling and VJP),
written from PAPER.md (citations in the C++ header).  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this module; the product
path (``paper_2512_13403_b200``) never does, and this module never imports the product.

All state arrays are numpy ``[5, nz, ny, nx]`` (rho, rho*vx, rho*vy, rho*vz, E); x is fastest.
State arithmetic is fp64; the dt recipe runs in the dtype of the array handed in (fp32 or fp64).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "dh_oracle.cpp"), os.path.join(_HERE, "dh_oracle.hpp")]
_LIB = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

LIMITERS = {"minmod": 0, "vanleer": 1, "mc": 2, "constant": 3}
RIEMANN = {"hllc": 0, "hll": 1, "rusanov": 2}
INTEGRATORS = {"vl2": 0, "heun": 1, "ssprk3": 2}
COOL_MODES = {"euler": 0, "trapezoid": 1, "masked": 2}
COOL_LAWS = {"powerlaw": 0, "twobranch": 1}


class _Params(ctypes.Structure):
    _fields_ = [
        ("gamma", ctypes.c_double),
        ("dx", ctypes.c_double * 3),
        ("rho_floor", ctypes.c_double),
        ("p_floor", ctypes.c_double),
        ("limiter", ctypes.c_int),
        ("riemann", ctypes.c_int),
        ("integrator", ctypes.c_int),
        ("cooling", ctypes.c_int),
        ("lambda0", ctypes.c_double),
        ("alpha", ctypes.c_double),
        ("t_floor", ctypes.c_double),
        ("cool_mode", ctypes.c_int),
        ("cool_nsub", ctypes.c_int),
        ("cool_law", ctypes.c_int),
        ("t_switch", ctypes.c_double),
        ("lambda1", ctypes.c_double),
        ("alpha1", ctypes.c_double),
        ("lambda2", ctypes.c_double),
        ("alpha2", ctypes.c_double),
        ("gamma0", ctypes.c_double),
        ("tab", ctypes.POINTER(ctypes.c_double)),
        ("ntab", ctypes.c_int),
        ("tab_logT0", ctypes.c_double),
        ("tab_dlogT", ctypes.c_double),
        ("f_sub", ctypes.c_double),
    ]


def build(force: bool = False) -> str:
    """Compile liboracle.so with g++ (``-ffp-contract=off`` so the dt recipe has no FMA)."""
    with _lock:
        stale = force or not os.path.exists(_LIB) or any(
            os.path.getmtime(s) > os.path.getmtime(_LIB) for s in _SRC
        )
        if stale:
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-ffp-contract=off", "-shared", "-fPIC",
                   _SRC[0], "-o", tmp]
            subprocess.run(cmd, check=True, cwd=_HERE)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        lib.dho_num_threads.restype = ctypes.c_int
        lib.dho_limiter.restype = ctypes.c_double
        lib.dho_limiter.argtypes = [ctypes.c_double, ctypes.c_double, ctypes.c_int]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().dho_num_threads())


def set_num_threads(n: int) -> None:
    _load().dho_set_num_threads(ctypes.c_int(int(n)))


def params(gamma=5.0 / 3.0, dx=None, shape=None, rho_floor=1e-10, p_floor=1e-10, limiter="minmod",
           riemann="hllc", integrator="vl2", cooling=False, lambda0=1e-3, alpha=0.5, t_floor=0.01,
           cool_mode="euler", cool_nsub=1, cool_law="powerlaw", t_switch=1.0, lambda1=0.0, alpha1=1.0, lambda2=0.0, alpha2=0.5,
           gamma0=0.0, table=None, f_sub=0.1):
    """Scheme parameters.  ``dx`` defaults to the unit box, dx_a = 1/n_a (reading A13)."""
    p = _Params()
    p.gamma = float(gamma)
    if dx is None:
        if shape is None:
            raise ValueError("give dx=(dx,dy,dz) or shape=(nz,ny,nx)")
        nz, ny, nx = shape[-3:]
        dx = (1.0 / nx, 1.0 / ny, 1.0 / nz)
    p.dx[0], p.dx[1], p.dx[2] = (float(d) for d in dx)
    p.rho_floor, p.p_floor = float(rho_floor), float(p_floor)
    p.limiter, p.riemann, p.integrator = LIMITERS[limiter], RIEMANN[riemann], INTEGRATORS[integrator]
    p.cooling = int(bool(cooling))
    p.lambda0, p.alpha, p.t_floor = float(lambda0), float(alpha), float(t_floor)
    # Eq. 23 sub-cycled ("euler", N_sub = cool_nsub) or the trapezoid of Eq. 22 (reading A20)
    p.cool_mode, p.cool_nsub = COOL_MODES[cool_mode], int(cool_nsub)
    if p.cool_nsub < 1:
        raise ValueError("cool_nsub must be >= 1")
    # Eqs. 17-19: Koyama-Inutsuka fit + uniform heating below t_switch, tabulated Lambda_CIE above it
    # (reading A25); table = (log10_T0, dlog10_T, [log10 Lambda at the nodes]); cool_mode "masked": reading A26
    p.cool_law = COOL_LAWS[cool_law]
    p.t_switch, p.lambda1, p.alpha1, p.lambda2, p.alpha2, p.gamma0 = (float(v) for v in (t_switch, lambda1, alpha1, lambda2, alpha2, gamma0))
    p.f_sub = float(f_sub)
    p.ntab = 0
    if table is not None:
        logT0, dlogT, vals = table
        arr = np.ascontiguousarray(vals, dtype=np.float64)
        p._table_keepalive = arr                      # the struct only holds a pointer
        p.tab = arr.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
        p.ntab, p.tab_logT0, p.tab_dlogT = int(arr.size), float(logT0), float(dlogT)
    if p.cool_law == 1 and p.ntab < 2:
        raise ValueError("cool_law='twobranch' needs a table with at least two nodes")
    return p


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _dims(U):
    assert U.ndim == 4 and U.shape[0] == 5, "state must be [5, nz, ny, nx]"
    _, nz, ny, nx = U.shape
    return ctypes.c_int(nx), ctypes.c_int(ny), ctypes.c_int(nz)


def cfl_dt(U, p, cfl=0.4):
    """Eq. A8 in the array's own dtype.  Returns (dt, smax[3]); raises on NaN/Inf."""
    lib = _load()
    U = np.ascontiguousarray(U)
    assert U.dtype in (np.float32, np.float64)
    dt = ctypes.c_double(0.0)
    smax = (ctypes.c_double * 3)()
    rc = lib.dho_cfl_dt(*_dims(U), ctypes.byref(p), ctypes.c_double(cfl),
                        ctypes.c_int(0 if U.dtype == np.float32 else 1), _ptr(U), ctypes.byref(dt), smax)
    if rc != 0:
        raise FloatingPointError("non-finite wave speed")
    return dt.value, np.array(list(smax))


def cool_dt(U, p, dt_hydro, c_cool=0.0, dt_max=0.0):
    """Eqs. 20-21: (min_x t_cool(x), min(dt_hydro, c_cool * that, dt_max)); t_cool in double,
    the three candidates compared in the array's dtype (reading A24); c_cool <= 0 / dt_max <= 0 switch a candidate off."""
    lib = _load()
    U = np.ascontiguousarray(U)
    assert U.dtype in (np.float32, np.float64)
    tmin = ctypes.c_double(0.0)
    dt = ctypes.c_double(0.0)
    lib.dho_cool_dt(*_dims(U), ctypes.byref(p), ctypes.c_int(0 if U.dtype == np.float32 else 1), _ptr(U),
                    ctypes.c_double(dt_hydro), ctypes.c_double(c_cool), ctypes.c_double(dt_max),
                    ctypes.byref(tmin), ctypes.byref(dt))
    return tmin.value, dt.value


def prims(U, p):
    lib = _load()
    U = _f64(U)
    W = np.empty_like(U)
    lib.dho_prims(*_dims(U), ctypes.byref(p), _ptr(U), _ptr(W))
    return W


def flux_divergence(U, p):
    """D(U) of Eq. A4."""
    lib = _load()
    U = _f64(U)
    D = np.empty_like(U)
    lib.dho_flux_divergence(*_dims(U), ctypes.byref(p), _ptr(U), _ptr(D))
    return D


def step(U, dt, p):
    """U^n -> U^{n+1}: two stages (+ cooling if p.cooling)."""
    lib = _load()
    U = _f64(U)
    out = np.empty_like(U)
    lib.dho_step(*_dims(U), ctypes.byref(p), _ptr(U), ctypes.c_double(dt), _ptr(out))
    return out


def step_jvp(U, V, dt, p):
    """(U^{n+1}, J V) by dual numbers through the same step code."""
    lib = _load()
    U, V = _f64(U), _f64(V)
    out, dout = np.empty_like(U), np.empty_like(U)
    lib.dho_step_jvp(*_dims(U), ctypes.byref(p), _ptr(U), _ptr(V), ctypes.c_double(dt), _ptr(out), _ptr(dout))
    return out, dout


def step_vjp(U, dt, g_out, p):
    """g_in = (dU^{n+1}/dU^n)^T g_out, dt held constant."""
    lib = _load()
    U, g_out = _f64(U), _f64(g_out)
    gin = np.empty_like(U)
    lib.dho_step_vjp(*_dims(U), ctypes.byref(p), _ptr(U), ctypes.c_double(dt), _ptr(g_out), _ptr(gin))
    return gin


def stage_vjp(U, tau, gV, p):
    """-tau J_D(U)^T gV for one stage V = B - tau D(U)."""
    lib = _load()
    U, gV = _f64(U), _f64(gV)
    gU = np.empty_like(U)
    lib.dho_stage_vjp(*_dims(U), ctypes.byref(p), _ptr(U), ctypes.c_double(tau), _ptr(gV), _ptr(gU))
    return gU


def cooling(U, dt, p):
    lib = _load()
    U = _f64(U)
    flat = np.ascontiguousarray(U.reshape(5, -1))
    out = np.empty_like(flat)
    lib.dho_cooling(ctypes.c_longlong(flat.shape[1]), ctypes.byref(p), ctypes.c_double(dt), _ptr(flat), _ptr(out))
    return out.reshape(U.shape)


def riemann(WL, WR, axis, p):
    """Batch of Riemann fluxes; WL, WR are [5, n] primitive (rho, vx, vy, vz, P)."""
    lib = _load()
    WL, WR = _f64(WL).reshape(5, -1), _f64(WR).reshape(5, -1)
    F = np.empty_like(WL)
    lib.dho_riemann(ctypes.c_longlong(WL.shape[1]), ctypes.byref(p), ctypes.c_int(axis), _ptr(WL), _ptr(WR), _ptr(F))
    return F


def reconstruct(W, p):
    """Face states along one periodic line; W is [5, n].  Returns (WL, WR) at faces i+1/2."""
    lib = _load()
    W = _f64(W)
    WL, WR = np.empty_like(W), np.empty_like(W)
    lib.dho_reconstruct(ctypes.c_int(W.shape[1]), ctypes.byref(p), _ptr(W), _ptr(WL), _ptr(WR))
    return WL, WR


def limiter(a, b, kind="minmod"):
    return float(_load().dho_limiter(float(a), float(b), LIMITERS[kind]))


def decision_margins(U, p):
    """[4, nz, ny, nx]: distance from the tie of every compare one evaluation of D(U) makes, relative to the rounding scale
    of its operands: slots 0-2 = limiter calls at the cell + Riemann compares at the face i+1/2 along x / y / z, slot 3 =
    the floors of prim().  Test infrastructure for the VJP parity check (dh_oracle.hpp, "Decision margins")."""
    lib = _load()
    U = _f64(U)
    M = np.empty((4,) + U.shape[1:], dtype=np.float64)
    lib.dho_decision_margins(*_dims(U), ctypes.byref(p), _ptr(U), _ptr(M))
    return M


def limiter_conditioning(U, p):
    """[3, nz, ny, nx]: s / (|a| + |b|) of the active slopes at every cell and axis (van Leer: the relative sensitivity of the
    limiter's derivative to rounding of the differences; zero for minmod / MC).  dh_oracle.hpp, "Conditioning of the limiter"."""
    lib = _load()
    U = _f64(U)
    C = np.empty((3,) + U.shape[1:], dtype=np.float64)
    lib.dho_limiter_conditioning(*_dims(U), ctypes.byref(p), _ptr(U), _ptr(C))
    return C


def cooling_margins(U1, dt, p):
    """[nz, ny, nx]: margins of the compares of the cooling update applied to the pre-cooling state U1."""
    lib = _load()
    U1 = _f64(U1)
    M = np.empty(U1.shape[1:], dtype=np.float64)
    lib.dho_cooling_margins(*_dims(U1), ctypes.byref(p), ctypes.c_double(dt), _ptr(U1), _ptr(M))
    return M


def cool_rate(Eth, rho, p):
    """Edot = n_H Gamma - n_H^2 Lambda of the law selected in p at thermal energy Eth and density rho."""
    lib = _load()
    lib.dho_cool_rate.restype = ctypes.c_double
    return float(lib.dho_cool_rate(ctypes.byref(p), ctypes.c_double(Eth), ctypes.c_double(rho)))


def lambda_table(T, p):
    """Lambda_CIE(T) of Eq. 19: log-log interpolation of p's table."""
    lib = _load()
    lib.dho_lambda_table.restype = ctypes.c_double
    return float(lib.dho_lambda_table(ctypes.byref(p), ctypes.c_double(T)))


def step_nocool(U, dt, p):
    """The pre-cooling state of a step: the hydro stages of step() without the cooling update."""
    lib = _load()
    U = _f64(U)
    out = np.empty_like(U)
    lib.dho_step_nocool(*_dims(U), ctypes.byref(p), _ptr(U), ctypes.c_double(dt), _ptr(out))
    return out


def cooling_table_vjp(U1, dt, g_out, p):
    """d sum(g_out_E * E_out) / d table nodes at the pre-cooling state U1, by dual numbers (ntab <= 32)."""
    lib = _load()
    U1, g_out = _f64(U1), _f64(g_out)
    gt = np.zeros(p.ntab, dtype=np.float64)
    rc = lib.dho_cooling_table_vjp(*_dims(U1), ctypes.byref(p), ctypes.c_double(dt), _ptr(U1), _ptr(g_out), _ptr(gt))
    if rc != 0:
        raise ValueError("cooling_table_vjp needs cool_law='twobranch' and a table of at most 32 nodes")
    return gt


def window_step(U_full, dt, p, lo, size, halo=4):
    """Windowed oracle: one step has a finite domain of dependence (+-4 cells per
    axis), so stepping a periodic-wrapped window of `size`+2*halo cells is exact on its interior.
    `lo`, `size` are (k, j, i) triples into the full periodic grid.  Returns [5, *size]."""
    idx = [np.arange(lo[a] - halo, lo[a] + size[a] + halo) % U_full.shape[1 + a] for a in range(3)]
    win = np.asarray(U_full)[:, idx[0][:, None, None], idx[1][None, :, None], idx[2][None, None, :]]
    out = step(win, dt, p)
    return out[:, halo:-halo, halo:-halo, halo:-halo]


def window_step_vjp(U_full, dt, g_full, p, lo, size, halo=8):
    """Windowed VJP: cotangent reach +-4, primal reach +-7 per axis for the two-stage step."""
    idx = [np.arange(lo[a] - halo, lo[a] + size[a] + halo) % U_full.shape[1 + a] for a in range(3)]
    sel = (slice(None), idx[0][:, None, None], idx[1][None, :, None], idx[2][None, None, :])
    out = step_vjp(np.asarray(U_full)[sel], dt, np.asarray(g_full)[sel], p)
    return out[:, halo:-halo, halo:-halo, halo:-halo]


def adjoint(U0, nsteps, g_final, p, cfl=0.4):
    """Adjoint of `nsteps` steps: the plain composition, no checkpoints.  Forward: dt_k from Eq. A8
    (in the array's own dtype, like cfl_dt) then one step, all states kept; reverse: step_vjp applied backwards with
    every dt_k held constant.  Returns (U_n, dL/dU_0, [dt_k])."""
    states, dts = [np.array(U0, copy=True)], []
    for _ in range(nsteps):
        dt, _ = cfl_dt(states[-1], p, cfl)
        dts.append(dt)
        states.append(step(states[-1], dt, p).astype(states[-1].dtype))
    g = np.asarray(g_final, dtype=np.float64)
    for k in range(nsteps - 1, -1, -1):
        g = step_vjp(states[k], dts[k], g, p)
    return states[-1], g, dts
