"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json `configs`).

This module is the ONLY code shared by the CUDA path's harness and the oracle's tests: it builds
initial-condition arrays and nothing else.  It contains none of the scheme's arithmetic (no primitive
conversion of evolving states, reconstruction, Riemann solver, update, CFL or cooling); the one formula
it uses is the paper's own definition of an initial state from (rho, u, p), Eq. 10.
The paper's real inputs (Athena++ ICs, SD93 table, reconstruction targets) are not available; these
fields stand in for them.  The recipe is restated in DESIGN.md.

Gaussian random fields follow PAPER.md:184-221 (Eqs. 3-10): white noise -> FFT -> multiply by
A(k) = |n|^{p/2} on the band k_min <= |n| <= k_max (Eqs. 4-5), k = 0 removed -> optional solenoidal
projection P_ij = delta_ij - k_i k_j / k^2 (Eq. 6) -> inverse FFT -> rescale (Eq. 9).

Everything is torch (CPU or CUDA) so that 512^3 / 1024^3 fields can be generated on the device;
the very same array is what both the oracle and the CUDA path receive.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import torch


@dataclass
class Workload:
    name: str
    U: torch.Tensor                 # [5, nz, ny, nx] conserved (rho, rho*vx, rho*vy, rho*vz, E)
    gamma: float
    steps: int
    cfl: float = 0.4
    cooling: bool = False
    lambda0: float = 1e-3
    alpha: float = 0.5
    t_floor: float = 0.01
    t_end: float | None = None
    extra: dict = field(default_factory=dict)


def _gen(seed: int, device) -> torch.Generator:
    g = torch.Generator(device=device)
    g.manual_seed(int(seed))
    return g


def _mode_numbers(n: int, device, half: bool = False) -> torch.Tensor:
    if half:
        return torch.arange(0, n // 2 + 1, device=device, dtype=torch.float64)
    return torch.fft.fftfreq(n, d=1.0 / n, device=device).to(torch.float64)


def _band_filter(shape, device, work_dtype, p: float, kmin: float, kmax: float):
    """A(k) = |n|^{p/2} inside the band, 0 outside (and at k=0); rfftn layout [nz, ny, nx//2+1]."""
    nz, ny, nx = shape
    kz = _mode_numbers(nz, device)[:, None, None]
    ky = _mode_numbers(ny, device)[None, :, None]
    kx = _mode_numbers(nx, device, half=True)[None, None, :]
    k2 = kz * kz + ky * ky + kx * kx
    kk = torch.sqrt(k2)
    amp = torch.where((kk >= kmin) & (kk <= kmax), kk.clamp_min(1e-30) ** (p / 2.0), torch.zeros_like(kk))
    return amp.to(work_dtype), (kz, ky, kx, k2)


def gaussian_random_field(shape, seed: int, device="cpu", work_dtype=torch.float64, p: float = -2.0,
                          kmin: float = 1.0, kmax: float | None = None, components: int = 1,
                          solenoidal: bool = False) -> torch.Tensor:
    """`components` real fields [c, nz, ny, nx] with spectrum |u_k|^2 ~ k^p on the band
    (PAPER.md:184-199); with `solenoidal` (needs 3 components) they are projected by Eq. 6.
    Returned un-normalised (callers rescale by Eq. 9 or to a target rms)."""
    nz, ny, nx = shape
    if kmax is None:
        kmax = float(min(16, min(shape) // 4))
    amp, (kz, ky, kx, k2) = _band_filter(shape, device, work_dtype, p, kmin, kmax)
    g = _gen(seed, device)
    hats = []
    for _ in range(components):
        w = torch.randn(shape, generator=g, device=device, dtype=work_dtype)
        hats.append(torch.fft.rfftn(w) * amp)
        del w
    if solenoidal:
        assert components == 3
        kvec = (kx.to(work_dtype), ky.to(work_dtype), kz.to(work_dtype))  # component order x, y, z
        inv_k2 = torch.where(k2 > 0, 1.0 / k2.clamp_min(1e-30), torch.zeros_like(k2)).to(work_dtype)
        div = (kvec[0] * hats[0] + kvec[1] * hats[1] + kvec[2] * hats[2]) * inv_k2
        for c in range(3):
            hats[c] = hats[c] - kvec[c] * div
        del div
    out = torch.empty((components,) + tuple(shape), device=device, dtype=work_dtype)
    for c in range(components):
        out[c] = torch.fft.irfftn(hats[c], s=shape)
        hats[c] = None
    return out


def conserved_from_primitive(rho, vel, p, gamma: float, dtype) -> torch.Tensor:
    """Eq. 10: m = rho u, E = p/(gamma-1) + rho|u|^2/2.  Evaluated in the working
    precision, then rounded once to `dtype`."""
    U = torch.empty((5,) + tuple(rho.shape), device=rho.device, dtype=dtype)
    U[0] = rho.to(dtype)
    ke = torch.zeros_like(rho)
    for c in range(3):
        U[1 + c] = (rho * vel[c]).to(dtype)
        ke += vel[c] * vel[c]
    U[4] = (p / (gamma - 1.0) + 0.5 * rho * ke).to(dtype)
    return U


def _cell_centres(n: int, device, dtype=torch.float64):
    return (torch.arange(n, device=device, dtype=dtype) + 0.5) / n


def smooth_waves(n: int = 32, seed: int = 1001, dtype=torch.float64, device="cpu") -> Workload:
    """Config 1: 32^3 fp64, gamma 5/3: rho = 1 + 0.1 sum of 8 seeded Fourier modes, p = 1, each
    velocity component an independent k^-2 Gaussian random field with rms 0.1; 10 steps."""
    gamma = 5.0 / 3.0
    shape = (n, n, n)
    g = _gen(seed, "cpu")
    x = _cell_centres(n, device)
    X, Y, Z = x[None, None, :], x[None, :, None], x[:, None, None]
    rho = torch.ones(shape, device=device, dtype=torch.float64)
    m = 0
    while m < 8:
        nvec = torch.randint(-3, 4, (3,), generator=g)
        a = 0.5 + 0.5 * torch.rand((), generator=g, dtype=torch.float64)
        ph = 2.0 * math.pi * torch.rand((), generator=g, dtype=torch.float64)
        if int(nvec.abs().sum()) == 0:
            continue
        rho = rho + 0.1 * float(a) * torch.cos(2.0 * math.pi * (int(nvec[0]) * X + int(nvec[1]) * Y + int(nvec[2]) * Z) + float(ph))
        m += 1
    vel = []
    for c in range(3):
        v = gaussian_random_field(shape, seed + 10 * (c + 1), device=device)[0]
        vel.append(v * (0.1 / v.pow(2).mean().sqrt()))
    p = torch.ones(shape, device=device, dtype=torch.float64)
    U = conserved_from_primitive(rho, vel, p, gamma, dtype)
    return Workload("smooth_waves_%d" % n, U, gamma, steps=10)


def sedov(n: int = 128, dtype=torch.float32, device="cpu", e_blast: float = 1.0, p_amb: float = 1e-5,
          r_dep_cells: float = 3.0) -> Workload:
    """Config 2: rho = 1, p = 1e-5, v = 0; energy E = 1 deposited as uniform pressure in the cells
    whose centre lies within 3 dx of the box centre; gamma 5/3; run to shock radius ~0.3
    (t_end = (0.3/1.15)^{5/2})."""
    gamma = 5.0 / 3.0
    shape = (n, n, n)
    x = _cell_centres(n, device)
    r2 = (x[None, None, :] - 0.5) ** 2 + (x[None, :, None] - 0.5) ** 2 + (x[:, None, None] - 0.5) ** 2
    inside = r2 < (r_dep_cells / n) ** 2
    ncell = int(inside.sum())
    p_in = (gamma - 1.0) * e_blast / (ncell * (1.0 / n) ** 3)
    rho = torch.ones(shape, device=device, dtype=torch.float64)
    p = torch.where(inside, torch.full_like(rho, p_in), torch.full_like(rho, p_amb))
    vel = [torch.zeros_like(rho) for _ in range(3)]
    U = conserved_from_primitive(rho, vel, p, gamma, dtype)
    t_end = (0.3 / 1.15) ** 2.5
    return Workload("sedov_%d" % n, U, gamma, steps=1000, t_end=t_end,
                    extra={"deposit_cells": ncell, "e_blast": e_blast})


def kelvin_helmholtz(n: int = 256, seed: int = 1003, dtype=torch.float32, device="cpu") -> Workload:
    """Config 3: shear layer rho = 2, vx = +0.5 for |y-0.5| < 0.25 else rho = 1, vx = -0.5; p = 2.5;
    vy = 0.01 * white noise * [exp(-(y-1/4)^2/0.0025) + exp(-(y-3/4)^2/0.0025)]; gamma 1.4; 50 steps
    (3D stand-in for the paper's 2D KH)."""
    gamma = 1.4
    shape = (n, n, n)
    y = _cell_centres(n, device)[None, :, None]
    inner = ((y - 0.5).abs() < 0.25).expand(shape)
    one = torch.ones(shape, device=device, dtype=torch.float64)
    rho = torch.where(inner, 2.0 * one, one)
    vx = torch.where(inner, 0.5 * one, -0.5 * one)
    w = torch.randn(shape, generator=_gen(seed, device), device=device, dtype=torch.float64)
    vy = 0.01 * w * (torch.exp(-((y - 0.25) ** 2) / 0.0025) + torch.exp(-((y - 0.75) ** 2) / 0.0025))
    vz = torch.zeros_like(one)
    U = conserved_from_primitive(rho, [vx, vy, vz], 2.5 * one, gamma, dtype)
    return Workload("kelvin_helmholtz_%d" % n, U, gamma, steps=50)


def turbulence(n: int = 512, seed: int = 1004, mach: float = 1.0, cooling: bool = True, steps: int = 20,
               dtype=torch.float32, device="cpu", work_dtype=None, sigma_ln: float = 0.5) -> Workload:
    """Configs 4 and 5: rho lognormal exp(sigma g - sigma^2/2) with g a unit-variance k^-2 Gaussian
    random field, p = 1, solenoidal k^-2 Gaussian random velocity scaled to rms Mach `mach` by Eq. 9
    (PAPER.md:216); config 4 adds Lambda(T) = n^2 1e-3 T^0.5 cooling with temperature floor 0.01."""
    gamma = 5.0 / 3.0
    shape = (n, n, n)
    if work_dtype is None:
        work_dtype = torch.float64 if n <= 256 else torch.float32
    g = gaussian_random_field(shape, seed, device=device, work_dtype=work_dtype)[0]
    g = g / g.pow(2).mean().sqrt()
    rho = torch.exp(sigma_ln * g - 0.5 * sigma_ln * sigma_ln)
    del g
    vel = gaussian_random_field(shape, seed + 1, device=device, work_dtype=work_dtype, components=3, solenoidal=True)
    p = torch.ones(shape, device=device, dtype=work_dtype)
    cs_mean = torch.sqrt(gamma * p / rho).mean()
    u_rms = (vel[0] ** 2 + vel[1] ** 2 + vel[2] ** 2).mean().sqrt()
    vel = vel * (mach * cs_mean / u_rms)      # Eq. 9
    U = conserved_from_primitive(rho, [vel[0], vel[1], vel[2]], p, gamma, dtype)
    name = "cooling_turbulence_%d" % n if cooling else "turbulence_%d_mach%g" % (n, mach)
    return Workload(name, U, gamma, steps=steps, cooling=cooling)


def cotangent(shape, seed: int = 2005, dtype=torch.float32, device="cpu") -> torch.Tensor:
    """Config 5's seeded white unit-Gaussian cotangent on all five conserved fields."""
    return torch.randn((5,) + tuple(shape[-3:]), generator=_gen(seed, device), device=device, dtype=dtype)


def cooling_table(seed: int = 1719, n: int = 24, log10_t_lo: float = 0.0, log10_t_hi: float = 2.0,
                  lambda_lo: float = 3.0e-2):
    """Synthetic stand-in for the tabulated collisional-ionisation-equilibrium cooling curve of Eq. 19 (the
    paper's SD93 table is not available): n nodes equally spaced in log10 T on [log10_t_lo, log10_t_hi]; log10 Lambda = a linear
    trend plus three seeded Gaussian bumps in log T (the shape of a line-cooling curve: peaks and valleys of about a decade),
    shifted so that the first node equals log10(lambda_lo) (the caller matches it to the low-temperature branch at the switch
    temperature, as the two branches of Eq. 17 meet in the KO15 prescription).  Returns (log10_t_lo, dlog10_T, values[n]) as
    Python floats / a float64 tensor: an INPUT of the cooling law, no arithmetic of the scheme."""
    g = torch.Generator(device="cpu")
    g.manual_seed(int(seed))
    r = torch.rand(10, generator=g, dtype=torch.float64)
    x = torch.linspace(0.0, 1.0, n, dtype=torch.float64)
    y = (r[0] - 0.5) * x
    for j in range(3):
        amp, cen, wid = -0.8 + 1.8 * r[1 + 3 * j], 0.1 + 0.8 * r[2 + 3 * j], 0.08 + 0.17 * r[3 + 3 * j]
        y = y + amp * (torch.exp(-((x - cen) / wid) ** 2) - torch.exp(-((0.0 - cen) / wid) ** 2))
    vals = math.log10(lambda_lo) + y
    return float(log10_t_lo), float((log10_t_hi - log10_t_lo) / (n - 1)), vals


def make_config(cfg: int, n: int | None = None, device="cpu", dtype=None) -> Workload:
    """BASELINE.json `configs[cfg]` (0-based), optionally at a reduced size `n` for tests."""
    if cfg == 0:
        return smooth_waves(n or 32, dtype=dtype or torch.float64, device=device)
    if cfg == 1:
        return sedov(n or 128, dtype=dtype or torch.float32, device=device)
    if cfg == 2:
        return kelvin_helmholtz(n or 256, dtype=dtype or torch.float32, device=device)
    if cfg == 3:
        return turbulence(n or 512, seed=1004, mach=1.0, cooling=True, steps=20, dtype=dtype or torch.float32, device=device)
    if cfg == 4:
        return turbulence(n or 1024, seed=1005, mach=2.0, cooling=False, steps=5, dtype=dtype or torch.float32, device=device)
    raise ValueError("cfg must be 0..4")
