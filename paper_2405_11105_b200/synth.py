"""Seeded synthetic IQ generator ("LCF synthetic IQ v1") and the five BASELINE.json configs.

This module serves BOTH the float64 oracle (tests only) and the CUDA path. It holds none of
the method's arithmetic (no windows, covariance, EVD, weights, projection): it only draws
seeded complex64 IQ cubes shaped like the paper's workloads and names the filter parameters
each BASELINE.json config asks for.

The paper's phantom / kidney / liver data ("Experimental Studies") are
private and not in the container; these cubes stand in for them.

Layout of every returned cube: complex64, C-order ``[N][Nx][Nz]`` (frame, lateral x, axial z;
z fastest) -- MATLAB's ``Ny x Nx x Nt`` column-major cube of PAPER.md:35, Casorati row
p = z + Nz*x.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

# threshold modes (values match include/lcf.h lcf_thresh_mode)
HARD_FIXED, HARD_ENERGY, SOFT_FIXED, SOFT_ENERGY, HARD_MEDIAN, SOFT_MEDIAN, HARD_CURVATURE, SOFT_CURVATURE, SOFT_ADAPTIVE, HARD_SLOPE, SOFT_SLOPE, HARD_SLOPE_DB, SOFT_SLOPE_DB, HARD_NCC, SOFT_NCC, HARD_FIXED_TOP, HARD_ENERGY_TOP = range(17)


@dataclass(frozen=True)
class DataSpec:
    Nz: int
    Nx: int
    N: int                      # frames per ensemble
    n_frames: int               # frames generated (== N except for the streaming config)
    seed: int
    tissue_db: float            # tissue power above blood, dB
    noise_db: float             # white noise power re tissue, dB (negative)
    motion: str                 # "const" (A = 0.2 px) | "ramp" (A(x) = x/(Nx-1) px)
    drift_px: float = 0.0       # extra linear axial drift over the whole sequence, px
    vessels: str = "random"     # "tubes" (config 0) | "random"
    n_vessels: int = 8
    rho: float = 0.9            # AR(1) correlation of the blood scatterers


@dataclass(frozen=True)
class FilterSpec:
    Kz: int
    Kx: int
    sigma_z: float              # <= 0 with a 1x1 grid: single all-ones window
    sigma_x: float
    trunc: float                # support |d| <= trunc*sigma per axis; <= 0: no truncation
    mode: int
    k_fixed: int = 0
    energy_frac: float = 0.995
    beta: float = 0.5
    precision: int = 0          # 0 = fp32 Gram+EVD, 1 = fp64 Gram+EVD
    cut_scale: float = 1.0      # beta of Eq. 7 (MEDIAN modes)


@dataclass(frozen=True)
class Config:
    name: str
    data: DataSpec
    filt: FilterSpec
    n_ensembles: int = 1
    stride: int = 0


def baseline_configs() -> list[Config]:
    """The five BASELINE.json configs (index = seed)."""
    return [
        Config("cfg0_tiny_local_3x3",
               DataSpec(64, 64, 32, 32, 0, 40.0, -60.0, "const", vessels="tubes"),
               FilterSpec(3, 3, 16.0, 16.0, 3.0, HARD_FIXED, k_fixed=4, precision=1)),
        Config("cfg1_global_evd",
               DataSpec(256, 256, 64, 64, 1, 50.0, -65.0, "const"),
               FilterSpec(1, 1, 0.0, 0.0, 0.0, HARD_FIXED, k_fixed=6, precision=1)),
        Config("cfg2_local_soft_8x8",
               DataSpec(256, 256, 128, 128, 2, 50.0, -65.0, "ramp"),
               FilterSpec(8, 8, 24.0, 24.0, 3.0, SOFT_ENERGY)),
        Config("cfg3_large_long_16x12",
               DataSpec(512, 384, 200, 200, 3, 60.0, -70.0, "ramp", n_vessels=20),
               FilterSpec(16, 12, 24.0, 24.0, 3.0, HARD_ENERGY)),
        Config("cfg4_streaming_10x10",
               DataSpec(256, 256, 100, 900, 4, 50.0, -65.0, "ramp", drift_px=2.0),
               FilterSpec(10, 10, 20.0, 20.0, 3.0, SOFT_ENERGY),
               n_ensembles=16, stride=50),
    ]


def scaled_config(cfg: Config, **data_overrides) -> Config:
    """Same recipe, different size (used by the parity tests for ragged/odd shapes)."""
    d = replace(cfg.data, **data_overrides)
    if "N" in data_overrides and "n_frames" not in data_overrides and cfg.n_ensembles == 1:
        d = replace(d, n_frames=d.N)
    return replace(cfg, data=d)


def _cn(rng: np.random.Generator, shape) -> np.ndarray:
    """Circular complex Gaussian CN(0, 1)."""
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * np.sqrt(0.5)


def vessel_mask(d: DataSpec, rng: np.random.Generator):
    """Returns (mask [Nx][Nz] int32 vessel id or -1, phase step per vessel)."""
    zz, xx = np.meshgrid(np.arange(d.Nz, dtype=np.float64),
                         np.arange(d.Nx, dtype=np.float64), indexing="xy")  # [Nx][Nz]
    vid = np.full((d.Nx, d.Nz), -1, dtype=np.int32)
    if d.vessels == "tubes":
        # two horizontal tubes of radius 3 px at z = 20 and z = 44 (scaled with Nz for resized variants)
        zc = (20.0 * d.Nz / 64.0, 44.0 * d.Nz / 64.0)
        for i, c in enumerate(zc):
            vid[np.abs(zz - c) <= 3.0] = i
        return vid, np.array([0.8, 0.8])
    phis = []
    for i in range(d.n_vessels):
        cz, cx = rng.uniform(0, d.Nz), rng.uniform(0, d.Nx)
        th = rng.uniform(0.0, np.pi)
        rad = rng.uniform(2.0, 6.0)
        phis.append(rng.uniform(0.3, 1.5))
        # distance from the infinite line through (cz, cx) with direction (cos th, sin th)
        dist = np.abs((zz - cz) * np.sin(th) - (xx - cx) * np.cos(th))
        vid[dist <= rad] = i            # later vessels overwrite earlier ones
    return vid, np.array(phis)


def generate_sequence(d: DataSpec) -> np.ndarray:
    """complex64 [n_frames][Nx][Nz]: tissue (rigidly shifted speckle) + AR(1) blood + white noise."""
    rng = np.random.Generator(np.random.PCG64(d.seed))
    T, Nx, Nz = d.n_frames, d.Nx, d.Nz
    # 1. tissue: unit-variance speckle, axial Fourier shift d(x, t)
    t0 = _cn(rng, (Nx, Nz))
    spec = np.fft.fft(t0, axis=1)                              # along z
    fz = np.fft.fftfreq(Nz)
    if d.motion == "const":
        amp = np.full(Nx, 0.2)
    elif d.motion == "ramp":
        amp = np.arange(Nx, dtype=np.float64) / max(Nx - 1, 1)
    else:
        raise ValueError(d.motion)
    vid, phis = vessel_mask(d, rng)
    inside = vid >= 0
    n_in = int(inside.sum())
    blood_amp = 10.0 ** (-d.tissue_db / 20.0)
    noise_amp = 10.0 ** (d.noise_db / 20.0)
    phase_step = np.exp(1j * phis[vid[inside]]) if n_in else None
    b = _cn(rng, n_in) if n_in else None
    out = np.empty((T, Nx, Nz), dtype=np.complex64)
    innov = np.sqrt(1.0 - d.rho ** 2)
    for t in range(T):
        disp = amp * np.sin(2.0 * np.pi * t / 32.0) + d.drift_px * t / max(T, 1)   # [Nx]
        frame = np.fft.ifft(spec * np.exp(-2j * np.pi * fz[None, :] * disp[:, None]), axis=1)
        if n_in:
            if t > 0:
                b = d.rho * phase_step * b + innov * _cn(rng, n_in)
            frame[inside] += blood_amp * b
        frame += noise_amp * _cn(rng, (Nx, Nz))
        out[t] = frame.astype(np.complex64)
    return out


def ensemble(seq: np.ndarray, cfg: Config, e: int = 0) -> np.ndarray:
    """Ensemble e of a sequence: a contiguous [N][Nx][Nz] view (no copy)."""
    s = e * cfg.stride
    return seq[s:s + cfg.data.N]


def generate(cfg: Config) -> np.ndarray:
    return generate_sequence(cfg.data)


def rank_r_clutter(Nz: int, Nx: int, N: int, r: int, seed: int) -> np.ndarray:
    """Exact rank-r cube S = A B^H (no blood, no noise), complex64 [N][Nx][Nz] (test input)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    A = _cn(rng, (Nx * Nz, r))
    B = _cn(rng, (N, r))
    S = A @ B.conj().T                       # [P][N]
    return np.ascontiguousarray(S.T.reshape(N, Nx, Nz)).astype(np.complex64)


def graded_rank_cube(Nz: int, Nx: int, N: int, r: int, step_db: float, noise_db: float, seed: int) -> np.ndarray:
    """r clutter components whose powers fall by step_db from one to the next, over white noise noise_db below the
    strongest: a spectrum with r well separated leading eigenvalues and a flat floor (test input for the cut-off
    rules that work on the leading eigenpairs).  complex64 [N][Nx][Nz]."""
    rng = np.random.Generator(np.random.PCG64(seed))
    A = _cn(rng, (Nx * Nz, r))
    B, _ = np.linalg.qr(_cn(rng, (N, r)))
    amp = 10.0 ** (-step_db * np.arange(r) / 20.0)
    S = (A * amp) @ B.conj().T + 10.0 ** (noise_db / 20.0) * _cn(rng, (Nx * Nz, N))
    return np.ascontiguousarray(S.T.reshape(N, Nx, Nz)).astype(np.complex64)


def random_cube(Nz: int, Nx: int, N: int, seed: int) -> np.ndarray:
    rng = np.random.Generator(np.random.PCG64(seed))
    return _cn(rng, (N, Nx, Nz)).astype(np.complex64)
