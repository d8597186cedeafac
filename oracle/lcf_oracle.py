"""ctypes binding of the float64 CPU oracle (oracle/lcf_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Argument marshalling only; all arithmetic is in the C file,
which cites the PAPER.md passage each function follows.  Shares nothing with the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "lcf_oracle.c"
_LIB = _HERE / "liblcf_oracle.so"
_lib = None

HARD_FIXED, HARD_ENERGY, SOFT_FIXED, SOFT_ENERGY, HARD_MEDIAN, SOFT_MEDIAN, HARD_CURVATURE, SOFT_CURVATURE, SOFT_ADAPTIVE, HARD_SLOPE, SOFT_SLOPE, HARD_SLOPE_DB, SOFT_SLOPE_DB, HARD_NCC, SOFT_NCC, HARD_FIXED_TOP, HARD_ENERGY_TOP = range(17)


def build(force: bool = False) -> Path:
    """gcc -O2 -fopenmp the oracle into oracle/liblcf_oracle.so (rebuilt when the source is newer)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        dp, fp, ip = C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int)
        L.lcf_oracle_num_threads.restype = C.c_int
        L.lcf_oracle_axis_windows.argtypes = [C.c_int, C.c_int, C.c_double, C.c_double, dp]
        L.lcf_oracle_axis_windows.restype = None
        L.lcf_oracle_gram.argtypes = [fp, C.c_int, C.c_int, C.c_int, dp, dp, dp]
        L.lcf_oracle_gram.restype = None
        L.lcf_oracle_jacobi.argtypes = [dp, C.c_int, dp, dp]
        L.lcf_oracle_jacobi.restype = C.c_int
        L.lcf_oracle_cutoff_energy.argtypes = [dp, C.c_int, C.c_double]
        L.lcf_oracle_cutoff_energy.restype = C.c_int
        L.lcf_oracle_cutoff_median.argtypes = [dp, C.c_int, C.c_double]
        L.lcf_oracle_cutoff_median.restype = C.c_int
        L.lcf_oracle_cutoff_curvature.argtypes = [dp, C.c_int, C.c_double]
        L.lcf_oracle_cutoff_curvature.restype = C.c_int
        L.lcf_oracle_cutoff_slope.argtypes = [dp, C.c_int, C.c_double]
        L.lcf_oracle_cutoff_slope.restype = C.c_int
        L.lcf_oracle_cutoff_slope_db.argtypes = [dp, C.c_int, C.c_double]
        L.lcf_oracle_cutoff_slope_db.restype = C.c_int
        L.lcf_oracle_left_singular_mag.argtypes = [fp, C.c_int, C.c_int, C.c_int, dp, dp, dp, dp, dp]
        L.lcf_oracle_left_singular_mag.restype = None
        L.lcf_oracle_cutoff_ncc.argtypes = [dp, C.c_size_t, C.c_int, C.c_int, dp]
        L.lcf_oracle_cutoff_ncc.restype = C.c_int
        L.lcf_oracle_weights.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, dp]
        L.lcf_oracle_weights.restype = None
        L.lcf_oracle_weights_adaptive.argtypes = [dp, C.c_int, C.c_double, dp]
        L.lcf_oracle_weights_adaptive.restype = None
        L.lcf_oracle_filter.argtypes = [dp, dp, C.c_int, dp]
        L.lcf_oracle_filter.restype = None
        L.lcf_oracle_project_pd.argtypes = [fp, C.c_int, C.c_int, C.c_int, dp, dp, dp, dp]
        L.lcf_oracle_project_pd.restype = None
        L.lcf_oracle_window.argtypes = [fp, C.c_int, C.c_int, C.c_int, dp, dp, C.c_int, C.c_int,
                                        C.c_double, C.c_double, C.c_double, dp, dp, dp, ip, dp, dp, dp, dp]
        L.lcf_oracle_window.restype = C.c_int
        L.lcf_oracle_combine.argtypes = [dp, C.c_int, C.c_size_t, dp, dp]
        L.lcf_oracle_combine.restype = None
        L.lcf_oracle_run.argtypes = [fp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double,
                                     C.c_double, C.c_double, C.c_int, C.c_int, C.c_double, C.c_double,
                                     C.c_double, dp, dp, ip, dp, dp, dp, dp]
        L.lcf_oracle_run.restype = C.c_int
        _lib = L
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _f(a):
    return a.ctypes.data_as(C.POINTER(C.c_float))


def _iq(iq: np.ndarray):
    """complex64 [N][Nx][Nz] -> (contiguous array kept alive, float*, N, Nx, Nz)."""
    a = np.ascontiguousarray(iq, dtype=np.complex64)
    assert a.ndim == 3
    N, Nx, Nz = a.shape
    return a, a.ctypes.data_as(C.POINTER(C.c_float)), N, Nx, Nz


def _c2d(z: np.ndarray) -> np.ndarray:
    """complex128 array -> contiguous interleaved float64 view holder."""
    return np.ascontiguousarray(z, dtype=np.complex128)


def num_threads() -> int:
    return int(_load().lcf_oracle_num_threads())


def axis_windows(n: int, K: int, sigma: float, trunc: float) -> np.ndarray:
    g = np.empty((K, n), dtype=np.float64)
    _load().lcf_oracle_axis_windows(n, K, float(sigma), float(trunc), _d(g))
    return g


def gram(iq: np.ndarray, gz: np.ndarray, gx: np.ndarray) -> np.ndarray:
    a, p, N, Nx, Nz = _iq(iq)
    gz = np.ascontiguousarray(gz, dtype=np.float64); gx = np.ascontiguousarray(gx, dtype=np.float64)
    assert gz.shape == (Nz,) and gx.shape == (Nx,)
    R = np.empty((N, N), dtype=np.complex128)
    _load().lcf_oracle_gram(p, N, Nx, Nz, _d(gz), _d(gx), _d(R))
    return R


def jacobi(R: np.ndarray):
    """-> (lam [N] descending, V [N][N] columns = eigenvectors, sweeps)."""
    R = _c2d(R)
    N = R.shape[0]
    lam = np.empty(N, dtype=np.float64)
    V = np.empty((N, N), dtype=np.complex128)
    sweeps = _load().lcf_oracle_jacobi(_d(R), N, _d(lam), _d(V))
    if sweeps < 0:
        raise RuntimeError("oracle Jacobi did not converge in 60 sweeps")
    return lam, V, sweeps


def cutoff_energy(lam: np.ndarray, frac: float) -> int:
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    return int(_load().lcf_oracle_cutoff_energy(_d(lam), lam.shape[0], float(frac)))


def cutoff_median(lam: np.ndarray, scale: float) -> int:
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    return int(_load().lcf_oracle_cutoff_median(_d(lam), lam.size, float(scale)))


def cutoff_slope(lam: np.ndarray, thresh: float) -> int:
    """Method 2 as printed: components before the curve lambda_n / lambda_1 first drops by less than thresh."""
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    return int(_load().lcf_oracle_cutoff_slope(_d(lam), lam.size, float(thresh)))


def cutoff_slope_db(lam: np.ndarray, thresh_db: float) -> int:
    """Named variant of method 2: the same rule on the curve in dB."""
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    return int(_load().lcf_oracle_cutoff_slope_db(_d(lam), lam.size, float(thresh_db)))


def left_singular_mag(iq: np.ndarray, gz: np.ndarray, gx: np.ndarray, lam: np.ndarray, V: np.ndarray) -> np.ndarray:
    """|u_i(p)| of the windowed data's left singular vectors: [Nx][Nz][N]."""
    a, p, N, Nx, Nz = _iq(iq)
    gz = np.ascontiguousarray(gz, dtype=np.float64); gx = np.ascontiguousarray(gx, dtype=np.float64)
    lam = np.ascontiguousarray(lam, dtype=np.float64); V = _c2d(V)
    U = np.empty((Nx, Nz, N), dtype=np.float64)
    _load().lcf_oracle_left_singular_mag(p, N, Nx, Nz, _d(gz), _d(gx), _d(lam), _d(V), _d(U))
    return U


def cutoff_ncc(Umag: np.ndarray, fn: int = 5):
    """Method 4 (Eq. 8): (k, ncc curve [N]) from |u_i(p)| given as [..., N] (any leading pixel shape)."""
    U = np.ascontiguousarray(Umag, dtype=np.float64)
    N = U.shape[-1]
    P = U.size // N
    ncc = np.empty(N, dtype=np.float64)
    k = int(_load().lcf_oracle_cutoff_ncc(_d(U), P, N, int(fn), _d(ncc)))
    return k, ncc


def cutoff_curvature(lam: np.ndarray, scale: float) -> int:
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    return int(_load().lcf_oracle_cutoff_curvature(_d(lam), lam.size, float(scale)))


def weights(N: int, soft: bool, c: int, beta: float) -> np.ndarray:
    wt = np.empty(N, dtype=np.float64)
    _load().lcf_oracle_weights(N, int(bool(soft)), int(c), float(beta), _d(wt))
    return wt


def weights_adaptive(lam: np.ndarray, beta: float) -> np.ndarray:
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    wt = np.empty(lam.size)
    _load().lcf_oracle_weights_adaptive(_d(lam), lam.size, float(beta), _d(wt))
    return wt


def filter_matrix(V: np.ndarray, wt: np.ndarray) -> np.ndarray:
    V = _c2d(V); wt = np.ascontiguousarray(wt, dtype=np.float64)
    N = V.shape[0]
    F = np.empty((N, N), dtype=np.complex128)
    _load().lcf_oracle_filter(_d(V), _d(wt), N, _d(F))
    return F


def project_pd(iq: np.ndarray, gz: np.ndarray, gx: np.ndarray, F: np.ndarray) -> np.ndarray:
    a, p, N, Nx, Nz = _iq(iq)
    gz = np.ascontiguousarray(gz, dtype=np.float64); gx = np.ascontiguousarray(gx, dtype=np.float64)
    F = _c2d(F)
    PDk = np.empty((Nx, Nz), dtype=np.float64)
    _load().lcf_oracle_project_pd(p, N, Nx, Nz, _d(gz), _d(gx), _d(F), _d(PDk))
    return PDk


def window(iq: np.ndarray, gz: np.ndarray, gx: np.ndarray, mode: int, k_fixed: int = 0,
           frac: float = 0.995, beta: float = 0.5, cut_scale: float = 1.0) -> dict:
    """One window end to end with every intermediate."""
    a, p, N, Nx, Nz = _iq(iq)
    gz = np.ascontiguousarray(gz, dtype=np.float64); gx = np.ascontiguousarray(gx, dtype=np.float64)
    R = np.empty((N, N), dtype=np.complex128); V = np.empty((N, N), dtype=np.complex128)
    F = np.empty((N, N), dtype=np.complex128)
    lam = np.empty(N); wt = np.empty(N); PDk = np.empty((Nx, Nz)); mean = C.c_double(0.0); c = C.c_int(0)
    sweeps = _load().lcf_oracle_window(p, N, Nx, Nz, _d(gz), _d(gx), int(mode), int(k_fixed), float(frac),
                                       float(beta), float(cut_scale), _d(R), _d(lam), _d(V), C.byref(c), _d(wt), _d(F),
                                       _d(PDk), C.byref(mean))
    if sweeps < 0:
        raise RuntimeError("oracle Jacobi did not converge")
    return dict(R=R, lam=lam, V=V, c=int(c.value), wt=wt, F=F, PDk=PDk, mean=float(mean.value), sweeps=sweeps)


def combine(PDk_all: np.ndarray):
    """[K][Nx][Nz] -> (PD [Nx][Nz], alpha [K])."""
    a = np.ascontiguousarray(PDk_all, dtype=np.float64)
    K = a.shape[0]
    P = int(np.prod(a.shape[1:]))
    alpha = np.empty(K); PD = np.empty(a.shape[1:], dtype=np.float64)
    _load().lcf_oracle_combine(_d(a), K, P, _d(alpha), _d(PD))
    return PD, alpha


def run(iq: np.ndarray, Kz: int, Kx: int, sigma_z: float, sigma_x: float, trunc: float, mode: int,
        k_fixed: int = 0, frac: float = 0.995, beta: float = 0.5, want_R: bool = False,
        want_F: bool = False, cut_scale: float = 1.0, want_V: bool = False) -> dict:
    """Whole path for one ensemble (OpenMP over windows)."""
    a, p, N, Nx, Nz = _iq(iq)
    K = Kz * Kx
    PD = np.empty((Nx, Nz)); lam = np.empty((K, N)); c = np.empty(K, dtype=np.int32); mean = np.empty(K)
    R = np.empty((K, N, N), dtype=np.complex128) if want_R else None
    F = np.empty((K, N, N), dtype=np.complex128) if want_F else None
    V = np.empty((K, N, N), dtype=np.complex128) if want_V else None
    rc = _load().lcf_oracle_run(p, N, Nx, Nz, Kz, Kx, float(sigma_z), float(sigma_x), float(trunc), int(mode),
                                int(k_fixed), float(frac), float(beta), float(cut_scale), _d(PD), _d(lam),
                                c.ctypes.data_as(C.POINTER(C.c_int)), _d(mean),
                                _d(R) if want_R else None, _d(F) if want_F else None, _d(V) if want_V else None)
    if rc != 0:
        raise RuntimeError(f"oracle Jacobi did not converge for window {-rc - 1}")
    return dict(PD=PD, lam=lam, c=c, mean=mean, R=R, F=F, V=V)


def run_config(iq: np.ndarray, filt, **kw) -> dict:
    """run() with a synth.FilterSpec-like object (fields Kz, Kx, sigma_z, sigma_x, trunc, mode, ...)."""
    return run(iq, filt.Kz, filt.Kx, filt.sigma_z, filt.sigma_x, filt.trunc, filt.mode, filt.k_fixed,
               filt.energy_frac, filt.beta, cut_scale=getattr(filt, "cut_scale", 1.0), **kw)
