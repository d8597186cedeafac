"""ctypes binding of liblcf.so (include/lcf.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels behind the C ABI.  PyTorch is used by callers for device memory and
streams; this module needs only raw pointers.

There is no CPU fallback: if liblcf.so is missing or does not load, `load()` raises.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

HERE = Path(__file__).resolve().parent
LIB_PATH = HERE / "liblcf.so"

HARD_FIXED, HARD_ENERGY, SOFT_FIXED, SOFT_ENERGY, HARD_MEDIAN, SOFT_MEDIAN, HARD_CURVATURE, SOFT_CURVATURE, SOFT_ADAPTIVE, HARD_SLOPE, SOFT_SLOPE, HARD_SLOPE_DB, SOFT_SLOPE_DB, HARD_NCC, SOFT_NCC, HARD_FIXED_TOP, HARD_ENERGY_TOP = range(17)
OK, ERR_INVALID_ARG, ERR_UNSUPPORTED, ERR_ALLOC, ERR_CUDA, ERR_NOT_CONVERGED = range(6)

EXPORTS = [
    "lcf_plan_create", "lcf_filter", "lcf_filter_batch", "lcf_filter_stream", "lcf_filter_host", "lcf_filter_host_batch", "lcf_plan_destroy", "lcf_num_windows",
    "lcf_get_eigenvalues", "lcf_get_cutoffs", "lcf_get_sweeps", "lcf_get_gram", "lcf_get_eigenvectors",
    "lcf_get_weights", "lcf_get_filters", "lcf_get_window_means", "lcf_set_timing", "lcf_get_stage_ms",
    "lcf_get_work", "lcf_measure_peak", "lcf_status_string", "lcf_last_error", "lcf_scale_exponent",
    "lcf_get_converged", "lcf_set_max_sweeps", "lcf_get_ncc",
]


class Windows(C.Structure):
    _fields_ = [("Kz", C.c_int), ("Kx", C.c_int), ("sigma_z", C.c_float), ("sigma_x", C.c_float),
                ("trunc_sigmas", C.c_float)]


class Thresh(C.Structure):
    _fields_ = [("mode", C.c_int), ("k_fixed", C.c_int), ("energy_frac", C.c_double), ("beta", C.c_double),
                ("precision", C.c_int), ("cut_scale", C.c_double)]


class Work(C.Structure):
    _fields_ = [("gram_flops", C.c_double), ("proj_flops", C.c_double), ("hbm_bytes", C.c_double),
                ("sum_Pk", C.c_double), ("launches", C.c_int), ("gram_tc", C.c_int), ("evd_chol", C.c_int),
                ("proj_tc", C.c_int), ("gram_tensor_flops", C.c_double), ("proj_tensor_flops", C.c_double)]


class LcfError(RuntimeError):
    def __init__(self, status: int, what: str):
        self.status = status
        super().__init__(f"{what}: {status_string(status)} (lcf_status {status})")


_lib = None


def load() -> C.CDLL:
    """dlopen liblcf.so; raises if it has not been built (python -m paper_2405_11105_b200.build)."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2405_11105_b200.build` "
                               "(there is no CPU fallback)")
        L = C.CDLL(str(LIB_PATH))
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.lcf_plan_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.POINTER(Windows), C.POINTER(Thresh)]
        L.lcf_filter.argtypes = [vp, vp, vp, vp]
        L.lcf_filter_host.argtypes = [vp, vp, vp, vp]
        L.lcf_filter_host_batch.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.c_int, vp]
        L.lcf_filter_stream.argtypes = [vp, vp, vp, C.c_int, vp]
        L.lcf_filter_batch.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), C.c_int, vp]
        L.lcf_plan_destroy.argtypes = [vp]
        L.lcf_num_windows.argtypes = [vp]
        for name in ("lcf_get_eigenvalues", "lcf_get_ncc", "lcf_get_gram", "lcf_get_eigenvectors", "lcf_get_weights",
                     "lcf_get_filters", "lcf_get_window_means"):
            getattr(L, name).argtypes = [vp, dp]
        L.lcf_get_cutoffs.argtypes = [vp, ip]
        L.lcf_get_sweeps.argtypes = [vp, ip]
        L.lcf_set_timing.argtypes = [vp, C.c_int]
        L.lcf_set_max_sweeps.argtypes = [vp, C.c_int]
        L.lcf_get_converged.argtypes = [vp, ip]
        L.lcf_get_stage_ms.argtypes = [vp, C.POINTER(C.c_float)]
        L.lcf_get_work.argtypes = [vp, C.POINTER(Work)]
        L.lcf_measure_peak.argtypes = [C.c_int, dp]
        L.lcf_status_string.argtypes = [C.c_int]
        L.lcf_status_string.restype = C.c_char_p
        L.lcf_last_error.argtypes = [vp]
        L.lcf_last_error.restype = C.c_char_p
        for name in EXPORTS:
            if name not in ("lcf_status_string", "lcf_last_error"):
                getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


def status_string(status: int) -> str:
    return load().lcf_status_string(int(status)).decode()


def scale_exponent(amax: float) -> int:
    """k such that amax * 2**k lies in [256, 512): the operand scaling of the tensor-core kernels."""
    L = load()
    L.lcf_scale_exponent.argtypes = [C.c_float]
    return int(L.lcf_scale_exponent(C.c_float(amax)))


def measure_peak(kind: int) -> float:
    """TFLOP/s of the FP32 FFMA (0), packed FFMA2 (1), FP64 DFMA (2) pipe or the tcgen05 fp16 tensor path (3) on the current device."""
    v = C.c_double(0.0)
    st = load().lcf_measure_peak(int(kind), C.byref(v))
    if st != OK:
        raise LcfError(st, "lcf_measure_peak")
    return float(v.value)


def _ptr(x) -> int:
    """Raw address of a torch tensor (data_ptr), numpy array or int."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return int(x.data_ptr())
    if isinstance(x, np.ndarray):
        return int(x.ctypes.data)
    raise TypeError(type(x))


def _stream(s) -> int:
    if s is None:
        return 0
    if isinstance(s, int):
        return s
    return int(s.cuda_stream)          # torch.cuda.Stream


class Plan:
    """lcf_plan_create / lcf_filter / lcf_plan_destroy plus the diagnostic getters."""

    def __init__(self, Nz: int, Nx: int, N: int, Kz: int, Kx: int, sigma_z: float, sigma_x: float, trunc: float,
                 mode: int, k_fixed: int = 0, energy_frac: float = 0.995, beta: float = 0.5, precision: int = 0,
                 cut_scale: float = 1.0):
        L = load()
        self._h = C.c_void_p(None)
        self.Nz, self.Nx, self.N, self.K = int(Nz), int(Nx), int(N), int(Kz) * int(Kx)
        w = Windows(int(Kz), int(Kx), float(sigma_z), float(sigma_x), float(trunc))
        t = Thresh(int(mode), int(k_fixed), float(energy_frac), float(beta), int(precision), float(cut_scale))
        st = L.lcf_plan_create(C.byref(self._h), int(Nz), int(Nx), int(N), C.byref(w), C.byref(t))
        if st != OK:
            self._h = C.c_void_p(None)
            raise LcfError(st, "lcf_plan_create")

    @classmethod
    def from_spec(cls, Nz: int, Nx: int, N: int, filt) -> "Plan":
        """filt: an object with the fields of synth.FilterSpec."""
        return cls(Nz, Nx, N, filt.Kz, filt.Kx, filt.sigma_z, filt.sigma_x, filt.trunc, filt.mode, filt.k_fixed,
                   filt.energy_frac, filt.beta, filt.precision, getattr(filt, "cut_scale", 1.0))

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load().lcf_plan_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.destroy()

    # ---- hot path ----
    def _check(self, t, what, numel, dtypes, cuda):
        """A tensor / array argument must be what the raw pointer is taken to be (an int address is trusted)."""
        if isinstance(t, int) or t is None:
            return
        dt = str(t.dtype).replace("torch.", "")
        if dt not in dtypes:
            raise TypeError(f"{what}: dtype {dt}, expected one of {dtypes}")
        n = int(t.numel()) if hasattr(t, "numel") else int(t.size)
        want = numel if dt.startswith("complex") or len(dtypes) == 1 else 2 * numel   # float32 view of complex64: (re, im) pairs
        if n != want:
            raise ValueError(f"{what}: {n} elements, expected {want}")
        contiguous = t.is_contiguous() if hasattr(t, "is_contiguous") else bool(t.flags["C_CONTIGUOUS"])
        if not contiguous:
            raise ValueError(f"{what}: not contiguous")
        if hasattr(t, "is_cuda") and bool(t.is_cuda) != cuda:
            raise ValueError(f"{what}: must be a {'CUDA' if cuda else 'host'} tensor")
        if not hasattr(t, "is_cuda") and cuda:
            raise ValueError(f"{what}: must be a CUDA tensor")

    def filter(self, iq_dev, pd_dev, stream=None):
        """iq_dev: complex64 device tensor [N][Nx][Nz] (or address); pd_dev: float32 [Nx][Nz]. Asynchronous."""
        self._check(iq_dev, "iq_dev", self.N * self.Nx * self.Nz, ("complex64", "float32"), True)
        self._check(pd_dev, "pd_dev", self.Nx * self.Nz, ("float32",), True)
        st = load().lcf_filter(self._h, _ptr(iq_dev), _ptr(pd_dev), _stream(stream))
        if st != OK:
            raise LcfError(st, "lcf_filter [" + load().lcf_last_error(self._h).decode() + "]")

    def filter_stream(self, iq_dev, pd_dev, stride: int, stream=None):
        """Sliding-window call: this ensemble is the previous streamed one advanced by `stride` frames. Asynchronous."""
        self._check(iq_dev, "iq_dev", self.N * self.Nx * self.Nz, ("complex64", "float32"), True)
        self._check(pd_dev, "pd_dev", self.Nx * self.Nz, ("float32",), True)
        st = load().lcf_filter_stream(self._h, _ptr(iq_dev), _ptr(pd_dev), int(stride), _stream(stream))
        if st != OK:
            raise LcfError(st, "lcf_filter_stream [" + load().lcf_last_error(self._h).decode() + "]")

    def filter_batch(self, iq_devs, pd_devs, stream=None):
        """Lists of device tensors: consecutive ensembles overlap on the plan's two lanes. Asynchronous."""
        n = len(iq_devs)
        if len(pd_devs) != n:
            raise ValueError("iq_devs and pd_devs differ in length")
        for a, b in zip(iq_devs, pd_devs):
            self._check(a, "iq_dev", self.N * self.Nx * self.Nz, ("complex64", "float32"), True)
            self._check(b, "pd_dev", self.Nx * self.Nz, ("float32",), True)
        ia = (C.c_void_p * n)(*[_ptr(x) for x in iq_devs])
        pa = (C.c_void_p * n)(*[_ptr(x) for x in pd_devs])
        st = load().lcf_filter_batch(self._h, ia, pa, n, _stream(stream))
        if st != OK:
            raise LcfError(st, "lcf_filter_batch [" + load().lcf_last_error(self._h).decode() + "]")

    def filter_host(self, iq_host, pd_host, stream=None):
        """Host buffers (numpy / pinned torch tensors); copies, filters, copies back, synchronises."""
        self._check(iq_host, "iq_host", self.N * self.Nx * self.Nz, ("complex64", "float32"), False)
        self._check(pd_host, "pd_host", self.Nx * self.Nz, ("float32",), False)
        st = load().lcf_filter_host(self._h, _ptr(iq_host), _ptr(pd_host), _stream(stream))
        if st != OK:
            raise LcfError(st, "lcf_filter_host")

    def filter_host_batch(self, iq_hosts, pd_hosts, stream=None):
        """Lists of host buffers (pinned): pipelined copies and kernels; returns when all are done."""
        n = len(iq_hosts)
        if len(pd_hosts) != n:
            raise ValueError("iq_hosts and pd_hosts differ in length")
        for a, b in zip(iq_hosts, pd_hosts):
            self._check(a, "iq_host", self.N * self.Nx * self.Nz, ("complex64", "float32"), False)
            self._check(b, "pd_host", self.Nx * self.Nz, ("float32",), False)
        ia = (C.c_void_p * n)(*[_ptr(x) for x in iq_hosts])
        pa = (C.c_void_p * n)(*[_ptr(x) for x in pd_hosts])
        st = load().lcf_filter_host_batch(self._h, ia, pa, n, _stream(stream))
        if st != OK:
            raise LcfError(st, "lcf_filter_host_batch [" + load().lcf_last_error(self._h).decode() + "]")

    def set_max_sweeps(self, n: int):
        st = load().lcf_set_max_sweeps(self._h, int(n))
        if st != OK:
            raise LcfError(st, "lcf_set_max_sweeps")

    def unconverged(self) -> int:
        """Window EVDs that hit the sweep cap since this was last asked (synchronises)."""
        n = C.c_int(0)
        st = load().lcf_get_converged(self._h, C.byref(n))
        if st not in (OK, ERR_NOT_CONVERGED):
            raise LcfError(st, "lcf_get_converged")
        return int(n.value)

    # ---- diagnostics ----
    def _get_d(self, fn, shape, allow_unconverged=False):
        out = np.empty(shape, dtype=np.float64)
        st = getattr(load(), fn)(self._h, out.ctypes.data_as(C.POINTER(C.c_double)))
        if st != OK and not (allow_unconverged and st == ERR_NOT_CONVERGED):
            raise LcfError(st, fn)
        return out

    def _get_i(self, fn, allow_unconverged=False):
        out = np.empty(self.K, dtype=np.int32)
        st = getattr(load(), fn)(self._h, out.ctypes.data_as(C.POINTER(C.c_int)))
        if st != OK and not (allow_unconverged and st == ERR_NOT_CONVERGED):
            raise LcfError(st, fn)
        return out

    def eigenvalues(self, **kw):
        return self._get_d("lcf_get_eigenvalues", (self.K, self.N), **kw)

    def cutoffs(self, **kw):
        return self._get_i("lcf_get_cutoffs", **kw)

    def sweeps(self, **kw):
        return self._get_i("lcf_get_sweeps", **kw)

    def weights(self, **kw):
        return self._get_d("lcf_get_weights", (self.K, self.N), **kw)

    def ncc(self, **kw):
        """NCC(k) curves of method 4, [K][N] (NCC-mode plans only)."""
        return self._get_d("lcf_get_ncc", (self.K, self.N), **kw)

    def window_means(self, **kw):
        return self._get_d("lcf_get_window_means", (self.K,), **kw)

    def gram(self, **kw):
        return self._get_d("lcf_get_gram", (self.K, self.N, self.N, 2), **kw).view(np.complex128)[..., 0]

    def eigenvectors(self, **kw):
        return self._get_d("lcf_get_eigenvectors", (self.K, self.N, self.N, 2), **kw).view(np.complex128)[..., 0]

    def filters(self, **kw):
        return self._get_d("lcf_get_filters", (self.K, self.N, self.N, 2), **kw).view(np.complex128)[..., 0]

    # ---- measurement ----
    def set_timing(self, enabled: bool):
        st = load().lcf_set_timing(self._h, int(bool(enabled)))
        if st != OK:
            raise LcfError(st, "lcf_set_timing")

    def stage_ms(self):
        ms = (C.c_float * 5)()
        st = load().lcf_get_stage_ms(self._h, ms)
        if st != OK:
            raise LcfError(st, "lcf_get_stage_ms")
        return dict(zip(("gram", "evd", "weights_projector", "projection", "combine"), [float(v) for v in ms]))

    def work(self) -> dict:
        w = Work()
        st = load().lcf_get_work(self._h, C.byref(w))
        if st != OK:
            raise LcfError(st, "lcf_get_work")
        return {k: getattr(w, k) for k, _ in Work._fields_}
