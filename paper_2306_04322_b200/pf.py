"""ctypes binding of libpf.so (include/pf.h): argument marshalling only -- every step of the
Fourier-spectral and finite-difference paths runs in the CUDA kernels of csrc/.

There is no CPU fallback: importing works anywhere (the library only needs the CUDA runtime that is
linked into it), but `Context(...)` raises PfError when no CUDA device is usable, and `lib()` raises
when libpf.so has not been built (python -m paper_2306_04322_b200.build).
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
SO_PATH = os.environ.get("PF_LIBPF") or os.path.join(_HERE, "libpf.so")      # PF_LIBPF: explicit path override

PF_F32, PF_F64 = 0, 1
PF_HOST, PF_DEVICE = 0, 1
PF_OK, PF_EINVAL, PF_ENOMEM, PF_ECUDA, PF_ESTATE, PF_EUNSUPPORTED = 0, -1, -2, -3, -4, -5

EXPORTS = ["pf_create", "pf_create_batch", "pf_batch_size", "pf_set_fields", "pf_step_fs", "pf_step_fd", "pf_get_fields", "pf_free_energy",
           "pf_free_energy_static", "pf_set_dt", "pf_launch_count", "pf_fp64_fma_peak", "pf_dsmem_read_rate", "pf_set_profiling", "pf_num_fs_kernels", "pf_fs_kernel_ms", "pf_launch_fs_kernel",
           "pf_fs_kernel_name", "pf_strerror", "pf_last_cuda_error", "pf_destroy"]


class PfParams(ctypes.Structure):
    _fields_ = [
        ("ndim", ctypes.c_int), ("n", ctypes.c_int * 3), ("n_eta", ctypes.c_int),
        ("dx", ctypes.c_double * 3), ("dt", ctypes.c_double),
        ("M", ctypes.c_double), ("L", ctypes.c_double),
        ("kappa_c", ctypes.c_double), ("kappa_eta", ctypes.c_double),
        ("rho2", ctypes.c_double), ("c_alpha", ctypes.c_double), ("c_beta", ctypes.c_double),
        ("w", ctypes.c_double), ("alpha", ctypes.c_double),
        ("precision", ctypes.c_int), ("k2_kind", ctypes.c_int),
        ("stream", ctypes.c_void_p),
    ]


class PfError(RuntimeError):
    def __init__(self, code: int, what: str, detail: str = ""):
        self.code = code
        super().__init__(f"{what}: {code} ({detail})" if detail else f"{what}: {code}")


_lib = None


def lib() -> ctypes.CDLL:
    """Loads libpf.so; raises if it is missing (no fallback of any kind)."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise FileNotFoundError(f"{SO_PATH} not built: run `python -m paper_2306_04322_b200.build`")
        L = ctypes.CDLL(SO_PATH)
        vp, pp = ctypes.c_void_p, ctypes.POINTER(PfParams)
        L.pf_create.restype = ctypes.c_int
        L.pf_create.argtypes = [pp, ctypes.POINTER(vp)]
        L.pf_create_batch.restype = ctypes.c_int
        L.pf_create_batch.argtypes = [pp, ctypes.c_int, ctypes.POINTER(vp)]
        L.pf_batch_size.restype = ctypes.c_int
        L.pf_batch_size.argtypes = [vp]
        L.pf_set_fields.restype = ctypes.c_int
        L.pf_set_fields.argtypes = [vp, vp, vp, ctypes.c_int]
        L.pf_get_fields.restype = ctypes.c_int
        L.pf_get_fields.argtypes = [vp, vp, vp, ctypes.c_int]
        L.pf_step_fs.restype = ctypes.c_int
        L.pf_step_fs.argtypes = [vp, ctypes.c_int]
        L.pf_step_fd.restype = ctypes.c_int
        L.pf_step_fd.argtypes = [vp, ctypes.c_int]
        L.pf_free_energy.restype = ctypes.c_int
        L.pf_free_energy.argtypes = [vp, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        L.pf_free_energy_static.restype = ctypes.c_int
        L.pf_free_energy_static.argtypes = [pp, vp, vp, ctypes.POINTER(ctypes.c_double)]
        L.pf_set_dt.restype = ctypes.c_int
        L.pf_set_dt.argtypes = [vp, ctypes.c_double]
        L.pf_launch_count.restype = ctypes.c_longlong
        L.pf_launch_count.argtypes = [vp]
        L.pf_fp64_fma_peak.restype = ctypes.c_int
        L.pf_fp64_fma_peak.argtypes = [ctypes.POINTER(ctypes.c_double)]
        L.pf_dsmem_read_rate.restype = ctypes.c_int
        L.pf_dsmem_read_rate.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_double)]
        L.pf_set_profiling.restype = ctypes.c_int
        L.pf_set_profiling.argtypes = [vp, ctypes.c_int]
        L.pf_num_fs_kernels.restype = ctypes.c_int
        L.pf_num_fs_kernels.argtypes = [vp]
        L.pf_fs_kernel_ms.restype = ctypes.c_double
        L.pf_fs_kernel_ms.argtypes = [vp, ctypes.c_int]
        L.pf_fs_kernel_name.restype = ctypes.c_char_p
        L.pf_fs_kernel_name.argtypes = [vp, ctypes.c_int]
        L.pf_launch_fs_kernel.restype = ctypes.c_int
        L.pf_launch_fs_kernel.argtypes = [vp, ctypes.c_int]
        L.pf_strerror.restype = ctypes.c_char_p
        L.pf_strerror.argtypes = [ctypes.c_int]
        L.pf_last_cuda_error.restype = ctypes.c_char_p
        L.pf_last_cuda_error.argtypes = [vp]
        L.pf_destroy.restype = None
        L.pf_destroy.argtypes = [vp]
        _lib = L
    return _lib


def make_params(n, n_eta=4, dx=1.0, dt=5e-3, M=5.0, L=5.0, kappa_c=3.0, kappa_eta=3.0, rho2=2.0,
                c_alpha=0.3, c_beta=0.7, w=1.0, alpha=5.0, precision="f64", k2_kind=0, stream=None) -> PfParams:
    """Parameters in the paper's notation; defaults are the paper's constants."""
    n = tuple(int(v) for v in n)
    ndim = len(n)
    dx = tuple(dx) if isinstance(dx, (tuple, list)) else (float(dx),) * ndim
    p = PfParams()
    p.ndim = ndim
    for d in range(3):
        p.n[d] = n[d] if d < ndim else 1
        p.dx[d] = dx[d] if d < ndim else 1.0
    p.n_eta, p.dt = int(n_eta), float(dt)
    p.M, p.L, p.kappa_c, p.kappa_eta = M, L, kappa_c, kappa_eta
    p.rho2, p.c_alpha, p.c_beta, p.w, p.alpha = rho2, c_alpha, c_beta, w, alpha
    p.precision = {"f64": PF_F64, "f32": PF_F32}[precision] if isinstance(precision, str) else int(precision)
    p.k2_kind = int(k2_kind)
    p.stream = ctypes.c_void_p(stream) if stream else None
    return p


def fp64_fma_peak() -> float:
    """Measured fp64 FMA rate of the current device, TFLOP/s (pf_fp64_fma_peak)."""
    out = ctypes.c_double()
    rc = lib().pf_fp64_fma_peak(ctypes.byref(out))
    if rc != PF_OK:
        raise PfError(rc, "pf_fp64_fma_peak", lib().pf_strerror(rc).decode())
    return float(out.value)


STATIC_MAX_POINTS = 1 << 24          # PF_STATIC_MAX_POINTS of pf.h


def free_energy_static(c, eta, n, **kw):
    """pf_free_energy_static: Eq. 1 with forward-difference gradients for fields that already sit on the device, for
    callers that may not allocate device memory (an application whose own pool owns the GPU, a monitor inside another
    solver's time loop, a no-allocation-after-start-up service). No context is created and the library allocates nothing:
    its working memory is a fixed array inside libpf.so, shared by all calls, which is why at most STATIC_MAX_POINTS grid
    points are accepted and why calls that overlap on the GPU must be serialised by the caller (see pf.h).
    c, eta: objects with data_ptr() (torch CUDA tensors of the dtype `precision` names; eta may be None when n_eta == 0);
    n and the keywords as for make_params. Returns the 3 + n_eta doubles of pf_free_energy(gradient_kind=1)."""
    p = make_params(n, **kw)
    out = (ctypes.c_double * (3 + p.n_eta))()
    rc = lib().pf_free_energy_static(ctypes.byref(p), c.data_ptr(), eta.data_ptr() if p.n_eta else None, out)
    if rc != PF_OK:
        raise PfError(rc, "pf_free_energy_static", lib().pf_strerror(rc).decode())
    return np.array(out[:], dtype=np.float64)


def dsmem_read_rate(cluster_size: int, remote: bool = True) -> float:
    """Measured distributed-shared-memory read rate, bytes per SM clock per SM (pf_dsmem_read_rate)."""
    out = ctypes.c_double()
    rc = lib().pf_dsmem_read_rate(int(cluster_size), int(bool(remote)), ctypes.byref(out))
    if rc != PF_OK:
        raise PfError(rc, "pf_dsmem_read_rate", lib().pf_strerror(rc).decode())
    return float(out.value)


class Context:
    """Thin RAII wrapper of pf_ctx. Host arrays are numpy, device arrays anything with `data_ptr()` (torch).
    nbatch = B > 0: pf_create_batch, B independent replicas per launch; fields are then c [B, ny, nx], eta [B, p, ny, nx]."""

    def __init__(self, n, nbatch=None, **kw):
        self.params = make_params(n, **kw)
        self.n = tuple(int(v) for v in n)
        self.n_eta = self.params.n_eta
        self.dtype = np.float64 if self.params.precision == PF_F64 else np.float32
        self.nbatch = None if nbatch is None else int(nbatch)
        self.shape = tuple(reversed(self.n))
        self._cshape = self.shape if nbatch is None else (self.nbatch,) + self.shape
        self._eshape = (self.n_eta,) + self.shape if nbatch is None else (self.nbatch, self.n_eta) + self.shape
        self._h = ctypes.c_void_p()
        if nbatch is None:
            rc, what = lib().pf_create(ctypes.byref(self.params), ctypes.byref(self._h)), "pf_create"
        else:
            rc, what = lib().pf_create_batch(ctypes.byref(self.params), self.nbatch, ctypes.byref(self._h)), "pf_create_batch"
        if rc != PF_OK:
            self._h = ctypes.c_void_p()
            raise PfError(rc, what, lib().pf_strerror(rc).decode())

    def _ck(self, rc, what):
        if rc != PF_OK:
            detail = lib().pf_strerror(rc).decode()
            if rc == PF_ECUDA:
                detail += ": " + lib().pf_last_cuda_error(self._h).decode()
            raise PfError(rc, what, detail)

    # ---- host (numpy) ----
    def set_fields(self, c, eta):
        c = np.ascontiguousarray(c, dtype=self.dtype).reshape(self._cshape)
        eta = np.ascontiguousarray(eta, dtype=self.dtype).reshape(self._eshape)
        self._ck(lib().pf_set_fields(self._h, c.ctypes.data, eta.ctypes.data if self.n_eta else None, PF_HOST), "pf_set_fields")

    def get_fields(self):
        c = np.empty(self._cshape, dtype=self.dtype)
        eta = np.empty(self._eshape, dtype=self.dtype)
        self._ck(lib().pf_get_fields(self._h, c.ctypes.data, eta.ctypes.data if self.n_eta else None, PF_HOST), "pf_get_fields")
        return c, eta

    # ---- device (objects exposing data_ptr(), e.g. torch CUDA tensors) ----
    def set_fields_device(self, c, eta):
        self._ck(lib().pf_set_fields(self._h, c.data_ptr(), eta.data_ptr() if self.n_eta else None, PF_DEVICE), "pf_set_fields")

    def get_fields_device(self, c, eta):
        self._ck(lib().pf_get_fields(self._h, c.data_ptr(), eta.data_ptr() if self.n_eta else None, PF_DEVICE), "pf_get_fields")

    def step_fs(self, nsteps: int):
        self._ck(lib().pf_step_fs(self._h, int(nsteps)), "pf_step_fs")

    def step_fd(self, nsteps: int):
        self._ck(lib().pf_step_fd(self._h, int(nsteps)), "pf_step_fd")

    def set_dt(self, dt: float):
        self._ck(lib().pf_set_dt(self._h, float(dt)), "pf_set_dt")

    def free_energy(self, gradient_kind: int = 0):
        out = (ctypes.c_double * (3 + self.n_eta))()
        self._ck(lib().pf_free_energy(self._h, int(gradient_kind), out), "pf_free_energy")
        return np.array(out[:], dtype=np.float64)

    def launch_count(self) -> int:
        return int(lib().pf_launch_count(self._h))

    def set_profiling(self, on):
        """Events around every kernel of a step (no graph replay); see pf.h."""
        self._ck(lib().pf_set_profiling(self._h, int(bool(on))), "pf_set_profiling")

    def launch_fs_kernel(self, which: int):
        """Timing aid (pf.h): queues only kernel `which` of a step; the fields are no trajectory afterwards."""
        self._ck(lib().pf_launch_fs_kernel(self._h, int(which)), "pf_launch_fs_kernel")

    def fs_kernel_names(self):
        return [lib().pf_fs_kernel_name(self._h, i).decode() for i in range(lib().pf_num_fs_kernels(self._h))]

    def fs_kernel_times(self):
        """[(name, ms)] of the most recent profiled pf_step_fs call."""
        k = lib().pf_num_fs_kernels(self._h)
        return [(lib().pf_fs_kernel_name(self._h, i).decode(), lib().pf_fs_kernel_ms(self._h, i)) for i in range(k)]

    def close(self):
        if self._h:
            lib().pf_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
