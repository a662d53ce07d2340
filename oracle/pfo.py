"""ORACLE binding (test infrastructure, not the product).

ctypes wrapper around oracle/pfo.c, the plain fp64 CPU implementation of arXiv 2306.04322 written
from PAPER.md.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module; the CUDA package never does.

`build()` compiles pfo.c with gcc into oracle/libpfo.so (building the checker is not using it).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libpfo.so")
_lib = None


def build(force: bool = False) -> str:
    src = os.path.join(_HERE, "pfo.c")
    hdr = os.path.join(_HERE, "pfo.h")
    if (not force and os.path.exists(_SO)
            and os.path.getmtime(_SO) >= max(os.path.getmtime(src), os.path.getmtime(hdr))):
        return _SO
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-o", _SO, src, "-lm"]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class _Params(ctypes.Structure):
    _fields_ = [
        ("ndim", ctypes.c_int), ("n", ctypes.c_int * 3), ("n_eta", ctypes.c_int),
        ("dx", ctypes.c_double * 3), ("dt", ctypes.c_double),
        ("M", ctypes.c_double), ("L", ctypes.c_double),
        ("kappa_c", ctypes.c_double), ("kappa_eta", ctypes.c_double),
        ("rho2", ctypes.c_double), ("c_alpha", ctypes.c_double), ("c_beta", ctypes.c_double),
        ("w", ctypes.c_double), ("alpha", ctypes.c_double),
        ("k2_kind", ctypes.c_int), ("dft_kind", ctypes.c_int),
    ]


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        dp = ctypes.POINTER(ctypes.c_double)
        pp = ctypes.POINTER(_Params)
        L.pfo_fchem.restype = ctypes.c_double
        L.pfo_fchem.argtypes = [pp, ctypes.c_double, dp]
        L.pfo_dfchem.restype = None
        L.pfo_dfchem.argtypes = [pp, ctypes.c_double, dp, dp, dp]
        L.pfo_dft1d_naive.restype = None
        L.pfo_dft1d_naive.argtypes = [ctypes.c_int, dp, dp, ctypes.c_int]
        L.pfo_fft1d_radix2.restype = None
        L.pfo_fft1d_radix2.argtypes = [ctypes.c_int, dp, ctypes.c_int]
        L.pfo_fftn.restype = ctypes.c_int
        L.pfo_fftn.argtypes = [ctypes.POINTER(ctypes.c_int), dp, ctypes.c_int, ctypes.c_int]
        L.pfo_k2_axis.restype = ctypes.c_double
        L.pfo_k2_axis.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_double, ctypes.c_int]
        L.pfo_laplacian.restype = None
        L.pfo_laplacian.argtypes = [pp, dp, dp]
        L.pfo_step_fs.restype = ctypes.c_int
        L.pfo_step_fs.argtypes = [pp, dp, dp, ctypes.c_int]
        L.pfo_step_fd.restype = ctypes.c_int
        L.pfo_step_fd.argtypes = [pp, dp, dp, ctypes.c_int]
        L.pfo_free_energy.restype = ctypes.c_int
        L.pfo_free_energy.argtypes = [pp, dp, dp, ctypes.c_int, dp]
        L.pfo_error_eq22.restype = ctypes.c_double
        L.pfo_error_eq22.argtypes = [ctypes.c_long, dp, dp]
        L.pfo_num_threads.restype = ctypes.c_int
        L.pfo_num_threads.argtypes = []
        _lib = L
    return _lib


def _dp(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


@dataclass
class Model:
    """Parameters in the paper's notation; defaults are the paper's constants."""
    n: tuple                      # (nx, ny) or (nx, ny, nz); arrays are indexed [z][y][x]
    n_eta: int = 4
    dx: tuple | float = 1.0
    dt: float = 5e-3
    M: float = 5.0
    L: float = 5.0
    kappa_c: float = 3.0
    kappa_eta: float = 3.0
    rho2: float = 2.0
    c_alpha: float = 0.3
    c_beta: float = 0.7
    w: float = 1.0
    alpha: float = 5.0
    k2_kind: int = 0
    dft_kind: int = 0
    _p: _Params = field(default=None, repr=False)

    def __post_init__(self):
        n = tuple(int(v) for v in self.n)
        ndim = len(n)
        assert ndim in (2, 3)
        dx = self.dx if isinstance(self.dx, (tuple, list)) else (self.dx,) * ndim
        self.n, self.dx = n, tuple(float(v) for v in dx)
        self._sync()

    def _sync(self):
        p = _Params()
        ndim = len(self.n)
        p.ndim = ndim
        for d in range(3):
            p.n[d] = self.n[d] if d < ndim else 1
            p.dx[d] = self.dx[d] if d < ndim else 1.0
        p.n_eta = self.n_eta
        p.dt = self.dt
        p.M, p.L, p.kappa_c, p.kappa_eta = self.M, self.L, self.kappa_c, self.kappa_eta
        p.rho2, p.c_alpha, p.c_beta, p.w, p.alpha = self.rho2, self.c_alpha, self.c_beta, self.w, self.alpha
        p.k2_kind, p.dft_kind = self.k2_kind, self.dft_kind
        self._p = p

    @property
    def shape(self):
        """numpy shape of one field: (ny, nx) or (nz, ny, nx)."""
        return tuple(reversed(self.n))

    @property
    def npoints(self):
        return int(np.prod(self.n))

    # ---- pointwise ----
    def fchem(self, c: float, eta) -> float:
        self._sync()
        e = np.ascontiguousarray(eta, dtype=np.float64)
        return float(lib().pfo_fchem(ctypes.byref(self._p), float(c), _dp(e)))

    def dfchem(self, c: float, eta):
        self._sync()
        e = np.ascontiguousarray(eta, dtype=np.float64)
        dc = ctypes.c_double(0.0)
        de = np.zeros(max(self.n_eta, 1), dtype=np.float64)
        lib().pfo_dfchem(ctypes.byref(self._p), float(c), _dp(e), ctypes.byref(dc), _dp(de))
        return dc.value, de[: self.n_eta].copy()

    # ---- whole-field operations (inputs are copied; fp64) ----
    def _fields(self, c, eta):
        c = np.array(c, dtype=np.float64, order="C").reshape(self.shape)
        eta = np.array(eta, dtype=np.float64, order="C").reshape((self.n_eta,) + self.shape)
        return c, eta

    def step_fs(self, c, eta, nsteps: int):
        self._sync()
        c, eta = self._fields(c, eta)
        rc = lib().pfo_step_fs(ctypes.byref(self._p), _dp(c), _dp(eta), int(nsteps))
        if rc != 0:
            raise RuntimeError("pfo_step_fs failed")
        return c, eta

    def step_fd(self, c, eta, nsteps: int):
        self._sync()
        c, eta = self._fields(c, eta)
        rc = lib().pfo_step_fd(ctypes.byref(self._p), _dp(c), _dp(eta), int(nsteps))
        if rc != 0:
            raise RuntimeError("pfo_step_fd failed")
        return c, eta

    def laplacian(self, u):
        self._sync()
        u = np.array(u, dtype=np.float64, order="C").reshape(self.shape)
        out = np.empty_like(u)
        lib().pfo_laplacian(ctypes.byref(self._p), _dp(u), _dp(out))
        return out

    def free_energy(self, c, eta, gradient_kind: int = 0):
        self._sync()
        c, eta = self._fields(c, eta)
        out = np.zeros(3 + self.n_eta, dtype=np.float64)
        rc = lib().pfo_free_energy(ctypes.byref(self._p), _dp(c), _dp(eta), int(gradient_kind), _dp(out))
        if rc != 0:
            raise RuntimeError("pfo_free_energy failed")
        return out

    def k2_axis(self, axis: int):
        return np.array([lib().pfo_k2_axis(self.k2_kind, self.n[axis], self.dx[axis], i)
                         for i in range(self.n[axis])])


def fftn(a: np.ndarray, sign: int = -1, naive: bool = False) -> np.ndarray:
    """Unnormalised transform of a complex array shaped (ny,nx) or (nz,ny,nx) with the oracle's own DFT/FFT."""
    z = np.array(a, dtype=np.complex128, order="C")
    shp = z.shape
    n3 = (ctypes.c_int * 3)(*([shp[-1], shp[-2], shp[-3] if z.ndim == 3 else 1]))
    buf = z.view(np.float64)
    rc = lib().pfo_fftn(n3, _dp(buf), int(sign), int(bool(naive)))
    if rc != 0:
        raise RuntimeError("pfo_fftn failed (size not a power of two?)")
    return z


def dft1d_naive(x: np.ndarray, sign: int = -1) -> np.ndarray:
    z = np.array(x, dtype=np.complex128, order="C")
    out = np.empty_like(z)
    lib().pfo_dft1d_naive(z.size, _dp(z.view(np.float64)), _dp(out.view(np.float64)), int(sign))
    return out


def fft1d_radix2(x: np.ndarray, sign: int = -1) -> np.ndarray:
    z = np.array(x, dtype=np.complex128, order="C")
    lib().pfo_fft1d_radix2(z.size, _dp(z.view(np.float64)), int(sign))
    return z


def error_eq22(phi: np.ndarray, ref: np.ndarray) -> float:
    """Eq. 22: sum (ref - phi)^2 / sum ref^2 over arrays sampled at the same points."""
    a = np.ascontiguousarray(phi, dtype=np.float64).ravel()
    b = np.ascontiguousarray(ref, dtype=np.float64).ravel()
    if a.size != b.size:
        raise ValueError("phi and ref must be sampled at the same points")
    v = float(lib().pfo_error_eq22(a.size, _dp(a), _dp(b)))
    if v < 0:
        raise RuntimeError("pfo_error_eq22 failed (empty input or zero reference)")
    return v


def num_threads() -> int:
    return int(lib().pfo_num_threads())
