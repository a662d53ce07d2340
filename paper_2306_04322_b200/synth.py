"""Seeded synthetic inputs (initial fields) shared by the tests, bench.py and smoke().

This module holds NO arithmetic of the method (no free-energy derivative, no transform, no update):
only initial conditions.  Both the CUDA path and the oracle are fed the arrays produced here.

* init A  -- the BASELINE.json configs' recipe: c = c0 + 0.01 U(-1,1), eta_i = 0.001 U(-1,1), U from a
  counter-based generator keyed by (seed, field, linear point index), so any traversal order or
  sharding reproduces the same field.
* init B  -- the paper's benchmark initial condition, Eqs. 4-5 sampled on x_j = j*dx,
  and its 3D extension Eq. 6 applied to the raw Eq. 5 field (the paper applies it to a
  pre-evolved field that is not available).  It gives eta = O(1) dynamics.
* band-limited noise -- random low-wavenumber Fourier modes, the same continuous function on any grid.
"""
from __future__ import annotations

import numpy as np

_U64 = np.uint64
_GOLD = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)


def counter_uniform(seed: int, field: int, index: np.ndarray) -> np.ndarray:
    """U(-1,1) as a pure function of (seed, field, index): a splitmix64-style finaliser over a
    64-bit counter; 53 mantissa bits -> doubles in [-1, 1)."""
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = idx * _GOLD + _U64(seed & 0xFFFFFFFFFFFFFFFF) * _M1 + _U64(field + 1) * _M2
        z = (z ^ (z >> _U64(30))) * _M1
        z = (z ^ (z >> _U64(27))) * _M2
        z = z ^ (z >> _U64(31))
        z = (z + _GOLD)
        z = (z ^ (z >> _U64(30))) * _M1
        z = (z ^ (z >> _U64(27))) * _M2
        z = z ^ (z >> _U64(31))
    u = (z >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    return 2.0 * u - 1.0


def init_a(n, n_eta: int, seed: int, c0: float = 0.5, amp_c: float = 0.01, amp_eta: float = 0.001):
    """Seeded noise init of the configs. n = (nx, ny) or (nx, ny, nz); returns c [.. ny, nx], eta [p, ...]."""
    shape = tuple(reversed(tuple(int(v) for v in n)))
    npts = int(np.prod(shape))
    idx = np.arange(npts, dtype=np.uint64)
    c = (c0 + amp_c * counter_uniform(seed, 0, idx)).reshape(shape)
    eta = np.empty((n_eta,) + shape, dtype=np.float64)
    for i in range(n_eta):
        eta[i] = (amp_eta * counter_uniform(seed, 1 + i, idx)).reshape(shape)
    return c, eta


# --- the paper's benchmark initial condition -------------------------------------------------
C0, EPS, ETA_NU, PSI = 0.5, 0.05, 0.1, 1.5


def _eq4(x, y):
    return C0 + EPS * (np.cos(0.105 * x) * np.cos(0.11 * y)
                       + (np.cos(0.13 * x) * np.cos(0.087 * y)) ** 2
                       + np.cos(0.025 * x - 0.15 * y) * np.cos(0.07 * x - 0.02 * y))


def _eq5(i, x, y):
    # exactly as printed at PAPER.md:61 (three cosine factors inside psi[...]^2)
    a = np.cos((0.01 * i) * x - 4.0) * np.cos((0.007 + 0.01 * i) * y)
    b = np.cos((0.11 + 0.01 * i) * x) * np.cos((0.11 + 0.01 * i) * y)
    t = (np.cos((0.046 + 0.001 * i) * x + (0.0405 + 0.001 * i) * y)
         * np.cos((0.031 + 0.001 * i) * x + (0.0405 + 0.001 * i) * y)
         * np.cos((0.031 + 0.001 * i) * x + (0.004 + 0.001 * i) * y))
    return ETA_NU * (a + b + PSI * t ** 2) ** 2


def init_b(n, n_eta: int, domain: float | None = None):
    """Eqs. 4-5 on an l x l domain (l = 200 in 2D), or Eq. 6 on l = 100 in 3D with c = c0.
    Returns (c, eta, dx)."""
    n = tuple(int(v) for v in n)
    if len(n) == 2:
        l = 200.0 if domain is None else float(domain)
        nx, ny = n
        dx = (l / nx, l / ny)
        x = (np.arange(nx) * dx[0])[None, :]
        y = (np.arange(ny) * dx[1])[:, None]
        c = _eq4(x, y) + 0.0 * (x + y)
        eta = np.stack([_eq5(i, x, y) + 0.0 * (x + y) for i in range(1, n_eta + 1)]) if n_eta else np.zeros((0, ny, nx))
        return np.ascontiguousarray(c), np.ascontiguousarray(eta), dx
    l = 100.0 if domain is None else float(domain)
    nx, ny, nz = n
    dx = (l / nx, l / ny, l / nz)
    x = (np.arange(nx) * dx[0])[None, None, :]
    y = (np.arange(ny) * dx[1])[None, :, None]
    z = (np.arange(nz) * dx[2])[:, None, None]
    c = np.full((nz, ny, nx), C0)
    eta = np.stack([0.5 * (1.0 + np.tanh(np.arctan(2.0 * _eq5(i, 2.0 * x, 2.0 * y) - 1.0)
                                         - ((z - l / 2.0) / 5.0) ** 4))
                    for i in range(1, n_eta + 1)]) if n_eta else np.zeros((0, nz, ny, nx))
    return c, np.ascontiguousarray(eta), dx


def band_limited(n, n_eta: int, seed: int, domain, kmax: int = 8, c0: float = 0.5,
                 amp_c: float = 0.05, amp_eta: float = 0.05):
    """Random Fourier modes |m_d| <= kmax with seeded amplitudes/phases on a periodic box of edge
    lengths `domain`; the same continuous function whatever the grid (used for grid-refinement runs)."""
    n = tuple(int(v) for v in n)
    ndim = len(n)
    domain = tuple(domain) if isinstance(domain, (tuple, list)) else (float(domain),) * ndim
    grids = np.meshgrid(*[np.arange(n[d]) * (domain[d] / n[d]) for d in reversed(range(ndim))], indexing="ij")
    coords = list(reversed(grids))                 # coords[d] varies along axis d (x fastest)
    nmodes = 24
    out = []
    for f in range(1 + n_eta):
        r = counter_uniform(seed, 100 + f, np.arange(nmodes * (ndim + 2), dtype=np.uint64)).reshape(nmodes, ndim + 2)
        u = np.zeros(tuple(reversed(n)))
        for m in range(nmodes):
            phase = np.pi * r[m, ndim]
            arg = phase
            for d in range(ndim):
                md = int(np.round(r[m, d] * kmax))
                arg = arg + 2.0 * np.pi * md / domain[d] * coords[d]
            u = u + r[m, ndim + 1] * np.cos(arg)
        u = u / nmodes ** 0.5
        out.append(u)
    c = c0 + amp_c * out[0]
    eta = np.stack([amp_eta * (1.0 + o) for o in out[1:]]) if n_eta else np.zeros((0,) + tuple(reversed(n)))
    return np.ascontiguousarray(c), np.ascontiguousarray(eta)
