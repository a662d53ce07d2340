"""Pins for the oracle's pointwise model, frequencies and stencil (SURVEY 8(c.6)(ii),(vii),(viii))."""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


def paper_values():
    out = {}
    with open(GOLD) as fh:
        for line in fh:
            line = line.split("#")[0].split()
            if len(line) == 2:
                out[line[0]] = float(line[1])
    return out


def test_default_constants_are_the_papers(oracle):
    pv = paper_values()
    m = oracle.Model(n=(8, 8))
    for k in ("kappa_c", "kappa_eta", "rho2", "c_alpha", "c_beta", "w", "alpha", "M", "L"):
        assert getattr(m, k) == pv[k], k
    assert m.n_eta == pv["p"]


def test_fchem_definition_special_values(oracle):
    # eta = 0 is the alpha matrix (h = g = 0), eta_i = 1 alone is beta (h = 1, g = 0)
    m = oracle.Model(n=(8, 8), n_eta=3)
    for c in (0.1, 0.3, 0.55, 0.9):
        assert np.isclose(m.fchem(c, [0, 0, 0]), m.rho2 * (c - m.c_alpha) ** 2, rtol=1e-15, atol=0)
        assert np.isclose(m.fchem(c, [0, 1, 0]), m.rho2 * (m.c_beta - c) ** 2, rtol=1e-15, atol=1e-18)
    # h is additive over variants, so the excess of two overlapping variants is the cross term alone:
    # w * alpha * (eta_1^2 eta_2^2 + eta_2^2 eta_1^2) = 2 alpha w (ordered double sum)
    assert np.isclose(m.fchem(0.3, [1, 1, 0]) - m.fchem(0.3, [1, 0, 0]) - (m.fchem(0.3, [0, 1, 0]) - m.fchem(0.3, [0, 0, 0])),
                      2 * m.alpha * m.w, rtol=1e-13)
    # h(1/2) = 1/2 (interpolation function symmetric), g(1/2) = 1/16
    assert np.isclose(m.fchem(0.5, [0.5, 0, 0]), m.rho2 * 0.04 + m.w / 16, rtol=1e-14)


@pytest.mark.parametrize("p", [1, 2, 4, 7])
def test_derivatives_are_central_differences_of_fchem(oracle, p):
    m = oracle.Model(n=(8, 8), n_eta=p)
    rng = np.random.default_rng(p)
    d = 1e-5
    for _ in range(25):
        c = rng.uniform(0.0, 1.0)
        eta = rng.uniform(-0.2, 1.2, size=p)
        dc, de = m.dfchem(c, eta)
        num_c = (m.fchem(c + d, eta) - m.fchem(c - d, eta)) / (2 * d)
        assert np.isclose(dc, num_c, rtol=0, atol=2e-8), (dc, num_c)
        for i in range(p):
            ep, em = eta.copy(), eta.copy()
            ep[i] += d
            em[i] -= d
            num = (m.fchem(c, ep) - m.fchem(c, em)) / (2 * d)
            assert np.isclose(de[i], num, rtol=0, atol=5e-8 * (1 + abs(num))), (i, de[i], num)


def test_derivative_special_values_and_fixed_points(oracle):
    m = oracle.Model(n=(8, 8), n_eta=3)
    dc, de = m.dfchem(0.42, [0, 0, 0])
    assert np.isclose(dc, 2 * m.rho2 * (0.42 - m.c_alpha), rtol=1e-15) and np.all(de == 0)
    dc, de = m.dfchem(0.42, [0, 1, 0])
    assert np.isclose(dc, -2 * m.rho2 * (m.c_beta - 0.42), rtol=1e-15) and np.all(np.abs(de) < 1e-15)
    # the two bulk equilibria: every derivative vanishes
    for c, eta in ((m.c_alpha, [0, 0, 0]), (m.c_beta, [0, 0, 1])):
        dc, de = m.dfchem(c, eta)
        assert abs(dc) < 1e-15 and np.all(np.abs(de) < 1e-15)


@pytest.mark.parametrize("n,dx", [(8, 1.0), (16, 0.37), (64, 2.0)])
def test_k2_axis(oracle, n, dx):
    m = oracle.Model(n=(n, n), dx=dx)
    # Eq. 16: the library's frequency vector, squared
    np.testing.assert_allclose(m.k2_axis(0), (2 * np.pi * np.fft.fftfreq(n, d=dx)) ** 2, rtol=1e-14, atol=0)
    # index vector as printed: [0..n/2, -(n/2-1)..-1]
    idx = np.array(list(range(0, n // 2 + 1)) + list(range(-(n // 2 - 1), 0)))
    np.testing.assert_allclose(m.k2_axis(0), (2 * np.pi * idx / (n * dx)) ** 2, rtol=1e-14)
    # Eq. 17 / Eq. 18 are the symbols of the 3-point and 5-point (4th-order) second differences:
    # apply the stencils to exp(i xi x) and read off the eigenvalue -k~^2.
    x = np.arange(n) * dx
    xi = 2 * np.pi * np.fft.fftfreq(n, d=dx)
    m.k2_kind = 1
    k2c2 = m.k2_axis(0)
    m.k2_kind = 2
    k2c4 = m.k2_axis(0)
    for j in range(n):
        e = np.exp(1j * xi[j] * x)
        d2 = (np.roll(e, -1) - 2 * e + np.roll(e, 1)) / dx ** 2
        d4 = (-np.roll(e, -2) + 16 * np.roll(e, -1) - 30 * e + 16 * np.roll(e, 1) - np.roll(e, 2)) / (12 * dx ** 2)
        assert np.allclose(d2, -k2c2[j] * e, rtol=0, atol=1e-11 / dx ** 2)
        assert np.allclose(d4, -k2c4[j] * e, rtol=0, atol=1e-11 / dx ** 2)


@pytest.mark.parametrize("n,dx", [((16, 8), (1.0, 0.5)), ((8, 16, 4), (0.7, 1.0, 1.3))])
def test_laplacian_equals_fourier_symbol(oracle, n, dx):
    # (vii): lap_h u = F^-1[-|xi_c2|^2 F u]  (Eq. 17/20), ties the stencil loops to the oracle's FFT
    m = oracle.Model(n=n, n_eta=1, dx=dx, k2_kind=1)
    rng = np.random.default_rng(3)
    u = rng.standard_normal(m.shape)
    lap = m.laplacian(u)
    k2 = m.k2_axis(0)[None, :] + m.k2_axis(1)[:, None]
    if len(n) == 3:
        k2 = k2[None, :, :] + m.k2_axis(2)[:, None, None]
    U = oracle.fftn(u.astype(complex), -1)
    via = oracle.fftn(-k2 * U, +1).real / u.size
    np.testing.assert_allclose(lap, via, rtol=0, atol=1e-12)
    # and a hand-typed stencil on one interior and one wrapped point
    if len(n) == 2:
        for (y, x) in ((3, 5), (0, 0), (n[1] - 1, n[0] - 1)):
            s = ((u[y, (x + 1) % n[0]] + u[y, x - 1] - 2 * u[y, x]) / dx[0] ** 2
                 + (u[(y + 1) % n[1], x] + u[y - 1, x] - 2 * u[y, x]) / dx[1] ** 2)
            assert np.isclose(lap[y, x], s, rtol=1e-13, atol=1e-13)


def test_spectral_laplacian_exact_on_band_limited(oracle):
    # (viii) "exponential convergence": with Eq. 16 frequencies the Laplacian of a
    # band-limited periodic function is exact to rounding, while the 5-point stencil is O(dx^2).
    nx, ny, l = 32, 16, 10.0
    m = oracle.Model(n=(nx, ny), n_eta=1, dx=(l / nx, l / ny))
    x = (np.arange(nx) * l / nx)[None, :]
    y = (np.arange(ny) * l / ny)[:, None]
    kx, ky = 2 * np.pi * 3 / l, 2 * np.pi * 2 / l
    u = np.sin(kx * x) * np.cos(ky * y) + 0.3 * np.cos(2 * kx * x)
    exact = -(kx ** 2 + ky ** 2) * np.sin(kx * x) * np.cos(ky * y) - 0.3 * 4 * kx ** 2 * np.cos(2 * kx * x)
    k2 = m.k2_axis(0)[None, :] + m.k2_axis(1)[:, None]
    spec = oracle.fftn(-k2 * oracle.fftn(u.astype(complex), -1), +1).real / u.size
    np.testing.assert_allclose(spec, exact, rtol=0, atol=1e-12)
    assert np.max(np.abs(m.laplacian(u) - exact)) > 1e-2
