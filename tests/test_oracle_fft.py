"""Pins for the oracle's own transforms: brute-force O(n^2) DFT, radix-2 FFT,
numpy.fft as the library routine, and identities the DFT must satisfy."""
import numpy as np
import pytest


def _rand_c(rng, shape):
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


@pytest.mark.parametrize("n", [1, 2, 3, 5, 8, 16, 30])
def test_naive_dft_is_the_definition(oracle, n):
    # the O(n^2) sum against the textbook matrix, typed out independently here
    rng = np.random.default_rng(n)
    x = _rand_c(rng, n)
    j = np.arange(n)
    Wf = np.exp(-2j * np.pi * np.outer(j, j) / n)
    np.testing.assert_allclose(oracle.dft1d_naive(x, -1), Wf @ x, rtol=0, atol=1e-12 * n)
    np.testing.assert_allclose(oracle.dft1d_naive(x, +1), Wf.conj() @ x, rtol=0, atol=1e-12 * n)


@pytest.mark.parametrize("n", [2, 4, 8, 64, 256, 2048])
def test_radix2_matches_naive_and_numpy(oracle, n):
    rng = np.random.default_rng(100 + n)
    x = _rand_c(rng, n)
    f = oracle.fft1d_radix2(x, -1)
    np.testing.assert_allclose(f, np.fft.fft(x), rtol=0, atol=1e-13 * n)
    np.testing.assert_allclose(oracle.fft1d_radix2(x, +1), np.fft.ifft(x) * n, rtol=0, atol=1e-13 * n)
    if n <= 256:
        np.testing.assert_allclose(f, oracle.dft1d_naive(x, -1), rtol=0, atol=1e-12 * n)


@pytest.mark.parametrize("shape", [(8, 8), (16, 16), (4, 8), (4, 4, 4), (8, 8, 8), (2, 4, 16)])
def test_fftn_radix2_vs_brute_force_vs_numpy(oracle, shape):
    rng = np.random.default_rng(sum(shape))
    a = _rand_c(rng, shape)
    fast = oracle.fftn(a, -1, naive=False)
    slow = oracle.fftn(a, -1, naive=True)
    ref = np.fft.fftn(a)
    np.testing.assert_allclose(fast, slow, rtol=0, atol=1e-13 * a.size)
    np.testing.assert_allclose(fast, ref, rtol=0, atol=1e-13 * a.size)
    # F^-1 F = N * identity (both unnormalised)
    back = oracle.fftn(fast, +1) / a.size
    np.testing.assert_allclose(back, a, rtol=0, atol=1e-13)


def test_fftn_non_power_of_two_needs_naive(oracle):
    a = np.ones((6, 6), dtype=complex)
    with pytest.raises(RuntimeError):
        oracle.fftn(a, -1, naive=False)
    np.testing.assert_allclose(oracle.fftn(a, -1, naive=True), np.fft.fftn(a), atol=1e-12)


def test_parseval_and_single_cosine(oracle):
    ny, nx = 16, 32
    rng = np.random.default_rng(7)
    a = _rand_c(rng, (ny, nx))
    A = oracle.fftn(a, -1)
    assert np.isclose(np.sum(np.abs(A) ** 2), a.size * np.sum(np.abs(a) ** 2), rtol=1e-13)
    # cos(2 pi (3 x/nx + 2 y/ny)) lands in exactly the bins (+3,+2) and (-3,-2) with amplitude N/2
    y, x = np.meshgrid(np.arange(ny), np.arange(nx), indexing="ij")
    u = np.cos(2 * np.pi * (3 * x / nx + 2 * y / ny))
    U = oracle.fftn(u.astype(complex), -1)
    expect = np.zeros((ny, nx), dtype=complex)
    expect[2, 3] = expect[ny - 2, nx - 3] = ny * nx / 2
    np.testing.assert_allclose(U, expect, rtol=0, atol=1e-11)


def test_axis_order_is_zyx(oracle):
    # a delta at (z,y,x) = (1,2,3) must produce the phase exp(-2 pi i (kz*1/nz + ky*2/ny + kx*3/nx))
    nz, ny, nx = 4, 8, 16
    a = np.zeros((nz, ny, nx), dtype=complex)
    a[1, 2, 3] = 1.0
    kz, ky, kx = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    expect = np.exp(-2j * np.pi * (kz * 1 / nz + ky * 2 / ny + kx * 3 / nx))
    np.testing.assert_allclose(oracle.fftn(a, -1), expect, rtol=0, atol=1e-13)
