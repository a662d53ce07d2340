"""Pins for the oracle's time steppers: closed-form amplification factors of
single Fourier modes, stability bounds against the paper's printed FD time steps, conservation of
mean c, monotone free energy, bulk fixed points, closed-form free-energy integrals, brute-force DFT."""
import numpy as np
import pytest

from paper_2306_04322_b200 import synth
from test_oracle_model import paper_values


def _mode(m, mvec):
    """cos(k.x) on the model's grid and the exact |k|^2 (Eq. 16/19) for integer mode numbers mvec."""
    axes = [np.arange(m.n[d]) * m.dx[d] for d in range(len(m.n))]
    k = [2 * np.pi * mvec[d] / (m.n[d] * m.dx[d]) for d in range(len(m.n))]
    if len(m.n) == 2:
        phase = k[0] * axes[0][None, :] + k[1] * axes[1][:, None]
    else:
        phase = k[0] * axes[0][None, None, :] + k[1] * axes[1][None, :, None] + k[2] * axes[2][:, None, None]
    return np.cos(phase), k


CASES = [((16, 16), (1.0, 1.0), (3, 0)), ((16, 8), (1.0, 0.5), (2, 3)), ((8, 32), (0.8, 1.1), (-1, 5)),
         ((8, 8, 16), (1.0, 0.7, 1.3), (1, 2, 3)), ((16, 16), (1.0, 1.0), (8, 8))]


@pytest.mark.parametrize("n,dx,mvec", CASES)
def test_fs_cahn_hilliard_mode_exact_amplification(oracle, n, dx, mvec):
    # (iii) with eta = 0: df/dc = 2 rho^2 (c - c_alpha) is linear, so one mode evolves EXACTLY as
    # A_c^n, A_c = (1 - 2 rho^2 M dt k^2) / (1 + M kappa_c dt k^4), for any amplitude (Eqs. 12, 14)
    m = oracle.Model(n=n, n_eta=2, dx=dx, dt=0.03)
    cosk, k = _mode(m, mvec)
    k2 = sum(v * v for v in k)
    A = (1 - 2 * m.rho2 * m.M * m.dt * k2) / (1 + m.M * m.kappa_c * m.dt * k2 * k2)
    c0, eps, steps = 0.45, 0.1, 4
    c, eta = m.step_fs(c0 + eps * cosk, np.zeros((2,) + m.shape), steps)
    np.testing.assert_allclose(c, c0 + eps * A ** steps * cosk, rtol=0, atol=2e-15)
    assert np.all(eta == 0)


@pytest.mark.parametrize("n,dx,mvec", CASES[:4])
def test_fs_allen_cahn_mode_linearised_amplification(oracle, n, dx, mvec):
    # eta_1 = eps cos(k.x), c = (c_alpha + c_beta)/2 (f^alpha = f^beta): d f/d eta = 2 w eta + O(eta^2), and the
    # quadratic term projects on modes 0 and 2k only -> A_eta = (1 - 2 w L dt)/(1 + L kappa_eta dt k^2)
    # with relative error O(eps^2)   (Eqs. 13, 15)
    m = oracle.Model(n=n, n_eta=2, dx=dx, dt=0.02)
    cosk, k = _mode(m, mvec)
    k2 = sum(v * v for v in k)
    A = (1 - 2 * m.w * m.L * m.dt) / (1 + m.L * m.kappa_eta * m.dt * k2)
    eps = 1e-4
    eta0 = np.zeros((2,) + m.shape)
    eta0[0] = eps * cosk
    c, eta = m.step_fs(np.full(m.shape, 0.5), eta0, 1)
    proj = 2 * np.mean(eta[0] * cosk) if any(2 * abs(mv) != nn for mv, nn in zip(mvec, n)) else np.mean(eta[0] * cosk)
    assert np.isclose(proj / eps, A, rtol=1e-7)
    assert np.max(np.abs(eta[1])) == 0.0


@pytest.mark.parametrize("kind", [1, 2])
def test_fs_fd_variants_use_the_modified_frequencies(oracle, kind):
    # FS-FD: the same step with |xi_c2|^2 / |xi_c4|^2; the mode still evolves exactly
    m = oracle.Model(n=(16, 32), n_eta=1, dx=(0.9, 0.6), dt=0.03, k2_kind=kind)
    mvec = (3, 5)
    cosk, k = _mode(m, mvec)
    if kind == 1:
        k2 = sum(2 * (1 - np.cos(k[d] * m.dx[d])) / m.dx[d] ** 2 for d in range(2))
    else:
        k2 = sum((15 - 16 * np.cos(k[d] * m.dx[d]) + np.cos(2 * k[d] * m.dx[d])) / (6 * m.dx[d] ** 2) for d in range(2))
    A = (1 - 2 * m.rho2 * m.M * m.dt * k2) / (1 + m.M * m.kappa_c * m.dt * k2 * k2)
    c, _ = m.step_fs(0.4 + 0.05 * cosk, np.zeros((1,) + m.shape), 3)
    np.testing.assert_allclose(c, 0.4 + 0.05 * A ** 3 * cosk, rtol=0, atol=2e-15)


@pytest.mark.parametrize("n,dx,mvec", CASES[:4])
def test_fd_mode_amplification(oracle, n, dx, mvec):
    # explicit FD: A_c = 1 - dt M k~^2 (2 rho^2 + kappa_c k~^2), A_eta = 1 - dt L (2 w + kappa_eta k~^2),
    # k~^2 the symbol of the 5/7-point Laplacian (Eq. 17/20)
    m = oracle.Model(n=n, n_eta=1, dx=dx, dt=1e-4)      # below the stability bound of every case
    cosk, k = _mode(m, mvec)
    kt2 = sum(2 * (1 - np.cos(k[d] * m.dx[d])) / m.dx[d] ** 2 for d in range(len(n)))
    Ac = 1 - m.dt * m.M * kt2 * (2 * m.rho2 + m.kappa_c * kt2)
    c, eta = m.step_fd(0.45 + 0.1 * cosk, np.zeros((1,) + m.shape), 3)
    np.testing.assert_allclose(c, 0.45 + 0.1 * Ac ** 3 * cosk, rtol=0, atol=5e-15)
    Ae = 1 - m.dt * m.L * (2 * m.w + m.kappa_eta * kt2)
    eps = 1e-4
    c, eta = m.step_fd(np.full(m.shape, 0.5), (eps * cosk)[None], 1)
    proj = 2 * np.mean(eta[0] * cosk)
    assert np.isclose(proj / eps, Ae, rtol=1e-7)


def _fd_bound(M, rho2, kappa_c, dxs):
    ktmax = sum(4.0 / d ** 2 for d in dxs)
    return 2.0 / (M * ktmax * (2 * rho2 + kappa_c * ktmax))


def test_fd_stability_bound_and_papers_time_steps(oracle):
    # (iv) the checkerboard (Nyquist) mode has the largest k~^2; FD is stable iff dt <= 2/(M k~max^2 (2 rho^2 + kappa_c k~max^2)).
    pv = paper_values()
    m = oracle.Model(n=(16, 16), n_eta=1, dx=1.0)
    bound = _fd_bound(m.M, m.rho2, m.kappa_c, (1.0, 1.0))
    assert np.isclose(bound, 1.786e-3, rtol=1e-3)
    y, x = np.meshgrid(np.arange(16), np.arange(16), indexing="ij")
    cb = (-1.0) ** (x + y)
    for fac, grows in ((0.98, False), (1.02, True)):
        m.dt = fac * bound
        c, _ = m.step_fd(0.5 + 1e-3 * cb, np.zeros((1, 16, 16)), 50)
        amp = np.max(np.abs(c - 0.5))
        assert (amp > 1e-3) == grows
    # the paper's printed 2D FD steps are 0.72-0.79 of this bound (they were found by trial and error
    # on eta = O(1) states); every printed 3D step is below it too.
    for n in (1024, 2048):
        ratio = pv[f"fd_dt_2d_{n}"] / _fd_bound(pv["M"], pv["rho2"], pv["kappa_c"], (pv["l_2d"] / n,) * 2)
        assert 0.70 < ratio < 0.80, (n, ratio)
    for n in (16, 32, 64, 128, 256):
        ratio = pv[f"fd_dt_3d_{n}"] / _fd_bound(pv["M"], pv["rho2"], pv["kappa_c"], (pv["l_3d"] / n,) * 3)
        assert 0.1 < ratio < 0.80, (n, ratio)
    # internal consistency of the printed ratios with the printed table entries
    assert np.isclose(1e-4 / pv["fd_dt_2d_1024"], pv["ratio_2d_1024_dt1e-4"], rtol=2e-3)
    assert np.isclose(5e-3 / pv["fd_dt_3d_128"], pv["ratio_3d_128_dt5e-3"], rtol=2e-3)


def test_fs_linear_stability_around_eta_zero(oracle):
    # explicit reaction term: |1 - 2 w L dt| < 1  <=>  dt < 1/(w L) = 0.2 for the eta k=0 mode
    for dt, stable in ((0.19, True), (0.21, False)):
        m = oracle.Model(n=(16, 16), n_eta=1, dt=dt)
        c, eta = synth.init_a((16, 16), 1, seed=5)
        c, eta = m.step_fs(c, eta, 400)
        if stable:
            assert np.all(np.isfinite(eta)) and np.max(np.abs(eta)) < 1e-3
        else:
            assert (not np.all(np.isfinite(eta))) or np.max(np.abs(eta)) > 1e-3


@pytest.mark.parametrize("ndim", [2, 3])
def test_mass_conservation_and_energy_decay_init_a(oracle, ndim):
    # (v) the k = 0 mode of c is untouched by Eq. 14; FD: sum lap mu = 0. (vi) F non-increasing
    n = (32, 32) if ndim == 2 else (16, 16, 8)
    c0, eta0 = synth.init_a(n, 2, seed=11)
    m = oracle.Model(n=n, n_eta=2, dx=1.0, dt=0.05)
    c, eta = c0, eta0
    mass0 = c0.mean()
    Fprev = m.free_energy(c, eta, 0)[0]
    for _ in range(10):
        c, eta = m.step_fs(c, eta, 3)
        assert abs(c.mean() - mass0) < 1e-14
        Fnow = m.free_energy(c, eta, 0)[0]
        assert Fnow <= Fprev + 1e-12 * abs(Fprev)
        Fprev = Fnow
    m.dt = 0.75 * _fd_bound(m.M, m.rho2, m.kappa_c, m.dx)
    c, eta = c0, eta0
    Fprev = m.free_energy(c, eta, 1)[0]
    for _ in range(10):
        c, eta = m.step_fd(c, eta, 20)
        assert abs(c.mean() - mass0) < 1e-14
        Fnow = m.free_energy(c, eta, 1)[0]
        assert Fnow <= Fprev + 1e-12 * abs(Fprev)
        Fprev = Fnow


def test_nontrivial_dynamics_init_b(oracle):
    # the paper's own initial condition (Eqs. 4-5) at its own dt (Table 1): eta grows towards 1,
    # energy decreases monotonically, mean c is conserved
    n, p = (64, 64), 4
    c, eta, dx = synth.init_b(n, p)
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3)
    mass0 = c.mean()
    Fprev = m.free_energy(c, eta, 0)[0]
    eta_init = eta.copy()
    for _ in range(8):
        c, eta = m.step_fs(c, eta, 50)
        Fnow = m.free_energy(c, eta, 0)[0]
        assert Fnow < Fprev
        Fprev = Fnow
        assert abs(c.mean() - mass0) < 1e-14
    # particles have formed: eta saturates near 1 and has moved O(1) away from the initial field
    assert 0.9 < eta.max() < 1.1 and np.abs(eta - eta_init).max() > 0.3 and np.all(np.isfinite(eta))


def test_bulk_equilibria_are_fixed_points(oracle):
    m = oracle.Model(n=(16, 8), n_eta=2, dt=0.05)
    for cval, e in ((m.c_alpha, (0.0, 0.0)), (m.c_beta, (0.0, 1.0))):
        c = np.full(m.shape, cval)
        eta = np.stack([np.full(m.shape, e[0]), np.full(m.shape, e[1])])
        for stepper in (m.step_fs, m.step_fd):
            c1, eta1 = stepper(c, eta, 5)
            np.testing.assert_allclose(c1, c, rtol=0, atol=1e-15)
            np.testing.assert_allclose(eta1, eta, rtol=0, atol=1e-15)


def test_free_energy_closed_forms(oracle):
    # eta = 0, c = c0 + a cos(k x): chem = V rho^2 ((c0-c_alpha)^2 + a^2/2); grad = V kappa_c a^2 k^2/4
    nx, ny, l = 32, 16, 12.0
    m = oracle.Model(n=(nx, ny), n_eta=2, dx=(l / nx, l / ny))
    k = 2 * np.pi * 3 / l
    x = (np.arange(nx) * l / nx)[None, :] + 0 * np.arange(ny)[:, None]
    c0, a = 0.45, 0.07
    c = c0 + a * np.cos(k * x)
    eta = np.zeros((2, ny, nx))
    V = l * l
    F0 = m.free_energy(c, eta, 0)
    assert np.isclose(F0[1], V * m.rho2 * ((c0 - m.c_alpha) ** 2 + a * a / 2), rtol=1e-13)
    assert np.isclose(F0[2], V * m.kappa_c * a * a * k * k / 4, rtol=1e-13)
    assert F0[3] == 0 and F0[4] == 0 and np.isclose(F0[0], F0[1] + F0[2], rtol=1e-15)
    F1 = m.free_energy(c, eta, 1)
    kt2 = 2 * (1 - np.cos(k * l / nx)) / (l / nx) ** 2
    assert np.isclose(F1[2], V * m.kappa_c * a * a * kt2 / 4, rtol=1e-13)
    # eta gradient term and the double well: eta_1 = b cos(k y) -> kappa_eta b^2 k^2 V / 4
    ky = 2 * np.pi * 2 / l
    y = (np.arange(ny) * l / ny)[:, None] + 0 * np.arange(nx)[None, :]
    eta[0] = 0.2 * np.cos(ky * y)
    F2 = m.free_energy(np.full((ny, nx), 0.5), eta, 0)
    assert np.isclose(F2[3], V * m.kappa_eta * 0.04 * ky * ky / 4, rtol=1e-13) and F2[4] == 0 and abs(F2[2]) < 1e-20


def test_fs_step_brute_force_dft_on_tiny_grids(oracle):
    # the same step with the O(n^2) DFT instead of the radix-2 FFT, and on a non-power-of-two grid
    c, eta = synth.init_a((8, 8), 2, seed=3)
    eta = eta * 300 + 0.3
    a = oracle.Model(n=(8, 8), n_eta=2, dt=0.004, dft_kind=0).step_fs(c, eta, 5)
    b = oracle.Model(n=(8, 8), n_eta=2, dt=0.004, dft_kind=1).step_fs(c, eta, 5)
    np.testing.assert_allclose(a[0], b[0], rtol=0, atol=1e-14)
    np.testing.assert_allclose(a[1], b[1], rtol=0, atol=1e-14)
    c, eta = synth.init_a((6, 5, 3), 1, seed=4)
    m = oracle.Model(n=(6, 5, 3), n_eta=1, dt=0.05, dft_kind=1)
    c1, eta1 = m.step_fs(c, eta, 3)
    assert abs(c1.mean() - c.mean()) < 1e-15 and np.all(np.isfinite(eta1))


def test_fs_step_cross_check_with_numpy_fft(oracle):
    # NOT a pin (it restates Eqs. 12-15), only a guard against indexing slips in the C loops:
    # the update typed with numpy broadcasting and the library FFT, anisotropic grid, eta = O(1)
    n, p = (16, 8, 4), 3
    dx = (1.0, 0.8, 1.25)
    c, eta, _ = synth.init_b(n, p)
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=4e-3)
    k2 = (m.k2_axis(0)[None, None, :] + m.k2_axis(1)[None, :, None] + m.k2_axis(2)[:, None, None])
    cc, ee = c.copy(), eta.copy()
    for _ in range(3):
        g = np.empty_like(cc)
        h = np.empty_like(ee)
        for idx in np.ndindex(cc.shape):
            g[idx], h[(slice(None),) + idx] = m.dfchem(cc[idx], ee[(slice(None),) + idx])
        cc = np.fft.ifftn((np.fft.fftn(cc) - m.dt * m.M * k2 * np.fft.fftn(g)) / (1 + m.dt * m.M * m.kappa_c * k2 ** 2)).real
        ee = np.stack([np.fft.ifftn((np.fft.fftn(ee[i]) - m.dt * m.L * np.fft.fftn(h[i])) / (1 + m.dt * m.L * m.kappa_eta * k2)).real
                       for i in range(p)])
    c1, eta1 = m.step_fs(c, eta, 3)
    np.testing.assert_allclose(c1, cc, rtol=0, atol=1e-14)
    np.testing.assert_allclose(eta1, ee, rtol=0, atol=1e-14)


def test_synth_generators_are_seeded_and_order_free():
    a1 = synth.init_a((16, 8), 2, seed=9)
    a2 = synth.init_a((16, 8), 2, seed=9)
    b = synth.init_a((16, 8), 2, seed=10)
    assert np.array_equal(a1[0], a2[0]) and np.array_equal(a1[1], a2[1]) and not np.array_equal(a1[0], b[0])
    # counter-based: a sub-range of indices reproduces the same values
    idx = np.arange(40, 60, dtype=np.uint64)
    assert np.array_equal(0.5 + 0.01 * synth.counter_uniform(9, 0, idx), a1[0].ravel()[40:60])
    u = synth.counter_uniform(1, 0, np.arange(200000, dtype=np.uint64))
    assert abs(u.mean()) < 0.01 and abs(u.var() - 1 / 3) < 0.01 and u.min() >= -1 and u.max() < 1
    c, eta, dx = synth.init_b((32, 32), 4)
    assert c.shape == (32, 32) and eta.shape == (4, 32, 32) and dx == (6.25, 6.25)
    assert np.isclose(c[0, 0], 0.5 + 0.05 * 3) and eta.min() >= 0


def test_free_energy_closed_forms_3d(oracle):
    # the 3D terms of the gradient energy (the dzu term of kind 1, the kz^2 term of kind 0), anisotropic box:
    # c = c0 + a cos(kz z) -> spectral: V kappa_c a^2 kz^2 / 4; forward differences: kz^2 -> 2 (1 - cos(kz dz)) / dz^2.
    # A y-mode in eta_1 and an oblique (x, z) mode in eta_2 make sure no axis is mistaken for another.
    nx, ny, nz = 16, 8, 32
    lx, ly, lz = 10.0, 6.0, 14.0
    dx = (lx / nx, ly / ny, lz / nz)
    m = oracle.Model(n=(nx, ny, nz), n_eta=2, dx=dx)
    V = lx * ly * lz
    x = (np.arange(nx) * dx[0])[None, None, :] + np.zeros((nz, ny, nx))
    y = (np.arange(ny) * dx[1])[None, :, None] + np.zeros((nz, ny, nx))
    z = (np.arange(nz) * dx[2])[:, None, None] + np.zeros((nz, ny, nx))
    kz, ky, kx = 2 * np.pi * 5 / lz, 2 * np.pi * 1 / ly, 2 * np.pi * 2 / lx
    kz2 = 2 * np.pi * 3 / lz
    c0, a, b1, b2 = 0.45, 0.07, 0.2, 0.1
    c = c0 + a * np.cos(kz * z)
    eta = np.stack([b1 * np.cos(ky * y), b2 * np.cos(kx * x + kz2 * z)])
    F0 = m.free_energy(c, eta, 0)
    assert np.isclose(F0[2], V * m.kappa_c * a * a * kz * kz / 4, rtol=1e-12)
    assert np.isclose(F0[3], V * m.kappa_eta * b1 * b1 * ky * ky / 4, rtol=1e-12)
    assert np.isclose(F0[4], V * m.kappa_eta * b2 * b2 * (kx * kx + kz2 * kz2) / 4, rtol=1e-12)
    F1 = m.free_energy(c, eta, 1)
    t = lambda k, d: 2 * (1 - np.cos(k * d)) / d ** 2
    assert np.isclose(F1[2], V * m.kappa_c * a * a * t(kz, dx[2]) / 4, rtol=1e-12)
    assert np.isclose(F1[3], V * m.kappa_eta * b1 * b1 * t(ky, dx[1]) / 4, rtol=1e-12)
    assert np.isclose(F1[4], V * m.kappa_eta * b2 * b2 * (t(kx, dx[0]) + t(kz2, dx[2])) / 4, rtol=1e-12)
    # FS-FD frequencies in the Parseval form (k2_kind 1 = Eq. 20) agree with the forward differences
    m1 = oracle.Model(n=(nx, ny, nz), n_eta=2, dx=dx, k2_kind=1)
    np.testing.assert_allclose(m1.free_energy(c, eta, 0)[2:], F1[2:], rtol=1e-12)


def test_eq22_closed_forms(oracle):
    # Eq. 22: ratio of squared L2 norms, no square root, no percent.
    n = 64
    x = 2 * np.pi * np.arange(n) / n
    A, B, a0 = 0.3, 0.25, 0.5
    # same mode, different amplitude: (A - B)^2 / A^2
    assert np.isclose(oracle.error_eq22(B * np.cos(3 * x), A * np.cos(3 * x)), (A - B) ** 2 / A ** 2, rtol=1e-13)
    # common mean, orthogonal modes: (A^2/2 + B^2/2) / (a0^2 + A^2/2); the reference (second argument) normalises
    e = oracle.error_eq22(a0 + B * np.cos(5 * x), a0 + A * np.cos(3 * x))
    assert np.isclose(e, (A * A / 2 + B * B / 2) / (a0 * a0 + A * A / 2), rtol=1e-13)
    e_swapped = oracle.error_eq22(a0 + A * np.cos(3 * x), a0 + B * np.cos(5 * x))
    assert np.isclose(e_swapped, (A * A / 2 + B * B / 2) / (a0 * a0 + B * B / 2), rtol=1e-13) and e_swapped != e
    assert oracle.error_eq22(np.ones(5), np.ones(5)) == 0.0
    # 2D arrays are flattened: a constant offset d against a unit reference -> d^2
    assert np.isclose(oracle.error_eq22(np.full((4, 6), 1.1), np.ones((4, 6))), 0.01, rtol=1e-12)
    with pytest.raises(RuntimeError):
        oracle.error_eq22(np.ones(4), np.zeros(4))


def test_harness_eq22_agrees_with_the_oracle(oracle):
    # accuracy.py and crossover.py report Eq. 22 through ONE harness function (paper_2306_04322_b200/metrics.py); it has
    # to be the quantity the oracle defines (and the closed forms above pin), including which argument normalises
    from paper_2306_04322_b200 import metrics
    rng = np.random.default_rng(22)
    for shape in ((50,), (12, 9), (5, 6, 7)):
        ref = 0.5 + 0.2 * rng.standard_normal(shape)
        phi = ref + 0.03 * rng.standard_normal(shape)
        assert np.isclose(metrics.eq22(phi, ref), oracle.error_eq22(phi, ref), rtol=1e-13)
        assert np.isclose(metrics.eq22_percent(phi, ref), 100.0 * oracle.error_eq22(phi, ref), rtol=1e-13)
        assert not np.isclose(metrics.eq22(phi, ref), oracle.error_eq22(ref, phi), rtol=1e-6)
