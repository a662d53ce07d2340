"""GPU parity of the Fourier-spectral step at the lengths and recipes SURVEY 8(c.7)/(d) lists as REQUIRED parity runs
(BASELINE.json configs[0..4]), through the C ABI against the CPU oracle, element by element.

  C1  64^2, p=2, init A seed 1, dt=0.05: 200 FS steps + the FD leg at 0.75 x the stability bound for the same T = 10 (7 467 steps)
  C2  512^2, p=4, init A seed 2 (c0 = 0.4), dt=0.05, the full 2000 steps  (the only parity run with a 512-long strided axis)
  C3  2048^2, p=4, init A seed 3, dt=0.05: 50 steps, fp64 and fp32 from the same (fp32-rounded) input; mass/energy over 1000 steps
  C4  256^3, p=2, init A seed 4, dt=0.1: 10 steps; and 10 steps of init B; 64^3 init B 200 steps
  C5  1024^2, p=2, dx in {0.5, 2}, band-limited seeded field; one large 50-step run of init B at 1024^2
plus the 3D variants no other test reaches: FS-FD frequencies (Eqs. 20/21), n_eta in {0, 4, 8}, fp32
beyond 32^3. Tolerances are north_star's: relative L-infinity 1e-10 (fp64), 1e-4 (fp32).
"""
import numpy as np
import pytest

from paper_2306_04322_b200 import pf, synth
from parity_util import make_init, rel_linf, run_both

pytestmark = pytest.mark.gpu

TOL64, TOL32 = 1e-10, 1e-4


def _check(oracle, tol, **kw):
    (gc, geta), (rc, reta) = run_both(oracle, **kw)
    assert np.all(np.isfinite(gc)) and np.all(np.isfinite(geta))
    err = rel_linf([gc, geta], [rc, reta])
    assert err < tol, f"rel Linf {err:.3e} >= {tol:g} for {kw}"
    return err


def _gpu_fs(n, p, dx, dt, c, eta, steps, precision="f64", k2_kind=0):
    with pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=precision, k2_kind=k2_kind) as ctx:
        ctx.set_fields(c, eta)
        ctx.step_fs(steps)
        return ctx.get_fields()


def test_c1_fd_leg_full_length(oracle):
    # configs[0]: "the same run with explicit FD at stable dt": dt = 0.75 x 1.786e-3, T = 10 -> 7 467 steps
    dt = 0.75 * 2.0 / (5 * 8 * (4 + 24))
    steps = int(round(10.0 / dt))
    assert steps == 7467
    (gc, geta), (rc, reta) = run_both(oracle, n=(64, 64), n_eta=2, init="A", steps=steps, dt=dt, method="fd", seed=1)
    assert rel_linf([gc, geta], [rc, reta]) < 1e-11


def test_c2_512_sq_p4_full_length(oracle):
    # configs[1]: 2D 512x512, c + 4 eta, init A seed 2 with c0 = 0.4, dt = 0.05, the full 2000 FS steps
    _check(oracle, TOL64, n=(512, 512), n_eta=4, init="A", steps=2000, dt=0.05, seed=2, c0=0.4)


def test_c2_512_sq_p4_init_b(oracle):
    # the same kernel instantiations (strided axis 512, x axis 512) on the eta = O(1) field
    _check(oracle, TOL64, n=(512, 512), n_eta=4, init="B", steps=100, dt=5e-3)


def test_c3_2048_sq_p4_50_steps_both_precisions(oracle):
    # configs[2]: 2048x2048, c + 4 eta, init A seed 3, dt = 0.05, fp64 and fp32 side by side, 50 steps against ONE oracle
    # run: both precisions start from the fp32-rounded input (exactly representable in fp64)
    n, p, dt = (2048, 2048), 4, 0.05
    c, eta = synth.init_a(n, p, seed=3)
    c = c.astype(np.float32).astype(np.float64)
    eta = eta.astype(np.float32).astype(np.float64)
    rc, reta = oracle.Model(n=n, n_eta=p, dx=1.0, dt=dt).step_fs(c, eta, 50)
    g64 = _gpu_fs(n, p, (1.0, 1.0), dt, c, eta, 50, "f64")
    assert rel_linf(g64, [rc, reta]) < TOL64
    g32 = _gpu_fs(n, p, (1.0, 1.0), dt, c, eta, 50, "f32")
    assert rel_linf(g32, [rc, reta]) < TOL32


@pytest.mark.parametrize("precision,mass_tol,e_tol", [("f64", 1e-13, 1e-12), ("f32", 2e-6, 1e-5)])
def test_c3_2048_sq_invariants_over_1000_steps(precision, mass_tol, e_tol):
    # properties that hold at any length: mean c conserved (the k = 0 mode is untouched by Eq. 14,
    # PAPER.md:112) and the free energy never increases, sampled every 100 steps of the full run
    n, p, dt = (2048, 2048), 4, 0.05
    c, eta = synth.init_a(n, p, seed=3)
    with pf.Context(n, n_eta=p, dx=(1.0, 1.0), dt=dt, precision=precision) as ctx:
        ctx.set_fields(c, eta)
        e_prev = ctx.free_energy(0)[0]
        for _ in range(10):
            ctx.step_fs(100)
            e = ctx.free_energy(0)[0]
            assert np.isfinite(e) and e <= e_prev + e_tol * abs(e_prev)
            e_prev = e
        gc, geta = ctx.get_fields()
    assert abs(float(gc.astype(np.float64).mean()) - float(c.mean())) < mass_tol
    assert np.all(np.isfinite(geta))


def test_c4_256_cubed_init_a_10_steps(oracle):
    # configs[3]: 3D 256^3, c + 2 eta, init A seed 4, dt = 0.1, 10 steps against the oracle, in the launch configuration
    # bench.py times
    _check(oracle, TOL64, n=(256, 256, 256), n_eta=2, init="A", steps=10, dt=0.1, seed=4)


def test_c4_256_cubed_init_b_10_steps(oracle):
    _check(oracle, TOL64, n=(256, 256, 256), n_eta=2, init="B", steps=10, dt=5e-3)


def test_3d_64_cubed_init_b_200_steps(oracle):
    # 64^3 p=2 200 steps on the eta = O(1) field (Eq. 6)
    _check(oracle, TOL64, n=(64, 64, 64), n_eta=2, init="B", steps=200, dt=5e-3)


def test_1024_sq_init_b_50_steps(oracle):
    # "one large 50-step run" -- the metric's 2D size
    _check(oracle, TOL64, n=(1024, 1024), n_eta=2, init="B", steps=50, dt=5e-3)


@pytest.mark.parametrize("dx", [0.5, 2.0])
def test_c5_1024_sq_band_limited_dx(oracle, dx):
    # configs[4]: 1024^2, c + 2 eta, dx in {0.5, 2}, band-limited seeded field, FS at 5 x the FD stability bound of the grid
    n, p = (1024, 1024), 2
    c, eta = synth.band_limited(n, p, seed=5, domain=(n[0] * dx, n[1] * dx), kmax=64)
    kt2 = 8.0 / dx ** 2
    dt = 5.0 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2))
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=dt).step_fs(c, eta, 20)
    g = _gpu_fs(n, p, (dx, dx), dt, c, eta, 20)
    assert rel_linf(g, [rc, reta]) < TOL64


@pytest.mark.parametrize("kind", [1, 2])
def test_3d_fs_fd_variants(oracle, kind):
    # Eqs. 20/21: the 3D FS-FD frequencies, anisotropic grid so no axis table can be swapped unnoticed
    _check(oracle, TOL64, n=(64, 32, 128), n_eta=2, init="B", steps=30, dt=5e-3, k2_kind=kind)


@pytest.mark.parametrize("n_eta", [0, 4, 8])
def test_3d_field_counts(oracle, n_eta):
    _check(oracle, TOL64, n=(32, 64, 32), n_eta=n_eta, init="B", steps=20, dt=5e-3)


@pytest.mark.parametrize("n,n_eta,steps", [((512, 512), 4, 50), ((256, 256), 4, 100), ((64, 64, 64), 2, 50)])
def test_fp32_mid_sizes(oracle, n, n_eta, steps):
    _check(oracle, TOL32, n=n, n_eta=n_eta, init="B", steps=steps, dt=5e-3, precision="f32")


@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("nx", [16, 32, 64, 128, 256, 512, 1024, 2048])
def test_every_accepted_parameter_set_steps(precision, nx):
    # pf_create must not accept what the kernels cannot launch (n_eta 0..8 x every nx x both precisions); values are
    # checked for finiteness here, element-wise parity of the extreme case is test_x_axis_2048_with_8_eta below
    for n_eta in range(0, 9):
        n = (nx, 16)
        c, eta, dx = synth.init_b(n, n_eta)
        with pf.Context(n, n_eta=n_eta, dx=dx, dt=5e-3, precision=precision) as ctx:
            ctx.set_fields(c, eta)
            ctx.step_fs(2)
            e = ctx.free_energy(0)
            gc, geta = ctx.get_fields()
        assert np.all(np.isfinite(gc)) and np.all(np.isfinite(geta)) and np.all(np.isfinite(e)), (nx, n_eta)
        n = (16, nx)
        c, eta, dx = synth.init_b(n, n_eta)
        with pf.Context(n, n_eta=n_eta, dx=dx, dt=5e-3, precision=precision) as ctx:
            ctx.set_fields(c, eta)
            ctx.step_fs(2)
            gc, geta = ctx.get_fields()
        assert np.all(np.isfinite(gc)) and np.all(np.isfinite(geta)), (nx, n_eta, "strided")


@pytest.mark.parametrize("n_eta", [6, 8])
def test_x_axis_2048_with_many_eta(oracle, n_eta):
    # nx = 2048 with 7 and 9 fields: the x kernel's widest CTA (VERDICT r1 item 3 / ADVICE: 1152 threads did not launch)
    _check(oracle, TOL64, n=(2048, 32), n_eta=n_eta, init="B", steps=10, dt=5e-3)
    _check(oracle, TOL32, n=(2048, 32), n_eta=n_eta, init="B", steps=10, dt=5e-3, precision="f32")
