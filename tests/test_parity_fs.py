"""GPU parity of the Fourier-spectral step (pf_step_fs through the C ABI) against the CPU oracle,
element by element on seeded inputs. Tolerances are north_star's: relative L-infinity 1e-10 (fp64),
1e-4 (fp32)."""
import numpy as np
import pytest

from parity_util import rel_linf, run_both

pytestmark = pytest.mark.gpu

TOL64, TOL32 = 1e-10, 1e-4


def _check(oracle, tol, **kw):
    (gc, geta), (rc, reta) = run_both(oracle, **kw)
    assert np.all(np.isfinite(gc)) and np.all(np.isfinite(geta))
    err = rel_linf([gc, geta], [rc, reta])
    assert err < tol, f"rel Linf {err:.3e} >= {tol:g} for {kw}"
    return err


def test_c1_64x64_init_a_200_steps(oracle):
    # BASELINE.json configs[0]: 2D 64x64, dx=1, c + 2 eta, fp64, dt=0.05, 200 FS steps
    _check(oracle, TOL64, n=(64, 64), n_eta=2, init="A", steps=200, dt=0.05)


def test_128x128_p4_init_b_400_steps(oracle):
    # the paper's benchmark initial condition (eta = O(1) dynamics), dt = 5e-3
    _check(oracle, TOL64, n=(128, 128), n_eta=4, init="B", steps=400, dt=5e-3)


@pytest.mark.parametrize("n,n_eta", [((16, 16), 1), ((32, 128), 1), ((256, 16), 3), ((64, 32), 0), ((128, 64), 8),
                                     ((512, 256), 2)])
def test_2d_shapes_and_field_counts(oracle, n, n_eta):
    _check(oracle, TOL64, n=n, n_eta=n_eta, init="B", steps=20, dt=5e-3)


@pytest.mark.parametrize("n", [(16, 16, 16), (32, 16, 64), (64, 32, 16)])
def test_3d_small(oracle, n):
    _check(oracle, TOL64, n=n, n_eta=2, init="B", steps=20, dt=5e-3)


def test_3d_64cubed_init_b(oracle):
    _check(oracle, TOL64, n=(64, 64, 64), n_eta=2, init="B", steps=40, dt=5e-3)


def test_3d_init_a_c4_shape_small(oracle):
    # configs[3] recipe (dt = 0.1, init A, c + 2 eta) on a 32^3 stand-in that the oracle finishes in seconds
    _check(oracle, TOL64, n=(32, 32, 32), n_eta=2, init="A", steps=50, dt=0.1, seed=4)


@pytest.mark.parametrize("kind", [1, 2])
def test_fs_fd_variants(oracle, kind):
    # Eqs. 17/18 frequencies
    _check(oracle, TOL64, n=(64, 128), n_eta=2, init="B", steps=30, dt=5e-3, k2_kind=kind)


def test_anisotropic_spacing(oracle):
    _check(oracle, TOL64, n=(64, 32), n_eta=2, init="A", steps=30, dt=0.02, dx=(0.7, 1.3))


def test_large_1024_sq(oracle):
    # the metric's size: several tiles per kernel, 5 steps (oracle ~ seconds per step)
    _check(oracle, TOL64, n=(1024, 1024), n_eta=2, init="B", steps=5, dt=5e-3)


def test_c4_256_cubed_two_steps_and_invariants(oracle):
    # BASELINE.json configs[3] at full size in the launch configuration bench.py times: element-wise parity after 2
    # steps (the oracle needs seconds per step), then properties that hold at any length: mean c conserved
    # (Eq. 14 leaves the k = 0 mode untouched) and the free energy does not increase
    from paper_2306_04322_b200 import pf, synth
    n, p = (256, 256, 256), 2
    _check(oracle, TOL64, n=n, n_eta=p, init="B", steps=2, dt=5e-3)
    c, eta, dx = synth.init_b(n, p)
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as ctx:
        ctx.set_fields(c, eta)
        e_prev = ctx.free_energy(0)[0]
        for _ in range(3):
            ctx.step_fs(10)
            e = ctx.free_energy(0)[0]
            assert e <= e_prev * (1 + 1e-12)
            e_prev = e
        gc, _ = ctx.get_fields()
    assert abs(gc.mean() - c.mean()) < 1e-13


def test_c3_2048_sq_p4(oracle):
    # BASELINE.json configs[2]: 2048 x 2048, c + 4 eta, fp64 and fp32 side by side (3 steps; the oracle is slow here)
    _check(oracle, TOL64, n=(2048, 2048), n_eta=4, init="B", steps=3, dt=5e-3)
    _check(oracle, TOL32, n=(2048, 2048), n_eta=4, init="B", steps=3, dt=5e-3, precision="f32")


def test_fp32_1024_sq_wide_column_blocks(oracle):
    # fp32 at ny = 1024 uses its own strided-kernel shape (16 elements per thread, four column pairs per CTA)
    _check(oracle, TOL32, n=(1024, 1024), n_eta=2, init="B", steps=5, dt=5e-3, precision="f32")
    _check(oracle, TOL32, n=(64, 1024), n_eta=1, init="B", steps=5, dt=5e-3, precision="f32")


def test_long_axes_2048(oracle):
    _check(oracle, TOL64, n=(2048, 32), n_eta=1, init="B", steps=10, dt=5e-3)
    _check(oracle, TOL64, n=(32, 2048), n_eta=1, init="B", steps=10, dt=5e-3)


def test_fp32_128_init_b_400_steps(oracle):
    _check(oracle, TOL32, n=(128, 128), n_eta=4, init="B", steps=400, dt=5e-3, precision="f32")


def test_fp32_3d(oracle):
    _check(oracle, TOL32, n=(32, 32, 32), n_eta=2, init="B", steps=50, dt=5e-3, precision="f32")


def test_unstable_dt_is_classified_the_same(oracle):
    # dt beyond the linear bound 0.2: both sides must blow up, values are not compared
    (gc, geta), (rc, reta) = run_both(oracle, n=(64, 64), n_eta=2, init="A", steps=400, dt=0.5)
    assert (not np.all(np.isfinite(rc))) or np.max(np.abs(rc)) > 1e6
    assert (not np.all(np.isfinite(gc))) or np.max(np.abs(gc)) > 1e6


@pytest.mark.parametrize("n,n_eta", [((1024, 1024), 2), ((512, 256), 4), ((64, 128, 32), 2)])
def test_repeated_runs_are_bitwise_identical(n, n_eta):
    # compute-sanitizer is closed on this pool: a data race in the exchange buffers, the warp-level barriers of the x
    # kernel or the parked g^ would show up as run-to-run differences; five runs must agree bit for bit
    from paper_2306_04322_b200 import pf, synth
    c, eta, dx = synth.init_b(n, n_eta)
    ref = None
    for _ in range(5):
        with pf.Context(n, n_eta=n_eta, dx=dx, dt=5e-3) as ctx:
            ctx.set_fields(c, eta)
            ctx.step_fs(12)
            out = ctx.get_fields()
        if ref is None:
            ref = out
        else:
            assert np.array_equal(ref[0], out[0]) and np.array_equal(ref[1], out[1])
