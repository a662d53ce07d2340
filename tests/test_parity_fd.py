"""GPU parity of the explicit finite-difference step (pf_step_fd) and of pf_free_energy against the oracle."""
import numpy as np
import pytest

from paper_2306_04322_b200 import pf
from parity_util import make_init, rel_linf, run_both

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("n,n_eta,steps", [((64, 64), 2, 500), ((32, 128), 4, 100), ((16, 32, 64), 2, 100), ((64, 32), 0, 50)])
def test_fd_parity_fp64(oracle, n, n_eta, steps):
    # dt = 0.75 x the linear Cahn-Hilliard stability limit of the grid, capped at 2e-3:
    # init B has dx = l/n (coarse) and eta = O(1), where the Allen-Cahn reaction term limits dt instead
    c, eta, dx = make_init("B", n, n_eta)
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = min(0.75 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2)), 2e-3)
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=n_eta, init="B", steps=steps, dt=dt, method="fd")
    assert rel_linf([gc, geta], [rc, reta]) < 1e-12


def test_fd_c1_noise_dx1(oracle):
    # configs[0] FD leg: dx = 1, dt = 0.75 * 1.786e-3
    (gc, geta), (rc, reta) = run_both(oracle, n=(64, 64), n_eta=2, init="A", steps=1000, dt=0.75 * 2.0 / (5 * 8 * (4 + 24)), method="fd")
    assert rel_linf([gc, geta], [rc, reta]) < 1e-12


@pytest.mark.parametrize("n,n_eta,steps", [((16, 16), 1, 50), ((32, 16), 8, 30), ((1024, 1024), 2, 20), ((2048, 64), 4, 20)])
def test_fd_fused_2d_tiles(oracle, n, n_eta, steps):
    # the fused shared-memory-halo kernel: smallest tiles (TX = 16, 32), most fields, and the crossover size
    # (configs[4] grid, 64 x 64 tiles of 64 x 16 points, halos wrapping in both directions)
    c, eta, dx = make_init("B", n, n_eta)
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = min(0.75 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2)), 2e-3)
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=n_eta, init="B", steps=steps, dt=dt, method="fd")
    assert rel_linf([gc, geta], [rc, reta]) < 1e-12


def test_fd_fp32(oracle):
    (gc, geta), (rc, reta) = run_both(oracle, n=(64, 64), n_eta=2, init="B", steps=200, dt=1e-3, method="fd", precision="f32")
    assert rel_linf([gc, geta], [rc, reta]) < 1e-4


def test_fs_then_fd_then_fs_state_handoff(oracle):
    n, p = (64, 32), 2
    c, eta, dx = make_init("B", n, p)
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=1e-3)
    with pf.Context(n, n_eta=p, dx=dx, dt=1e-3) as ctx:
        ctx.set_fields(c, eta)
        ctx.step_fs(7); ctx.step_fd(5); ctx.step_fs(3)
        gc, geta = ctx.get_fields()
    rc, reta = m.step_fs(c, eta, 7)
    rc, reta = m.step_fd(rc, reta, 5)
    rc, reta = m.step_fs(rc, reta, 3)
    assert rel_linf([gc, geta], [rc, reta]) < 1e-10


@pytest.mark.parametrize("n", [(64, 128), (32, 16, 64)])
@pytest.mark.parametrize("kind", [0, 1])
def test_free_energy(oracle, n, kind):
    p = 3
    c, eta, dx = make_init("B", n, p)
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3)
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as ctx:
        ctx.set_fields(c, eta)
        e0 = ctx.free_energy(kind)
        ctx.step_fs(10)
        e1 = ctx.free_energy(kind)
        gc, geta = ctx.get_fields()
    np.testing.assert_allclose(e0, m.free_energy(c, eta, kind), rtol=1e-11)
    rc, reta = m.step_fs(c, eta, 10)
    np.testing.assert_allclose(e1, m.free_energy(rc, reta, kind), rtol=1e-9)
    assert e1[0] < e0[0]                      # monotone decrease
    assert rel_linf([gc, geta], [rc, reta]) < 1e-10


@pytest.mark.parametrize("n,n_eta,steps", [((16, 16, 16), 1, 40), ((32, 16, 64), 3, 30), ((64, 64, 64), 2, 20), ((128, 32, 256), 2, 6)])
def test_fd_fused_3d_planes(oracle, n, n_eta, steps):
    # the plane-marching 3D kernel: both tile shapes (16 x 16, 32 x 8), one and several z chunks, rings wrapping in z
    c, eta, dx = make_init("B", n, n_eta)
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = min(0.75 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2)), 2e-3)
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=n_eta, init="B", steps=steps, dt=dt, method="fd")
    assert rel_linf([gc, geta], [rc, reta]) < 1e-12


@pytest.mark.parametrize("n,n_eta,steps,precision", [
    ((64, 16, 16), 0, 30, "f64"), ((64, 16, 32), 1, 30, "f64"), ((128, 64, 16), 2, 25, "f64"), ((64, 32, 64), 3, 20, "f64"),
    ((256, 16, 64), 4, 10, "f64"), ((64, 64, 128), 2, 12, "f64"), ((64, 64, 64), 6, 10, "f64"),
    ((128, 32, 64), 2, 40, "f32"), ((64, 16, 32), 4, 40, "f32")])
def test_fd_3d_pair_marching_kernel(oracle, n, n_eta, steps, precision):
    # fd3d_kernels.cu (nx >= 64, up to four order parameters: two points per thread, z neighbours in registers): every
    # field count it serves, tiles that wrap in x and y (nx = 64: one tile per row; ny = 16: two tiles per column),
    # several z chunks with rings that wrap in z, both precisions; six order parameters take the older kernel
    c, eta, dx = make_init("B", n, n_eta)
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = min(0.75 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2)), 2e-3)
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=n_eta, init="B", steps=steps, dt=dt, method="fd", precision=precision)
    assert rel_linf([gc, geta], [rc, reta]) < (1e-12 if precision == "f64" else 1e-5)


def test_fd_3d_anisotropic_spacing_noise(oracle):
    # seeded noise (every point differs from its neighbours) and three different spacings: a transposed stencil weight
    # or a wrong neighbour in the pair code shows up at once
    n, dx = (64, 32, 16), (1.0, 0.8, 1.25)
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = 0.5 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2))
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=2, init="A", steps=50, dt=dt, method="fd", dx=dx)
    assert rel_linf([gc, geta], [rc, reta]) < 1e-12


@pytest.mark.parametrize("n,n_eta,steps,precision", [((64, 16), 0, 40, "f64"), ((64, 64), 8, 30, "f64"), ((128, 32), 5, 30, "f64"),
                                                     ((256, 16), 3, 30, "f64"), ((64, 128), 1, 30, "f64"), ((128, 64), 4, 60, "f32"),
                                                     ((64, 32), 7, 30, "f32")])
def test_fd_2d_pair_kernel(oracle, n, n_eta, steps, precision):
    # fd2d_kernels.cu (nx >= 64, ny >= 16: two points per thread in two rows): every field count, one tile per row / per column
    # (the halo wraps onto the tile itself), both precisions
    c, eta, dx = make_init("B", n, n_eta)
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = min(0.75 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2)), 2e-3)
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=n_eta, init="B", steps=steps, dt=dt, method="fd", precision=precision)
    assert rel_linf([gc, geta], [rc, reta]) < (1e-12 if precision == "f64" else 1e-5)


def test_fd_2d_pair_kernel_noise_anisotropic(oracle):
    n, dx = (128, 64), (1.0, 0.7)
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = 0.5 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2))
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=2, init="A", steps=80, dt=dt, method="fd", dx=dx)
    assert rel_linf([gc, geta], [rc, reta]) < 1e-12
