"""GPU parity of the 3D Fourier-spectral step when a STRIDED axis (y or z) is longer than 256, through the C ABI against
the CPU oracle (the 3D transform of PAPER.md:141-146, the update of Eqs. 12-15).

pf_create accepts every power of two in 16..2048 on every axis; in 3D that selects the strided kernels
col_kernel<T, {512, 1024, 2048}, ..., COL_3D_MIDFWD | COL_3D_LAST | COL_3D_MIDINV | COL_3D_ENERGY> -- among them the fp32
shapes with 16 elements per thread and the carried-c^ indexing of the z kernel at those lengths -- which no test with
ny, nz <= 256 launches. Element-wise cases first, then a sweep of every accepted long-axis shape
for launchability and finiteness, then pf_free_energy in fp32.
"""
import numpy as np
import pytest

from paper_2306_04322_b200 import pf, synth
from parity_util import rel_linf, run_both

pytestmark = pytest.mark.gpu

TOL64, TOL32 = 1e-10, 1e-4


@pytest.mark.parametrize("n", [(16, 16, 1024), (16, 1024, 16), (32, 2048, 16), (16, 32, 2048), (16, 512, 512), (64, 16, 512)])
def test_long_strided_axis_fp64(oracle, n):
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=2, init="B", steps=8, dt=5e-3)
    err = rel_linf([gc, geta], [rc, reta])
    assert err < TOL64, (n, err)


@pytest.mark.parametrize("n", [(16, 16, 2048), (16, 2048, 16), (32, 1024, 32), (32, 16, 1024), (16, 512, 16), (16, 16, 512)])
def test_long_strided_axis_fp32(oracle, n):
    (gc, geta), (rc, reta) = run_both(oracle, n=n, n_eta=2, init="B", steps=8, dt=5e-3, precision="f32")
    err = rel_linf([gc, geta], [rc, reta])
    assert err < TOL32, (n, err)


@pytest.mark.parametrize("n,n_eta", [((16, 2048, 16), 8), ((16, 16, 2048), 8), ((16, 1024, 16), 0), ((16, 16, 1024), 0)])
def test_long_strided_axis_field_counts(oracle, n, n_eta):
    # most and fewest fields at the longest columns, and a read-out in the middle (the carried c^ survives pf_get_fields)
    c, eta, dx = synth.init_b(n, n_eta)
    m = oracle.Model(n=n, n_eta=n_eta, dx=dx, dt=5e-3)
    with pf.Context(n, n_eta=n_eta, dx=dx, dt=5e-3) as ctx:
        ctx.set_fields(c, eta)
        ctx.step_fs(3)
        ctx.get_fields()
        ctx.step_fs(3)
        gc, geta = ctx.get_fields()
    rc, reta = m.step_fs(c, eta, 6)
    assert rel_linf([gc, geta], [rc, reta]) < TOL64


@pytest.mark.parametrize("precision", ["f64", "f32"])
@pytest.mark.parametrize("long_n", [512, 1024, 2048])
def test_every_accepted_3d_long_axis_shape_steps(precision, long_n):
    # pf_create must not accept a 3D shape the kernels cannot launch: each axis in turn at long_n, n_eta in {0, 2, 8},
    # two steps, both gradient kinds of pf_free_energy (the COL_3D_ENERGY shapes), finiteness of everything
    for axis in range(3):
        n = [16, 16, 16]
        n[axis] = long_n
        n = tuple(n)
        for n_eta in (0, 2, 8):
            c, eta, dx = synth.init_b(n, n_eta)
            with pf.Context(n, n_eta=n_eta, dx=dx, dt=5e-3, precision=precision) as ctx:
                ctx.set_fields(c, eta)
                ctx.step_fs(2)
                e0 = ctx.free_energy(0)
                e1 = ctx.free_energy(1)
                ctx.step_fs(1)
                gc, geta = ctx.get_fields()
            assert np.all(np.isfinite(gc)) and np.all(np.isfinite(geta)), (n, n_eta)
            assert np.all(np.isfinite(e0)) and np.all(np.isfinite(e1)), (n, n_eta)
            # the chemical part is the same sum in both kinds; the gradient parts differ by the discretisation only
            assert abs(e0[1] - e1[1]) <= 1e-5 * abs(e1[1]), (n, n_eta)


@pytest.mark.parametrize("n", [(64, 128), (32, 16, 64), (16, 512, 16), (16, 16, 1024)])
@pytest.mark.parametrize("kind", [0, 1])
def test_free_energy_fp32(oracle, n, kind):
    # the fp32 instantiations of energy_kernel and COL_*_ENERGY against the oracle, from the same fp32-rounded fields:
    # pointwise arithmetic in fp32 (relative error ~1e-7 per term), accumulation in fp64 -> rtol 1e-5
    p = 3
    c, eta, dx = synth.init_b(n, p)
    c32 = c.astype(np.float32).astype(np.float64)
    e32 = eta.astype(np.float32).astype(np.float64)
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3)
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3, precision="f32") as ctx:
        ctx.set_fields(c, eta)
        e = ctx.free_energy(kind)
    np.testing.assert_allclose(e, m.free_energy(c32, e32, kind), rtol=1e-5)
