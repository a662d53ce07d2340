"""GPU parity of batched contexts (pf_create_batch, include/pf.h): B independent replicas advanced by the same launches.
Every replica must evolve exactly as the oracle evolves it on its own (the paper's small-grid remark,
PAPER.md:265)."""
import ctypes

import numpy as np
import pytest

from paper_2306_04322_b200 import pf, synth
from parity_util import rel_linf

pytestmark = pytest.mark.gpu


def _stack(inits):
    return np.stack([c for c, _ in inits]), np.stack([e for _, e in inits])


def test_batch_of_c1_replicas_fs_200_steps(oracle):
    # configs[0] (64^2, c + 2 eta, seeded noise, dt = 0.05) five times over with different seeds and mean compositions
    n, p, B = (64, 64), 2, 5
    inits = [synth.init_a(n, p, seed=10 + b, c0=0.4 + 0.05 * b) for b in range(B)]
    c0, e0 = _stack(inits)
    with pf.Context(n, n_eta=p, dx=1.0, dt=0.05, nbatch=B) as ctx:
        ctx.set_fields(c0, e0)
        l0 = ctx.launch_count()
        ctx.step_fs(200)
        steps_launches = ctx.launch_count() - l0
        gc, ge = ctx.get_fields()
    m = oracle.Model(n=n, n_eta=p, dx=(1.0, 1.0), dt=0.05)
    for b in range(B):
        rc, re_ = m.step_fs(c0[b], e0[b], 200)
        assert rel_linf([gc[b], ge[b]], [rc, re_]) < 1e-10, b
    # the replicas ride in the launches of one simulation: two kernels per step (+ the one-off transforms of the start)
    assert steps_launches <= 2 * 200 + 2


@pytest.mark.parametrize("n,p,B,steps,precision,tol", [((128, 64), 4, 3, 60, "f64", 1e-10), ((32, 128), 1, 7, 40, "f64", 1e-10),
                                                       ((256, 256), 4, 2, 30, "f64", 1e-10), ((64, 64), 2, 9, 100, "f32", 1e-4),
                                                       ((16, 16), 8, 33, 25, "f64", 1e-10), ((1024, 32), 0, 2, 10, "f64", 1e-10)])
def test_batch_fs_init_b_shapes(oracle, n, p, B, steps, precision, tol):
    # eta = O(1) dynamics (Eqs. 4-5), every replica with its own perturbation; ragged column-block counts, one and many
    # items per CTA of the last-axis schedule, both precisions
    c, eta, dx = synth.init_b(n, p)
    rng = np.random.default_rng(7)
    c0 = np.stack([c + 0.02 * rng.standard_normal(c.shape) for _ in range(B)])
    e0 = np.stack([eta + 0.01 * rng.standard_normal(eta.shape) for _ in range(B)])
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3, precision=precision, nbatch=B) as ctx:
        ctx.set_fields(c0, e0)
        ctx.step_fs(steps)
        gc, ge = ctx.get_fields()
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3)
    for b in range(B):
        ci, ei = c0[b], e0[b]
        if precision == "f32":
            ci, ei = ci.astype(np.float32).astype(np.float64), ei.astype(np.float32).astype(np.float64)
        rc, re_ = m.step_fs(ci, ei, steps)
        assert rel_linf([gc[b], ge[b]], [rc, re_]) < tol, b


def test_batch_fd_and_state_handoff(oracle):
    # explicit FD steps of a batch (one launch per step for all replicas), then FS, then FD again
    n, p, B = (64, 32), 2, 4
    c, eta, dx = synth.init_b(n, p)
    rng = np.random.default_rng(3)
    c0 = np.stack([c + 0.02 * rng.standard_normal(c.shape) for _ in range(B)])
    e0 = np.stack([eta + 0.01 * rng.standard_normal(eta.shape) for _ in range(B)])
    kt2 = sum(4.0 / d ** 2 for d in dx)
    dt = min(0.5 * 2.0 / (5.0 * kt2 * (4.0 + 3.0 * kt2)), 2e-3)
    with pf.Context(n, n_eta=p, dx=dx, dt=dt, nbatch=B) as ctx:
        ctx.set_fields(c0, e0)
        ctx.step_fd(40); ctx.step_fs(6); ctx.step_fd(15)
        gc, ge = ctx.get_fields()
        with pytest.raises(pf.PfError) as ei:
            ctx.free_energy(0)
        assert ei.value.code == pf.PF_EUNSUPPORTED
        assert pf.lib().pf_batch_size(ctx._h) == B
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=dt)
    for b in range(B):
        rc, re_ = m.step_fd(c0[b], e0[b], 40)
        rc, re_ = m.step_fs(rc, re_, 6)
        rc, re_ = m.step_fd(rc, re_, 15)
        assert rel_linf([gc[b], ge[b]], [rc, re_]) < 1e-10, b


def test_batch_of_one_equals_single_context_bitwise():
    n, p = (128, 128), 2
    c, eta, dx = synth.init_b(n, p)
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as a, pf.Context(n, n_eta=p, dx=dx, dt=5e-3, nbatch=1) as b:
        a.set_fields(c, eta); b.set_fields(c[None], eta[None])
        a.step_fs(25); b.step_fs(25)
        ac, ae = a.get_fields(); bc, be = b.get_fields()
    assert np.array_equal(ac, bc[0]) and np.array_equal(ae, be[0])


def test_batch_rejects_more_planes_than_a_grid_dimension_holds():
    # 3D: the planes of all replicas are blockIdx.y of the y kernels (at most 65535)
    h = ctypes.c_void_p()
    q = pf.make_params((32, 32, 32), n_eta=2)
    assert pf.lib().pf_create_batch(ctypes.byref(q), 4096, ctypes.byref(h)) == pf.PF_EUNSUPPORTED


@pytest.mark.parametrize("n,p,B,steps,precision,tol", [((16, 16, 16), 2, 5, 40, "f64", 1e-10), ((32, 32, 32), 2, 4, 30, "f64", 1e-10),
                                                       ((64, 32, 16), 4, 3, 20, "f64", 1e-10), ((32, 16, 64), 0, 6, 20, "f64", 1e-10),
                                                       ((32, 32, 32), 2, 3, 30, "f32", 1e-4), ((64, 64, 64), 1, 2, 10, "f64", 1e-10)])
def test_batch_3d_fs(oracle, n, p, B, steps, precision, tol):
    # 3D batches (the paper's small 3D grids, Table 2 / PAPER.md:267): replicas are further planes of the x and y kernels and
    # further column blocks (blockIdx.y) of the z kernel with its carried c^; anisotropic shapes so no stride can be swapped
    c, eta, dx = synth.init_b(n, p)
    rng = np.random.default_rng(11)
    c0 = np.stack([c + 0.02 * rng.standard_normal(c.shape) for _ in range(B)])
    e0 = np.stack([eta + 0.01 * rng.standard_normal(eta.shape) for _ in range(B)])
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3, precision=precision, nbatch=B) as ctx:
        ctx.set_fields(c0, e0)
        l0 = ctx.launch_count()
        ctx.step_fs(steps // 2)
        mid = ctx.get_fields()                       # read-out in the middle: the carried spectra survive it
        ctx.step_fs(steps - steps // 2)
        launches = ctx.launch_count() - l0
        gc, ge = ctx.get_fields()
    assert gc.shape == (B,) + tuple(reversed(n)) and ge.shape == (B, p) + tuple(reversed(n)) and mid[0].shape == gc.shape
    assert launches <= 4 * steps + 6                 # the launches of ONE simulation
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3)
    for b in range(B):
        ci, ei = c0[b], e0[b]
        if precision == "f32":
            ci, ei = ci.astype(np.float32).astype(np.float64), ei.astype(np.float32).astype(np.float64)
        rc, re_ = m.step_fs(ci, ei, steps)
        assert rel_linf([gc[b], ge[b]], [rc, re_]) < tol, b


@pytest.mark.parametrize("n", [(64, 32, 32), (16, 16, 32)])
def test_batch_3d_fd_and_handoff(oracle, n):
    # explicit FD on a 3D batch (one launch per replica and step; both 3D FD kernels: nx >= 64 marching, nx < 64 fused) and
    # the FS -> FD -> FS hand-off
    p, B = 2, 3
    c, eta, dx = synth.init_b(n, p)
    rng = np.random.default_rng(12)
    c0 = np.stack([c + 0.02 * rng.standard_normal(c.shape) for _ in range(B)])
    e0 = np.stack([eta + 0.01 * rng.standard_normal(eta.shape) for _ in range(B)])
    with pf.Context(n, n_eta=p, dx=dx, dt=1e-3, nbatch=B) as ctx:
        ctx.set_fields(c0, e0)
        ctx.step_fs(4); ctx.step_fd(6); ctx.step_fs(3)
        gc, ge = ctx.get_fields()
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=1e-3)
    for b in range(B):
        rc, re_ = m.step_fs(c0[b], e0[b], 4)
        rc, re_ = m.step_fd(rc, re_, 6)
        rc, re_ = m.step_fs(rc, re_, 3)
        assert rel_linf([gc[b], ge[b]], [rc, re_]) < 1e-10, b
