"""GPU parity of the cluster-resident small-grid kernel (sgrid_kernels.cu): all steps of a pf_step_fs(n) call in one
launch, state in the distributed shared memory of a thread-block cluster. Square grids up to 64^2 take this path by
default; PF_RESIDENT=0 / PF_SG_CLUSTER=<n> (read at pf_create) select the two-kernel path / the resident path with
clusters of at least n CTAs for every size the kernel serves (32^2 .. 256^2; 256^2 in fp64 with c + 2 eta or more does not fit a
cluster since c^ is carried: those cases check parity on the two-kernel path they fall back to and then skip)."""
import numpy as np
import pytest

from paper_2306_04322_b200 import pf, synth
from parity_util import rel_linf

pytestmark = pytest.mark.gpu


def _run(n, p, calls, dx, dt, c, eta, precision="f64", nbatch=None):
    with pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=precision, nbatch=nbatch) as ctx:
        ctx.set_fields(c, eta)
        l0 = ctx.launch_count()
        for k in calls:
            ctx.step_fs(k)
        launches = ctx.launch_count() - l0
        gc, ge = ctx.get_fields()
    return gc, ge, launches


@pytest.mark.parametrize("nn,p,precision,tol", [(32, 2, "f64", 1e-10), (64, 2, "f64", 1e-10), (64, 4, "f64", 1e-10), (128, 4, "f64", 1e-10),
                                                (128, 0, "f64", 1e-10), (256, 0, "f64", 1e-10), (256, 2, "f64", 1e-10), (256, 4, "f64", 1e-10),
                                                (64, 8, "f64", 1e-10), (64, 2, "f32", 1e-4), (256, 4, "f32", 1e-4)])
def test_resident_steps_match_the_oracle(oracle, monkeypatch, nn, p, precision, tol):
    monkeypatch.delenv("PF_RESIDENT", raising=False)
    monkeypatch.setenv("PF_SG_CLUSTER", "8")             # resident path for every size (default: up to 64^2)
    n = (nn, nn)
    c, eta, dx = synth.init_b(n, p)
    calls = (1, 9, 50)                                   # the state leaves and re-enters shared memory between calls
    gc, ge, launches = _run(n, p, calls, dx, 5e-3, c, eta, precision)
    ci, ei = (c, eta) if precision == "f64" else (c.astype(np.float32).astype(np.float64), eta.astype(np.float32).astype(np.float64))
    rc, re_ = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3).step_fs(ci, ei, sum(calls))
    assert rel_linf([gc, ge], [rc, re_]) < tol
    if launches > 6:                                     # first call of ONE step: x transform, carried spectrum, two kernels;
        # then one launch per call
        pytest.skip(f"grid {nn}^2 with {p + 1} fields does not fit a cluster on this device: two-kernel path ({launches} launches)")


@pytest.mark.parametrize("cs", [1, 2, 4, 8, 16])
def test_every_cluster_size_gives_the_same_fields(oracle, monkeypatch, cs):
    n, p = (64, 64), 2
    c, eta = synth.init_a(n, p, seed=1)
    monkeypatch.setenv("PF_SG_CLUSTER", str(cs))
    gc, ge, launches = _run(n, p, (200,), 1.0, 0.05, c, eta)
    assert launches == 2
    rc, re_ = oracle.Model(n=n, n_eta=p, dx=(1.0, 1.0), dt=0.05).step_fs(c, eta, 200)
    assert rel_linf([gc, ge], [rc, re_]) < 1e-10


def test_resident_and_two_kernel_paths_agree_and_hand_over(oracle, monkeypatch):
    n, p = (128, 128), 2
    c, eta, dx = synth.init_b(n, p)
    monkeypatch.setenv("PF_RESIDENT", "0")
    ac, ae, la = _run(n, p, (40,), dx, 5e-3, c, eta)
    monkeypatch.delenv("PF_RESIDENT")
    monkeypatch.setenv("PF_SG_CLUSTER", "16")
    bc, be, lb = _run(n, p, (40,), dx, 5e-3, c, eta)
    assert la >= 80 and lb == 2
    assert rel_linf([ac, ae], [bc, be]) < 1e-12
    # FD steps between resident calls (real fields <-> z-form hand-off), default policy on a 64^2 grid
    monkeypatch.delenv("PF_SG_CLUSTER")
    n = (64, 64)
    c, eta, dx = synth.init_b(n, p)
    with pf.Context(n, n_eta=p, dx=dx, dt=1e-3) as ctx:
        ctx.set_fields(c, eta)
        l0 = ctx.launch_count()
        ctx.step_fs(5); ctx.step_fd(7); ctx.step_fs(4)
        assert ctx.launch_count() - l0 == 1 + 1 + 1 + 7 + 1 + 1        # set -> z-form, resident, get, 7 FD, set, resident
        gc, ge = ctx.get_fields()
    m = oracle.Model(n=n, n_eta=p, dx=dx, dt=1e-3)
    rc, re_ = m.step_fs(c, eta, 5)
    rc, re_ = m.step_fd(rc, re_, 7)
    rc, re_ = m.step_fs(rc, re_, 4)
    assert rel_linf([gc, ge], [rc, re_]) < 1e-10


def test_resident_batch(oracle, monkeypatch):
    monkeypatch.delenv("PF_RESIDENT", raising=False)
    monkeypatch.delenv("PF_SG_CLUSTER", raising=False)
    n, p, B = (64, 64), 2, 6
    inits = [synth.init_a(n, p, seed=20 + b, c0=0.45 + 0.02 * b) for b in range(B)]
    c0, e0 = np.stack([c for c, _ in inits]), np.stack([e for _, e in inits])
    gc, ge, launches = _run(n, p, (100,), 1.0, 0.05, c0, e0, nbatch=B)
    assert launches == 2
    m = oracle.Model(n=n, n_eta=p, dx=(1.0, 1.0), dt=0.05)
    for b in range(B):
        rc, re_ = m.step_fs(c0[b], e0[b], 100)
        assert rel_linf([gc[b], ge[b]], [rc, re_]) < 1e-10, b
