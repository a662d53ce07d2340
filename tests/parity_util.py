"""Shared helpers of the GPU parity tests: run the same seeded input through the CUDA path (C ABI via
paper_2306_04322_b200.pf) and through the CPU oracle (oracle/pfo.c), and compare field by field."""
import numpy as np

from paper_2306_04322_b200 import pf, synth


def make_init(kind, n, n_eta, seed=1, c0=0.5):
    """Returns (c, eta, dx). kind 'A' = the configs' seeded noise (dx = 1), 'B' = Eqs. 4-6 of the paper."""
    if kind == "A":
        c, eta = synth.init_a(n, n_eta, seed, c0=c0)
        return c, eta, (1.0,) * len(n)
    c, eta, dx = synth.init_b(n, n_eta)
    return c, eta, dx


def rel_linf(gpu, ref):
    """Joint relative L-infinity over all fields (SURVEY 8(c.5) 'error norm for parity')."""
    num = max(float(np.max(np.abs(g.astype(np.float64) - r))) if r.size else 0.0 for g, r in zip(gpu, ref))
    den = max(float(np.max(np.abs(r))) if r.size else 0.0 for r in ref)
    return num / den


def run_both(oracle, n, n_eta, init, steps, dt, method="fs", precision="f64", k2_kind=0, seed=1, c0=0.5,
             dx=None, model_kw=None):
    c0_, eta0, dx0 = make_init(init, n, n_eta, seed, c0)
    dx = dx0 if dx is None else dx
    kw = dict(model_kw or {})
    m = oracle.Model(n=n, n_eta=n_eta, dx=dx, dt=dt, k2_kind=k2_kind, **kw)
    ctx = pf.Context(n, n_eta=n_eta, dx=dx, dt=dt, precision=precision, k2_kind=k2_kind, **kw)
    try:
        ctx.set_fields(c0_, eta0)
        if precision == "f32":      # the oracle starts from the same rounded input
            c0_ = c0_.astype(np.float32).astype(np.float64)
            eta0 = eta0.astype(np.float32).astype(np.float64)
        if method == "fs":
            ctx.step_fs(steps)
            rc, reta = m.step_fs(c0_, eta0, steps)
        else:
            ctx.step_fd(steps)
            rc, reta = m.step_fd(c0_, eta0, steps)
        gc, geta = ctx.get_fields()
    finally:
        ctx.close()
    return (gc, geta), (rc, reta)
