"""FS-vs-FD crossover on B200 (BASELINE.json configs[4]; paper section 3.2, and Eq. 22).

    python -m paper_2306_04322_b200.crossover [--ndim 2] [--n 1024] [--n-eta 2] [--dx 0.5 1 2] [--out results.json]
    python -m paper_2306_04322_b200.crossover --ndim 3 --n 128 --dx 1      (3D: 128^3 against FS on 256^3)

For every grid spacing dx: the same band-limited seeded field (synth.band_limited: one continuous function, so it
can also be sampled on the 2n x 2n reference grid) is advanced to a fixed physical time T = 240 x dt_FD,lim(dx) with
  * explicit FD at 0.75 x dt_FD,lim   (dt_FD,lim = 2 / (M k~2max (2 rho2 + kappa_c k~2max)), k~2max = 4 d/dx^2: the linear
    stability bound of the 5/7-point scheme in d dimensions; the paper's own FD steps are 0.72-0.79 of it),
  * semi-implicit FS at dt = m x dt_FD,lim, m in {1,2,3,4,5,6,8,10},
  * a reference: FS on the (2n)^2 grid (dx/2) at dt = dt_FD,lim/4,
all through the C ABI (pf.Context). Reported per run: device time (CUDA events), time per step, and the error of
Eq. 22, E_phi = sum (phi - phi_ref)^2 / sum phi_ref^2 for phi = c and phi = sum_i eta_i, on the coarse grid points.
The break-even time-step ratio is (FS time per step) / (FD time per step): FS wins when dt_FS/dt_FD exceeds it
(paper on an RTX 2080 Ti: 5.2-6.5 in 2D; 2.3-4.3 in 3D). Needs a CUDA device and torch (for events only).
"""
from __future__ import annotations

import argparse
import json

import numpy as np


from .metrics import eq22  # noqa: E402  (Eq. 22; one harness definition, checked against the oracle's in tests/)


def run(ctx, steps, torch):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    steps()
    e1.record()
    torch.cuda.synchronize()
    return e0.elapsed_time(e1)


def main():
    import torch
    from . import pf, synth

    ap = argparse.ArgumentParser()
    ap.add_argument("--ndim", type=int, default=2, choices=[2, 3])
    ap.add_argument("--n", type=int, default=1024)
    ap.add_argument("--n-eta", type=int, default=2)
    ap.add_argument("--dx", type=float, nargs="+", default=[0.5, 1.0, 2.0])
    ap.add_argument("--seed", type=int, default=5)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    M, kc, rho2 = 5.0, 3.0, 2.0
    n, p, nd = a.n, a.n_eta, a.ndim
    shape, shape2, half = (n,) * nd, (2 * n,) * nd, (slice(None, None, 2),) * nd
    stream = torch.cuda.current_stream().cuda_stream
    results = []
    for dx in a.dx:
        L = n * dx
        k2max = 4.0 * nd / dx ** 2
        lim = 2.0 / (M * k2max * (2 * rho2 + kc * k2max))
        T = 240 * lim
        c0, e0 = synth.band_limited(shape, p, a.seed, L, kmax=8)
        cr, er = synth.band_limited(shape2, p, a.seed, L, kmax=8)
        with pf.Context(shape2, n_eta=p, dx=dx / 2, dt=lim / 4, stream=stream) as ref:
            ref.set_fields(cr, er)
            ms_ref = run(ref, lambda: ref.step_fs(960), torch)
            rc, re_ = ref.get_fields()
        rc, rs = rc[half], re_.sum(0)[half]
        rows = []
        with pf.Context(shape, n_eta=p, dx=dx, dt=0.75 * lim, stream=stream) as fd:
            fd.set_fields(c0, e0)
            ms = run(fd, lambda: fd.step_fd(320), torch)
            gc, ge = fd.get_fields()
            rows.append({"method": "FD", "dt_over_lim": 0.75, "dt": 0.75 * lim, "steps": 320, "ms": ms, "ms_per_step": ms / 320,
                         "E_c": eq22(gc, rc), "E_eta": eq22(ge.sum(0), rs), "finite": bool(np.isfinite(gc).all())})
        for m in (1, 2, 3, 4, 5, 6, 8, 10):
            with pf.Context(shape, n_eta=p, dx=dx, dt=m * lim, stream=stream) as fs:
                fs.set_fields(c0, e0)
                fs.step_fs(2)                                  # graph capture + warm-up, then restart from the same field
                fs.set_fields(c0, e0)
                ms = run(fs, lambda: fs.step_fs(240 // m), torch)
                gc, ge = fs.get_fields()
                fin = bool(np.isfinite(gc).all() and np.isfinite(ge).all())
                rows.append({"method": "FS", "dt_over_lim": m, "dt": m * lim, "steps": 240 // m, "ms": ms,
                             "ms_per_step": ms / (240 // m), "E_c": eq22(gc, rc) if fin else None,
                             "E_eta": eq22(ge.sum(0), rs) if fin else None, "finite": fin})
        fd_step = rows[0]["ms_per_step"]
        fs_step = float(np.median([r["ms_per_step"] for r in rows[1:]]))
        results.append({"dx": dx, "ndim": nd, "n": n, "n_eta": p, "T": T, "dt_fd_lim": lim, "reference": {"grid": 2 * n, "dt": lim / 4, "steps": 960, "ms": ms_ref},
                        "fs_ms_per_step": fs_step, "fd_ms_per_step": fd_step,
                        "break_even_dt_ratio": fs_step / fd_step, "runs": rows})
        print(f"dx={dx}: FS {fs_step * 1e3:.1f} us/step, FD {fd_step * 1e3:.1f} us/step, break-even dt_FS/dt_FD = {fs_step / fd_step:.2f}", flush=True)
        for r in rows:
            print(f"   {r['method']} dt={r['dt']:.3e} ({r['dt_over_lim']} x lim) steps={r['steps']:4d} time={r['ms']:.2f} ms "
                  f"E_c={r['E_c']} E_eta={r['E_eta']}", flush=True)
    if a.out:
        with open(a.out, "w") as fh:
            json.dump(results, fh, indent=1)


if __name__ == "__main__":
    main()
