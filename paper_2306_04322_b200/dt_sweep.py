"""Time-step sweep of BASELINE.json configs[1] on B200 (SURVEY 8(d) run C2; the paper's trial-and-error search for the largest stable
time step).

    python -m paper_2306_04322_b200.dt_sweep [--n 512] [--n-eta 4] [--steps 2000] [--out results.json]

2D n x n grid, dx = 1, c + 4 eta_i, fp64, seeded noise (c0 = 0.4, seed 2; synth.init_a). For every dt in
{0.01, 0.02, 0.05, 0.1, 0.15, 0.19, 0.2, 0.25, 0.5, 1.0}: `steps` semi-implicit Fourier-spectral steps through the C ABI, then
  * whether the fields are still finite (and, if not, the first checkpoint of 100 steps at which they were not),
  * mean of c (conserved by the method: the k = 0 mode of Eq. 14 is untouched), max |eta|, device time.
With the paper's coefficients the explicit reaction term of the Allen-Cahn equation makes eta = 0 linearly unstable for
dt > 2 / (2 w L) = 0.2: "non-finite" beyond that is the expected outcome, recorded, not a failure.
The explicit FD path runs the same physical time T = steps * dt (capped at --fd-max-steps) at 0.75 x its linear stability limit
1.786e-3 (dx = 1) for the cost comparison. Needs a CUDA device; numpy only inspects the fields.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

DTS = (0.01, 0.02, 0.05, 0.1, 0.15, 0.19, 0.2, 0.25, 0.5, 1.0)


def main():
    from . import pf, synth

    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=512)
    ap.add_argument("--n-eta", type=int, default=4)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--fd-max-steps", type=float, default=2e5)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    n, p = (a.n, a.n), a.n_eta
    c0, e0 = synth.init_a(n, p, seed=2, c0=0.4)
    fd_dt = 0.75 * 2.0 / (5.0 * 8.0 * (4.0 + 3.0 * 8.0))
    rows = []
    print(f"{'dt':>6} {'outcome':>22} {'mean c':>20} {'max|eta|':>12} {'FS s':>8} {'FD steps':>9} {'FD s':>8}")
    for dt in DTS:
        with pf.Context(n, n_eta=p, dx=1.0, dt=dt) as ctx:
            ctx.set_fields(c0, e0)
            t0 = time.perf_counter()
            first_bad = None
            done = 0
            while done < a.steps:
                k = min(100, a.steps - done)
                ctx.step_fs(k)
                done += k
                c, eta = ctx.get_fields()
                if first_bad is None and not (np.isfinite(c).all() and np.isfinite(eta).all()):
                    first_bad = done
            sec = time.perf_counter() - t0
        finite = first_bad is None
        fd_steps = int(min(a.fd_max_steps, round(a.steps * dt / fd_dt)))
        with pf.Context(n, n_eta=p, dx=1.0, dt=fd_dt) as fd:
            fd.set_fields(c0, e0)
            t0 = time.perf_counter()
            fd.step_fd(fd_steps)
            fc, fe = fd.get_fields()
            fsec = time.perf_counter() - t0
        row = {"dt": dt, "steps": a.steps, "finite": finite, "first_non_finite_checkpoint": first_bad,
               "mean_c": float(np.mean(c)) if finite else None, "max_abs_eta": float(np.max(np.abs(eta))) if finite and p else None,
               "fs_seconds_incl_checkpoint_readouts": sec, "fd_dt": fd_dt, "fd_steps": fd_steps,
               "fd_covers_T": bool(fd_steps * fd_dt >= a.steps * dt * 0.999), "fd_seconds": fsec,
               "fd_finite": bool(np.isfinite(fc).all() and np.isfinite(fe).all())}
        rows.append(row)
        outcome = "finite" if finite else f"non-finite by step {first_bad}"
        mc = f"{row['mean_c']:.15f}" if finite else "-"
        me = f"{row['max_abs_eta']:.3e}" if finite and p else "-"
        print(f"{dt:>6g} {outcome:>22} {mc:>20} {me:>12} {sec:>8.2f} {fd_steps:>9d} {fsec:>8.2f}", flush=True)
    if a.out:
        with open(a.out, "w") as fh:
            json.dump({"n": a.n, "n_eta": p, "steps": a.steps, "runs": rows}, fh, indent=1)


if __name__ == "__main__":
    main()
