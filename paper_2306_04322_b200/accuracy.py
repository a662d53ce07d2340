"""The paper's accuracy study on B200 (section 3.3, Fig. 6, Eq. 22).

    python -m paper_2306_04322_b200.accuracy [--grids 128 256 512 1024] [--ref-grid 2048] [--ref-dt 1e-4]
                                             [--t-end 100] [--fd-max-steps 5e6] [--out results.json]

Benchmark of the paper: l = 200, c + 4 order parameters, initial condition Eqs. 4-5 evolved from
t = 1 to t = 100. The paper first evolves the (non-periodic) Eq. 5 field from t = 0 to t = 1 with FD "on a fine spatial
grid and small time step" without giving either; the stand-in here is the semi-implicit Fourier-spectral
step on the reference grid at the reference time step. The t = 1 field is then sampled on every coarser grid (the grids
nest) and advanced to t_end with
  * FS (Eq. 16), FS-FD O(dl^2) (Eq. 17) and FS-FD O(dl^4) (Eq. 18) at dt = 5e-3 and 1e-3 (Table 1),
  * explicit FD at 0.75 x its linear stability limit (the paper's own steps are 0.72-0.79 of it), capped at 2e-3 where the
    Allen-Cahn reaction term is the limit; skipped where it would need more than --fd-max-steps steps,
and compared with the reference (FS on the reference grid at the reference dt) through Eq. 22,
E_phi = sum (phi - phi_ref)^2 / sum phi_ref^2 with phi = c and phi = sum_i eta_i, printed in percent as in the paper.
The paper prints two values to compare with: E_c = 2.03 %, E_eta = 7.74 % for FD and FS-FD O(dl^2) on 128^2.
Everything runs through the C ABI (pf.Context); numpy only samples and compares.
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np


from .metrics import eq22_percent  # noqa: E402  (Eq. 22; one harness definition, checked against the oracle's in tests/)


def advance(pf, n, p, dx, dt, t_span, c, eta, method="fs", k2_kind=0):
    """Returns (c, eta, steps, seconds) after advancing by t_span with a whole number of steps of size ~dt."""
    steps = max(1, int(round(t_span / dt)))
    dt = t_span / steps
    with pf.Context((n, n), n_eta=p, dx=(dx, dx), dt=dt, k2_kind=k2_kind) as ctx:
        ctx.set_fields(c, eta)
        t0 = time.perf_counter()
        done = 0
        while done < steps:                      # chunks keep the launch queue short
            k = min(20000, steps - done)
            (ctx.step_fs if method == "fs" else ctx.step_fd)(k)
            done += k
        out_c, out_eta = ctx.get_fields()
        return out_c, out_eta, steps, time.perf_counter() - t0


def restrict(u, r, how):
    """A periodic fine-grid field u[..., ny, nx] on the grid that keeps every r-th point (the grids nest). Harness code:
    PAPER.md:65 does not say how the t = 1 field reaches the coarse grids.
      sample    point sampling u[::r, ::r] (aliases what the coarse grid cannot carry);
      spectral  Fourier truncation: the modes |k| < n/2 of the fine field, evaluated on the coarse points;
      average   mean over the coarse cell centred on each coarse point (trapezoid weights, periodic)."""
    if r == 1 or how == "sample":
        return np.ascontiguousarray(u[..., ::r, ::r])
    ny, nx = u.shape[-2:]
    my, mx = ny // r, nx // r
    if how == "spectral":
        U = np.fft.fft2(u)
        ky, kx = np.fft.fftfreq(ny, 1.0 / ny), np.fft.fftfreq(nx, 1.0 / nx)
        keep = (np.abs(ky)[:, None] < my / 2) & (np.abs(kx)[None, :] < mx / 2)
        iy, ix = np.nonzero(np.abs(ky) < my / 2)[0], np.nonzero(np.abs(kx) < mx / 2)[0]
        V = np.zeros(u.shape[:-2] + (my, mx), dtype=complex)
        V[..., (ky[iy].astype(int) % my)[:, None], (kx[ix].astype(int) % mx)[None, :]] = (U * keep)[..., iy[:, None], ix[None, :]]
        return np.ascontiguousarray(np.fft.ifft2(V).real / (r * r))
    if how == "average":
        w = np.ones(r + 1)
        w[0] = w[-1] = 0.5
        w /= w.sum()
        out = u
        for axis in (-2, -1):
            out = sum(wk * np.roll(out, r // 2 - k, axis=axis) for k, wk in enumerate(w))
        return np.ascontiguousarray(out[..., ::r, ::r])
    raise ValueError(how)


def main():
    from . import pf, synth

    ap = argparse.ArgumentParser()
    ap.add_argument("--grids", type=int, nargs="+", default=[128, 256, 512, 1024])
    ap.add_argument("--ref-grid", type=int, default=2048)
    ap.add_argument("--ref-dt", type=float, default=1e-4)
    ap.add_argument("--t-end", type=float, default=100.0)
    ap.add_argument("--fd-max-steps", type=float, default=5e6)
    ap.add_argument("--pre", default="fs", choices=["fs", "fd"],
                    help="pre-evolution t = 0 -> 1 on the reference grid: the FS step at --ref-dt (stand-in) or, as the paper "
                         "describes it (PAPER.md:65), explicit FD at 0.75 x its stability limit on that grid (sensitivity run)")
    ap.add_argument("--restrict", nargs="+", default=["sample"], choices=["sample", "spectral", "average"],
                    help="how the t = 1 field of the reference grid is put on the coarse grids (PAPER.md:65 is silent); the "
                         "coarse results are always compared with the reference at the coarse points")
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    p, length = 4, 200.0
    M, kc, rho2 = 5.0, 3.0, 2.0
    nr = a.ref_grid
    c0, eta0, dx0 = synth.init_b((nr, nr), p)
    assert abs(dx0[0] - length / nr) < 1e-12
    # stand-in for the paper's pre-evolution, then the reference run
    if a.pre == "fd":
        k2r = 8.0 / (length / nr) ** 2
        pre_dt = min(0.75 * 2.0 / (M * k2r * (2 * rho2 + kc * k2r)), 2e-3)
    else:
        pre_dt = a.ref_dt
    c1, eta1, s, sec = advance(pf, nr, p, length / nr, pre_dt, 1.0, c0, eta0, a.pre)
    print(f"pre-evolution t=0..1 on {nr}^2, dt={pre_dt:g}: {s} {a.pre.upper()} steps in {sec:.1f} s", flush=True)
    cr, er, s, sec = advance(pf, nr, p, length / nr, a.ref_dt, a.t_end - 1.0, c1, eta1)
    print(f"reference     t=1..{a.t_end:g} on {nr}^2, dt={a.ref_dt:g}: {s} FS steps in {sec:.1f} s "
          f"(finite: {bool(np.isfinite(cr).all())})", flush=True)
    rows = []
    print(f"{'grid':>6} {'method':>14} {'dt':>10} {'steps':>9} {'seconds':>8} {'E_c %':>11} {'E_eta %':>11}")
    for how, n in [(h, g) for h in a.restrict for g in a.grids]:
        if len(a.restrict) > 1 or how != "sample":
            print(f"# t = 1 field restricted to {n}^2 by: {how}", flush=True)
        r = nr // n
        dx = length / n
        ci, ei = restrict(c1, r, how), restrict(eta1, r, how)
        rc, rs = cr[::r, ::r], er.sum(0)[::r, ::r]
        k2max = 8.0 / dx ** 2
        dt_fd = min(0.75 * 2.0 / (M * k2max * (2 * rho2 + kc * k2max)), 2e-3)
        runs = [("FS", "fs", 0, 5e-3), ("FS-FD O(dl^2)", "fs", 1, 5e-3), ("FS-FD O(dl^4)", "fs", 2, 5e-3),
                ("FS", "fs", 0, 1e-3), ("FS-FD O(dl^2)", "fs", 1, 1e-3), ("FS-FD O(dl^4)", "fs", 2, 1e-3),
                ("FD", "fd", 0, dt_fd)]
        for name, method, kind, dt in runs:
            if method == "fd" and (a.t_end - 1.0) / dt > a.fd_max_steps:
                print(f"{n:>6} {name:>14} {dt:>10.3e}   skipped: {(a.t_end - 1.0) / dt:.2e} steps", flush=True)
                continue
            gc, ge, steps, sec = advance(pf, n, p, dx, dt, a.t_end - 1.0, ci, ei, method, kind)
            fin = bool(np.isfinite(gc).all() and np.isfinite(ge).all())
            row = {"grid": n, "restrict": how, "method": name, "dt": dt, "steps": steps, "seconds": sec, "finite": fin,
                   "E_c_percent": eq22_percent(gc, rc) if fin else None,
                   "E_eta_percent": eq22_percent(ge.sum(0), rs) if fin else None}
            rows.append(row)
            ec = f"{row['E_c_percent']:.4e}" if fin else "non-finite"
            ee = f"{row['E_eta_percent']:.4e}" if fin else "non-finite"
            print(f"{n:>6} {name:>14} {dt:>10.3e} {steps:>9d} {sec:>8.2f} {ec:>11} {ee:>11}", flush=True)
    if a.out:
        with open(a.out, "w") as fh:
            json.dump({"ref_grid": nr, "ref_dt": a.ref_dt, "pre": a.pre, "pre_dt": pre_dt, "t_end": a.t_end, "runs": rows}, fh, indent=1)


if __name__ == "__main__":
    main()
