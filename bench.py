#!/usr/bin/env python
"""bench.py -- throughput of the Fourier-spectral (FS) step of arXiv 2306.04322 on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 1024sq|256cube|2048sq|2048sq_f32|512sq|256sq|64sq]
                    [--impl ours|reference]

A "step" is one FS time step (all kernels of SURVEY 8(a): x-pass with the nonlinear evaluation, strided passes with
the spectral update) of one simulation. At the L2-resident sizes the timed loop cycles through R independent
replicas of the simulation so that consecutive steps never find their inputs in L2 (timing rule "inputs larger than
L2"); the single-simulation (L2-resident) figure is reported next to it. Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOADS = {
    # name: (n, n_eta, precision, init, dt, description)
    "1024sq": ((1024, 1024), 2, "f64", "B", 5e-3, "2D 1024x1024, c + 2 eta, fp64 (the metric's 2D size; configs[4] grid)"),
    "256cube": ((256, 256, 256), 2, "f64", "B", 5e-3, "3D 256^3, c + 2 eta, fp64 (the metric's 3D size; configs[3] grid)"),
    "2048sq": ((2048, 2048), 4, "f64", "B", 5e-3, "2D 2048x2048, c + 4 eta, fp64 (configs[2])"),
    "2048sq_f32": ((2048, 2048), 4, "f32", "B", 5e-3, "2D 2048x2048, c + 4 eta, fp32 (configs[2])"),
    "512sq": ((512, 512), 4, "f64", "B", 5e-3, "2D 512x512, c + 4 eta, fp64 (configs[1] grid)"),
    "256sq": ((256, 256), 4, "f64", "B", 5e-3, "2D 256x256, c + 4 eta, fp64 (paper Table 1 grid; its FS run of PAPER.md:286)"),
    "64sq": ((64, 64), 2, "f64", "A", 0.05, "2D 64x64, c + 2 eta, fp64 (configs[0])"),
}
DEFAULT_STEPS = {"1024sq": 20000, "256cube": 1500, "2048sq": 3000, "2048sq_f32": 5000, "512sq": 40000, "256sq": 60000, "64sq": 100000}
L2_BYTES = 126e6
PROF_REPEAT = 8
METRIC = "FS steps/s (Gpoint-updates/s and achieved HBM GB/s alongside)"


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def make_fields(wl):
    from paper_2306_04322_b200 import synth
    n, p, prec, init, dt, _ = WORKLOADS[wl]
    if init == "A":
        c, eta = synth.init_a(n, p, seed=1)
        dx = (1.0,) * len(n)
    else:
        c, eta, dx = synth.init_b(n, p)
    return c, eta, dx


def bytes_model(n, p, w):
    """Algorithmic bytes per FS step and per kernel launch. R = bytes of one real field (= one
    z-form array), S = bytes of one half spectrum, F = p + 1.
    survey: SURVEY 8(d): one read + one write of every field per 1-D pass + the u^ read of the update, attributed to the
            kernel that performs the pass: x kernel (a6 + a1 + a2) 2F(R+S); 2D y kernel (a4 + a5) 5FS;
            3D y-forward (a3) 2FS, z kernel (a4 + a5) 5FS, y-inverse (a5) 2FS.  Sum: 2D F(2R+7S), 3D F(2R+11S).
    design: what the kernels of this design have to move (z-form state, cross-step fusion, g^ parked in L2)."""
    F = p + 1
    N = int(np.prod(n))
    R = N * w
    S = (n[0] // 2 + 1) * (N // n[0]) * 2 * w
    if len(n) == 2:
        survey = {"row_c2r_nonlinear_r2c": 2 * F * (R + S), "col_y_fft_update_ifft": 5 * F * S}
        design = {"row_c2r_nonlinear_r2c": 2 * F * R, "col_y_fft_update_ifft": (3 + 2 * p) * R}
    else:
        P2 = ((n[0] // 2 + 1 + 15) // 16) * 16
        Sp = P2 * n[1] * n[2] * 2 * w          # one padded half-spectrum array as stored
        survey = {"row_c2r_nonlinear_r2c": 2 * F * (R + S), "col_y_fwd": 2 * F * S, "col_z_fft_update_ifft": 5 * F * S,
                  "col_y_inv": 2 * F * S}
        design = {"row_c2r_nonlinear_r2c": 2 * F * R, "col_y_fwd": F * (R + Sp),
                  "col_z_fft_update_ifft": (3 + 2 * p) * Sp, "col_y_inv": F * (Sp + R)}
    return survey, design


# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the ncu --set full captures
# summarised under profiles/ (key: workload -> kernel -> bytes)
NCU_TRAFFIC = {
    # profiles/r1_ncu_full_1024sq.md (the L2 keeps part of what the previous kernel wrote: traffic < algorithmic bytes)
    "1024sq": {"row_c2r_nonlinear_r2c": 25221120 + 512, "col_y_fft_update_ifft": 33624320 + 27136},
    # profiles/r1_ncu_full_256cube.md
    "256cube": {"row_c2r_nonlinear_r2c": 402713856 + 353691904, "col_y_fwd": 408681216 + 364982528,
                "col_z_fft_update_ifft": 604053248 + 545553920, "col_y_inv": 427836160 + 358318336},
}


class ClockSampler:
    FIELDS = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.tmp = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.tmp, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.tmp.flush()
        rows = [r.split(",") for r in open(self.tmp.name).read().strip().splitlines() if r.count(",") >= 6]
        os.unlink(self.tmp.name)
        if not rows:
            return out
        try:
            sm = sorted(float(r[0]) for r in rows)
            out["sm_mhz"] = sm[len(sm) // 2]
            out["sm_max_mhz"] = float(rows[0][1])
            out["power_w_max"] = max(float(r[2]) for r in rows)
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            out["reasons"] = [nm for i, nm in enumerate(names) if any(r[3 + i].strip() == "Active" for r in rows)]
            out["samples"] = len(rows)
        except Exception:
            pass
        return out


def run_reference(args):
    """The oracle (oracle/pfo.c, as it stands) on the host cores: the base contract's reference arm for this tier."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import pfo
    pfo.build()
    n, p, prec, init, dt, desc = WORKLOADS[args.workload]
    c, eta, dx = make_fields(args.workload)
    m = pfo.Model(n=n, n_eta=p, dx=dx, dt=dt)
    budget = float(os.environ.get("PF_REF_BUDGET_S", "150"))
    t_all = time.time()
    for _ in range(min(args.warmup, 1)):
        c, eta = m.step_fs(c, eta, 1)
    t0 = time.time()
    done = 0
    while done < args.steps and (done == 0 or (time.time() - t_all) + (time.time() - t0) / done < budget):
        c, eta = m.step_fs(c, eta, 1)
        done += 1
    el = time.time() - t0
    val = done / el
    N = int(np.prod(n))
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "steps/s", "n_gpus": args.gpus, "steps": done,
            "warmup": min(args.warmup, 1), "ms_per_step": 1e3 * el / done, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "init": init, "dt": dt, "note": "CPU oracle; steps bounded by a time budget"},
            "gpoint_updates_per_s": val * N / 1e9,
            "cpu_baseline": {"value": val, "unit": "steps/s", "cores": pfo.num_threads(), "kind": "oracle",
                             "sample": f"{done} full FS steps of the same workload"},
            "e2e": {"value": val, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def cufft_side_reference(torch, n, p, prec, dx, dt, c0, eta0, stream, steps=20):
    """Side reference only (north_star): the same FS step assembled from cuFFT (torch.fft.rfftn/irfftn) and elementwise
    torch ops, timed in the same process. Not part of the product path and not compared for parity here."""
    dev = torch.device("cuda")
    tdt = torch.float64 if prec == "f64" else torch.float32
    M_, L_, kc, ke, rho2, ca, cb, w_, al = 5.0, 5.0, 3.0, 3.0, 2.0, 0.3, 0.7, 1.0, 5.0
    nd = len(n)
    with torch.cuda.stream(stream):
        c = torch.as_tensor(c0, dtype=tdt, device=dev)
        eta = torch.as_tensor(eta0, dtype=tdt, device=dev)
        k2 = None
        for d in range(nd):                       # array axis nd-1-d has length n[d] (x fastest)
            ax = nd - 1 - d
            freq = torch.fft.rfftfreq(n[d], d=dx[d]) if ax == nd - 1 else torch.fft.fftfreq(n[d], d=dx[d])
            kk = (2 * np.pi * freq.to(tdt).to(dev)) ** 2
            shape = [1] * nd
            shape[ax] = kk.numel()
            k2 = kk.reshape(shape) if k2 is None else k2 + kk.reshape(shape)
        dc = 1.0 / (1.0 + dt * M_ * kc * k2 * k2)
        de = 1.0 / (1.0 + dt * L_ * ke * k2)
        ch = torch.fft.rfftn(c)
        eh = torch.fft.rfftn(eta, dim=tuple(range(1, nd + 1)))
        dims = tuple(range(-nd, 0))

        def step(ch, eh):
            c = torch.fft.irfftn(ch, s=c0.shape, dim=dims)
            eta = torch.fft.irfftn(eh, s=c0.shape, dim=dims)
            h = (eta ** 3 * (6 * eta ** 2 - 15 * eta + 10)).sum(0)
            s2 = (eta ** 2).sum(0)
            g = 2 * rho2 * ((c - ca) * (1 - h) - (cb - c) * h)
            fba = rho2 * ((cb - c) ** 2 - (c - ca) ** 2)
            hh = fba * 30 * eta ** 2 * (1 - eta) ** 2 + w_ * (2 * eta * (1 - eta) * (1 - 2 * eta) + 4 * al * eta * (s2 - eta ** 2))
            gh = torch.fft.rfftn(g, dim=dims)
            hh = torch.fft.rfftn(hh, dim=dims)
            return (ch - dt * M_ * k2 * gh) * dc, (eh - dt * L_ * hh) * de

        for _ in range(3):
            ch, eh = step(ch, eh)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(steps):
            ch, eh = step(ch, eh)
        e1.record(stream)
        torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    return {"value": 1e3 / ms, "unit": "steps/s", "ms_per_step": ms, "steps": steps,
            "what": "torch.fft.rfftn/irfftn (cuFFT) + elementwise torch ops, single simulation, same workload"}


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2306_04322_b200 import pf, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pf.lib()                                   # fails loudly if libpf.so is missing

    n, p, prec, init, dt, desc = WORKLOADS[args.workload]
    w = 8 if prec == "f64" else 4
    F, N = p + 1, int(np.prod(n))
    R = N * w
    c0, eta0, dx = make_fields(args.workload)
    # replicas only: every rank advances its own independent simulations
    state_bytes = (F + 1) * R if len(n) == 2 else 3 * F * R
    reps = 1 if state_bytes > 2 * L2_BYTES else int(np.ceil(2.5 * L2_BYTES / state_bytes))
    stream = torch.cuda.Stream()
    ctxs = [pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=prec, stream=stream.cuda_stream) for _ in range(reps)]
    for i, cx in enumerate(ctxs):
        cx.set_fields(replicas.perturb(c0, rank, i, reps), eta0)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def run_steps(k, which):
        # one step of each replica in turn; a call is asynchronous (graph replay of one step)
        for s in range(k):
            which[s % len(which)].step_fs(1)

    def timed(k, which):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        run_steps(k, which)
        e1.record(stream)
        barrier()
        return replicas.max_over_ranks(e0.elapsed_time(e1), device="cuda")

    K, W = args.steps, max(args.warmup, 3)
    run_steps(W * len(ctxs), ctxs)
    sampler = ClockSampler(torch.cuda.current_device()) if rank == 0 else None
    l0 = sum(cx.launch_count() for cx in ctxs)
    ms = timed(K, ctxs)
    launches = sum(cx.launch_count() for cx in ctxs) - l0
    clocks = sampler.stop() if sampler else {}
    value = replicas.job_throughput(K, ms, world)

    # single simulation, state resident in L2 where it fits (reported, not the headline)
    ms_res = timed(K, ctxs[:1])
    resident = replicas.job_throughput(K, ms_res, world)

    # per-kernel device times: CUDA events on the context's stream, recorded by the library around PROF_REPEAT back-to-back
    # launches of each kernel (pf_set_profiling), same replica cycling as the timed region. Timing only: the replicas'
    # fields are not a trajectory afterwards (the e2e leg below sets fields again).
    for cx in ctxs:
        cx.set_profiling(PROF_REPEAT)
    acc, cnt = {}, 0
    for s in range(min(K, 20 * len(ctxs))):
        cx = ctxs[s % len(ctxs)]
        cx.step_fs(1)
        for name, t in cx.fs_kernel_times():
            acc[name] = acc.get(name, 0.0) + t
        cnt += 1
    for cx in ctxs:
        cx.set_profiling(0)
    kms = {k: v / cnt for k, v in acc.items()}
    ksurvey, kdesign = bytes_model(n, p, w)
    survey_bytes, design_bytes = sum(ksurvey.values()), sum(kdesign.values())
    peak, peak_src = peaks()
    dom = max(kms, key=kms.get)
    achieved = ksurvey[dom] / (kms[dom] * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": NCU_TRAFFIC.get(args.workload, {}).get(dom), "peak_source": peak_src,
                "algorithmic_bytes_per_launch": ksurvey[dom],
                "algorithmic_bytes_note": "SURVEY 8(d) per-pass bytes of the passes this kernel fuses (see DESIGN.md section 5)",
                "design_bytes_per_launch": kdesign[dom],
                "achieved_vs_design_bytes": kdesign[dom] / (kms[dom] * 1e-3) / 1e9,
                "kernel_ms": kms[dom], "kernels_ms": kms, "kernel_timing": f"events around {PROF_REPEAT} back-to-back launches of one kernel on one replica (L2 warm after the first; the step time above is the cold-L2 figure)",
                "kernel_share_of_step": kms[dom] / sum(kms.values())}
    step_ms = ms / K
    step_roofline = {"bytes_per_step_survey_8d": survey_bytes, "bytes_per_step_this_design": design_bytes,
                     "achieved_vs_survey_bytes_gbs": survey_bytes / (step_ms * 1e-3) / 1e9,
                     "frac_vs_survey_bytes": survey_bytes / (step_ms * 1e-3) / 1e9 / peak,
                     "achieved_vs_design_bytes_gbs": design_bytes / (step_ms * 1e-3) / 1e9,
                     "frac_vs_design_bytes": design_bytes / (step_ms * 1e-3) / 1e9 / peak}

    # end to end through the C ABI with HOST buffers: set (H2D) + 1 step + get (D2H), pinned host memory
    tdt = torch.float64 if prec == "f64" else torch.float32
    hc = torch.empty(tuple(reversed(n)), dtype=tdt).pin_memory()
    he = torch.empty((p,) + tuple(reversed(n)), dtype=tdt).pin_memory()
    hc.numpy()[...] = c0
    he.numpy()[...] = eta0
    L = pf.lib()
    cx = ctxs[0]
    ke = max(3, min(K, 20))
    def e2e_step():
        L.pf_set_fields(cx._h, hc.data_ptr(), he.data_ptr(), pf.PF_HOST)
        L.pf_step_fs(cx._h, 1)
        L.pf_get_fields(cx._h, hc.data_ptr(), he.data_ptr(), pf.PF_HOST)
    for _ in range(2):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(ke):
        e2e_step()
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    e2e_s = replicas.max_over_ranks(e2e_s, device="cuda")
    serial_e2e = world * ke / e2e_s
    # the same loop for two independent simulations from two host threads (own context, stream and pinned buffers
    # each): the H2D copy of one overlaps the D2H copy of the other (PCIe is full duplex)
    import threading
    cxs2 = [pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=prec) for _ in range(2)]
    bufs2 = []
    for _ in range(2):
        bc = torch.empty(tuple(reversed(n)), dtype=tdt).pin_memory()
        be = torch.empty((p,) + tuple(reversed(n)), dtype=tdt).pin_memory()
        bc.numpy()[...] = c0
        be.numpy()[...] = eta0
        bufs2.append((bc, be))

    def worker(i, steps):
        h, (bc, be) = cxs2[i]._h, bufs2[i]
        for _ in range(steps):
            L.pf_set_fields(h, bc.data_ptr(), be.data_ptr(), pf.PF_HOST)
            L.pf_step_fs(h, 1)
            L.pf_get_fields(h, bc.data_ptr(), be.data_ptr(), pf.PF_HOST)

    for i in range(2):
        worker(i, 2)
    barrier()
    t0 = time.perf_counter()
    th = [threading.Thread(target=worker, args=(i, ke)) for i in range(2)]
    for t in th:
        t.start()
    for t in th:
        t.join()
    torch.cuda.synchronize()
    e2e2_s = replicas.max_over_ranks(time.perf_counter() - t0, device="cuda")
    for cx2 in cxs2:
        cx2.close()
    e2e = {"value": world * 2 * ke / e2e2_s, "unit": "steps/s", "h2d_bytes_per_step": F * R, "d2h_bytes_per_step": F * R,
           "steps": 2 * ke, "contexts": 2, "one_context_value": serial_e2e,
           "note": "pf_set_fields(HOST) + pf_step_fs(1) + pf_get_fields(HOST) per step, pinned host buffers; two independent "
                   "simulations driven from two host threads so that uploads and downloads overlap; one_context_value = the same loop for one simulation"}

    line = {"metric": METRIC, "value": value, "unit": "steps/s", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": prec,
            "data": "synthetic",
            "config": {"workload": desc, "init": "Eqs. 4-6 benchmark field (synth.init_b)" if init == "B" else "seeded noise (synth.init_a)",
                       "dt": dt, "replicas_per_gpu": reps, "parallelism": "independent replicas per GPU, no collective",
                       "l2": (f"timed loop cycles {reps} independent replicas ({reps * state_bytes / 1e6:.0f} MB of state > 126 MB L2)"
                              if reps > 1 else f"state {state_bytes / 1e6:.0f} MB per step exceeds the 126 MB L2")},
            "gpoint_updates_per_s": value * N / 1e9,
            "field_point_updates_per_s_G": value * N * F / 1e9,
            "l2_resident_single_simulation": {"value": resident, "unit": "steps/s", "gpoint_updates_per_s": resident * N / 1e9},
            "roofline": roofline, "step_roofline": step_roofline, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks}

    # independent simulations advanced concurrently on two streams (the paper's sweeps are independent runs, DESIGN.md
    # "Multi-GPU"): kernels of different simulations fill each other's tails. Reported beside the headline, which stays
    # the one-stream figure. Timed with events on `stream`, which waits for the second stream's last step.
    concurrent = None
    if len(ctxs) >= 2:
        stream2 = torch.cuda.Stream()
        half = max(1, len(ctxs) // 2)
        ctxs2 = [pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=prec, stream=stream2.cuda_stream) for _ in range(half)]
        for i, cx in enumerate(ctxs2):
            cx.set_fields(replicas.perturb(c0, rank, i, half), eta0)
            cx.step_fs(W)
        grpa = ctxs[:half]
        for i, cx in enumerate(grpa):          # the profiling leg left these replicas without a valid trajectory
            cx.set_fields(replicas.perturb(c0, rank, i, reps), eta0)
            cx.step_fs(W)
        barrier()
        c0e, c1e, c2e = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        c0e.record(stream)
        stream2.wait_event(c0e)
        for s in range(K // 2):
            grpa[s % half].step_fs(1)
            ctxs2[s % half].step_fs(1)
        c2e.record(stream2)
        stream.wait_event(c2e)
        c1e.record(stream)
        barrier()
        cms = replicas.max_over_ranks(c0e.elapsed_time(c1e), device="cuda")
        concurrent = {"streams": 2, "value": replicas.job_throughput(2 * (K // 2), cms, world), "unit": "steps/s",
                      "us_per_step": 1e3 * cms / (2 * (K // 2)),
                      "note": "two independent simulations in flight at a time, one per stream; every simulation still advances step by step"}
        for cx in ctxs2:
            cx.close()

    # comparison path: explicit FD steps of one simulation of the same grid, device-timed
    fd = pf.Context(n, n_eta=p, dx=dx, dt=1e-6, precision=prec, stream=stream.cuda_stream)
    fd.set_fields(c0, eta0)
    kfd = max(20, min(2000, K // 4))
    fd.step_fd(20)
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    f0.record(stream)
    fd.step_fd(kfd)
    f1.record(stream)
    barrier()
    fd_ms = f0.elapsed_time(f1) / kfd
    fd.close()
    fd_bytes = 2 * F * R                      # fused kernels: every field read once and written once per step
    if concurrent:
        line["concurrent_replicas"] = concurrent
    line["fd_comparison_path"] = {"value": 1e3 / fd_ms, "unit": "steps/s", "us_per_step": 1e3 * fd_ms, "steps": kfd,
                                  "algorithmic_bytes_per_step": fd_bytes, "achieved_gbs": fd_bytes / (fd_ms * 1e-3) / 1e9,
                                  "note": "explicit forward-Euler 5/7-point step (pf_step_fd), single simulation (L2 resident below ~60 MB of state)",
                                  "fs_over_fd_time_per_step": step_ms / fd_ms}

    if rank == 0 and not args.no_cufft:
        line["cufft_side_reference"] = cufft_side_reference(torch, n, p, prec, dx, dt, c0, eta0, stream)

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        from oracle import pfo
        pfo.build()
        m = pfo.Model(n=n, n_eta=p, dx=dx, dt=dt)
        cc, ee = c0, eta0
        t0 = time.time()
        k = 0
        while k < 3 or (time.time() - t0 < 10 and k < 50):
            cc, ee = m.step_fs(cc, ee, 1)
            k += 1
            if time.time() - t0 > 40:
                break
        el = time.time() - t0
        line["cpu_baseline"] = {"value": k / el, "unit": "steps/s", "cores": pfo.num_threads(), "kind": "oracle",
                                "sample": f"{k} full FS steps of the same workload ({el:.1f} s)"}
    for cx in ctxs:
        cx.close()
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="default: enough steps for a >= 1 s timed region")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="1024sq", choices=sorted(WORKLOADS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT side reference")
    args = ap.parse_args()
    if args.steps is None:
        args.steps = DEFAULT_STEPS[args.workload] if args.impl == "ours" else 20
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
