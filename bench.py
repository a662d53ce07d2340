#!/usr/bin/env python
"""bench.py -- throughput of the Fourier-spectral (FS) step of arXiv 2306.04322 on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--also NAME ...] [--impl ours|reference]

A "step" is one FS time step (all kernels of SURVEY 8(a): x-pass with the nonlinear evaluation, strided passes with
the spectral update) of one simulation. At the L2-resident sizes the timed loop cycles through R independent
replicas of the simulation so that consecutive steps never find their inputs in L2 (timing rule "inputs larger than
L2"). The timed region of K steps is repeated B >= 5 times; `value` is the median batch.
Prints ONE JSON line: the headline workload (1024sq, the metric's 2D size) at the top level and the metric's other
size (256cube), configs[2] (2048sq, 2048sq_f32) and configs[1]'s grid (512sq) measured in the same invocation under "workloads".

--gpus N > 1 outside torchrun re-executes itself under torch.distributed.run with N ranks (replicas only, no
data-path collective).
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
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
    "128sq": ((128, 128), 4, "f64", "B", 5e-3, "2D 128x128, c + 4 eta, fp64 (paper Table 1 grid)"),
    "64sq": ((64, 64), 2, "f64", "A", 0.05, "2D 64x64, c + 2 eta, fp64 (configs[0])"),
    "128cube": ((128, 128, 128), 2, "f64", "B", 5e-3, "3D 128^3, c + 2 eta, fp64 (paper Table 2 grid)"),
    "64cube": ((64, 64, 64), 2, "f64", "B", 5e-3, "3D 64^3, c + 2 eta, fp64 (paper Table 2 grid)"),
}
# steps per timed batch when --steps is not given (>= 200); the batch is repeated >= 5 times
DEFAULT_STEPS = {"1024sq": 2000, "256cube": 200, "2048sq": 400, "2048sq_f32": 600, "512sq": 4000, "256sq": 6000, "128sq": 8000,
                 "64sq": 10000, "128cube": 1000, "64cube": 4000}
L2_BYTES = 126e6
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
    design: what the kernels of this design have to move (z-form state, cross-step fusion, c^ carried between steps as in
            Algorithm 1): the last-axis kernel reads g^ and the carried c^, writes the carried c^ and the z-form of c (4 arrays)
            and reads + writes every eta (2p arrays): (4 + 2p) R in 2D, (4 + 2p) Sp in 3D. Where the schedule splits a
            Cahn-Hilliard block over two CTAs (C_FWD / C_INV) the carried c^ is read once more: at most one array on top
            (design_upper)."""
    F = p + 1
    N = int(np.prod(n))
    R = N * w
    S = (n[0] // 2 + 1) * (N // n[0]) * 2 * w
    if len(n) == 2:
        survey = {"row_c2r_nonlinear_r2c": 2 * F * (R + S), "col_y_fft_update_ifft": 5 * F * S}
        design = {"row_c2r_nonlinear_r2c": 2 * F * R, "col_y_fft_update_ifft": (4 + 2 * p) * R}
    else:
        P2 = ((n[0] // 2 + 1 + 15) // 16) * 16
        Sp = P2 * n[1] * n[2] * 2 * w          # one padded half-spectrum array as stored
        survey = {"row_c2r_nonlinear_r2c": 2 * F * (R + S), "col_y_fwd": 2 * F * S, "col_z_fft_update_ifft": 5 * F * S,
                  "col_y_inv": 2 * F * S}
        design = {"row_c2r_nonlinear_r2c": 2 * F * R, "col_y_fwd": F * (R + Sp),
                  "col_z_fft_update_ifft": (4 + 2 * p) * Sp, "col_y_inv": F * (Sp + R)}
    return survey, design


def kernel_source_hash(kernel=None):
    """Hash of the sources a kernel is built from (kernel=None: of every kernel file). An ncu traffic figure under profiles/
    is quoted only while the files of ITS kernel still hash to the value the capture step stored beside it."""
    from paper_2306_04322_b200 import ncu_traffic as nt
    return nt.source_hash(kernel)


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu --set full summary
    (profiles/ncu_traffic.json; entries are written by `python -m paper_2306_04322_b200.ncu_traffic`, never by hand).
    None when the sources of that kernel have changed since its capture."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as fh:
            t = json.load(fh)
        ent = t["traffic"].get(workload, {}).get(kernel)
        if not isinstance(ent, dict):
            return None, "no capture of this kernel for this workload in profiles/ncu_traffic.json"
        if ent.get("source_hash") != kernel_source_hash(kernel):
            return None, f"profiles/ncu_traffic.json: captured from other sources of this kernel ({ent.get('source_hash')})"
        return ent["dram_bytes_per_launch"], ent.get("capture", t.get("capture"))
    except Exception as e:
        return None, f"no profiles/ncu_traffic.json ({type(e).__name__})"


# environment variables that make pf_create pick other kernels or launch paths (A/B runs)
SWITCHES = ["PF_WCOL", "PF_COL2D_LEGACY", "PF_COL2D_NOTICKET", "PF_COL3D_PARK", "PF_FD2D_LEGACY", "PF_FD3D_LEGACY", "PF_NO_GRAPH",
            "PF_RESIDENT", "PF_SG_CLUSTER"]


def live_switches():
    """Every PF_* variable of the environment (name -> value) and the subset that changes the code path."""
    seen = {k: v for k, v in sorted(os.environ.items()) if k.startswith("PF_")}
    return seen, [k for k in seen if k in SWITCHES]


class ClockSampler:
    """SM clock, power and clock-event reasons sampled through NVML by a host thread every ~2 ms while the timed batches run
    (a timed region can be as short as 1 ms, far below what `nvidia-smi -lms` resolves), plus one sample taken right
    after the last batch was queued. Falls back to one-shot nvidia-smi queries when NVML is unavailable."""

    REASONS = {0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap"}

    def __init__(self, torch_device_index):
        self.samples = []
        self.stop_flag = False
        self.h = None
        self.idx = torch_device_index
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = str(torch.cuda.get_device_properties(torch_device_index).uuid)
                self.h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid).encode() if not uuid.startswith("GPU-") else uuid.encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(torch_device_index)
            self.max_sm = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.h = None
        self.thread = threading.Thread(target=self._run, daemon=True)

    def _one(self):
        nv = self.nv
        sm = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
        try:
            reasons = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
        except Exception:
            reasons = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
        try:
            pw = nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0
        except Exception:
            pw = None
        return sm, reasons, pw

    def _run(self):
        while not self.stop_flag:
            try:
                self.samples.append(self._one())
            except Exception:
                break
            time.sleep(0.002)

    def start(self):
        if self.h is not None:
            self.thread.start()
        return self

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "how": "NVML polled every ~2 ms by a host thread during the timed batches"}
        if self.h is None:
            return self._smi(out)
        try:
            self.samples.append(self._one())          # the queue of the last batch is still draining here
        except Exception:
            pass
        self.stop_flag = True
        self.thread.join(timeout=2)
        if not self.samples:
            return self._smi(out)
        sm = sorted(s[0] for s in self.samples)
        bits = 0
        for s in self.samples:
            bits |= s[1]
        out.update(sm_mhz=sm[len(sm) // 2], sm_min_mhz=sm[0], sm_max_mhz=self.max_sm, samples=len(sm),
                   reasons=[nm for b, nm in self.REASONS.items() if bits & b])
        pws = [s[2] for s in self.samples if s[2] is not None]
        if pws:
            out["power_w_max"] = max(pws)
        return out

    def _smi(self, out):
        try:
            q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
                "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"
            r = subprocess.run(["nvidia-smi", "-i", str(self.idx), f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=10).stdout.strip().split(",")
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            out.update(sm_mhz=float(r[0]), sm_max_mhz=float(r[1]), power_w_max=float(r[2]),
                       reasons=[nm for i, nm in enumerate(names) if r[3 + i].strip() == "Active"],
                       how="one nvidia-smi query right after the timed batches (NVML unavailable)")
        except Exception:
            pass
        return out


def oracle_timing(wl, budget_s, threads=None):
    """The oracle as it stands (oracle/pfo.c) on the host cores: full FS steps of the workload until budget_s is spent."""
    import ctypes
    from oracle import pfo
    pfo.build()
    n, p, prec, init, dt, _ = WORKLOADS[wl]
    c, eta, dx = make_fields(wl)
    m = pfo.Model(n=n, n_eta=p, dx=dx, dt=dt)
    gomp, before = None, pfo.num_threads()
    if threads is not None:
        try:                                          # the oracle's OpenMP runtime; nothing in oracle/ is changed
            gomp = ctypes.CDLL("libgomp.so.1")
            gomp.omp_set_num_threads(int(threads))
        except Exception:
            return None
    used = pfo.num_threads()
    t0 = time.time()
    k = 0
    while k < 2 or (time.time() - t0 < budget_s and k < 200):
        c, eta = m.step_fs(c, eta, 1)
        k += 1
        if time.time() - t0 > 3 * budget_s:
            break
    el = time.time() - t0
    if gomp is not None:
        gomp.omp_set_num_threads(int(before))
    return {"value": k / el, "unit": "steps/s", "cores": used, "kind": "oracle",
            "sample": f"{k} full FS steps of the same workload ({el:.1f} s)"}


def run_reference(args):
    """The oracle (oracle/pfo.c, as it stands) on the host cores: the base contract's reference arm for this tier.
    Under torchrun rank 0 alone runs and prints; the other ranks exit 0 without work."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    from oracle import pfo
    pfo.build()
    n, p, prec, init, dt, desc = WORKLOADS[args.workload]
    c, eta, dx = make_fields(args.workload)
    m = pfo.Model(n=n, n_eta=p, dx=dx, dt=dt)
    budget = float(os.environ.get("PF_REF_BUDGET_S", "150"))
    t_all = time.time()
    W = min(args.warmup, 1)
    for _ in range(W):
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
            "warmup": W, "ms_per_step": 1e3 * el / done, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": desc, "init": init_name(init), "dt": dt,
                       "note": "CPU oracle (oracle/pfo.c as it stands); steps bounded by a time budget"},
            "gpoint_updates_per_s": val * N / 1e9,
            "cpu_baseline": {"value": val, "unit": "steps/s", "cores": pfo.num_threads(), "kind": "oracle",
                             "sample": f"{done} full FS steps of the same workload"},
            "e2e": {"value": val, "unit": "steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


def init_name(init):
    return "Eqs. 4-6 benchmark field (synth.init_b)" if init == "B" else "seeded noise (synth.init_a)"


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


def stats(vals):
    v = sorted(vals)
    return {"min": v[0], "median": v[len(v) // 2] if len(v) % 2 else 0.5 * (v[len(v) // 2 - 1] + v[len(v) // 2]), "max": v[-1], "n": len(v)}


def measure_workload(wl, K, W, env, full=True):
    """All device measurements of one workload. Returns the dict of a JSON line (headline keys + details).
    env: torch, dist, pf, replicas, rank, world, stream."""
    torch, dist, pf, replicas = env["torch"], env["dist"], env["pf"], env["replicas"]
    rank, world, stream = env["rank"], env["world"], env["stream"]
    n, p, prec, init, dt, desc = WORKLOADS[wl]
    w = 8 if prec == "f64" else 4
    F, N = p + 1, int(np.prod(n))
    R = N * w
    c0, eta0, dx = make_fields(wl)
    # replicas only: every rank advances its own independent simulations
    state_bytes = (F + 1) * R if len(n) == 2 else 3 * F * R
    reps = 1 if state_bytes > 2 * L2_BYTES else int(np.ceil(2.5 * L2_BYTES / state_bytes))
    ctxs = [pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=prec, stream=stream.cuda_stream) for _ in range(reps)]

    def reset_fields(group, count):
        for i, cx in enumerate(group):
            cx.set_fields(replicas.perturb(c0, rank, i, count), eta0)

    reset_fields(ctxs, reps)
    torch.cuda.synchronize()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(stream)
        fn()
        e1.record(stream)
        barrier()
        return replicas.max_over_ranks(e0.elapsed_time(e1), device="cuda")

    def fs_steps(k, which):
        for s in range(k):                     # one step of each replica in turn: asynchronous plain launches (programmatic
            which[s % len(which)].step_fs(1)   # stream serialization); pf_step_fs replays its graph only for calls of >= 8 steps

    nbatch = max(5, min(50, int(np.ceil(1000 / K))))
    fs_steps(max(W, 3) * len(ctxs), ctxs)
    sampler = ClockSampler(torch.cuda.current_device()).start() if rank == 0 else None
    l0 = sum(cx.launch_count() for cx in ctxs)
    batches = [timed(lambda: fs_steps(K, ctxs)) for _ in range(nbatch)]
    launches = (sum(cx.launch_count() for cx in ctxs) - l0) // nbatch
    clocks = sampler.stop() if sampler else {}
    bst = stats(batches)
    ms = bst["median"]
    value = replicas.job_throughput(K, ms, world)
    step_ms = ms / K

    # single simulation, state resident in L2 where it fits (reported, not the headline)
    res_b = [timed(lambda: fs_steps(K, ctxs[:1])) for _ in range(5)]
    resident = replicas.job_throughput(K, stats(res_b)["median"], world)

    # the launch path a long run takes: ONE pf_step_fs(K8) call on one simulation = replays of the captured 8-step graph
    # (pf.h), beside the same simulation advanced by K8 single-step calls (plain launches) above
    K8 = max(8, (K // 8) * 8)
    ctxs[0].step_fs(8)
    gr_b = [timed(lambda: ctxs[0].step_fs(K8)) for _ in range(5)]
    graph_replay = replicas.job_throughput(K8, stats(gr_b)["median"], world)

    # per-kernel device times, L2-cold like the step: kernel k of every replica in turn (pf_launch_fs_kernel) between two
    # events on the stream, repeated; the replicas' fields are no trajectory afterwards (they are set again below)
    names = ctxs[0].fs_kernel_names()
    kms = {}
    rounds = max(2, int(np.ceil(40 / len(ctxs))))
    for k, name in enumerate(names):
        def one_kernel():
            for _ in range(rounds):
                for cx in ctxs:
                    cx.launch_fs_kernel(k)
        one_kernel()
        ts = [timed(one_kernel) for _ in range(5)]
        kms[name] = stats(ts)["median"] / (rounds * len(ctxs))
    reset_fields(ctxs, reps)
    ksurvey, kdesign = bytes_model(n, p, w)
    survey_bytes, design_bytes = sum(ksurvey.values()), sum(kdesign.values())
    peak, peak_src = peaks()
    dom = max(kms, key=kms.get)
    achieved = ksurvey[dom] / (kms[dom] * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(wl, dom)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": ksurvey[dom],
                "algorithmic_bytes_note": "SURVEY 8(d) per-pass bytes of the passes this kernel fuses (see DESIGN.md section 5)",
                "design_bytes_per_launch": kdesign[dom],
                "achieved_vs_design_bytes": kdesign[dom] / (kms[dom] * 1e-3) / 1e9,
                "frac_vs_design_bytes": kdesign[dom] / (kms[dom] * 1e-3) / 1e9 / peak,
                "kernel_ms": kms[dom], "kernels_ms": kms,
                "kernel_timing": f"CUDA events on the launch stream around {rounds * len(ctxs)} launches of this kernel alone, "
                                 f"one per replica in turn ({len(ctxs)} replicas: L2-cold like the step), launched as in a step "
                                 f"(programmatic stream serialization: prologues overlap the previous launch's tail)",
                "kernel_share_of_step": kms[dom] / sum(kms.values())}
    if roofline["frac"] > 1.0:
        roofline["note"] = ("frac > 1 on the SURVEY 8(d) per-pass bytes: this kernel fuses passes whose intermediate results never "
                            "leave the SM, so it moves fewer bytes than the per-pass count; frac_vs_design_bytes is the HBM utilisation")
    step_roofline = {"bytes_per_step_survey_8d": survey_bytes, "bytes_per_step_this_design": design_bytes,
                     "achieved_vs_survey_bytes_gbs": survey_bytes / (step_ms * 1e-3) / 1e9,
                     "frac_vs_survey_bytes": survey_bytes / (step_ms * 1e-3) / 1e9 / peak,
                     "achieved_vs_design_bytes_gbs": design_bytes / (step_ms * 1e-3) / 1e9,
                     "frac_vs_design_bytes": design_bytes / (step_ms * 1e-3) / 1e9 / peak}

    line = {"metric": METRIC, "value": value, "unit": "steps/s", "n_gpus": world, "steps": K, "warmup": max(W, 3),
            "ms_per_step": step_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": prec,
            "data": "synthetic",
            "config": {"workload": desc, "init": init_name(init), "dt": dt, "replicas_per_gpu": reps,
                       "parallelism": "independent replicas per GPU, no collective",
                       "l2": (f"timed loop cycles {reps} independent replicas ({reps * state_bytes / 1e6:.0f} MB of state > 126 MB L2)"
                              if reps > 1 else f"state {state_bytes / 1e6:.0f} MB per step exceeds the 126 MB L2")},
            "timed_batches": {"steps_per_batch": K, "batches": nbatch, "ms": bst,
                              "steps_per_s": {"min": replicas.job_throughput(K, bst["max"], world),
                                              "median": value, "max": replicas.job_throughput(K, bst["min"], world)},
                              "note": "value = the median batch; every batch is K steps bracketed by barrier + synchronize, CUDA events on the launch stream, max over ranks"},
            "gpoint_updates_per_s": value * N / 1e9,
            "field_point_updates_per_s_G": value * N * F / 1e9,
            "l2_resident_single_simulation": {"value": resident, "unit": "steps/s", "gpoint_updates_per_s": resident * N / 1e9,
                                              "how": "one simulation, K calls of pf_step_fs(1): plain launches"},
            "graph_replay_single_simulation": {"value": graph_replay, "unit": "steps/s", "steps_per_call": K8,
                                               "how": "the same simulation, ONE pf_step_fs(K8) call per batch: replays of the 8-step CUDA graph "
                                                      "(2D grids up to 64^2: the cluster-resident kernel instead)"},
            "roofline": roofline, "step_roofline": step_roofline, "gpu_launches": int(launches), "clocks": clocks}

    # end to end through the C ABI with HOST buffers: set (H2D) + 1 step + get (D2H), pinned host memory, ONE simulation
    tdt = torch.float64 if prec == "f64" else torch.float32
    L = pf.lib()

    def host_buffers():
        bc = torch.empty(tuple(reversed(n)), dtype=tdt).pin_memory()
        be = torch.empty((p,) + tuple(reversed(n)), dtype=tdt).pin_memory()
        bc.numpy()[...] = c0
        be.numpy()[...] = eta0
        return bc, be

    def e2e_loop(h, bufs, steps):
        bc, be = bufs
        for _ in range(steps):
            L.pf_set_fields(h, bc.data_ptr(), be.data_ptr(), pf.PF_HOST)
            L.pf_step_fs(h, 1)
            L.pf_get_fields(h, bc.data_ptr(), be.data_ptr(), pf.PF_HOST)

    ke = max(3, min(K, 20))
    bufs = host_buffers()
    e2e_loop(ctxs[0]._h, bufs, 2)
    barrier()
    t0 = time.perf_counter()
    e2e_loop(ctxs[0]._h, bufs, ke)
    torch.cuda.synchronize()
    e2e_s = replicas.max_over_ranks(time.perf_counter() - t0, device="cuda")
    e2e = {"value": world * ke / e2e_s, "unit": "steps/s", "h2d_bytes_per_step": F * R, "d2h_bytes_per_step": F * R,
           "steps": ke, "contexts": 1,
           "note": "pf_set_fields(HOST) + pf_step_fs(1) + pf_get_fields(HOST) per step of ONE simulation, pinned host buffers, "
                   "host wall clock around the loop (PCIe bound)"}
    if full:
        # two independent simulations from two host threads (own context, stream and pinned buffers each): the upload of
        # one overlaps the download of the other (PCIe is full duplex). Reported beside the single-simulation value.
        cxs2 = [pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=prec) for _ in range(2)]
        bufs2 = [host_buffers() for _ in range(2)]
        for i in range(2):
            e2e_loop(cxs2[i]._h, bufs2[i], 2)
        barrier()
        t0 = time.perf_counter()
        th = [threading.Thread(target=e2e_loop, args=(cxs2[i]._h, bufs2[i], ke)) for i in range(2)]
        for t in th:
            t.start()
        for t in th:
            t.join()
        torch.cuda.synchronize()
        e2e2_s = replicas.max_over_ranks(time.perf_counter() - t0, device="cuda")
        for cx2 in cxs2:
            cx2.close()
        e2e["two_contexts_value"] = world * 2 * ke / e2e2_s
    line["e2e"] = e2e

    # independent simulations advanced concurrently on two streams (the paper's sweeps are independent runs, DESIGN.md
    # "Multi-GPU"): kernels of different simulations fill each other's tails. Reported beside the headline, which stays
    # the one-stream figure. Timed with events on `stream`, which waits for the second stream's last step.
    if full and len(ctxs) >= 2:
        stream2 = torch.cuda.Stream()
        half = max(1, len(ctxs) // 2)
        ctxs2 = [pf.Context(n, n_eta=p, dx=dx, dt=dt, precision=prec, stream=stream2.cuda_stream) for _ in range(half)]
        reset_fields(ctxs2, half)
        for cx in ctxs2:
            cx.step_fs(W)
        grpa = ctxs[:half]
        for cx in grpa:
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
        line["concurrent_replicas"] = {"streams": 2, "value": replicas.job_throughput(2 * (K // 2), cms, world), "unit": "steps/s",
                                       "us_per_step": 1e3 * cms / (2 * (K // 2)),
                                       "note": "two independent simulations in flight at a time, one per stream; every simulation still advances step by step"}
        for cx in ctxs2:
            cx.close()

    # comparison path: explicit FD steps, same replica cycling as the FS loop (L2-cold against L2-cold)
    for cx in ctxs:
        cx.set_dt(1e-6)
    reset_fields(ctxs, reps)

    def fd_steps(k, which):
        for s in range(k):
            which[s % len(which)].step_fd(1)

    kfd = max(20 * len(ctxs), min(2000, K))
    fd_steps(3 * len(ctxs), ctxs)
    fd_ms = stats([timed(lambda: fd_steps(kfd, ctxs)) for _ in range(5)])["median"] / kfd
    fd_res_ms = stats([timed(lambda: fd_steps(kfd, ctxs[:1])) for _ in range(3)])["median"] / kfd
    fd_bytes = 2 * F * R                      # fused kernels: every field read once and written once per step
    line["fd_comparison_path"] = {"value": 1e3 / fd_ms, "unit": "steps/s", "us_per_step": 1e3 * fd_ms, "steps": kfd,
                                  "algorithmic_bytes_per_step": fd_bytes, "achieved_gbs": fd_bytes / (fd_ms * 1e-3) / 1e9,
                                  "frac_of_hbm_peak": fd_bytes / (fd_ms * 1e-3) / 1e9 / peak,
                                  "l2_resident_single_simulation_us_per_step": 1e3 * fd_res_ms,
                                  "note": f"explicit forward-Euler 5/7-point step (pf_step_fd), one launch per step, cycling the same {len(ctxs)} replicas as the FS loop",
                                  "fs_over_fd_time_per_step": step_ms / fd_ms}
    for cx in ctxs:
        cx.set_dt(dt)

    if rank == 0 and full and not env["args"].no_cufft:
        line["cufft_side_reference"] = cufft_side_reference(torch, n, p, prec, dx, dt, c0, eta0, stream)
    for cx in ctxs:
        cx.close()
    return line


def small_grid_measurements(env):
    """SURVEY 8(f)-4 (the paper's small-grid remark): configs[0]'s grid (64^2, c + 2 eta, fp64, seeded noise,
    dt = 0.05) as ONE simulation -- cluster-resident kernel (default up to 64^2: pf_step_fs(K) is one launch) against the
    two-kernel path (PF_RESIDENT=0 at pf_create) -- and as a batch of 64 replicas in one context (pf_create_batch)
    against a loop over 64 contexts."""
    torch, pf, stream = env["torch"], env["pf"], env["stream"]
    from paper_2306_04322_b200 import synth
    n, p, K = (64, 64), 2, 2000

    def timed(fn):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        fn()
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1)

    def single(resident, n=n, p=p):
        old = os.environ.get("PF_RESIDENT")
        if not resident:
            os.environ["PF_RESIDENT"] = "0"
        try:
            c, eta = synth.init_a(n, p, seed=1)
            with pf.Context(n, n_eta=p, dx=1.0, dt=0.05, stream=stream.cuda_stream) as cx:
                cx.set_fields(c, eta)
                cx.step_fs(50)
                l0 = cx.launch_count()
                ms = stats([timed(lambda: cx.step_fs(K)) for _ in range(5)])["median"]
                launches = (cx.launch_count() - l0) // 5
        finally:
            if old is None:
                os.environ.pop("PF_RESIDENT", None)
            else:
                os.environ["PF_RESIDENT"] = old
        return {"value": 1e3 * K / ms, "unit": "steps/s", "us_per_step": 1e3 * ms / K, "launches_per_call_of_%d_steps" % K: int(launches)}

    out = {"workload": "2D 64x64, c + 2 eta, fp64, seeded noise, dt = 0.05 (configs[0])",
           "single_simulation_cluster_resident": single(True), "single_simulation_two_kernel_path": single(False),
           "single_256sq_c_4eta_two_kernel_path": single(True, (256, 256), 4),
           "single_128sq_c_4eta_two_kernel_path": single(True, (128, 128), 4)}
    # the paper's small 3D grids (Table 2; 16^3 and 32^3 "increase significantly"): one
    # simulation, c + 2 eta, fp64, four launches per step replayed as an 8-step graph -- launch-latency bound, reported as is
    for m in (16, 32, 64):
        r = single(True, (m, m, m), 2)
        r["frac_of_hbm_roofline_on_survey_8d_bytes"] = (3 * (2 * m ** 3 * 8 + 11 * (m // 2 + 1) * m * m * 16)) * r["value"] / 1e9 / peaks()[0]
        out[f"single_{m}cube_c_2eta"] = r
    B = 64
    inits = [synth.init_a(n, p, seed=100 + b) for b in range(B)]
    c0, e0 = np.stack([c for c, _ in inits]), np.stack([e for _, e in inits])
    with pf.Context(n, n_eta=p, dx=1.0, dt=0.05, nbatch=B, stream=stream.cuda_stream) as cx:
        cx.set_fields(c0, e0)
        cx.step_fs(20)
        msb = stats([timed(lambda: cx.step_fs(K // 4)) for _ in range(5)])["median"] / (K // 4)
    cxs = [pf.Context(n, n_eta=p, dx=1.0, dt=0.05, stream=stream.cuda_stream) for _ in range(B)]
    for b, cx in enumerate(cxs):
        cx.set_fields(c0[b], e0[b])
        cx.step_fs(4)

    def loop():
        for _ in range(20):
            for cx in cxs:
                cx.step_fs(1)
    msl = stats([timed(loop) for _ in range(3)])["median"] / 20
    for cx in cxs:
        cx.close()
    out["batch_of_64_replicas"] = {"one_context_replica_steps_per_s": 1e3 * B / msb, "us_per_step_of_all_replicas": 1e3 * msb,
                                   "loop_over_64_contexts_replica_steps_per_s": 1e3 * B / msl, "ratio": msl / msb,
                                   "note": "pf_create_batch(nbatch=64) + pf_step_fs(K) against pf_step_fs(1) on 64 contexts in turn"}
    # 3D: 64 replicas of 32^3 (c + 2 eta) in one context against a loop over 64 contexts
    n3 = (32, 32, 32)
    inits = [synth.init_a(n3, p, seed=200 + b) for b in range(B)]
    c0, e0 = np.stack([c for c, _ in inits]), np.stack([e for _, e in inits])
    with pf.Context(n3, n_eta=p, dx=1.0, dt=0.05, nbatch=B, stream=stream.cuda_stream) as cx:
        cx.set_fields(c0, e0)
        cx.step_fs(16)
        msb = stats([timed(lambda: cx.step_fs(200)) for _ in range(5)])["median"] / 200
    cxs = [pf.Context(n3, n_eta=p, dx=1.0, dt=0.05, stream=stream.cuda_stream) for _ in range(B)]
    for b, cx in enumerate(cxs):
        cx.set_fields(c0[b], e0[b])
        cx.step_fs(4)
    msl = stats([timed(loop) for _ in range(3)])["median"] / 20
    for cx in cxs:
        cx.close()
    out["batch_of_64_replicas_32cube"] = {"one_context_replica_steps_per_s": 1e3 * B / msb, "us_per_step_of_all_replicas": 1e3 * msb,
                                          "loop_over_64_contexts_replica_steps_per_s": 1e3 * B / msl, "ratio": msl / msb,
                                          "frac_of_hbm_roofline_on_survey_8d_bytes": B * 3 * (2 * 32 ** 3 * 8 + 11 * 17 * 32 * 32 * 16) / (msb * 1e-3) / 1e9 / peaks()[0],
                                          "note": "pf_create_batch(nbatch=64) on 32^3 + pf_step_fs(200) against pf_step_fs(1) on 64 contexts in turn"}
    return out


def spawn_ranks(args, argv):
    """python bench.py --gpus N outside torchrun: re-execute under torch.distributed.run with N ranks on this node."""
    port = 29500 + (os.getpid() % 2000)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + argv
    return subprocess.call(cmd)


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2306_04322_b200 import pf, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if os.environ.get("PF_LIBPF") and not args.allow_lib_override:
        raise SystemExit("PF_LIBPF is set: bench.py times the product library only (ablation builds: --allow-lib-override)")
    seen, live = live_switches()
    if live and not args.allow_switches:
        raise SystemExit(f"{', '.join(live)} set in the environment: these pick other kernels / launch paths than the product's "
                         "defaults; bench.py times the defaults only (A/B runs: --allow-switches)")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    pf.lib()                                   # fails loudly if libpf.so is missing
    env = {"torch": torch, "dist": dist, "pf": pf, "replicas": replicas, "rank": rank, "world": world,
           "stream": torch.cuda.Stream(), "args": args}

    K = args.steps if args.steps is not None else DEFAULT_STEPS[args.workload]
    line = measure_workload(args.workload, K, args.warmup, env, full=True)
    if rank == 0:
        line["fp64_fma_peak_tflops"] = {"measured": pf.fp64_fma_peak(),
                                        "nominal_from_unit_counts": 148 * 64 * 2 * 1.965e9 / 1e12,
                                        "how": "pf_fp64_fma_peak: independent DFMA chains, 4 x 1024 threads per SM, best of 3 launches"}
    line["library"] = {"path": pf.SO_PATH, "override": bool(os.environ.get("PF_LIBPF")), "kernel_source_hash": kernel_source_hash(),
                       "switches": seen, "switches_changing_the_code_path": live}

    if rank == 0 and world == 1 and args.workload == "1024sq" and not args.no_small_grids:
        line["small_grids"] = small_grid_measurements(env)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        allc = oracle_timing(args.workload, 8.0)
        one = oracle_timing(args.workload, 4.0, threads=1)
        line["cpu_baseline"] = dict(allc, single_thread=one)

    others = {}
    for wl in args.also:
        if wl == args.workload:
            continue
        Ko = min(K, DEFAULT_STEPS[wl]) if args.steps is not None else DEFAULT_STEPS[wl]
        sub = measure_workload(wl, Ko, args.warmup, env, full=False)
        if rank == 0 and world == 1 and not args.no_cpu_baseline:
            sub["cpu_baseline"] = oracle_timing(wl, 5.0)
        others[wl] = sub
    if others:
        line["workloads"] = others
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None, help="steps per timed batch (default: >= 200, per workload)")
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--workload", default="1024sq", choices=sorted(WORKLOADS))
    ap.add_argument("--also", nargs="*", default=None, choices=sorted(WORKLOADS),
                    help="further workloads measured in the same invocation and reported under 'workloads' "
                         "(default: 256cube, 2048sq, 2048sq_f32 and 512sq beside the default headline, none otherwise)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cufft", action="store_true", help="skip the cuFFT side reference")
    ap.add_argument("--no-small-grids", action="store_true", help="skip the 64^2 single-simulation / batch measurements")
    ap.add_argument("--allow-lib-override", action="store_true", help="accept PF_LIBPF (ablation builds; never for a reported number)")
    ap.add_argument("--allow-switches", action="store_true", help="accept PF_* A/B switches in the environment (never for a reported number)")
    args = ap.parse_args()
    if args.also is None:
        args.also = ["256cube", "2048sq", "2048sq_f32", "512sq"] if args.workload == "1024sq" else []
    if args.gpus > 1 and "RANK" not in os.environ:
        raise SystemExit(spawn_ranks(args, sys.argv[1:]))
    if args.impl == "reference":
        if args.steps is None:
            args.steps = 20
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
