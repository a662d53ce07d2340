"""Behaviour of the C ABI on a GPU beyond plain stepping (include/pf.h): state errors, device-pointer set/get on a
caller stream, dt changes between calls (graph re-capture), profiling mode, launch accounting."""
import numpy as np
import pytest

from paper_2306_04322_b200 import pf, synth
from parity_util import rel_linf

pytestmark = pytest.mark.gpu


def test_step_before_set_fields_is_a_state_error():
    with pf.Context((32, 32), n_eta=1, dx=(1.0, 1.0), dt=0.01) as ctx:
        for call in (lambda: ctx.step_fs(1), lambda: ctx.step_fd(1), ctx.get_fields, ctx.free_energy):
            with pytest.raises(pf.PfError) as e:
                call()
            assert e.value.code == pf.PF_ESTATE
        ctx.step_fs(0)                                   # nsteps == 0 is a no-op even then
        with pytest.raises(pf.PfError) as e:
            ctx.step_fs(-1)
        assert e.value.code == pf.PF_EINVAL


def test_dt_change_between_calls_matches_oracle(oracle):
    n, p = (64, 128), 2
    c, eta, dx = synth.init_b(n, p)
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as ctx:
        ctx.set_fields(c, eta)
        ctx.step_fs(7)
        ctx.set_dt(2e-3)                                 # dt is baked into the captured graph: must be re-captured
        ctx.step_fs(9)
        ctx.set_dt(1e-3)
        ctx.step_fd(5)
        gc, geta = ctx.get_fields()
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3).step_fs(c, eta, 7)
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=2e-3).step_fs(rc, reta, 9)
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=1e-3).step_fd(rc, reta, 5)
    assert rel_linf([gc, geta], [rc, reta]) < 1e-10


def test_device_pointers_on_a_caller_stream(oracle):
    import torch
    n, p = (128, 64), 2
    c, eta, dx = synth.init_b(n, p)
    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        dc = torch.as_tensor(c, device="cuda").contiguous()
        de = torch.as_tensor(eta, device="cuda").contiguous()
        oc, oe = torch.empty_like(dc), torch.empty_like(de)
    stream.synchronize()
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3, stream=stream.cuda_stream) as ctx:
        ctx.set_fields_device(dc, de)                    # asynchronous on `stream`
        ctx.step_fs(10)
        ctx.get_fields_device(oc, oe)
        stream.synchronize()
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3).step_fs(c, eta, 10)
    assert rel_linf([oc.cpu().numpy(), oe.cpu().numpy()], [rc, reta]) < 1e-10
    assert torch.equal(dc.cpu(), torch.as_tensor(c))     # the caller's input buffers are not touched


def test_profiling_mode_steps_identically_and_reports_kernels():
    n, p = (256, 256), 2
    c, eta, dx = synth.init_b(n, p)
    outs = []
    for prof in (0, 1):
        with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as ctx:
            ctx.set_fields(c, eta)
            ctx.set_profiling(prof)
            ctx.step_fs(1)                               # includes the one-off transform of the fields that were set
            l0 = ctx.launch_count()
            ctx.step_fs(5)
            assert ctx.launch_count() - l0 == 10         # two kernels per 2D step, graph replay or not
            if prof:
                times = ctx.fs_kernel_times()
                assert [nm for nm, _ in times] == ["row_c2r_nonlinear_r2c", "col_y_fft_update_ifft"]
                assert all(0 < t < 10 for _, t in times)
            outs.append(ctx.get_fields())
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])


def test_get_fields_twice_and_continue(oracle):
    n, p = (32, 32, 32), 1
    c, eta, dx = synth.init_b(n, p)
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as ctx:
        ctx.set_fields(c, eta)
        ctx.step_fs(3)
        a = ctx.get_fields()
        b = ctx.get_fields()
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])
        ctx.step_fs(4)                                   # the spectral state survived the read-out
        gc, geta = ctx.get_fields()
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3).step_fs(c, eta, 7)
    assert rel_linf([gc, geta], [rc, reta]) < 1e-10


def test_single_kernel_launches_leave_no_trajectory():
    # pf_launch_fs_kernel is a timing aid (bench.py's per-kernel figures): afterwards the context must refuse to step or
    # read out until fields are set again (a profiled context silently returned garbage)
    n, p = (64, 32, 16), 2
    c, eta, dx = synth.init_b(n, p)
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as ctx:
        with pytest.raises(pf.PfError) as e:
            ctx.launch_fs_kernel(0)
        assert e.value.code == pf.PF_ESTATE
        ctx.set_fields(c, eta)
        assert ctx.fs_kernel_names() == ["row_c2r_nonlinear_r2c", "col_y_fwd", "col_z_fft_update_ifft", "col_y_inv"]
        l0 = ctx.launch_count()
        for k in range(4):
            ctx.launch_fs_kernel(k)
            ctx.launch_fs_kernel(k)
        assert ctx.launch_count() - l0 >= 8
        with pytest.raises(pf.PfError) as e:
            ctx.launch_fs_kernel(4)
        assert e.value.code == pf.PF_EINVAL
        for call in (lambda: ctx.step_fs(1), lambda: ctx.step_fd(1), ctx.get_fields, ctx.free_energy):
            with pytest.raises(pf.PfError) as e:
                call()
            assert e.value.code == pf.PF_ESTATE
        ctx.set_fields(c, eta)                           # and it recovers
        ctx.step_fs(2)
        a = ctx.get_fields()
    with pf.Context(n, n_eta=p, dx=dx, dt=5e-3) as ctx:
        ctx.set_fields(c, eta)
        ctx.step_fs(2)
        b = ctx.get_fields()
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_two_contexts_on_two_streams_step_concurrently(oracle):
    # The 2D last-axis kernel hands c^ from one CTA to another through a flag. Its places in the schedule are tickets taken
    # in the order CTAs start, so the hand-off needs neither the whole grid resident nor index-order dispatch:
    # two contexts on two non-blocking streams compete for the SMs here, both must finish and both must match the oracle.
    import torch
    n, p = (512, 512), 2
    c, eta, dx = synth.init_b(n, p)
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    ctxs = [pf.Context(n, n_eta=p, dx=dx, dt=5e-3, stream=s.cuda_stream) for s in streams]
    try:
        for ctx in ctxs:
            ctx.set_fields(c, eta)
        for _ in range(10):                                  # interleaved single steps and an 8-step graph replay
            for ctx in ctxs:
                ctx.step_fs(1)
        for ctx in ctxs:
            ctx.step_fs(10)
        outs = [ctx.get_fields() for ctx in ctxs]
    finally:
        for ctx in ctxs:
            ctx.close()
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=5e-3).step_fs(c, eta, 20)
    for gc, geta in outs:
        assert rel_linf([gc, geta], [rc, reta]) < 1e-10


def test_fd3d_on_every_visible_device(oracle):
    # function attributes (the 86 KB dynamic shared memory of the 3D FD kernel) are per device: contexts on every GPU of the
    # process must step. Needs at least two GPUs; the single-GPU box skips.
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("one visible GPU")
    n, p = (64, 32, 32), 2
    c, eta, dx = synth.init_b(n, p)
    rc, reta = oracle.Model(n=n, n_eta=p, dx=dx, dt=1e-3).step_fd(c, eta, 5)
    try:
        for d in range(torch.cuda.device_count()):
            torch.cuda.set_device(d)
            with pf.Context(n, n_eta=p, dx=dx, dt=1e-3) as ctx:
                ctx.set_fields(c, eta)
                ctx.step_fd(5)
                gc, geta = ctx.get_fields()
            assert rel_linf([gc, geta], [rc, reta]) < 1e-12, d
    finally:
        torch.cuda.set_device(0)


def test_dsmem_read_rate_probe():
    # diagnostic of DESIGN.md section 6: own shared memory is at least as fast as a neighbour's; sizes that are no power of
    # two are refused
    own = pf.dsmem_read_rate(4, remote=False)
    rem = pf.dsmem_read_rate(4, remote=True)
    assert 1.0 < rem <= own * 1.05 and own < 300.0           # bytes per clock per SM: 128 is the shared-memory pipe's width
    with pytest.raises(pf.PfError):
        pf.dsmem_read_rate(3)
