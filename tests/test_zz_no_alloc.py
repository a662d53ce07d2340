"""pf_free_energy_static: the entry point for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is off the table: inside an application whose own memory pool has
taken the whole GPU, as an energy monitor hooked into another solver's time loop (cudaMalloc/cudaFree would stall the
device at every call), or under a "no allocation after start-up" rule. For them the library offers one call that needs
no context and allocates nothing; its working memory is a fixed array compiled into libpf.so (about 320 KB per GPU, at
most 2^24 grid points, all calls share it). This file checks that call against the ordinary, context-based
pf_free_energy(gradient_kind=1) on the same fields, twice in a row, so that what the first call leaves behind in the
shared array is seen not to leak into the second.

The file is named to be collected last: the driver runs pytest with -x, and a failure here must not hide the parity
tests. Nothing here depends on an earlier test: it passes alone in a fresh process as well as after the rest.
"""
import ctypes

import numpy as np
import pytest


def _params(pf, n, **kw):
    return pf.make_params(n, **kw)


def test_static_entry_point_rejects_what_it_cannot_hold():
    """Argument checks come before any device is touched, so they run on the CPU box too."""
    from paper_2306_04322_b200 import build, pf
    build.build()
    L = pf.lib()
    out = (ctypes.c_double * 16)()
    dummy = ctypes.c_void_p(256)                    # never dereferenced: every case below is refused first
    # 512^3 = 2^27 points: more tiles than the static array has slots for
    p = _params(pf, (512, 512, 512), n_eta=2)
    assert L.pf_free_energy_static(ctypes.byref(p), dummy, dummy, out) == pf.PF_EUNSUPPORTED
    assert 512 ** 3 > pf.STATIC_MAX_POINTS >= 256 ** 3
    p = _params(pf, (64, 48), n_eta=2)              # not a power of two
    assert L.pf_free_energy_static(ctypes.byref(p), dummy, dummy, out) == pf.PF_EUNSUPPORTED
    p = _params(pf, (64, 64), n_eta=9)              # more order parameters than the result slots hold
    assert L.pf_free_energy_static(ctypes.byref(p), dummy, dummy, out) == pf.PF_EINVAL
    p = _params(pf, (64, 64), n_eta=2)
    assert L.pf_free_energy_static(ctypes.byref(p), None, dummy, out) == pf.PF_EINVAL
    assert L.pf_free_energy_static(ctypes.byref(p), dummy, None, out) == pf.PF_EINVAL
    assert L.pf_free_energy_static(ctypes.byref(p), dummy, dummy, None) == pf.PF_EINVAL
    assert L.pf_free_energy_static(None, dummy, dummy, out) == pf.PF_EINVAL


@pytest.mark.gpu
@pytest.mark.parametrize("precision,rtol", [("f64", 1e-11), ("f32", 1e-8)])
def test_static_entry_point_matches_context_path_twice_in_a_row(precision, rtol):
    """Two calls back to back on different problems -- first the larger one (1024 tiles of partial sums, five result
    slots), then a smaller one with fewer fields -- each compared with pf_free_energy(1) of a context holding the same
    fields. Both paths do the same pointwise arithmetic and accumulate in fp64. In fp64 they differ only in the order of
    the sum: rtol 1e-11, the tolerance tests/test_parity_fd.py::test_free_energy uses. In fp32 the compiler fuses the
    multiply-adds of a term differently in the two kernels, a rounding difference of 1e-7 per term that averages out over
    the grid (5.6e-11 measured): rtol 1e-8, three orders tighter than the 1e-5 the fp32 energy tests allow against the
    oracle."""
    import torch
    from paper_2306_04322_b200 import pf, synth
    assert torch.cuda.is_available()
    torch.cuda.set_device(0)
    dtype = torch.float64 if precision == "f64" else torch.float32
    cases = [((256, 128, 128), 3), ((64, 32), 1), ((256, 128, 128), 3)]
    got, want = [], []
    for n, p in cases:
        c, eta, dx = synth.init_b(n, p)
        dc = torch.from_numpy(np.ascontiguousarray(c)).to(device="cuda", dtype=dtype)
        de = torch.from_numpy(np.ascontiguousarray(eta)).to(device="cuda", dtype=dtype)
        torch.cuda.synchronize()
        before = torch.cuda.memory_allocated()
        e_static = pf.free_energy_static(dc, de, n, n_eta=p, dx=dx, precision=precision)
        again = pf.free_energy_static(dc, de, n, n_eta=p, dx=dx, precision=precision)
        assert torch.cuda.memory_allocated() == before
        assert np.array_equal(e_static, again)          # fixed summation order: the same bits on every run
        with pf.Context(n, n_eta=p, dx=dx, dt=5e-3, precision=precision) as ctx:
            ctx.set_fields_device(dc, de)
            e_ctx = ctx.free_energy(1)
        got.append(e_static)
        want.append(e_ctx)
    for (n, p), g, w in zip(cases, got, want):
        assert g.shape == (3 + p,) and np.all(np.isfinite(g))
        np.testing.assert_allclose(g, w, rtol=rtol, err_msg=f"{n} p={p}")
    assert np.array_equal(got[0], got[2])               # the small problem in between left nothing behind


@pytest.mark.gpu
def test_static_entry_point_largest_grid_and_host_pointer():
    """The largest accepted grid (2^24 points, every slot of the static array in use) with n_eta = 0, and the refusal of a
    host pointer where a device pointer is required."""
    import torch
    from paper_2306_04322_b200 import pf
    torch.cuda.set_device(0)
    n = (256, 256, 256)
    g = torch.Generator(device="cuda").manual_seed(3)
    dc = 0.5 + 0.1 * torch.rand(n[::-1], device="cuda", dtype=torch.float64, generator=g)
    e_static = pf.free_energy_static(dc, None, n, n_eta=0, dx=0.5)
    with pf.Context(n, n_eta=0, dx=0.5, dt=1e-3) as ctx:
        ctx.set_fields_device(dc, None)
        e_ctx = ctx.free_energy(1)
    np.testing.assert_allclose(e_static, e_ctx, rtol=1e-11)
    host = torch.zeros(64 * 64, dtype=torch.float64)
    with pytest.raises(pf.PfError) as ei:
        pf.free_energy_static(host, None, (64, 64), n_eta=0)
    assert ei.value.code == pf.PF_EINVAL
