"""CPU-side checks of the C ABI: libpf.so builds, loads and exports every symbol include/pf.h declares;
argument validation that needs no GPU."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libpf():
    from paper_2306_04322_b200 import build, pf
    build.build()
    return pf


def test_every_declared_symbol_is_exported(libpf):
    hdr = open(os.path.join(ROOT, "include", "pf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pf_[a-z_0-9]+)\s*\(", hdr))
    assert {"pf_create", "pf_set_fields", "pf_step_fs", "pf_step_fd", "pf_get_fields", "pf_free_energy",
            "pf_destroy"} <= declared
    L = libpf.lib()
    for name in sorted(declared):
        assert hasattr(L, name), f"{name} declared in pf.h but not exported by libpf.so"
    assert declared == set(libpf.EXPORTS)


def test_params_struct_matches_header_order(libpf):
    hdr = open(os.path.join(ROOT, "include", "pf.h")).read()
    body = hdr[hdr.index("typedef struct {"):hdr.index("} pf_params;")]
    body = re.sub(r"/\*.*?\*/", "", body, flags=re.S)
    names = []
    for decl in body.split(";"):
        decl = decl.replace("typedef struct {", "").strip()
        if not decl:
            continue
        decl = re.sub(r"^(int|double|void)\s*\*?", "", decl)
        names += [re.sub(r"\[.*\]", "", v).strip().lstrip("*") for v in decl.split(",")]
    assert names == [f[0] for f in libpf.PfParams._fields_]


def test_argument_validation_without_gpu(libpf):
    L = libpf.lib()
    h = ctypes.c_void_p()
    assert L.pf_create(None, ctypes.byref(h)) == libpf.PF_EINVAL
    p = libpf.make_params((64, 64), n_eta=2)
    assert L.pf_create(ctypes.byref(p), None) == libpf.PF_EINVAL
    for bad, code in [(dict(n=(64, 48)), libpf.PF_EUNSUPPORTED), (dict(n=(8, 64)), libpf.PF_EUNSUPPORTED),
                      (dict(n=(4096, 64)), libpf.PF_EUNSUPPORTED), (dict(n=(64, 64), dt=0.0), libpf.PF_EINVAL),
                      (dict(n=(64, 64), dx=-1.0), libpf.PF_EINVAL), (dict(n=(64, 64), n_eta=9), libpf.PF_EINVAL),
                      (dict(n=(64, 64), k2_kind=3), libpf.PF_EINVAL), (dict(n=(64, 64), precision=7), libpf.PF_EINVAL)]:
        q = libpf.make_params(**bad)
        assert L.pf_create(ctypes.byref(q), ctypes.byref(h)) == code, bad
    # batched contexts (pf_create_batch): replica count 1..4096, in 3D at most 65535 planes over all replicas; checked before
    # any device is touched
    q = libpf.make_params((64, 64), n_eta=2)
    assert L.pf_create_batch(ctypes.byref(q), 0, ctypes.byref(h)) == libpf.PF_EINVAL
    assert L.pf_create_batch(ctypes.byref(q), 5000, ctypes.byref(h)) == libpf.PF_EINVAL
    assert L.pf_create_batch(None, 4, ctypes.byref(h)) == libpf.PF_EINVAL
    q3 = libpf.make_params((32, 32, 32), n_eta=2)
    assert L.pf_create_batch(ctypes.byref(q3), 4096, ctypes.byref(h)) == libpf.PF_EUNSUPPORTED
    assert L.pf_batch_size(None) == 0
    assert L.pf_step_fs(None, 1) == libpf.PF_EINVAL
    assert L.pf_launch_count(None) == 0
    L.pf_destroy(None)
    assert L.pf_strerror(libpf.PF_ESTATE) == b"no fields set"


def test_no_cpu_fallback_without_device(libpf):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(libpf.PfError) as ei:
        libpf.Context((64, 64), n_eta=2)
    assert ei.value.code == libpf.PF_ECUDA


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2306_04322_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "pfo.h" not in src, f
