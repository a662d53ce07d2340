"""Runs the host emulation of the CUDA path's thread-cooperative Stockham FFT (csrc/fft_core.cuh): the
per-thread stage / exchange functions executed phase by phase on the CPU against a naive long-double DFT
(tests/host/fft_core_host_test.cu). Host logic only; no GPU."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_fft_core_emulated_on_host(tmp_path):
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "fft_core_host_test")
    subprocess.run([nvcc, "-std=c++17", "-O1", "-arch=sm_100a", "-diag-suppress", "20011,20014", "-o", exe,
                    os.path.join(ROOT, "tests", "host", "fft_core_host_test.cu")], check=True, capture_output=True)
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout[-3000:]
    assert "ALL OK" in r.stdout


def test_exchange_buffer_index_map_on_host(tmp_path):
    """csrc/col_buf.cuh: the swizzled exchange buffer of the strided kernels addresses every cell once, delivers the
    Stockham scatter to the registers fft_core.cuh expects, and is free of shared-memory bank conflicts."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "col_buf_host_test")
    subprocess.run([nvcc, "-std=c++17", "-O1", "-arch=sm_100a", "-diag-suppress", "20011,20014", "-o", exe,
                    os.path.join(ROOT, "tests", "host", "col_buf_host_test.cu")], check=True, capture_output=True)
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0, r.stdout[-3000:]
    assert "ALL OK" in r.stdout
