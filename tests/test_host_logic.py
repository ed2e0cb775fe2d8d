"""Host logic of the CUDA path that needs no GPU: the butterflies and radix schedules of the fast kernel family
(soa_core.cuh is host/device code) are compiled with nvcc for the host and checked against the DFT definition."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_butterflies_and_schedules_on_the_host(tmp_path):
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc) and shutil.which("nvcc") is None:
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "check_soa_core")
    src = os.path.join(ROOT, "tests", "host", "check_soa_core.cu")
    subprocess.run([nvcc if os.path.exists(nvcc) else "nvcc", "-O1", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a",
                    "-o", exe, src], check=True, capture_output=True)
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 0 and r.stdout.strip() == "OK", r.stdout + r.stderr
