"""The data movement of the 3-pass ("T1") structure at C3, measured (profiles/r2_05_dsmem_t1.md):
tests/host/dsmem_plane_exchange.cu holds one pair plane in an 8-CTA cluster and gathers / scatters the z columns through
distributed shared memory.  The test checks that the round trip returns every element (with the stand-in transform's
sign) and prints the measured time per plane."""
import os
import shutil
import subprocess

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_plane_exchange_through_distributed_shared_memory(tmp_path, capsys):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc) and shutil.which("nvcc") is None:
        pytest.skip("nvcc not available")
    exe = str(tmp_path / "dsmem_plane_exchange")
    src = os.path.join(ROOT, "tests", "host", "dsmem_plane_exchange.cu")
    subprocess.run([nvcc if os.path.exists(nvcc) else "nvcc", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-o", exe, src],
                   check=True, capture_output=True)
    r = subprocess.run([exe], capture_output=True, text=True, timeout=120)
    assert r.returncode == 0 and r.stdout.startswith("OK"), r.stdout + r.stderr
    with capsys.disabled():
        print("\n[t1 exchange] " + r.stdout.strip())
