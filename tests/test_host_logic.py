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


def test_byte_model_of_the_roofline():
    """bench.py: stage_bytes is the 5-pass (T2) byte model of SURVEY.md 8(d) that the roofline fractions are computed
    from: C3 fp32 1.42 GB per apply with 507 MB in the z stage, 338 B per cell; one-cell-thick meshes have no z padding."""
    import sys
    sys.path.insert(0, ROOT)
    import bench
    sb = bench.stage_bytes((256, 256, 64), 4)
    nc = 256 * 256 * 64
    assert sb[0] == sb[4] == 3 * nc * 4 + 3 * 257 * 64 * 256 * 8
    assert sb[1] == sb[3] == 3 * 257 * 64 * 256 * 8 + 3 * 257 * 64 * 512 * 8
    assert sb[2] == 2 * 3 * 257 * 64 * 512 * 8 + 6 * 257 * 257 * 65 * 4 == 507262488
    assert sum(sb) == 1416377880 and 337 < sum(sb) / nc < 339
    assert sum(bench.stage_bytes((256, 256, 64), 8)) == 2 * sum(sb)
    film = bench.stage_bytes((1024, 1024, 1), 4)
    assert film[2] == 2 * 3 * 1025 * 2048 * 8 + 6 * 1025 * 1025 * 4          # Nz = 1: no z padding, kpz = 1
