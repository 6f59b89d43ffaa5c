"""Probes that back figures quoted in profiles/ (not parity tests): built from committed sources and run on the GPU."""
import os
import shutil
import subprocess

import pytest

pytestmark = pytest.mark.gpu

HERE = os.path.dirname(os.path.abspath(__file__))


def test_dsmem_alltoall_probe(tmp_path):
    """tests/probes/dsmem_alltoall.cu: clocks per all-to-all exchange in a 16-CTA cluster for bulk copies (from one
    warp / one per warp) and for remote stores (profiles/r02a_summary.md section 7).  Asserts only that every
    method moved the right data; the printed table is the measurement."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    exe = str(tmp_path / "dsmem_alltoall")
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-o", exe,
                           os.path.join(HERE, "probes", "dsmem_alltoall.cu")])
    out = subprocess.run([exe], capture_output=True, text=True, timeout=120).stdout
    print(out)
    lines = [l for l in out.splitlines() if l.startswith("method")]
    assert len(lines) == 12
    for l in lines:
        assert "no error" in l and "MISMATCH" not in l, l


def test_fft_issue_rate_probe(tmp_path):
    """tests/probes/fft_issue_rate.cu: throughput of the library's line transform alone for 4..16 warps per SM and the
    warp -> scheduler map (profiles/r02b_summary.md).  The program checks its own ratios (14 warps as slow as 16,
    two warps of one scheduler twice a lone warp); the printed table is the measurement."""
    nvcc = shutil.which("nvcc") or "/usr/local/cuda/bin/nvcc"
    if not os.path.exists(nvcc):
        pytest.skip("nvcc not available on this box")
    exe = str(tmp_path / "fft_issue_rate")
    subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17",
                           "--expt-relaxed-constexpr", "-o", exe, os.path.join(HERE, "probes", "fft_issue_rate.cu")])
    r = subprocess.run([exe], capture_output=True, text=True, timeout=300)
    print(r.stdout)
    assert r.returncode == 0 and "probe ok" in r.stdout, r.stdout[-2000:]
