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
