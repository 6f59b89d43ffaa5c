"""Build libshg.so (the C-ABI CUDA library) in-tree for sm_100a with nvcc.

    python -m paper_2410_04994_b200.build [--force] [--verbose]

One object per line length (64..1024) plus the host API, compiled in parallel, linked into
``paper_2410_04994_b200/libshg.so``.  nvcc cross-compiles without a GPU.  Environment: ``NVCC`` (compiler
path), ``SHG_NVCC_EXTRA`` (extra nvcc flags, e.g. ``-Xptxas -v`` or a ``-D`` for an experiment).
"""
from __future__ import annotations

import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
LIB = os.path.join(HERE, "libshg.so")
LIB_DIAG = os.path.join(HERE, "libshg_diag.so")   # bench.py's measuring equipment (include/shg_diag.h), not the product
SIZES = (64, 128, 256, 512, 1024)
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
         "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"] + os.environ.get("SHG_NVCC_EXTRA", "").split()


def _sources():
    deps = [os.path.join(CSRC, f) for f in sorted(os.listdir(CSRC))]
    deps.append(os.path.join(os.path.dirname(HERE), "include", "shg.h"))
    deps.append(os.path.join(os.path.dirname(HERE), "include", "shg_diag.h"))
    return deps


def _digest() -> str:
    h = hashlib.sha256()
    for p in _sources():
        with open(p, "rb") as f:
            h.update(p.encode() + b"\0" + f.read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()


KERNEL_SOURCES = ("fft_reg.cuh", "shg_device.cuh", "shg_cluster.cuh", "shg_inst.cu", "shg_params.h", "shg_launch.h")


def kernel_digest() -> str:
    """16 hex digits that name the device code of the z-loop kernels (sources + compiler flags).  Written next to each
    row of profiles/roofline_traffic.csv, so that bench.py can tell whether an ncu capture belongs to the code it times."""
    h = hashlib.sha256()
    for f in KERNEL_SOURCES:
        with open(os.path.join(CSRC, f), "rb") as fh:
            h.update(f.encode() + b"\0" + fh.read())
    h.update(" ".join(FLAGS).encode())
    return h.hexdigest()[:16]


def _run(cmd, verbose):
    if verbose:
        print(" ".join(cmd), flush=True)
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stdout + r.stderr


def build(force: bool = False, verbose: bool = False, ptxas_info: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    stamp = os.path.join(OBJ, "stamp")
    dig = _digest()
    if not force and os.path.exists(LIB) and os.path.exists(LIB_DIAG) and os.path.exists(stamp) and open(stamp).read() == dig:
        return LIB
    extra = ["-Xptxas", "-v"] if ptxas_info else []
    jobs = []
    for n in SIZES:
        o = os.path.join(OBJ, "shg_inst_%d.o" % n)
        jobs.append(([NVCC, *FLAGS, *extra, "-DSHG_N=%d" % n, "-c", os.path.join(CSRC, "shg_inst.cu"), "-o", o], o))
    for name in ("shg_api", "shg_static"):
        o = os.path.join(OBJ, name + ".o")
        jobs.append(([NVCC, *FLAGS, *extra, "-c", os.path.join(CSRC, name + ".cu"), "-o", o], o))
    diag_o = os.path.join(OBJ, "shg_diag.o")
    diag_job = ([NVCC, *FLAGS, *extra, "-c", os.path.join(CSRC, "shg_diag.cu"), "-o", diag_o], diag_o)
    logs = []
    with cf.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
        for out in ex.map(lambda j: _run(j[0], verbose), jobs + [diag_job]):
            logs.append(out)
    tmp = LIB + ".%d.tmp" % os.getpid()
    _run([NVCC, "-shared", "-o", tmp, *[j[1] for j in jobs], "-cudart", "static"], verbose)
    os.replace(tmp, LIB)
    tmp = LIB_DIAG + ".%d.tmp" % os.getpid()
    _run([NVCC, "-shared", "-o", tmp, diag_o, "-cudart", "static"], verbose)
    os.replace(tmp, LIB_DIAG)
    with open(stamp, "w") as f:
        f.write(dig)
    if ptxas_info:
        print("\n".join(logs))
    return LIB


if __name__ == "__main__":
    if "--kernel-digest" in sys.argv:
        print(kernel_digest())
        sys.exit(0)
    path = build(force="--force" in sys.argv, verbose="--verbose" in sys.argv, ptxas_info="--ptxas" in sys.argv)
    print(path)
