#!/usr/bin/env python
"""Writes tests/golden/cfg5_oracle_summary.json: what the CPU oracle (oracle/, fp64) computes for the FULL
BASELINE.json config 5 (1024 x 1024, 10 000 z-steps, 1 GiB temperature array) -- the run the oracle cannot
repeat inside a test (about 1.5 core-hours).  Calls ONLY oracle/ and the seeded input generator; nothing here
comes from the CUDA path.

    python tests/golden/make_cfg5_golden.py [--nz 10000]

Stored in the .json: SH efficiency, the powers at z = L, the rms amplitude of both output fields, the power
history at every 100th node, and both output fields at 96 seeded sample points.  Stored beside it in
cfg5_oracle_sample.npz: both output fields at 65 536 distinct grid points drawn uniformly from the whole grid with a
fixed seed (flat indices iy * nx + ix in `idx`; complex128 rounded to complex64: 3e-8 relative, against a 2e-4
parity bar), the power sum |A_j|^2 of each of the 16 x 16 tiles of 64 x 64 points (fp64), and the power history at
EVERY node -- the GPU test computes the relative L2 error of each field over the sample, compares the 256 tile
powers per field and all 10 001 history nodes.  (Until round 3 the sample was the lattice iy = 1 + 4 p, ix = 2 + 4 q,
which meets only 8 of the 32 lanes and 2 of the 8 strip columns of the kernels' data layout; a uniform draw meets
every residue of ix and iy modulo 32, and the tile sums see every point.)
Paper passages the oracle follows: see oracle/shg_oracle.c (PAPER.md:72-73 Eq. 2, :136, :157-161).
"""
import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2410_04994_b200 import workloads as wl  # noqa: E402  (input generator only)


SAMPLE_SEED, SAMPLE_N, TILE = 241004994, 65536, 64


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--nz", type=int, default=None)
    ap.add_argument("--out", default=os.path.join(os.path.dirname(os.path.abspath(__file__)),
                                                  "cfg5_oracle_summary.json"))
    a = ap.parse_args()
    w = wl.make("cfg5", nz=a.nz)
    g = w["grid"]
    o = oracle.Oracle(g, w["crystal"], w["beams"])
    o.set_temperature(w["T"], w["T_uniform"], w["per_member"])
    t0 = time.time()
    a1, a2 = o.propagate(w["A1"].astype(np.complex128))
    dt = time.time() - t0
    h = o.power_history(0)
    rng = np.random.default_rng(55)
    n = g["nx"]
    # half of the samples near the beam (where the field is), half anywhere on the grid
    near = rng.integers(n // 2 - n // 8, n // 2 + n // 8, size=(48, 2))
    anyw = rng.integers(0, n, size=(48, 2))
    pts = np.concatenate([near, anyw])
    samples = [[int(iy), int(ix), float(a1[0, iy, ix].real), float(a1[0, iy, ix].imag),
                float(a2[0, iy, ix].real), float(a2[0, iy, ix].imag)] for iy, ix in pts]
    out = {
        "config": "cfg5", "nz": g["nz"], "nx": g["nx"], "ny": g["ny"], "nzt": g["nzt"],
        "oracle_seconds": dt, "oracle_threads": oracle.num_threads(),
        "eta": float(h[-1, 1] / (h[0, 0] + h[0, 1])),
        "P1_0": float(h[0, 0]), "P2_0": float(h[0, 1]), "P1_L": float(h[-1, 0]), "P2_L": float(h[-1, 1]),
        "A1_rms": float(np.sqrt(np.mean(np.abs(a1) ** 2))), "A2_rms": float(np.sqrt(np.mean(np.abs(a2) ** 2))),
        "A1_l2": float(np.linalg.norm(a1.ravel())), "A2_l2": float(np.linalg.norm(a2.ravel())),
        "history_stride": 100, "history": h[::100].tolist(),
        "samples": samples,
    }
    with open(a.out, "w") as f:
        json.dump(out, f, indent=1)
    smp = a.out.replace("_summary.json", "_sample.npz")
    ny, nx = g["ny"], g["nx"]
    idx = np.sort(np.random.default_rng(SAMPLE_SEED).choice(ny * nx, SAMPLE_N, replace=False)).astype(np.int32)

    def tiles(f):
        return (np.abs(f) ** 2).reshape(ny // TILE, TILE, nx // TILE, TILE).sum(axis=(1, 3))
    np.savez_compressed(smp, seed=SAMPLE_SEED, idx=idx, tile=TILE,
                        A1=a1[0].ravel()[idx].astype(np.complex64), A2=a2[0].ravel()[idx].astype(np.complex64),
                        tiles1=tiles(a1[0]), tiles2=tiles(a2[0]),
                        history=np.asarray(h, dtype=np.float64))
    print("wrote %s (%.0f s on %d threads): eta = %.9f" % (a.out, dt, out["oracle_threads"], out["eta"]))


if __name__ == "__main__":
    main()
