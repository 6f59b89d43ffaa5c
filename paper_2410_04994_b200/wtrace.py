"""Per-warp timeline of the row pass (diagnostic, needs a library built with the SHG_WTRACE stamps):

    SHG_NVCC_EXTRA=-DSHG_WTRACE python -m paper_2410_04994_b200.build --force
    python -m paper_2410_04994_b200.wtrace [cfg5] [OPTION=VALUE ...]
    python -m paper_2410_04994_b200.build --force          # back to the product build

In that build lane 0 of every warp stamps the SM clock at eight points of its row item of z-steps 100..163 into the
tail of the SHG_OPT_TRACE buffer (csrc/shg_device.cuh: SHG_WT).  This module runs one propagate of a single
simulation with 4100 z-steps, reads the buffer and prints, for the CTAs that hold the most rows, the mean stamp of
every warp relative to the release of the device-wide barrier before the pass.  (A clock read after a bar.sync is
the time the barrier was ISSUED, not released: read the barrier columns with that in mind.)  profiles/r02b_summary.md
quotes its output.
"""
from __future__ import annotations

import sys

import numpy as np

NAMES = ["item starts", "loads issued", "F_x^-1 done", "lines in smem, pair barrier issued", "nonlinear step done",
         "pair barrier 2 issued", "F_x done", "hx multiply done, stores issued"]


def main(argv):
    import torch
    from . import shg, workloads as wl

    name = argv[0] if argv and "=" not in argv[0] else "cfg5"
    w = wl.make(name, nz=4100)
    assert w["grid"]["batch"] == 1
    ctx = shg.Shg(w["grid"], w["crystal"], w["beams"])
    ctx.set_option(shg.OPT_TRACE, 4096)
    ctx.set_option(shg.OPT_CLUSTER, 0)
    for a in argv:
        if "=" in a:
            k, v = a.split("=")
            ctx.set_option(int(k), int(v))
    if w["grid"]["nzt"] > 0:
        Td = torch.from_numpy(w["T"]).cuda()
        ctx.set_temperature(Td)
    else:
        ctx.set_temperature(None, w["T_uniform"])
    A1 = torch.from_numpy(w["A1"]).cuda()
    for _ in range(2):
        ctx.propagate(A1)
        torch.cuda.synchronize()
    raw = ctx.read_trace()
    G = raw.shape[1]
    tr = raw.reshape(-1)
    base = tr[:200 * G * 8].reshape(200, G, 2, 4)
    wt = tr[200 * G * 8: 200 * G * 8 + 64 * G * 16 * 8].reshape(64, G, 16, 8)
    if not wt.any():
        raise SystemExit("no warp stamps in the trace buffer: build the library with SHG_NVCC_EXTRA=-DSHG_WTRACE")
    rel1 = base[99:163, :, 1, 1]            # release of the barrier after the column pass of step n - 1
    arr0 = base[100:164, :, 0, 0]           # the CTA's arrival at the barrier after the row pass of step n
    rows = w["grid"]["ny"] // (2 if w["grid"]["nx"] <= 128 else 1)       # row items (Geo::HG rows each)
    nrow = (rows * (np.arange(G) + 1)) // G - (rows * np.arange(G)) // G
    sel = nrow == nrow.max()
    d = (wt[:, sel] - rel1[:, sel][:, :, None, None]).astype(np.float64)
    busy = [w_ for w_ in range(16) if wt[0, np.nonzero(sel)[0][0], w_].any()]
    print("%s: %d CTAs with %d row items; SM clocks after the barrier release, mean over 64 z-steps and these CTAs"
          % (name, int(sel.sum()), int(nrow.max())))
    print("warp sched " + " ".join("%8d" % i for i in range(8)))
    for w_ in busy:
        print("%4d %5d " % (w_, w_ % 4) + " ".join("%8.0f" % x for x in d[:, :, w_].mean((0, 1))))
    for i, nm in enumerate(NAMES):
        print("[%d] %s" % (i, nm))
    print("CTA arrives at the barrier after the pass: %.0f" % (arr0[:, sel] - rel1[:, sel]).mean())
    ctx.close()


if __name__ == "__main__":
    main(sys.argv[1:])
