"""Short runs of every kernel family of libshg, for compute-sanitizer (memcheck / racecheck / synccheck).

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

Not a pytest file: the parity tests prove the numbers, this only drives each kernel once or twice at a length a
sanitizer gets through in seconds, with the spin limit of the device-wide barriers off (SHG_OPT_SPIN_LIMIT = 0: a
sanitizer slows the kernels by one to two orders of magnitude).  Every case is run twice and the two results must be
the same bits -- a race that the tool does not model (global memory between CTAs) would most likely show up there.
On the B200 pool of round 3 compute-sanitizer is closed (profiles/r03_sanitizer.md has the refusal and what stands in for
it); run without the tool, the script is still a quick self-check of every kernel family.
"""
import os
import sys

import numpy as np
import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
from paper_2410_04994_b200 import shg                      # noqa: E402
from paper_2410_04994_b200 import workloads as wl          # noqa: E402

KERNELS = {0: "k_row + k_col", 1: "k_persist", 2: "k_persist_flat", 3: "k_persist_pipe", 4: "k_cluster",
           5: "k_persist_paper"}

# (label, workload, nz, make() keywords, Shg() keywords, options, heat planes, expected shg_last_kernel or None)
CASES = [
    ("per-pass launches, 128 x 128", "cfg2", 3, {}, {"persistent": False}, {}, 0, 0),
    ("per-pass launches, 1024 x 1024", "cfg5", 2, {}, {"persistent": False}, {}, 0, 0),
    ("cluster kernel, 64 x 64", "cfg1", 4, {}, {}, {}, 0, 4),
    ("cluster kernel, 128 x 128", "cfg2", 3, {}, {}, {}, 0, 4),
    ("cluster kernel, 64 x 64, 8 CTAs", "cfg1", 4, {}, {}, {shg.OPT_CLUSTER: 8}, 0, 4),
    ("persistent dense, 128 x 128 batch 4", "cfg4", 3, {"batch": 4}, {}, {shg.OPT_CLUSTER: 0, shg.OPT_PIPELINE: 0}, 0, None),
    ("persistent dense, 1024 x 1024", "cfg5", 2, {}, {}, {}, 0, 1),
    ("persistent sparse, 256 x 256", "cfg3", 3, {}, {}, {}, 0, 2),
    ("pipelined batched, 128 x 128 batch 5", "cfg4", 3, {"batch": 5}, {}, {shg.OPT_CLUSTER: 0, shg.OPT_PIPELINE: 2}, 0, 3),
    ("pipelined batched, 256 x 256 batch 3", "stream256", 3, {"batch": 3}, {}, {shg.OPT_PIPELINE: 2}, 0, 3),
    ("pipelined batched, 1024 x 1024 batch 2", "stream1024", 2, {"batch": 2}, {}, {shg.OPT_PIPELINE: 2}, 0, 3),
    ("paper's ordering, persistent", "cfg2", 3, {}, {}, {shg.OPT_SCHEME: 1}, 0, 5),
    ("heat output, persistent 128 x 128", "cfg2", 4, {}, {}, {}, 2, None),
    ("heat output, per-pass 256 x 256", "cfg3", 3, {}, {"persistent": False}, {}, 1, 0),
]


def run(label, name, nz, mk, ck, options, nq, want):
    w = wl.make(name, nz=nz, **mk)
    g = w["grid"]
    results = []
    for rep in range(2):
        ctx = shg.Shg(g, w["crystal"], w["beams"], **ck)
        ctx.set_option(shg.OPT_SPIN_LIMIT, 0)
        for k, v in options.items():
            ctx.set_option(k, v)
        if g["nzt"] > 0:
            T = torch.from_numpy(w["T"]).cuda()
            ctx.set_temperature(T, per_member=w["per_member"])
        else:
            ctx.set_temperature(None, w["T_uniform"])
        Q = None
        if nq:
            Q = torch.zeros((g["batch"], nq, g["ny"], g["nx"]), dtype=torch.float32, device="cuda")
            ctx.set_heat_output(Q)
        o1, o2 = ctx.propagate(torch.from_numpy(w["A1"]).cuda())
        ctx.synchronize()
        hist = ctx.power_history(0)
        kern = ctx.last_kernel()
        assert want is None or kern == want, "%s ran %s, expected %s" % (label, KERNELS[kern], KERNELS[want])
        a1, a2 = o1.cpu().numpy(), o2.cpu().numpy()
        assert np.isfinite(a1).all() and np.isfinite(a2).all() and np.isfinite(hist).all(), label
        results.append((a1, a2, hist, None if Q is None else Q.cpu().numpy()))
        ctx.close()
    for x, y in zip(results[0], results[1]):
        assert x is None or np.array_equal(x, y), "%s: two runs differ" % label
    print("ok  %-42s %s" % (label, KERNELS[kern]), flush=True)
    return kern


def main():
    assert torch.cuda.is_available()
    seen = {run(*case) for case in CASES}
    assert seen == set(KERNELS), "kernel families not reached: %s" % sorted(set(KERNELS) - seen)
    # the context-free power integral in static scratch
    A = torch.randn((5, 64, 96, 2), device="cuda")
    out = torch.zeros((5, 2), dtype=torch.float64, device="cuda")
    for _ in range(2):
        shg.field_power_static(torch.view_as_complex(A), None, 1.0, 1.0, out)
    torch.cuda.synchronize()
    assert np.allclose(out[:, 0].cpu().numpy(), (A.double() ** 2).sum(dim=(1, 2, 3)).cpu().numpy(), rtol=1e-12)
    print("ok  shg_field_power_static", flush=True)
    print("all cases done")


if __name__ == "__main__":
    main()
