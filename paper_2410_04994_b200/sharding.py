"""Multi-GPU plumbing.  Batch members are independent simulations (no exchange step anywhere in the
path), so a sweep is sharded by member across ranks with NO data-path collective; the only communication
is gathering the per-member efficiencies (a few doubles) at the end.  A single simulation does not shard
(two all-to-all transposes per z-step over <= 16 MB of state would be latency bound): "replicas only".
"""
from __future__ import annotations

import numpy as np


def member_range(n_members: int, rank: int, world: int) -> range:
    """Contiguous, balanced split: the first (n_members % world) ranks get one extra member."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    base, extra = divmod(n_members, world)
    lo = rank * base + min(rank, extra)
    return range(lo, lo + base + (1 if rank < extra else 0))


def shard_workload(w: dict, rank: int, world: int) -> dict:
    """The slice of a batched workload (workloads.make output) that `rank` owns."""
    r = member_range(w["grid"]["batch"], rank, world)
    out = dict(w)
    out["beams"] = [w["beams"][b] for b in r]
    out["A1"] = w["A1"][r.start:r.stop]
    out["grid"] = dict(w["grid"], batch=len(r))
    if w.get("T") is not None and w.get("per_member"):
        out["T"] = w["T"].reshape(w["grid"]["batch"], -1)[r.start:r.stop]
    out["members"] = r
    return out


def gather_member_values(local: np.ndarray, n_members: int, rank: int, world: int, group=None) -> np.ndarray:
    """All ranks receive the full per-member vector (e.g. the efficiency map of a sweep).
    Uses torch.distributed (nccl or gloo) when world > 1; identity otherwise."""
    local = np.asarray(local, dtype=np.float64)
    if world == 1:
        return local.copy()
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    sizes = [len(member_range(n_members, r, world)) for r in range(world)]
    pad = max(sizes)
    buf = torch.zeros(pad, dtype=torch.float64, device=dev)
    buf[:len(local)] = torch.from_numpy(local).to(dev)
    outs = [torch.zeros(pad, dtype=torch.float64, device=dev) for _ in range(world)]
    dist.all_gather(outs, buf, group=group)
    return np.concatenate([o[:s].cpu().numpy() for o, s in zip(outs, sizes)])


def _member_efficiencies(part: dict, options=None, stream=None) -> np.ndarray:
    """Propagate the members of `part` on the current CUDA device and return their SH conversion efficiencies."""
    import torch
    from . import shg
    g = part["grid"]
    ctx = shg.Shg(g, part["crystal"], part["beams"])
    try:
        for k, v in (options or {}).items():
            ctx.set_option(k, v)
        if g["nzt"] > 0:
            T = part["T"]
            ctx.set_temperature(T if isinstance(T, torch.Tensor) and T.is_cuda else torch.from_numpy(np.ascontiguousarray(T)).cuda(),
                                per_member=part["per_member"])
        else:
            ctx.set_temperature(None, part["T_uniform"])
        A1 = torch.from_numpy(np.ascontiguousarray(part["A1"])).cuda()
        if stream is not None:
            # the uploads above ran on torch's current stream: the propagate on `stream` must come after them
            stream.wait_stream(torch.cuda.current_stream())
        ctx.propagate(A1, stream=stream)
        ctx.synchronize()
        return np.array([ctx.efficiency(b) for b in range(g["batch"])])
    finally:
        ctx.close()


def sweep(w: dict, rank: int = 0, world: int = 1, group=None, options=None, stream=None) -> np.ndarray:
    """A parameter sweep (BASELINE.json configs[3]; the paper runs one simulation per process): propagate
    this rank's share of the members of the batched workload `w` (workloads.make output) in ONE launch sequence of
    libshg and return the SH conversion efficiency P2(L) / (P1(0) + P2(0)) of EVERY member on every rank.
    options: {shg.OPT_*: value}.  A rank whose share is empty (fewer members than ranks) propagates nothing and
    still takes part in the gather.  Needs the CUDA library; there is no other path."""
    part = shard_workload(w, rank, world) if world > 1 else w
    if part["grid"]["batch"] == 0:
        local = np.empty(0, dtype=np.float64)
    else:
        local = _member_efficiencies(part, options, stream)
    return gather_member_values(local, w["grid"]["batch"], rank, world, group)
