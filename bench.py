#!/usr/bin/env python
"""bench.py -- SSFM throughput of libshg on B200 (BASELINE.json metric: grid-point z-steps per second).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg5] [--impl reference]

A "step" is one pass of the whole hot path over one workload: one shg_propagate (opening half-step, the nz
fused z-steps, closing half-step, power history) of the named BASELINE.json config on synthetic seeded input.
Prints ONE JSON line (rank 0).  See DESIGN.md §7 for what each key means and how the roofline numbers are
formed.  `--impl reference` times the CPU oracle (oracle/, fp64, as it stands) on the host cores instead.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ssfm_grid_point_z_steps_per_s"
UNIT = "pt-steps/s"
NOMINAL_HBM_GBS = 8000.0            # the ~8 TB/s BASELINE.json names (context only)
FALLBACK_HBM_GBS = 6650.0           # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
# fp32 FMA peak for the "alu" side figure: 148 SMs x 128 lanes x 2 flop x 1.965 GHz
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg5", help="cfg2 | cfg3 | cfg4 | cfg5 (default: the largest single-GPU config) | stream256 | stream1024 "
                         "(sweeps whose field state is larger than L2)")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--nz", type=int, default=None, help="override the z-step count (profiling runs only; "
                    "a number measured with --nz is not the config's)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--per-pass", action="store_true", help="two launches per z-step instead of the persistent kernel")
    ap.add_argument("--opt", action="append", default=[], metavar="K=V",
                    help="shg_set_option(K, V) before the run (option numbers of include/shg.h; measurements only)")
    ap.add_argument("--no-others", action="store_true",
                    help="skip the short timed runs of the other workloads (key other_workloads)")
    ap.add_argument("--shard-members", action="store_true",
                    help="N > 1 with a batched workload: split the members over the ranks (strong scaling) instead "
                         "of running one replica per rank")
    return ap.parse_args()


def measured_peak_hbm():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy kernel)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic_bytes(workload: str, nz: int):
    """(bytes, source): dram__bytes_read.sum + dram__bytes_write.sum of the dominant kernel, per launch, from the
    committed ncu capture (profiles/roofline_traffic.csv: workload,nz,kernel,dram_bytes_per_launch,kernel_digest).
    A row counts only when its digest is the one of the device code being timed (build.kernel_digest()): a capture
    of other code gives bytes = None."""
    from paper_2410_04994_b200 import build as shg_build
    p = os.path.join(ROOT, "profiles", "roofline_traffic.csv")
    if not os.path.exists(p):
        return None, "no capture (profiles/roofline_traffic.csv is missing)"
    dig = shg_build.kernel_digest()
    for line in open(p):
        f = [s.strip() for s in line.split(",")]
        if len(f) >= 4 and f[0] == workload and f[1].isdigit():
            if len(f) < 5 or f[4] != dig:
                return None, ("stale: the capture in profiles/roofline_traffic.csv is of kernel sources %s, this build "
                              "is %s" % (f[4] if len(f) >= 5 else "without a digest", dig))
            # scale linearly in the z-step count when the capture used a shorter run of the same kernel
            return float(f[3]) * nz / int(f[1]), (
                "static: ncu dram__bytes_read.sum + dram__bytes_write.sum of this kernel in the capture committed as "
                "profiles/roofline_traffic.csv (same kernel sources, digest %s; not re-measured in this run)" % dig)
    return None, "no capture of this workload in profiles/roofline_traffic.csv"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.f = None
        self.p = None

    def start(self):
        try:
            self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None
        return self

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw = [], [], []
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.f:
            c = [s.strip() for s in line.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        try:
            os.unlink(self.f.name)
        except OSError:
            pass
        if sm:
            # "under load" = samples at or above the median (the sampler also sees the gaps between steps)
            s = sorted(sm)
            out.update(sm_mhz=s[len(s) // 2], sm_max_mhz=max(mx), power_w_max=max(pw), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


# ------------------------------------------------------------------------------------------------
# CPU oracle timing (reported baseline; the oracle as it stands, never tuned for this)
# ------------------------------------------------------------------------------------------------
def time_oracle_sample(w_full, budget_s: float, nz_probe: int = 1):
    """Time oracle.propagate on a bounded sample of the workload: the same grid, crystal, beams, input field
    and temperature array, but only `nz_s` z-steps (dz = L/nz_s), nz_s chosen from a 1-step probe so that the
    run takes about `budget_s` seconds.  Returns (pt_steps_per_s, cores, description, seconds)."""
    import numpy as np
    import oracle
    from paper_2410_04994_b200 import workloads as wl

    g = w_full["grid"]
    # members: a sweep is sampled by its first members (they are independent)
    nb = min(g["batch"], 4)
    npts = g["nx"] * g["ny"] * nb

    def run(nz_s):
        ws = wl.make(w_full["name"], nz=nz_s, batch=nb) if w_full["name"] == "cfg4" else \
            (w_full if nz_s == g["nz"] else _with_nz(w_full, nz_s))
        o = oracle.Oracle(ws["grid"], ws["crystal"], ws["beams"])
        o.set_temperature(ws["T"], ws["T_uniform"], ws["per_member"])
        a1 = ws["A1"].astype(np.complex128)
        t0 = time.perf_counter()
        o.propagate(a1)
        dt = time.perf_counter() - t0
        o.close()
        return dt

    t_probe = run(nz_probe)
    per_step = max(t_probe / nz_probe, 1e-6)
    nz_s = int(max(1, min(g["nz"], budget_s / per_step)))
    dt = run(nz_s) if nz_s > nz_probe else t_probe
    if nz_s <= nz_probe:
        nz_s = nz_probe
    desc = ("%s grid %dx%d, %d member(s), same input field and temperature array, rerun with "
            "%d of %d z-steps (%.1f s)" % (w_full["name"], g["nx"], g["ny"], nb, nz_s, g["nz"], dt))
    return npts * nz_s / dt, oracle.num_threads(), desc, dt


def cpu_context():
    """Host CPU model and the oracle's build line, for the reported CPU baseline."""
    model = "unknown"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count(), "build": "gcc -O2 -std=c99 -fopenmp (no -ffast-math)"}


def _with_nz(w, nz_s):
    """Same workload with a different z-step count.  Configs whose T planes sit on the step nodes (nzt = nz+1)
    are regenerated; a fixed-plane-count T (cfg5) is reused as is (it is interpolated in z)."""
    from paper_2410_04994_b200 import workloads as wl
    g = w["grid"]
    if g["nzt"] == g["nz"] + 1:
        return wl.make(w["name"], nz=nz_s)
    out = dict(w)
    out["grid"] = dict(g, nz=nz_s)
    return out


def run_reference(args):
    """--impl reference: the oracle on the host cores, same config / metric / unit; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2410_04994_b200 import workloads as wl
    import oracle
    oracle.build()
    w = wl.make(args.workload, nz=args.nz)
    total = max(1, args.steps + args.warmup)
    budget = min(20.0, 150.0 / total)          # whole run ends within a few minutes
    vals, desc, cores = [], "", 1
    for i in range(total):
        v, cores, desc, dt = time_oracle_sample(w, budget)
        if i >= args.warmup:
            vals.append((v, dt))
    value = sum(v for v, _ in vals) / len(vals)
    g = w["grid"]
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(d for _, d in vals) / len(vals),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": workload_label(w), "nx": g["nx"], "ny": g["ny"], "nz": g["nz"], "batch": g["batch"],
                   "nzt": g["nzt"]},
        "cpu_baseline": dict({"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc},
                             **cpu_context()),
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


def workload_label(w):
    labels = {"cfg1": "BASELINE.json configs[0]: 64x64, 200 z-steps",
              "cfg2": "BASELINE.json configs[1]: 128x128, 1000 z-steps, absorption + T array",
              "cfg3": "BASELINE.json configs[2]: 256x256, 4000 z-steps, T array",
              "cfg4": "BASELINE.json configs[3]: 64 x (128x128, 1000 z-steps) parameter sweep",
              "cfg5": "BASELINE.json configs[4]: 1024x1024, 10000 z-steps, 1 GiB T array",
              "stream256": "throughput regime (SURVEY 8(f) rank 3): 192 x (256x256), 201 MB of fields > L2",
              "stream1024": "throughput regime (SURVEY 8(f) rank 3): 16 x (1024x1024), 268 MB of fields > L2"}
    return labels.get(w["name"], w["name"])


# ------------------------------------------------------------------------------------------------
# B200 arm
# ------------------------------------------------------------------------------------------------
def kernel_label(ctx, g, per_pass):
    k = ctx.last_kernel()
    if k == 4:
        return "k_cluster<%d,%d>" % (g["nx"], ctx.last_cluster_size())
    names = {1: "k_persist", 2: "k_persist_flat", 3: "k_persist_pipe", 5: "k_persist_paper"}
    if k in names:
        return "%s<%d>" % (names[k], g["nx"])
    return "k_row+k_col"


def time_workload(name, steps, warmup, args, sync, nz=None, members=None):
    """Device-resident timing of `steps` propagates of one workload (after `warmup`): returns the numbers the JSON
    line is built from.  members = (rank, world): run only this rank's share of a batched workload."""
    import torch
    from paper_2410_04994_b200 import shg
    from paper_2410_04994_b200 import workloads as wl
    from paper_2410_04994_b200.sharding import shard_workload

    w = wl.make(name, nz=nz)
    if members is not None:
        w = shard_workload(w, *members)
    g = w["grid"]
    B = g["batch"]
    pts = g["nx"] * g["ny"] * g["nz"] * B
    ctx = shg.Shg(g, w["crystal"], w["beams"], persistent=not args.per_pass)
    for kv in args.opt:
        k, v = kv.split("=")
        ctx.set_option(int(k), int(v))
    ctx.enable_timing(True)
    stream = torch.cuda.current_stream()
    A1 = torch.from_numpy(w["A1"]).cuda()
    Td = None
    if g["nzt"] > 0:
        Td = torch.from_numpy(w["T"]).cuda()
        ctx.set_temperature(Td, per_member=w["per_member"])
    else:
        ctx.set_temperature(None, w["T_uniform"])
    O1, O2 = torch.empty_like(A1), torch.empty_like(A1)
    for _ in range(warmup):
        ctx.propagate(A1, None, O1, O2)
    sync()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    ev[0].record(stream)
    for _ in range(steps):
        ctx.propagate(A1, None, O1, O2)
    ev[1].record(stream)
    sync()
    ctx.synchronize()                                  # reports a failed run (barrier timeout) instead of timing it
    return dict(w=w, g=g, B=B, pts=pts, ctx=ctx, A1=A1, Td=Td, O1=O1, O2=O2, stream=stream,
                ms_total=ev[0].elapsed_time(ev[1]), main_loop_ms=ctx.last_main_loop_ms(),
                launches=ctx.last_launch_count(), kernel=kernel_label(ctx, g, args.per_pass))


def roofline_of(r, fp32_measured, fp32_distinct, traffic):
    """The dominant kernel's roofline entry: algorithmic flops (or bytes) of one launch over the
    CUDA-event time of the z-loop kernel."""
    from paper_2410_04994_b200 import workloads as wl
    peak, peak_src = measured_peak_hbm()
    w, pts = r["w"], r["pts"]
    b_alg = wl.algorithmic_bytes_per_point_step(w)
    f_alg = wl.algorithmic_flops_per_point_step(w)
    t_loop = r["main_loop_ms"] * 1e-3
    achieved_tf = f_alg * pts / t_loop / 1e12
    achieved = b_alg * pts / t_loop / 1e9
    return {
        "bound": "alu", "achieved": achieved_tf, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
        "frac": achieved_tf / FP32_PEAK_TFLOPS, "traffic": traffic[0], "traffic_source": traffic[1],
        "peak_source": "derived: 148 SMs x 128 fp32 lanes x 2 flops x 1.965 GHz (DESIGN.md 7)",
        "kernel": r["kernel"], "kernel_ms_per_launch": r["main_loop_ms"],
        "us_per_z_step": 1e3 * r["main_loop_ms"] / r["g"]["nz"],
        "algorithmic_flops_per_pt_step": f_alg,
        "fp32_peak_tflops_measured": fp32_measured,
        # FFMA with three distinct register operands (what butterflies and RK4 stages are): the register file feeds
        # ~2/3 of the operand-reuse rate, so this is the ceiling the kernel's instruction mix can actually reach
        "fp32_peak_tflops_measured_distinct_operands": fp32_distinct,
        "frac_of_distinct_operand_peak": (achieved_tf / fp32_distinct) if fp32_distinct else None,
        "hbm": {"achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "peak_source": peak_src,
                "algorithmic_bytes_per_pt_step": b_alg, "frac_of_nominal_8TBs": achieved / NOMINAL_HBM_GBS,
                "two_pass_traffic_GBs": None if r["kernel"].startswith("k_cluster") else
                (b_alg + 32.0) * pts / t_loop / 1e9},
        "note": "the field state (<= 16 MB) is L2-resident (k_cluster: shared-memory-resident) across z-steps, so "
                "dram bytes are far below the algorithmic bytes",
    }


def run_b200(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2410_04994_b200 import shg
    from paper_2410_04994_b200 import workloads as wl
    from paper_2410_04994_b200.sharding import gather_member_values

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # Default: every rank runs one full replica of the workload (simulations are independent: no data-path
    # collective; weak scaling).  --shard-members: the members of a sweep are split over the ranks (strong
    # scaling), the efficiency map is gathered at the end.  DESIGN.md 8.
    shard = args.shard_members and world > 1
    if shard and wl.make(args.workload, nz=1)["grid"]["batch"] < world:
        raise SystemExit("bench.py --shard-members: %s has fewer members than ranks (%d)" % (args.workload, world))
    sampler = ClockSampler(local).start() if rank == 0 else None
    r = time_workload(args.workload, args.steps, args.warmup, args, barrier, nz=args.nz,
                      members=(rank, world) if shard else None)
    clocks = sampler.stop() if sampler else None
    w, g, B, ctx, stream = r["w"], r["g"], r["B"], r["ctx"], r["stream"]
    launches = r["launches"] * args.steps
    eta_local = np.array([ctx.efficiency(b) for b in range(B)])
    t = torch.tensor([r["ms_total"]], dtype=torch.float64, device="cuda")
    pts_all = torch.tensor([float(r["pts"])], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        if shard:
            dist.all_reduce(pts_all, op=dist.ReduceOp.SUM)
        else:
            pts_all *= world
    ms_step = float(t.item()) / args.steps
    value = float(pts_all.item()) / (ms_step * 1e-3)
    eta_map = None
    if shard:
        total_members = int(round(float(pts_all.item()) / (g["nx"] * g["ny"] * g["nz"])))
        eta_map = gather_member_values(eta_local, total_members, rank, world)

    # ---- end to end through the host-buffer entry points: pinned host inputs -> device -> result on the host
    def time_e2e(ctx, w, g, B, stream, steps, warmup):
        """ms for `steps` end-to-end steps (host temperature array + host fields in, fields + history out), and
        the bytes moved per step."""
        hA1 = torch.from_numpy(w["A1"]).pin_memory()
        hO1, hO2 = torch.empty_like(hA1).pin_memory(), torch.empty_like(hA1).pin_memory()
        hT = torch.from_numpy(w["T"]).pin_memory() if g["nzt"] > 0 else None
        h2d = hA1.numel() * 8 + (hT.numel() * 4 if hT is not None else 0)
        d2h = 2 * hA1.numel() * 8 + B * (g["nz"] + 1) * 2 * 8

        def e2e_step():
            if hT is not None:
                ctx.set_temperature(hT, per_member=w["per_member"], stream=stream)
            else:
                ctx.set_temperature(None, w["T_uniform"])
            ctx.propagate_host(hA1, None, hO1, hO2, stream=stream)
            return ctx.power_history(0)            # synchronises the stream and reads the history back

        for _ in range(warmup):
            e2e_step()
        barrier()
        t0 = time.perf_counter()
        ev2 = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        ev2[0].record(stream)
        for _ in range(steps):
            e2e_step()
        ev2[1].record(stream)
        barrier()
        wall_ms = (time.perf_counter() - t0) * 1e3
        # host work (history read-back) sits between device work, so take the larger of the two clocks
        return max(ev2[0].elapsed_time(ev2[1]), wall_ms), h2d, d2h

    e2e = None
    if not args.no_e2e:
        ms_e2e, h2d, d2h = time_e2e(ctx, w, g, B, stream, args.steps, max(1, min(args.warmup, 2)))
        t2 = torch.tensor([ms_e2e], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t2, op=dist.ReduceOp.MAX)
        e2e = {"value": float(pts_all.item()) / (float(t2.item()) / args.steps * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": float(t2.item()) / args.steps,
               "api": "shg_set_temperature_host + shg_propagate_host + shg_power_history (pinned host buffers)"}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (the z-loop kernel: k_persist / k_cluster, or the k_row/k_col pairs)
    from paper_2410_04994_b200 import diag              # libshg_diag.so: measuring equipment, not the product library
    fp32_measured = diag.measure_fp32_peak()            # register-only FFMA kernel, CUDA events
    fp32_distinct = diag.measure_fp32_peak_distinct()
    roofline = roofline_of(r, fp32_measured, fp32_distinct, ncu_traffic_bytes(w["name"], g["nz"]))

    cpu = None
    if not args.no_cpu_baseline and world == 1:
        import oracle
        oracle.build()
        v, cores, desc, dt = time_oracle_sample(w, 15.0)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
        cpu.update(cpu_context())
        # the same oracle on one thread (single-thread and all-core figures), a shorter sample
        oracle.set_num_threads(1)
        try:
            v1, _, desc1, _ = time_oracle_sample(w, 6.0)
        finally:
            oracle.set_num_threads(cores)
        cpu["single_thread"] = {"value": v1, "sample": desc1}

    # ---- the other workloads, briefly (same timing method; BASELINE.json names "the 256x256-and-larger configs",
    # SURVEY 7 H2 asks for the batched runs): device-resident, 3 warm-ups + 3 timed propagates each
    others = None
    if not args.no_others and world == 1 and args.nz is None and not args.opt:
        ctx.close()
        del r
        torch.cuda.empty_cache()
        others = {}
        for name in ("cfg1", "cfg2", "cfg3", "cfg4", "cfg5", "stream256", "stream1024"):
            if name == args.workload:
                continue
            smp = ClockSampler(local).start()
            ro = time_workload(name, 3, 3, args, barrier)
            ck = smp.stop()
            rf = roofline_of(ro, fp32_measured, fp32_distinct, ncu_traffic_bytes(name, ro["g"]["nz"]))
            others[name] = {
                "workload": workload_label(ro["w"]), "value": ro["pts"] / (ro["ms_total"] / 3 * 1e-3), "unit": UNIT,
                "ms_per_step": ro["ms_total"] / 3, "us_per_z_step": rf["us_per_z_step"], "kernel": ro["kernel"],
                "roofline_frac": rf["frac"], "frac_of_distinct_operand_peak": rf["frac_of_distinct_operand_peak"],
                "hbm_frac": rf["hbm"]["frac"], "two_pass_traffic_GBs": rf["hbm"]["two_pass_traffic_GBs"],
                "gpu_launches_per_step": ro["launches"], "eta_member0": ro["ctx"].efficiency(0),
                "e2e": None,
                "clocks": {k: ck.get(k) for k in ("sm_mhz", "sm_max_mhz", "reasons")},
            }
            if not args.no_e2e:
                # the same end-to-end measurement as the headline's, 1 warm-up + 2 timed steps
                ms2, h2d_o, d2h_o = time_e2e(ro["ctx"], ro["w"], ro["g"], ro["B"], ro["stream"], 2, 1)
                others[name]["e2e"] = {"value": ro["pts"] / (ms2 / 2 * 1e-3), "unit": UNIT, "ms_per_step": ms2 / 2,
                                       "h2d_bytes_per_step": int(h2d_o), "d2h_bytes_per_step": int(d2h_o)}
            ro["ctx"].close()
            del ro
            torch.cuda.empty_cache()

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if shard else "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_label(w), "nx": g["nx"], "ny": g["ny"], "nz": g["nz"], "batch": B,
                   "nzt": g["nzt"], "launch": "per-pass" if args.per_pass else "persistent",
                   "parallelism": ("members sharded over %d ranks, no data-path collective" % world) if shard else
                                  ("replicas x%d (no collective)" % world),
                   "l2": "inputs larger than L2 where the config has a T array (cfg5: 1 GiB); the 16 MB field state "
                         "is L2-resident by construction of the z-sequential method, no flush between steps"},
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
        "eta_member0": float(eta_local[0]),
        "other_workloads": others,
        "paper_context": "paper reports GPU/CPU speedup only: ~40x (17-43x), GTX 1650 vs i7-9700 (PAPER.md:13,272,312)",
    }
    if eta_map is not None:
        line["eta_map"] = [float(x) for x in eta_map]
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
