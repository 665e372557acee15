#!/usr/bin/env python
"""bench.py — throughput of the subcycled RK4 AMR step on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--mode sub|uniform] [--impl reference]

One "step" = one coarse step of the whole hierarchy (sc_step): every level's RK4 level-steps, all ghost
fills and restrictions. Default workload: BASELINE.json configs[4] ("large scalar-wave hierarchy for the
bandwidth roofline": 6 levels x 256^3, fp64, subcycled), the configuration the metric's "% of HBM
roofline" is quoted on; it fits one GPU (12 GB). Prints ONE JSON line.

N > 1 (launched by torchrun, one rank per GPU): the path does not shard (north_star: one GPU, no
collectives) -> N independent replicas, "scaling": "weak"; NCCL is used only for the barrier and the
max-over-ranks of the device time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_2503_09629_b200 import workloads as wl  # noqa: E402

METRIC = "grid-point updates/s (all levels, fp64 RK4)"
UNIT = "updates/s"


def pick_workload(idx: int, sigma: float = 0.0, cut: int = 1, fd_order: int = 4, opts=None):
    w = {1: wl.cfg1, 2: lambda: wl.cfg2(128), 3: wl.cfg3, 4: wl.cfg4, 5: wl.cfg5}[idx]()
    if cut > 1:
        w = wl.cut_finest(w, cut)
    if fd_order == 8:
        w.ghost, w.fd_order = 4, 8
        w.name += " + 8th-order FD (ghost 4)"
    if sigma:
        w.ko_sigma = sigma
        w.name += f" + Kreiss-Oliger sigma={sigma}"
    for k, v in (opts or {}).items():  # NEXT-3 / NEXT-4 options: ko_order, integrator, outer_bc, interp, vertex, ghost
        if v is not None and v != getattr(w, k):
            setattr(w, k, v)
            w.name += f" + {k}={v}"
    if w.ko_sigma and (w.ko_order == 9 or (w.ko_order == 0 and w.fd_order == 8)) and w.ghost < 5:
        w.ghost = 5  # delta^10 reads five ghost layers
        w.name += " (ghost 5)"
    return w


def workload_opts(args):
    return {"ko_order": args.ko_order, "integrator": args.integrator, "outer_bc": args.outer_bc,
            "interp": args.interp, "vertex": args.vertex, "ghost": args.ghost}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# ------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands on the host cores, bounded sample
# ------------------------------------------------------------------------------------------------
def oracle_sample(w, max_levels: int):
    """The first `max_levels` levels of the workload (same boxes, same inputs, same discretisation)."""
    if w.nlevels <= max_levels:
        return w, f"all {w.nlevels} levels"
    boxes = [b for b in w.boxes if b.level < max_levels]
    s = wl.Workload(w.name + f" [levels 0..{max_levels - 1}]", boxes, w.domain_cells, w.nfields, w.ghost,
                    w.xlo, w.xhi, w.coupling, w.coarse_steps, w.init, ko_sigma=w.ko_sigma, fd_order=w.fd_order)
    for k in ("integrator", "outer_bc", "ko_order", "interp", "vertex"):  # the NEXT-3 / NEXT-4 options
        setattr(s, k, getattr(w, k))
    return s, f"SAMPLE: levels 0..{max_levels - 1} of {w.nlevels} ({'+'.join(str(b.n[0]) + '^3' for b in boxes)})"


def cpu_model() -> str:
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def time_oracle(w, steps: int, warmup: int, sub: bool, max_levels: int, threads: int = 0):
    """The oracle as it stands on `threads` host threads (0 = all), on a bounded sample of the workload."""
    import oracle

    oracle.build()
    allthreads = oracle.max_threads()
    if threads > 0:
        oracle.set_threads(threads)
    s, what = oracle_sample(w, max_levels)
    H = oracle.OracleHierarchy.from_workload(s)
    for _ in range(warmup):
        H.step(s.dt_coarse, sub)
    t0 = time.perf_counter()
    for _ in range(steps):
        H.step(s.dt_coarse, sub)
    dt = time.perf_counter() - t0
    used = oracle.max_threads()
    H.close()
    if threads > 0:
        oracle.set_threads(allthreads)
    upd = s.updates_per_coarse_step(sub) * steps
    return {"value": upd / dt, "unit": UNIT, "cores": used, "kind": "oracle", "cpu": cpu_model(),
            "flags": "g++ -O2 -fopenmp, no fast-math",
            "sample": f"{what}, {steps} coarse step(s), {'subcycled' if sub else 'uniform'}, {dt:.1f} s",
            "_seconds": dt, "_steps": steps, "_levels": s.nlevels, "_updates_per_step": s.updates_per_coarse_step(sub)}


def config_dict(w, sub: bool, world: int):
    """The `config` object of the JSON line; the same for the GPU arm and the reference arm."""
    return {"workload": w.name, "mode": "subcycled" if sub else "uniform", "ghost": w.ghost, "nfields": w.nfields,
            "ko_sigma": w.ko_sigma, "fd_order": w.fd_order, "ko_order": w.ko_order, "integrator": w.integrator,
            "outer_bc": w.outer_bc, "interp": w.interp, "vertex": w.vertex, "dt_coarse": w.dt_coarse,
            "updates_per_step": w.updates_per_coarse_step(sub), "zone_cycles_per_step": w.zone_cycles_per_coarse_step(),
            "l2": "inputs larger than L2 (state and stage buffers of every level stream through once per launch)",
            "parallelism": "replicas only" if world > 1 else "1 GPU"}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = pick_workload(args.config, args.sigma, args.cut_finest, args.fd_order, workload_opts(args))
    sub = args.mode == "sub"
    r = time_oracle(w, max(1, args.steps), min(args.warmup, 1), sub, max_levels=args.oracle_levels)
    ms = 1e3 * r.pop("_seconds") / r.pop("_steps")
    # The config is the GPU arm's (the contract), but what was TIMED is a sample of it: say so in the config itself, so
    # that ms_per_step is never read as the time of the full workload (value is a rate and compares per update).
    cfg = config_dict(w, sub, 1)
    lev, upd = r.pop("_levels"), r.pop("_updates_per_step")
    cfg.update({"sampled": lev < w.nlevels, "sample_levels": lev, "sample_updates_per_step": upd,
                "ms_per_step_is": "one coarse step of the SAMPLE (sample_updates_per_step updates), not of the workload"
                                  if lev < w.nlevels else "one coarse step of the workload"})
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": cfg,
            "note": "CPU oracle (as it stands, all host threads) on a bounded SAMPLE of the workload: " + r["sample"],
            "cpu_baseline": r,
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# clocks sampling
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except Exception:
            self.p.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 6:
                continue
            try:
                sm.append(float(t[0]))
                mx.append(float(t[1]))
            except ValueError:
                continue
            for nm, v in zip(names, t[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
# N > 1: replicas only. The only cross-rank arithmetic of the bench: the step time is
# the MAX over ranks, the value the work of all replicas divided by it.
def max_over_ranks(x: float, dist, device) -> float:
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world: int, units_per_step: float, steps: int, seconds: float) -> float:
    return world * units_per_step * steps / seconds


def run_gpu(args):
    import torch

    import paper_2503_09629_b200 as sc

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — libsubcycle has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    w = pick_workload(args.config, args.sigma, args.cut_finest, args.fd_order, workload_opts(args))
    sub = args.mode == "sub"
    dt = w.dt_coarse
    H = sc.Hierarchy(w.boxes, w.domain_cells, w.nfields, w.ghost, w.xlo, w.xhi, w.coupling, device=f"cuda:{local}",
                     ko_sigma=w.ko_sigma, fd_order=w.fd_order, ko_order=w.ko_order, integrator=w.integrator,
                     outer_bc=w.outer_bc, interp=w.interp, vertex=w.vertex)

    # inputs: seeded synthetic state, staged in pinned host memory (also the e2e source buffers)
    host_in, host_out = {}, {}
    for l in range(w.nlevels):
        for ib in range(len(w.level_boxes(l))):
            for c in range(w.ncomp):
                a = w.initial_state(l, ib, c)
                t = torch.empty(a.shape, dtype=torch.float64).pin_memory()
                t.numpy()[...] = a
                host_in[(l, ib, c)] = t
    state_bytes = sum(t.numel() * 8 for t in host_in.values())
    for k, t in host_in.items():
        H.sc_set_state(*k, t.numpy())
    H.synchronize()

    st = H.stream
    upd_step = w.updates_per_coarse_step(sub)

    # ---- device-resident timing: W warm-up steps, then exactly K steps between two events ----------
    for _ in range(args.warmup):
        H.sc_step(dt, sub)
    barrier()
    n0 = H.sc_launch_count()
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for _ in range(args.steps):
        H.sc_step(dt, sub)
    e1.record(st)
    barrier()
    ms_total = e0.elapsed_time(e1)
    clocks = sampler.stop()
    launches = H.sc_launch_count() - n0
    ms_total = max_over_ranks(ms_total, dist, f"cuda:{local}")
    value = whole_job_value(world, upd_step, args.steps, ms_total * 1e-3)

    # ---- per-kernel roofline: same steps launched one by one with an event pair per kernel ---------
    peak, peak_src = measured_peaks()
    H.sc_profile(True)
    for _ in range(max(1, min(args.steps, 2))):
        H.sc_step(dt, sub)
    kinds = {}
    for i, name in enumerate(H.KERNEL_KINDS):
        n, ms, by = H.sc_profile_read(i)
        if n:
            kinds[name] = {"launches": n, "ms_total": ms, "avg_us": 1e3 * ms / n,
                           "algorithmic_GBps": by / (ms * 1e-3) / 1e9, "frac": by / (ms * 1e-3) / 1e9 / peak,
                           "bytes_per_launch": by / n}
    H.sc_profile(False)
    dom = max(kinds, key=lambda k: kinds[k]["ms_total"])
    ksum = sum(k["ms_total"] for k in kinds.values())
    wkey = f"cfg{args.config}/{args.mode}/sigma{args.sigma:g}/cut{args.cut_finest}/fd{args.fd_order}"
    if (w.ko_order, w.integrator, w.outer_bc, w.interp, w.vertex) != (0, 4, 0, 0, 0):
        wkey += f"/ko{w.ko_order}/rk{w.integrator}/bc{w.outer_bc}/ip{w.interp}/v{w.vertex}"
    # the practical ceiling of THIS device for a plain streaming kernel with a stage kernel's read/write mix over one
    # 256^3-sized array set (sc_debug_stream): context for the roofline fractions, which stay against the copy peak
    ceiling = None
    if rank == 0:
        ceiling = {f"R{r}W{wr}": round(H.sc_debug_stream(r, wr, 16 << 20), 1) for r, wr in ((1, 1), (2, 2), (4, 3))}
        ceiling["unit"], ceiling["what"] = "GB/s", "plain grid-stride double2 kernel, R arrays read + W written, 128 MiB each, best of 5"

    def roof(kind):
        k = kinds[kind]
        tr = ncu_traffic(kind, wkey)
        return {"bound": "hbm", "kernel": kind, "achieved": k["algorithmic_GBps"], "peak": peak, "unit": "GB/s",
                "frac": k["frac"], "traffic": tr["bytes_per_launch"] if tr else None,
                "traffic_source": tr["source"] if tr else "no ncu --set full capture of this kernel source under profiles/",
                "peak_source": peak_src, "frac_of_nominal_8TBps": k["algorithmic_GBps"] / 8000.0,
                "share_of_step": k["ms_total"] / ksum, "bytes_per_launch": k["bytes_per_launch"],
                "avg_launch_us": k["avg_us"]}
    roofline = roof(dom)
    # north_star sets a bar on the ghost-fill kernel as well: its roofline entry next to the dominant kernel's
    roofline_ghost = roof("ghost_dense_prolong") if "ghost_dense_prolong" in kinds else None

    # ---- the OTHER mode in the same run: north_star's bar "subcycling beats the non-subcycled hierarchy step by at
    # least the level-work ratio minus 15 %" (read as 0.85 x ratio, and as ratio - 0.15) ------------------
    other = None
    if args.other_mode_steps > 0:
        osub = not sub
        for _ in range(3):
            H.sc_step(dt, osub)
        barrier()
        o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        o0.record(st)
        for _ in range(args.other_mode_steps):
            H.sc_step(dt, osub)
        o1.record(st)
        barrier()
        oms = max_over_ranks(o0.elapsed_time(o1), dist, f"cuda:{local}") / args.other_mode_steps
        ms_sub = ms_total / args.steps if sub else oms
        ms_uni = oms if sub else ms_total / args.steps
        ratio = w.updates_per_coarse_step(False) / w.updates_per_coarse_step(True)
        other = {"ms_per_step_subcycled": ms_sub, "ms_per_step_uniform": ms_uni, "uniform_steps_timed": args.other_mode_steps if sub else args.steps,
                 "speedup_vs_uniform": ms_uni / ms_sub, "level_work_ratio": ratio,
                 "bar_0.85_x_ratio": 0.85 * ratio, "bar_ratio_minus_0.15": ratio - 0.15,
                 "meets_bar": bool(ms_uni / ms_sub >= max(0.85 * ratio, ratio - 0.15))}

    # ---- end to end through the C ABI with HOST buffers: H2D of the whole state, step, D2H ---------
    for k, t in host_in.items():
        host_out[k] = torch.empty(t.shape, dtype=torch.float64).pin_memory()
    e2e_steps = max(1, min(args.steps, 3))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        for k, t in host_in.items():
            H.sc_set_state(*k, t.numpy())
        H.sc_step(dt, sub)
        for k, t in host_out.items():
            H.sc_read_level(*k, t.numpy())
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, dist, f"cuda:{local}")
    e2e = {"value": whole_job_value(world, upd_step, e2e_steps, e2e_s), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
           "d2h_bytes_per_step": state_bytes, "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps}
    finite = all(bool(torch.isfinite(t).all()) for t in host_out.values())
    graph_stats = H.sc_debug_graph_stats()
    H.close()

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return 0

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = time_oracle(w, 1, 0, sub, max_levels=args.oracle_levels)
        cpu.pop("_seconds"), cpu.pop("_steps")
        cpu["sample_levels"], cpu["sample_updates_per_step"] = cpu.pop("_levels"), cpu.pop("_updates_per_step")
        if not args.no_cpu_1thread:  # one thread and all threads
            one = time_oracle(w, 1, 0, sub, max_levels=args.oracle_levels, threads=1)
            cpu["value_1thread"] = one["value"]
            cpu["sample_1thread"] = one["sample"]

    # model bytes of the whole step for the whole-step roofline fraction
    step_bytes = sum(k["bytes_per_launch"] * k["launches"] for k in kinds.values()) / max(1, min(args.steps, 2))
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_total / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(w, sub, world), "arena_GB": H.arena_bytes / 1e9,
            "roofline": roofline, "roofline_ghost": roofline_ghost, "sub_vs_uniform": other, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
            "kernels": kinds, "zone_cycles_per_s": world * w.zone_cycles_per_coarse_step() * args.steps / (ms_total * 1e-3),
            "step_algorithmic_GB": step_bytes / 1e9,
            "step_roofline_frac": step_bytes / (ms_total / args.steps * 1e-3) / 1e9 / peak,
            "stream_ceiling": ceiling, "graph": graph_stats, "finite": finite}
    print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    return 0


# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of a kernel kind, from the committed
# `ncu --set full` capture listed in profiles/traffic.csv. A row counts only while the kernel's SOURCE FILE still has
# the hash the capture was taken with (first 16 hex digits of its sha256) and the workload key matches; otherwise the
# line says null — a later kernel change can never carry an old figure along.
KIND_SOURCES = {"rk_stage": "stage_tma.cu", "ghost_dense_prolong": "ghost_tma.cu", "restrict": "restrict_zmarch.cu",
                "periodic_fill": "kernels_basic.cu"}


def ncu_traffic(kind: str, wkey: str):
    import csv
    import hashlib
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    src = os.path.join(ROOT, "paper_2503_09629_b200", "csrc", KIND_SOURCES.get(kind, ""))
    if not (os.path.exists(path) and os.path.isfile(src)):
        return None
    sha = hashlib.sha256(open(src, "rb").read()).hexdigest()[:16]
    with open(path, newline="") as f:
        for row in csv.DictReader(f):
            if row["kind"] == kind and row["workload"] == wkey and row["source_sha256_16"] == sha:
                return {"bytes_per_launch": float(row["dram_bytes_per_launch"]),
                        "source": f"profiles/{row['capture']} ({row['source_file']} sha256 {sha})"}
    return None


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--mode", default="sub", choices=["sub", "uniform"])
    ap.add_argument("--sigma", type=float, default=0.0,
                    help="Kreiss-Oliger dissipation strength (PAPER.md eqs 35-36); 0 = the configs as BASELINE states them")
    ap.add_argument("--cut-finest", type=int, default=1,
                    help="cut the finest level into this many abutting slabs that exchange ghosts (NEXT-2 variant)")
    ap.add_argument("--fd-order", type=int, default=4, choices=[4, 8],
                    help="8: the paper's BBH discretisation (PAPER.md:125): 8th-order centred differences, ghost width 4")
    ap.add_argument("--ko-order", type=int, default=None, choices=[0, 5, 9], help="dissipation order (0: eq 36, r = fd order)")
    ap.add_argument("--integrator", type=int, default=None, choices=[4, 3, 2], help="RK4 (default) / RK3 / RK2 (reading S28)")
    ap.add_argument("--outer-bc", type=int, default=None, choices=[0, 1], help="0 periodic (default), 1 radiative (S29)")
    ap.add_argument("--interp", type=int, default=None, choices=[0, 1], help="1: 9-/10-point interpolation (S30)")
    ap.add_argument("--vertex", type=int, default=None, choices=[0, 1], help="1: vertex-centred grids (S31)")
    ap.add_argument("--ghost", type=int, default=None, choices=[2, 3, 4, 5])
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--oracle-levels", type=int, default=2,
                    help="levels of the workload the CPU oracle is timed on (bounded sample)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-cpu-1thread", action="store_true", help="skip the one-thread leg of cpu_baseline")
    ap.add_argument("--other-mode-steps", type=int, default=3,
                    help="coarse steps of the OTHER mode timed in the same run for speedup_vs_uniform (0 = skip)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "b200":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
