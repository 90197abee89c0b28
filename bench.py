#!/usr/bin/env python
"""bench.py -- throughput of the checkerboard CPM sweep on B200 (copy attempts/s, MCS/s).

A "step" is one Monte Carlo step (one pass of the whole hot path: 2^d phase-steps of the sweep
kernel, the snapshot refresh, the Act decay) over the synthetic workload C4 of BASELINE.json
(3D 1024^3, ~1M cells, 20% frozen obstacle network, adhesion+volume+perimeter, Act on 10% of the
cells) -- the configuration the north_star's target is quoted on.  Inputs are seeded and synthetic
(cpm_inputs); the lattice (4 GiB) is far larger than L2, so no L2 flush is needed between steps.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--dims XxYxZ]

N > 1: one process per GPU (torchrun), independent replicas (the path does not shard on one
problem: "replicas only"), barrier + max-over-ranks timing, value = aggregate.
`--impl reference` times the CPU oracle (the deliberately plain baseline) on a bounded sample.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "copy_attempts_per_s"
UNIT = "attempts/s"
# algorithmic bytes per copy attempt of the sweep kernel in THIS layout:
# id word read + write-back (4+4 B), Act byte read + write-back (1+1 B)
BYTES_PER_ATTEMPT_ACT = 10.0
BYTES_PER_ATTEMPT_NOACT = 8.0
# SURVEY.md 8(d)'s model (float32 Act field, explicit decay folded in): 8 B / 16 B
SURVEY_BYTES_ACT, SURVEY_BYTES_NOACT = 16.0, 8.0


def parse_dims(s):
    return tuple(int(v) for v in s.lower().split("x"))


def env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


def measured_peak_gbs():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.gpu = gpu_index
        self.proc = None
        self.path = "/tmp/cpm_bench_clocks_%d_%d.csv" % (os.getpid(), gpu_index)

    def start(self):
        try:
            self.f = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            self.f.close()
            sm, mx, reasons = [], [], set()
            for line in open(self.path):
                t = [v.strip() for v in line.split(",")]
                if len(t) < 9:
                    continue
                try:
                    sm.append(float(t[1])); mx.append(float(t[2]))
                except ValueError:
                    continue
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), t[5:9]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            os.remove(self.path)
            if sm:
                out = {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "reasons": sorted(reasons),
                       "samples": len(sm)}
        except Exception:
            pass
        return out


def build_workload(name, dims, rank):
    import cpm_inputs as ci
    cfg = ci.make_config(name, dims=dims)
    if rank:
        cfg["params"]["seed"] = int(cfg["params"]["seed"]) + 7919 * rank   # independent replica
    return cfg


def reduce_over_ranks(times, counts, world, device):
    """Replicas only: the job's time is the MAX over ranks of each device time,
    its launch count the SUM; no data-path collective.  Identity for one rank."""
    if world <= 1:
        return [float(v) for v in times], [int(v) for v in counts]
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    c = torch.tensor(list(counts), dtype=torch.int64, device=device)
    dist.all_reduce(c)
    return [float(v) for v in t.tolist()], [int(v) for v in c.tolist()]


def oracle_rate(cfg, sample_dims, n_mcs, warm=0):
    """Attempts/s of the oracle, as it stands, on a corner crop of the workload (one host core)."""
    import cpm_inputs as ci
    from oracle import binding as ob
    crop = ci.crop_config(cfg, sample_dims)
    o = ob.Oracle(crop["dims"], max_cells=crop["max_cells"], **crop["params"])
    o.set_lattice(crop["ids"], crop["frozen"], crop["cell_type"])
    if warm:
        o.step(warm)
    t0 = time.perf_counter()
    o.step(n_mcs)
    dt = time.perf_counter() - t0
    n = int(np.prod(sample_dims)) * n_mcs
    return n / dt, dt


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, bounded sample per step."""
    if rank != 0:
        return
    dims = parse_dims(args.dims) if args.dims else (1024, 1024, 1024)
    sample = tuple(min(d, 128) for d in dims)
    gen_dims = tuple(min(d, 256) for d in dims)       # the crop only needs the corner of the workload
    cfg = build_workload(args.config, gen_dims, 0)
    import cpm_inputs as ci
    from oracle import binding as ob
    crop = ci.crop_config(cfg, sample)
    o = ob.Oracle(crop["dims"], max_cells=crop["max_cells"], **crop["params"])
    o.set_lattice(crop["ids"], crop["frozen"], crop["cell_type"])
    o.step(args.warmup)
    t0 = time.perf_counter()
    o.step(args.steps)
    dt = time.perf_counter() - t0
    n_step = int(np.prod(sample))
    value = n_step * args.steps / dt
    sample_txt = "corner crop %s of the %s workload, 1 MCS per step" % ("x".join(map(str, sample)), args.config)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": "%s %s (oracle on a bounded sample)" % (args.config, "x".join(map(str, dims))),
                   "sample": sample_txt},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample_txt},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "mcs_per_s_on_sample": args.steps / dt,
    }
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="C4")
    ap.add_argument("--dims", default=None, help="override the lattice size, e.g. 256x256x256")
    ap.add_argument("--subsection", type=int, default=0, help="checkerboard subsection edge S; 0 = scheduler's choice")
    ap.add_argument("--mode", type=int, default=0, help="0 deterministic (default), 1 live atomics")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    rank, world, local = env_int("RANK", 0), env_int("WORLD_SIZE", 1), env_int("LOCAL_RANK", 0)
    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    import paper_2312_09317_b200 as pk

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the CUDA path is the only implementation")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    dims = parse_dims(args.dims) if args.dims else None
    t_gen = time.perf_counter()
    cfg = build_workload(args.config, dims, rank)
    t_gen = time.perf_counter() - t_gen
    dims = cfg["dims"]
    N = int(np.prod(dims))
    params = dict(cfg["params"])
    params["subsection"] = args.subsection   # 0: the library's scheduler chooses (3D: 4, 2D: 8)
    act_on = params.get("max_act") is not None and any(int(v) != 0 for v in params["max_act"])

    # pinned host buffers: the inputs of the end-to-end leg and the result buffer
    ids_h = torch.from_numpy(cfg["ids"].view(np.int32).reshape(-1)).pin_memory()
    frozen_h = torch.from_numpy(cfg["frozen"].reshape(-1)).pin_memory() if cfg["frozen"] is not None else None
    ctype_h = torch.from_numpy(cfg["cell_type"]).pin_memory()
    out_h = torch.empty(N, dtype=torch.int32).pin_memory()

    g = pk.CPM(dims, max_cells=cfg["max_cells"], mode=args.mode, device=local, **params)
    g.set_lattice(ids_h, frozen_h, ctype_h)
    sched = g.get_schedule()
    info0 = g.get_launch_info()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput ----
    g.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    g.set_kernel_timing(True)
    l0 = g.get_launch_info()["launches"]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.step(args.steps)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    sweep_ms, sweep_n = g.get_kernel_timing(reset=True)
    g.set_kernel_timing(False)
    launches = g.get_launch_info()["launches"] - l0
    clocks = sampler.stop()
    counters = g.get_counters()

    # ---- end to end through the C ABI with HOST buffers: H2D of the inputs, MCS, D2H of the lattice ----
    e2e_steps = max(1, min(args.e2e_steps, args.steps))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        g.set_lattice(ids_h, frozen_h, ctype_h)
        g.step(1)
        g.get_lattice(out_h)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    h2d = ids_h.numel() * 4 + (frozen_h.numel() if frozen_h is not None else 0) + ctype_h.numel()
    d2h = out_h.numel() * 4

    (ms, e2e_s, sweep_ms), (launches,) = reduce_over_ranks([ms, e2e_s, sweep_ms], [launches], world, "cuda")

    if rank == 0:
        value = world * N * args.steps / (ms * 1e-3)
        e2e_value = world * N * e2e_steps / e2e_s
        peak, peak_src = measured_peak_gbs()
        bpa = BYTES_PER_ATTEMPT_ACT if act_on else BYTES_PER_ATTEMPT_NOACT
        attempts_per_launch = N * args.steps / max(sweep_n, 1)
        avg_launch_s = (sweep_ms * 1e-3) / max(sweep_n, 1)
        achieved = bpa * attempts_per_launch / avg_launch_s / 1e9
        survey_bpa = SURVEY_BYTES_ACT if act_on else SURVEY_BYTES_NOACT
        traffic = None
        # dram bytes per sweep launch from the committed ncu --set full capture (profiles/traffic_per_launch.csv)
        tpath = os.path.join(ROOT, "profiles", "traffic_per_launch.csv")
        if os.path.exists(tpath):
            try:
                key = "%s_%s" % (args.config, "x".join(map(str, dims)))
                for row in open(tpath).read().splitlines()[1:]:
                    f = row.split(",")
                    if f[0] == key and int(f[1]) == sched["S"]:
                        traffic = int(f[2])
            except Exception:
                traffic = None
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int64", "data": "synthetic",
            "config": {"workload": "%s %s" % (args.config, "x".join(map(str, dims))), "cells": int(cfg["max_cells"]),
                       "mode": "deterministic" if args.mode == 0 else "live_atomics", "subsection": sched["S"],
                       "attempts_per_activation": sched["k"], "phase_steps_per_mcs": sched["phase_steps_per_mcs"],
                       "act": bool(act_on), "l2": "inputs larger than L2 (no flush needed)",
                       "parallelism": "replicas x%d" % world, "input_generation_s": round(t_gen, 1)},
            "mcs_per_s": world * args.steps / (ms * 1e-3),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "traffic": traffic, "kernel": "sweep_pool_kernel" if info0["pooled"] else "sweep_kernel", "bytes_per_attempt": bpa,
                         "launches_timed": int(sweep_n), "avg_launch_ms": 1e3 * avg_launch_s, "peak_source": peak_src,
                         "kernel_share_of_step": sweep_ms / ms,
                         "frac_with_survey_model_bytes": survey_bpa * attempts_per_launch / avg_launch_s / 1e9 / peak},
            "counters": {"evaluated_frac": counters["evaluated"] / max(counters["attempts"], 1),
                         "accepted_frac": counters["accepted"] / max(counters["attempts"], 1)},
        }
        if not args.no_cpu_baseline:
            sample = tuple(min(d, 256 if len(dims) == 3 else 4096) for d in dims)
            n_mcs = 3
            try:
                v, dt = oracle_rate(cfg, sample, n_mcs)
                line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                                        "sample": "corner crop %s of the workload, first %d MCS (%.1f s)" % (
                                            "x".join(map(str, sample)), n_mcs, dt)}
            except Exception as ex:  # the baseline is a reported extra, never a reason to lose the bench line
                line["cpu_baseline"] = {"value": None, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": "failed: %r" % (ex,)}
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
