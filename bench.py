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
# ALGORITHMIC bytes per copy attempt, SURVEY.md 8(d)'s model: id word read + write-back
# = 8 B; with the Act extension + 8 B (float32 Act read + write-back, decay folded in) = 16 B.  roofline.achieved
# and roofline.frac use this figure.
SURVEY_BYTES_ACT, SURVEY_BYTES_NOACT = 16.0, 8.0
# what THIS layout has to move per attempt (extra key roofline.frac_layout_bytes): id word read + write-back
# (4 + 4 B), Act byte read + write-back (1 + 1 B)
LAYOUT_BYTES_ACT, LAYOUT_BYTES_NOACT = 10.0, 8.0
BURN_IN_MCS = 10          # 10 MCS burn-in before anything is timed (the first MCS are a transient)
CPU_SAMPLE_3D, CPU_SAMPLE_2D = 256, 4096   # edge of the corner crop both oracle legs run


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
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=self.f,
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


def source_hash():
    """SHA-256 over the sources of the sweep kernels (cpm_device.cuh, cpm_pool_kernel.cuh): ties a stored ncu figure
    to the code it was taken on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2312_09317_b200", "csrc")
    for name in ("cpm_device.cuh", "cpm_pool_kernel.cuh"):   # the files the sweep kernels are made of
        with open(os.path.join(d, name), "rb") as f:
            h.update(name.encode()); h.update(f.read())
    return h.hexdigest()[:16]


def static_capture(config, dims, S):
    """DRAM bytes per sweep launch (and warp-instructions per attempt) from the committed `ncu --set full` capture,
    profiles/traffic_per_launch.csv.  It is a STATIC figure: it is only reported when the capture was taken on the
    very kernel sources being timed (source_hash), otherwise traffic is null."""
    tpath = os.path.join(ROOT, "profiles", "traffic_per_launch.csv")
    try:
        rows = [r.split(",") for r in open(tpath).read().splitlines()]
        hdr, rows = rows[0], rows[1:]
        key = "%s_%s" % (config, "x".join(map(str, dims)))
        cur = source_hash()
        for f in rows:
            r = dict(zip(hdr, f))
            if r["workload"] == key and int(r["subsection"]) == S:
                if r.get("source_hash") != cur:
                    return None, "stale: %s was captured on sources %s, timed sources are %s" % (r.get("source"), r.get("source_hash"), cur), None
                wipa = float(r["warp_instr_per_attempt"]) if r.get("warp_instr_per_attempt") else None
                alu = float(r["alu_pipe_active_pct_under_ncu"]) if r.get("alu_pipe_active_pct_under_ncu") else None
                return int(r["dram_bytes_per_sweep_launch"]), "static ncu capture %s (sources %s)" % (r.get("source"), cur), {"warp_instr_per_attempt": wipa, "alu_pipe_active_pct_under_ncu": alu}
    except Exception:
        pass
    return None, "no capture for this workload", None


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


def host_info():
    """What SURVEY.md 8(d) asks to print beside the oracle's time: core count and CPU model of the box."""
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.lower().startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"nproc": os.cpu_count(), "cpu_model": model}


def cpu_sample_dims(dims):
    return tuple(min(d, CPU_SAMPLE_3D if len(dims) == 3 else CPU_SAMPLE_2D) for d in dims)


def make_oracle(cfg, sample_dims, params):
    """The oracle, as it stands, on a corner crop of the workload, with the schedule of the GPU leg (same S, k)."""
    import cpm_inputs as ci
    from oracle import binding as ob
    crop = ci.crop_config(cfg, sample_dims)
    o = ob.Oracle(crop["dims"], max_cells=crop["max_cells"], **params)
    o.set_lattice(crop["ids"], crop["frozen"], crop["cell_type"])
    if crop.get("field") is not None:
        o.set_chemotaxis_field(crop["field"])
    return o


def oracle_rate(cfg, sample_dims, params, n_mcs, warm=0):
    """Attempts/s of the oracle on the crop (one host core), over n_mcs MCS after `warm` untimed ones."""
    o = make_oracle(cfg, sample_dims, params)
    if warm:
        o.step(warm)
    t0 = time.perf_counter()
    o.step(n_mcs)
    dt = time.perf_counter() - t0
    n = int(np.prod(sample_dims)) * n_mcs
    return n / dt, dt


def sample_text(sample, cfg_name, first, n_mcs):
    return "corner crop %s of the %s workload, MCS %d..%d of the run, 1 MCS per step, one core" % (
        "x".join(map(str, sample)), cfg_name, first + 1, first + n_mcs)


def run_reference(args, rank, world):
    """--impl reference: the oracle on the host cores, bounded sample per step."""
    if rank != 0:
        return
    cfg = build_workload(args.config, parse_dims(args.dims) if args.dims else None, 0)   # the workload of the ours arm
    dims = cfg["dims"]
    sample = cpu_sample_dims(dims)                    # the same crop the cpu_baseline leg of the ours arm runs
    params = dict(cfg["params"]); params["subsection"] = args.subsection
    value, dt = oracle_rate(cfg, sample, params, args.steps, warm=args.warmup)
    n_step = int(np.prod(sample))
    sample_txt = sample_text(sample, args.config, args.warmup, args.steps)
    hi = host_info()
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int64", "data": "synthetic",
        "config": {"workload": "%s %s (oracle on a bounded sample)" % (args.config, "x".join(map(str, dims))),
                   "sample": sample_txt},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample_txt,
                         "nproc": hi["nproc"], "cpu_model": hi["cpu_model"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "mcs_per_s_on_sample": args.steps / dt,
    }
    print(json.dumps(line))


def run_speed_accuracy_map(args):
    """--map: the S x switching-frequency speed / accuracy map of the paper's 2D circular chemotaxis workload
    (Fig 6E) as a markdown table on stdout.
    accuracy side: an ensemble of `--ensemble` seeds of C7 at 128x128 (one cell circling in the tangential field), 200 MCS;
    per-pixel occupancy q (fraction of runs in which the pixel is covered by a cell at the end) against the occupancy p of
    the SERIAL schedule (S = 128: the whole lattice is one region, i.e. the update order of the serial CPM), as the mean
    binary cross-entropy in bits, probabilities clipped to [1/2n, 1 - 1/2n]; accuracy = 1 - cross-entropy (the paper's axis).
    speed side: copy attempts/s of the same (S, k) on C7 at `--dims` (default 4096x4096), 10 MCS after 10 burn-in."""
    import torch
    import cpm_inputs as ci
    import paper_2312_09317_b200 as pk
    n_ens, n_mcs = args.ensemble, 200
    small = ci.make_config("C7", dims=(128, 128))

    def occupancy(S, k, seed0):
        streams = [torch.cuda.Stream() for _ in range(8)]
        ctxs = []
        for i in range(n_ens):
            p = dict(small["params"]); p.update(subsection=S, attempts_per_activation=k, seed=seed0 + i)
            with torch.cuda.stream(streams[i % len(streams)]):
                g = pk.CPM(small["dims"], max_cells=small["max_cells"], **p)
                g.set_lattice(small["ids"], None, small["cell_type"])
                g.set_chemotaxis_field(small["field"])
                g.step(n_mcs)
                ctxs.append(g)
        torch.cuda.synchronize()
        occ = np.zeros(small["ids"].shape, dtype=np.float64)
        for g in ctxs:
            occ += (g.get_lattice() != 0)
        return occ / n_ens

    def cross_entropy(p, q):
        eps = 1.0 / (2 * n_ens)
        q = np.clip(q, eps, 1 - eps)
        return float(-(p * np.log2(q) + (1 - p) * np.log2(1 - q)).mean())

    p_serial = occupancy(128, 0, 1000)
    p_serial2 = occupancy(128, 0, 500000)          # an independent serial ensemble: the noise floor of the measure
    big_dims = parse_dims(args.dims) if args.dims else (4096, 4096)
    big = ci.make_config("C7", dims=big_dims)
    N = int(np.prod(big_dims))
    rows = []
    for S in (2, 4, 8, 16):
        for k in sorted({max(S * S // div, 1) for div in (1, 4, 16)}, reverse=True):
            q = occupancy(S, k, 1000)
            ce = cross_entropy(p_serial, q)
            p = dict(big["params"]); p.update(subsection=S, attempts_per_activation=k)
            g = pk.CPM(big["dims"], max_cells=big["max_cells"], **p)
            g.set_lattice(big["ids"], None, big["cell_type"])
            g.set_chemotaxis_field(big["field"])
            g.step(BURN_IN_MCS)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); g.step(10); e1.record(); torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 10
            rows.append((S, k, g.get_schedule()["phase_steps_per_mcs"], N / (ms * 1e-3), ms, ce, 1 - ce))
            del g
    print("| S | k | phase-steps / MCS | attempts/s (C7 %s) | ms / MCS | cross-entropy vs serial (bits / pixel) | accuracy |" % "x".join(map(str, big_dims)))
    print("|---:|---:|---:|---:|---:|---:|---:|")
    for r in rows:
        print("| %d | %d | %d | %.3g | %.3f | %.4f | %.4f |" % r)
    print()
    print("serial ensemble against itself (entropy of p, the lower bound): %.4f bits / pixel; against an independent serial "
          "ensemble (noise floor at %d runs): %.4f bits / pixel" % (cross_entropy(p_serial, p_serial), n_ens, cross_entropy(p_serial, p_serial2)))


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
    ap.add_argument("--no-live", action="store_true", help="skip the extra LIVE-mode measurement")
    ap.add_argument("--map", action="store_true", help="print the speed / accuracy map of the C7 chemotaxis workload instead of the bench line")
    ap.add_argument("--ensemble", type=int, default=64, help="--map: runs per ensemble")
    args = ap.parse_args()
    if args.map:
        run_speed_accuracy_map(args)
        return
    args.warmup = max(args.warmup, BURN_IN_MCS)   # both arms: the same burn-in, so the same MCS window is timed

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

    field_h = torch.from_numpy(cfg["field"].reshape(-1)).pin_memory() if cfg.get("field") is not None else None
    g = pk.CPM(dims, max_cells=cfg["max_cells"], mode=args.mode, device=local, **params)
    g.set_lattice(ids_h, frozen_h, ctype_h)
    if field_h is not None:
        g.set_chemotaxis_field(field_h)
    sched = g.get_schedule()
    info0 = g.get_launch_info()

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident throughput ----
    # the clock sampler starts before the burn-in (the same kernels on the same workload) so that nvidia-smi is already
    # polling when the timed region, a fraction of a second long, begins; it stops after the graph replay
    sampler = ClockSampler(local)
    sampler.start()
    g.step(args.warmup)
    barrier()
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
    counters = g.get_counters()
    # the same K steps again the way cpm_step runs them for a user: one CUDA graph per MCS, no per-launch events
    g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    g0.record()
    g.step(args.steps)
    g1.record()
    barrier()
    graph_ms = g0.elapsed_time(g1)
    clocks = sampler.stop()
    graph_window = [args.warmup + args.steps + 1, args.warmup + 2 * args.steps]   # later MCS than the timed region: the workload relaxes

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

    (ms, e2e_s, sweep_ms, graph_ms), (launches,) = reduce_over_ranks([ms, e2e_s, sweep_ms, graph_ms], [launches], world, "cuda")

    # ---- extra: the paper-faithful LIVE mode (atomics on live per-cell values, L51-53) on the same workload ----
    live = None
    if args.mode == 0 and not args.no_live:
        del g
        gl = pk.CPM(dims, max_cells=cfg["max_cells"], mode=1, device=local, **params)
        gl.set_lattice(ids_h, frozen_h, ctype_h)
        if field_h is not None:
            gl.set_chemotaxis_field(field_h)
        gl.step(args.warmup)
        barrier()
        f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        n_live = min(args.steps, 5)
        f0.record()
        gl.step(n_live)
        f1.record()
        barrier()
        live_ms = f0.elapsed_time(f1)
        (live_ms,), _ = reduce_over_ranks([live_ms], [0], world, "cuda")
        live = {"value": world * N * n_live / (live_ms * 1e-3), "unit": UNIT, "ms_per_step": live_ms / n_live, "steps": n_live}
        del gl

    if rank == 0:
        value = world * N * args.steps / (ms * 1e-3)
        e2e_value = world * N * e2e_steps / e2e_s
        peak, peak_src = measured_peak_gbs()
        bpa = SURVEY_BYTES_ACT if act_on else SURVEY_BYTES_NOACT
        layout_bpa = LAYOUT_BYTES_ACT if act_on else LAYOUT_BYTES_NOACT
        attempts_per_launch = N * args.steps / max(sweep_n, 1)
        avg_launch_s = (sweep_ms * 1e-3) / max(sweep_n, 1)
        achieved = bpa * attempts_per_launch / avg_launch_s / 1e9
        kernel_name = "sweep_pool_kernel" if info0["pooled"] else "sweep_kernel"
        traffic, traffic_src, prof = static_capture(args.config, dims, sched["S"])
        roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": traffic_src, "kernel": kernel_name, "bytes_per_attempt": bpa,
                "launches_timed": int(sweep_n), "avg_launch_ms": 1e3 * avg_launch_s, "peak_source": peak_src,
                "kernel_share_of_step": sweep_ms / ms,
                "frac_layout_bytes": layout_bpa * attempts_per_launch / avg_launch_s / 1e9 / peak,
                "layout_bytes_per_attempt": layout_bpa,
                # what limits the kernel today is not HBM: issue slots and barrier latency
                "limiter": "integer alu pipe and instruction issue (DESIGN.md section 7), not HBM"}
        if prof and prof.get("warp_instr_per_attempt"):
            # the plain-ALU side SURVEY.md 8(d) asks for: warp-instructions issued per second against
            # SMs x 4 schedulers x SM clock (one warp-instruction per scheduler and cycle)
            sm_mhz = clocks.get("sm_mhz") or 1965.0
            issue_peak = 148 * 4 * sm_mhz * 1e6
            roof["alu"] = {"warp_instr_per_attempt": prof["warp_instr_per_attempt"],
                           "achieved": prof["warp_instr_per_attempt"] * attempts_per_launch / avg_launch_s,
                           "peak": issue_peak, "unit": "warp-instr/s",
                           "frac": prof["warp_instr_per_attempt"] * attempts_per_launch / avg_launch_s / issue_peak,
                           "alu_pipe_active_pct_under_ncu": prof.get("alu_pipe_active_pct_under_ncu"),
                           "note": "warp_instr_per_attempt is the static capture's (one launch of MCS 11); later MCS evaluate and accept fewer attempts, so this fraction is an upper estimate for a window that extends beyond MCS 20",
                           "source": traffic_src}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "int64", "data": "synthetic",
            "config": {"workload": "%s %s" % (args.config, "x".join(map(str, dims))), "cells": int(cfg["max_cells"]),
                       "mode": "deterministic" if args.mode == 0 else "live_atomics", "subsection": sched["S"],
                       "attempts_per_activation": sched["k"], "phase_steps_per_mcs": sched["phase_steps_per_mcs"],
                       "act": bool(act_on), "l2": "inputs larger than L2 (no flush needed)", "burn_in_mcs": args.warmup,
                       "parallelism": "replicas x%d" % world, "input_generation_s": round(t_gen, 1)},
            "mcs_per_s": world * args.steps / (ms * 1e-3),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps},
            "gpu_launches": int(launches),
            # the timed region above launches the kernels one by one with an event pair around every sweep launch;
            # this is the same K steps replayed as CUDA graphs (what cpm_step does when per-launch timing is off)
            "graph_replay": {"value": world * N * args.steps / (graph_ms * 1e-3), "unit": UNIT, "ms_per_step": graph_ms / args.steps,
                             "mcs_window": graph_window},
            "clocks": clocks,
            "roofline": roof,
            "counters": {"evaluated_frac": counters["evaluated"] / max(counters["attempts"], 1),
                         "accepted_frac": counters["accepted"] / max(counters["attempts"], 1)},
        }
        if live is not None:
            line["live_mode"] = live
        if not args.no_cpu_baseline:
            sample = cpu_sample_dims(dims)
            hi = host_info()
            n_mcs = min(args.steps, 10)
            base = {"unit": UNIT, "cores": 1, "kind": "oracle", "nproc": hi["nproc"], "cpu_model": hi["cpu_model"]}
            try:
                v, dt = oracle_rate(cfg, sample, params, n_mcs, warm=args.warmup)
                base.update({"value": v, "sample": sample_text(sample, args.config, args.warmup, n_mcs) + " (%.1f s timed)" % dt})
            except Exception as ex:  # the baseline is a reported extra, never a reason to lose the bench line
                base.update({"value": None, "sample": "failed: %r" % (ex,)})
            line["cpu_baseline"] = base
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
