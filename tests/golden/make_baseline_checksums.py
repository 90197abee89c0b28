"""Writes tests/golden/baseline_oracle_checksums.json: SHA-256 checksums of the ORACLE's state on the BASELINE.json
workloads at their FULL sizes and run lengths ("bit-exact parity: every MCS for C1; every 10 MCS for
C2/C3"), and on the SURVEY 8(f) workloads C6 / C7:

    C2  256^3, 200 MCS, a checkpoint every 10 MCS          C3  256^3 with Act, 500 MCS, every 50 MCS
    C5  16384^2, S = 16 and S = 32, 10 MCS each            C6  256^3 persistence collective, 100 MCS, every 20 MCS
    C7  1024^2 circular chemotaxis, 100 MCS, every 20 MCS

Calls only oracle/ and the seeded input generators (cpm_inputs/); nothing here comes from the CUDA path.  Run from the
repo root; each run is one process on one core (C3: ~15 min, C5: ~6 min per S, the others a few minutes):

    python tests/golden/make_baseline_checksums.py              # all runs, one after the other
    python tests/golden/make_baseline_checksums.py C2 C6        # only these (merged into the existing file)

The schedule is the scheduler's choice (subsection = 0; S = 4 in 3D, 8 in 2D) unless a run names S; deterministic mode.
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "baseline_oracle_checksums.json")

# key -> (config, dims or None = the config's own, subsection, checkpoints)
RUNS = {
    "C2": ("C2", None, 0, list(range(10, 201, 10))),
    "C3": ("C3", None, 0, list(range(50, 501, 50))),
    "C5_S16": ("C5", None, 16, [5, 10]),
    "C5_S32": ("C5", None, 32, [5, 10]),
    "C6": ("C6", None, 0, list(range(20, 101, 20))),
    "C7": ("C7", None, 0, list(range(20, 101, 20))),
}


def sha(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def state_record(s, act, pers):
    """Checksums of everything the C ABI can read back (the oracle here; the CUDA path in tests/test_gpu_fullsize.py)."""
    st = s.get_cell_stats()
    rec = {"lattice": sha(s.get_lattice())}
    if act:
        rec["act"] = sha(s.get_act())
    if pers:
        rec["persistence"] = sha(s.get_persistence())      # the doubles of Eq 6-7, bit for bit
    for k in ("volume", "perimeter", "sum_x", "sum_y", "sum_z"):
        rec[k] = sha(st[k])
    rec["counters"] = s.get_counters()
    return rec


def input_record(cfg):
    p = cfg["params"]
    rec = {"ids": sha(cfg["ids"]), "cell_type": sha(cfg["cell_type"]), "max_cells": int(cfg["max_cells"]),
           "J": np.asarray(p["J"]).tolist(), "seed": int(p["seed"])}
    if cfg.get("field") is not None:
        rec["field"] = sha(cfg["field"])
    return rec


def flags_of(cfg):
    p = cfg["params"]
    act = p.get("max_act") is not None and any(int(v) != 0 for v in p["max_act"])
    pers = p.get("lambda_pers") is not None and any(int(v) != 0 for v in p["lambda_pers"])
    return act, pers


def build(key):
    import cpm_inputs as ci
    name, dims, S, checkpoints = RUNS[key]
    cfg = ci.make_config(name, dims=dims)
    params = dict(cfg["params"]); params["subsection"] = S
    return cfg, params, checkpoints


def run(key):
    from oracle import binding as ob
    t0 = time.time()
    cfg, params, checkpoints = build(key)
    act, pers = flags_of(cfg)
    o = ob.Oracle(cfg["dims"], max_cells=cfg["max_cells"], **params)
    o.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
    if cfg.get("field") is not None:
        o.set_chemotaxis_field(cfg["field"])
    rec = {"config": RUNS[key][0], "dims": list(cfg["dims"]), "subsection": RUNS[key][2], "schedule": o.get_schedule(),
           "inputs": input_record(cfg), "mcs": {}}
    print("%s: generated %s in %.0f s" % (key, cfg["dims"], time.time() - t0), flush=True)
    done = 0
    for m in checkpoints:
        o.step(m - done)
        done = m
        rec["mcs"][str(m)] = state_record(o, act, pers)
        print("  %s MCS %d at %.0f s" % (key, m, time.time() - t0), flush=True)
    return rec


def main():
    which = sys.argv[1:] or list(RUNS)
    out = {}
    if os.path.exists(OUT):
        with open(OUT) as f:
            out = json.load(f)
    for key in which:
        out[key] = run(key)
        with open(OUT, "w") as f:
            json.dump(out, f, indent=1, sort_keys=True)
            f.write("\n")
    print("wrote", OUT)


if __name__ == "__main__":
    main()
