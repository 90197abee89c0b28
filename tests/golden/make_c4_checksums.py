"""Writes tests/golden/c4_oracle_checksums.json: SHA-256 checksums of the ORACLE's state on BASELINE
config 4 ("for C4 the first >= 2 MCS in full plus a lattice/stat checksum at the end of
a 512^3 scaled copy run to 100 MCS"; BASELINE.md same sentence).

Calls only oracle/ and the seeded input generators (cpm_inputs/).  Nothing here comes from the CUDA
path.  Run from the repo root (takes ~25 min and ~16 GB of RAM on one core):

    python tests/golden/make_c4_checksums.py            # both runs
    python tests/golden/make_c4_checksums.py 512        # only the 512^3 x 100 MCS run
    python tests/golden/make_c4_checksums.py 1024       # only the 1024^3 x 2 MCS run

The schedule is the one bench.py times: subsection = 0 (scheduler's choice, S = 4, k = 64), deterministic
mode.  Every record also carries the checksums of the generated INPUTS, so that a drift of the generators
(numpy / scipy version) is reported as such and not as a parity failure.
"""
import hashlib
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
OUT = os.path.join(os.path.dirname(os.path.abspath(__file__)), "c4_oracle_checksums.json")

N_SLABS = 8


def sha(a):
    return hashlib.sha256(np.ascontiguousarray(a).tobytes()).hexdigest()


def slab_hashes(a3):
    """SHA-256 of N_SLABS equal slabs along z (localises a mismatch) -- a3 has shape (z, y, x)."""
    z = a3.shape[0]
    step = z // N_SLABS
    return [sha(a3[i * step:(i + 1) * step]) for i in range(N_SLABS)]


def state_record(s):
    """Checksums of everything the C ABI can read back (used for the oracle here and, in
    tests/test_gpu_fullsize.py, for the CUDA path)."""
    st = s.get_cell_stats()
    rec = {"lattice": slab_hashes(s.get_lattice()), "act": slab_hashes(s.get_act())}
    for k in ("volume", "perimeter", "sum_x", "sum_y", "sum_z"):
        rec[k] = sha(st[k])
    rec["counters"] = s.get_counters()
    return rec


def input_record(cfg):
    p = cfg["params"]
    return {"ids": sha(cfg["ids"]), "frozen": sha(cfg["frozen"]), "cell_type": sha(cfg["cell_type"]),
            "max_cells": int(cfg["max_cells"]), "J": np.asarray(p["J"]).tolist(), "seed": int(p["seed"]),
            "target_P": [int(v) for v in p["target_P"]]}


def run(dims, checkpoints):
    import cpm_inputs as ci
    from oracle import binding as ob
    t0 = time.time()
    cfg = ci.make_config("C4", dims=dims)
    params = dict(cfg["params"]); params["subsection"] = 0
    o = ob.Oracle(cfg["dims"], max_cells=cfg["max_cells"], **params)
    o.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
    rec = {"dims": list(dims), "schedule": o.get_schedule(), "inputs": input_record(cfg), "mcs": {}}
    print("generated %s in %.0f s" % (dims, time.time() - t0), flush=True)
    done = 0
    for m in checkpoints:
        o.step(m - done)
        done = m
        rec["mcs"][str(m)] = state_record(o)
        print("  MCS %d at %.0f s" % (m, time.time() - t0), flush=True)
    return rec


def main():
    which = sys.argv[1:] or ["512", "1024"]
    out = json.load(open(OUT)) if os.path.exists(OUT) else {}
    out["_about"] = ("SHA-256 checksums of the CPU oracle's state on BASELINE config 4 (SURVEY.md 8(d), BASELINE.md); "
                     "written by tests/golden/make_c4_checksums.py, which calls only oracle/ and cpm_inputs/")
    if "512" in which:
        out["512"] = run((512, 512, 512), [1, 2, 5, 10, 20, 50, 100])
        json.dump(out, open(OUT, "w"), indent=1, sort_keys=True)
    if "1024" in which:
        out["1024"] = run((1024, 1024, 1024), [1, 2])
        json.dump(out, open(OUT, "w"), indent=1, sort_keys=True)


if __name__ == "__main__":
    main()
