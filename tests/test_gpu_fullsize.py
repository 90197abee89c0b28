"""BASELINE config 4 at the sizes SURVEY.md 8(d) / BASELINE.md name for the full-size parity check:
"for C4 the first >= 2 MCS in full plus a lattice/stat checksum at the end of a 512^3 scaled copy run to
100 MCS".  The CUDA path (through the C ABI, in the launch configuration bench.py times: subsection = 0,
deterministic mode, Act on) is compared with the ORACLE's state, recorded as SHA-256 checksums of every
array the C ABI can read back (lattice and Act field in 8 z-slabs, V, P, coordinate sums, counters) by
tests/golden/make_c4_checksums.py, a committed script that calls only oracle/ and the seeded input
generators.  Equal SHA-256 of the raw bytes = equal element by element.  The oracle needs ~150 s per MCS
at 1024^3 and ~16 s at 512^3 on one core, which is why its side is stored and not recomputed here.

All tests here need a B200 (`-m gpu`)."""
import importlib.util
import json
import os

import numpy as np
import pytest

import helpers as H

pytestmark = pytest.mark.gpu

GOLDEN_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _golden_tools():
    spec = importlib.util.spec_from_file_location("make_c4_checksums", os.path.join(GOLDEN_DIR, "make_c4_checksums.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


@pytest.fixture(scope="module")
def pk():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2312_09317_b200 as m
    m.load_library()
    return m


@pytest.fixture(scope="module")
def golden():
    with open(os.path.join(GOLDEN_DIR, "c4_oracle_checksums.json")) as f:
        return json.load(f)


def _start(pk, cfg):
    params = dict(cfg["params"]); params["subsection"] = 0
    g = pk.CPM(cfg["dims"], max_cells=cfg["max_cells"], **params)
    g.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
    return g


def _check_against_golden(pk, golden_rec, cfg):
    tools = _golden_tools()
    # the generators must have produced the inputs the oracle ran on: otherwise this is a drift of numpy /
    # scipy, not a parity failure
    assert tools.input_record(cfg) == golden_rec["inputs"], "generated inputs differ from the ones the golden run used"
    g = _start(pk, cfg)
    assert g.get_schedule() == golden_rec["schedule"]
    assert g.get_launch_info()["pooled"]
    done = 0
    for m in sorted(int(k) for k in golden_rec["mcs"]):
        g.step(m - done)
        done = m
        got, want = tools.state_record(g), golden_rec["mcs"][str(m)]
        for key in want:
            assert got[key] == want[key], "C4 %s after %d MCS: %s differs from the oracle's checksum" % (cfg["dims"], m, key)
    return g


def test_C4_512_cubed_100_mcs_equals_oracle_checksums(pk, golden):
    """512^3 scaled copy of config 4, 100 MCS, compared with the oracle after 1, 2, 5, 10, 20, 50 and 100 MCS."""
    import cpm_inputs as ci
    cfg = ci.make_config("C4", dims=(512, 512, 512))
    _check_against_golden(pk, golden["512"], cfg)


def test_C4_full_size_equals_oracle_and_properties(pk, golden):
    """BASELINE config 4 at its full size (1024^3, ~1.04 M cells, 20 % obstacles) in bench.py's launch
    configuration: (o) after MCS 1 and MCS 2 every array equals the oracle's (checksums, see the module
    docstring); and what must hold at any size: (i) the volume and coordinate-sum tallies equal a recount of
    the lattice (the paper's invariant, L57, L288); (ii) perimeters equal a recount for every cell that lies
    inside a 128^3 corner block; (iii) obstacle voxels never change and no cell disappears; (iv) a second
    context with the same seed reproduces the state bit for bit (counter-based RNG, deterministic mode)."""
    import cpm_inputs as ci
    cfg = ci.make_config("C4")
    assert cfg["dims"] == (1024, 1024, 1024)
    n = cfg["max_cells"] + 1

    g = _check_against_golden(pk, golden["1024"], cfg)     # (o); leaves the context after 2 MCS
    lat = g.get_lattice()
    assert g.get_schedule()["S"] == 4
    st = g.get_cell_stats()
    c = g.get_counters()
    assert c["attempts"] == 2 * 1024 ** 3 and 0 < c["accepted"] < c["evaluated"] < c["attempts"]
    assert (lat != cfg["ids"]).any()

    # (i) volumes and coordinate sums, slab by slab
    V = np.zeros(n, np.int64); sx = np.zeros(n, np.int64); sy = np.zeros(n, np.int64); sz = np.zeros(n, np.int64)
    xs = np.arange(1024, dtype=np.float64)
    for z0 in range(0, 1024, 32):
        blk = lat[z0:z0 + 32].reshape(-1).astype(np.int64)
        V += np.bincount(blk, minlength=n)
        sx += np.bincount(blk, weights=np.tile(xs, 32 * 1024), minlength=n).astype(np.int64)
        sy += np.bincount(blk, weights=np.tile(np.repeat(xs, 1024), 32), minlength=n).astype(np.int64)
        sz += np.bincount(blk, weights=np.repeat(xs[z0:z0 + 32], 1024 * 1024), minlength=n).astype(np.int64)
    for a in (V, sx, sy, sz):
        a[0] = 0
    np.testing.assert_array_equal(st["volume"].astype(np.int64), V)
    np.testing.assert_array_equal(st["sum_x"].astype(np.int64), sx)
    np.testing.assert_array_equal(st["sum_y"].astype(np.int64), sy)
    np.testing.assert_array_equal(st["sum_z"].astype(np.int64), sz)

    # (ii) perimeters of the cells that lie strictly inside the 128^3 corner block
    B = 128
    blk = lat[:B, :B, :B]
    Vb, Pb, _, _, _ = H.recount(blk, cfg["max_cells"], 3)
    face = np.zeros(n, bool)
    for sl in (blk[-1], blk[:, -1], blk[:, :, -1]):     # faces towards the rest of the lattice
        face[np.unique(sl)] = True
    inside = (Vb > 0) & (Vb == V) & ~face
    inside[0] = False
    assert inside.sum() > 500
    np.testing.assert_array_equal(st["perimeter"].astype(np.int64)[inside], Pb[inside])

    # (iii) obstacles and conservation
    fz = cfg["frozen"].astype(bool)
    assert (lat[fz] == cfg["ids"][fz]).all()
    V0 = np.bincount(cfg["ids"].reshape(-1).astype(np.int64), minlength=n)
    assert ((V[1:] > 0) == (V0[1:] > 0)).all()

    # (iv) reproducibility
    del g
    g2 = _start(pk, cfg)
    g2.step(2)
    assert np.array_equal(lat, g2.get_lattice())
    st2 = g2.get_cell_stats()
    for k in st:
        np.testing.assert_array_equal(st[k], st2[k])


# ---- every other workload at its full size and run length (tests/golden/make_baseline_checksums.py) ----
def _baseline_tools():
    spec = importlib.util.spec_from_file_location("make_baseline_checksums", os.path.join(GOLDEN_DIR, "make_baseline_checksums.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return mod


@pytest.mark.parametrize("key", ["C2", "C3", "C5_S16", "C5_S32", "C6", "C7"])
def test_workloads_at_full_size_and_length_equal_oracle_checksums(pk, key):
    """BASELINE configs 2, 3, 5 and the SURVEY 8(f) workloads C6, C7 at the sizes and run lengths BASELINE.json / the paper
    name (C2: 256^3 x 200 MCS, C3: 256^3 x 500 MCS with Act, C5: 16384^2 at S = 16 and 32, C6: 256^3 x 100 MCS with
    persistence, C7: 1024^2 x 100 MCS with chemotaxis): at every checkpoint (every 10 MCS for C2) the SHA-256
    of every array the C ABI reads back -- lattice, Act, V, P, coordinate sums, persistence doubles, counters -- equals
    the oracle's, recorded by the committed script that calls only oracle/."""
    tools = _baseline_tools()
    with open(os.path.join(GOLDEN_DIR, "baseline_oracle_checksums.json")) as f:
        rec = json.load(f)[key]
    cfg, params, checkpoints = tools.build(key)
    assert tools.input_record(cfg) == rec["inputs"], "generated inputs differ from the ones the golden run used"
    act, pers = tools.flags_of(cfg)
    g = pk.CPM(cfg["dims"], max_cells=cfg["max_cells"], **params)
    g.set_lattice(cfg["ids"], cfg["frozen"], cfg["cell_type"])
    if cfg.get("field") is not None:
        g.set_chemotaxis_field(cfg["field"])
    assert g.get_schedule() == rec["schedule"]
    done = 0
    for m in sorted(int(k) for k in rec["mcs"]):
        g.step(m - done)
        done = m
        got, want = tools.state_record(g, act, pers), rec["mcs"][str(m)]
        for k2 in want:
            assert got[k2] == want[k2], "%s after %d MCS: %s differs from the oracle's checksum" % (key, m, k2)
