"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these compares the oracle with itself or with the CUDA path: the expected side is a
brute-force definition (helpers.brute_force_H, helpers.recount), a closed form, a published
known-answer vector, or a limit case.
"""
import math
import os

import numpy as np
import pytest

import helpers as H

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _tiny_case(ob, rng, dims, n_cells, periodic=(0, 0, 0), frozen_frac=0.1, subsection=None, mode=0,
               lamP=(0, 3, 2), T=20.0, seed=7, act=False):
    nd = len(dims)
    shape = tuple(reversed(dims))
    ids = rng.integers(0, n_cells + 1, size=shape).astype(np.uint32)
    frozen = (rng.random(shape) < frozen_frac).astype(np.uint8)
    cell_type = np.zeros(n_cells + 1, dtype=np.uint8)
    cell_type[1:] = rng.integers(1, 3, size=n_cells)
    J = np.array([[0, 7, -3], [7, 11, 16], [-3, 16, 5]], dtype=np.int32)
    lamV, tgtV = [0, 4, 6], [0, 9, 14]
    tgtP = [0, 30, 41]
    kw = dict(J=J, lambda_V=lamV, target_V=tgtV, lambda_P=list(lamP), target_P=tgtP, T=T, seed=seed,
              subsection=subsection or dims[0], mode=mode, max_cells=n_cells, periodic=periodic)
    if act:
        kw.update(lambda_act=[0, 200, 90], max_act=[0, 40, 17])
    o = ob.Oracle(dims, **kw)
    o.set_lattice(ids, frozen, cell_type)
    return o, ids, frozen, cell_type, J, lamV, tgtV, list(lamP), tgtP


# ------------------------------------------------------------------------------------- P1 --
@pytest.mark.parametrize("dims,periodic,sub", [
    ((6, 6), (0, 0, 0), 6), ((6, 6), (1, 0, 0), 3), ((6, 6), (1, 1, 0), 3),
    ((5, 5, 5), (0, 0, 0), 5), ((4, 4, 4), (0, 1, 1), 2), ((4, 8, 4), (1, 1, 1), 2),
])
def test_P1_incremental_dH_equals_bruteforce(oracle_mod, dims, periodic, sub):
    """dH(adhesion, volume, perimeter) == H(after) - H(before), H from Eq 1 + Eq 3 brute force."""
    rng = np.random.default_rng(11 + sum(dims))
    o, ids, frozen, ct, J, lamV, tgtV, lamP, tgtP = _tiny_case(oracle_mod, rng, dims, 4, periodic, subsection=sub)
    nd = len(dims)
    nNb = 8 if nd == 2 else 26
    N = int(np.prod(dims))
    checked = 0
    statuses = set()
    for it in range(400):
        t = int(rng.integers(N)); nb = int(rng.integers(nNb))
        st, dH, dA = o.probe(t, nb)
        statuses.add(st)
        assert dA == 0  # Act off
        if st != 1:
            continue
        lat0 = o.get_lattice().copy()
        H0 = H.brute_force_H(lat0, ct, J, lamV, tgtV, lamP, tgtP, nd, periodic)
        o.force_copy(t, nb)
        lat1 = o.get_lattice()
        assert (lat0 != lat1).sum() == 1
        H1 = H.brute_force_H(lat1, ct, J, lamV, tgtV, lamP, tgtP, nd, periodic)
        assert dH == H1 - H0, (it, t, nb, dH, H1 - H0)
        checked += 1
        if checked >= 60:
            break
    assert checked >= 30
    assert 0 in statuses


def test_P1_early_outs_and_frozen(oracle_mod):
    """same cell / frozen target / frozen source are early-outs (a4, reading S14); a frozen
    neighbour still enters adhesion and perimeter (covered by the brute force above)."""
    ob = oracle_mod
    ids = np.array([[1, 1, 2, 0], [1, 2, 2, 0], [0, 0, 0, 0], [0, 0, 0, 0]], dtype=np.uint32)
    frozen = np.zeros((4, 4), np.uint8); frozen[0, 2] = 1
    J = np.array([[0, 5], [5, 9]], np.int32)
    o = ob.Oracle((4, 4), J=J, lambda_V=[0, 1], target_V=[0, 3], max_cells=2, subsection=4)
    o.set_lattice(ids, frozen, np.array([0, 1, 1], np.uint8))
    offs = H.moore_offsets(2)
    nb_of = {o_: i for i, o_ in enumerate(offs)}
    # target (0,0) source (1,0): same cell
    assert o.probe(0, nb_of[(1, 0, 0)])[0] == 0
    # target (2,0) is frozen
    assert o.probe(2, nb_of[(-1, 0, 0)])[0] == 0
    # target (1,0), source (2,0) frozen
    assert o.probe(1, nb_of[(1, 0, 0)])[0] == 0
    # target (1,0), source (1,1) = cell 2 -> evaluated
    assert o.probe(1, nb_of[(0, 1, 0)])[0] == 1
    # target (0,0), source (-1,0) outside = medium -> evaluated (medium copies in)
    assert o.probe(0, nb_of[(-1, 0, 0)])[0] == 1
    np.testing.assert_array_equal(ob.neighbour_offsets(2), np.array(offs))
    np.testing.assert_array_equal(ob.neighbour_offsets(3), np.array(H.moore_offsets(3)))


# -------------------------------------------------------------------------------- P2, P5 --
def _check_tallies(o, max_cells, nd, periodic=(0, 0, 0)):
    st = o.get_cell_stats()
    V, P, sx, sy, sz = H.recount(o.get_lattice(), max_cells, nd, periodic)
    np.testing.assert_array_equal(st["volume"].astype(np.int64), V)
    np.testing.assert_array_equal(st["perimeter"].astype(np.int64), P)
    np.testing.assert_array_equal(st["sum_x"].astype(np.int64), sx)
    np.testing.assert_array_equal(st["sum_y"].astype(np.int64), sy)
    np.testing.assert_array_equal(st["sum_z"].astype(np.int64), sz)
    return V


@pytest.mark.parametrize("mode", [0, 1])
def test_P2_P5_tallies_equal_recount_and_conservation_C1(oracle_mod, mode):
    """Paper L57: the tracked size always equals the number of sites the cell occupies; P5:
    no cell disappears and sum of volumes + medium == N."""
    import cpm_inputs as ci
    c = ci.make_config("C1")
    o = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], mode=mode, **c["params"])
    o.set_lattice(c["ids"], c["frozen"], c["cell_type"])
    N = int(np.prod(c["dims"]))
    alive0 = None
    for m in range(30):
        V = _check_tallies(o, c["max_cells"], 2)
        lat = o.get_lattice()
        assert V.sum() + int((lat == 0).sum()) == N
        alive = int((V[1:] > 0).sum())
        alive0 = alive if alive0 is None else alive0
        assert alive == alive0 == 64
        o.step(1)
    cnt = o.get_counters()
    assert cnt["attempts"] == 30 * N and cnt["mcs"] == 30


@pytest.mark.parametrize("periodic", [(0, 0, 0), (1, 1, 1)])
def test_P2_tallies_3d_perimeter_frozen(oracle_mod, periodic):
    import cpm_inputs as ci
    c = ci.make_config("C2", dims=(32, 32, 32))
    rng = np.random.default_rng(5)
    frozen = (rng.random(c["ids"].shape) < 0.05).astype(np.uint8)
    o = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], periodic=periodic, **c["params"])
    o.set_lattice(c["ids"], frozen, c["cell_type"])
    ids0 = c["ids"].copy()
    for m in range(4):
        _check_tallies(o, c["max_cells"], 3, periodic)
        o.step(1)
    _check_tallies(o, c["max_cells"], 3, periodic)
    lat = o.get_lattice()
    assert (lat != ids0).any()
    # frozen voxels never change (reading S14)
    np.testing.assert_array_equal(lat[frozen == 1], ids0[frozen == 1])


# ------------------------------------------------------------------------------------- P3 --
def _trace_run(ob, T, n_mcs=6, mode=0, seed=3):
    import cpm_inputs as ci
    c = ci.make_config("C1", dims=(64, 64))
    p = dict(c["params"]); p["T"] = T; p["seed"] = seed
    o = ob.Oracle(c["dims"], max_cells=c["max_cells"], mode=mode, **p)
    o.set_lattice(c["ids"], c["frozen"], c["cell_type"])
    buf, cnt = o.trace(64 * 64 * n_mcs)
    o.step(n_mcs)
    o.stop_trace()
    return buf[: int(cnt[0])], o


def test_P3_metropolis_limits(oracle_mod):
    """T = 0: no uphill move is ever accepted; T = +inf: every evaluated move is accepted."""
    tr, o = _trace_run(oracle_mod, 0.0)
    ev = tr[tr[:, 2] == 1]
    assert len(ev) > 100
    assert (ev[ev[:, 3] > 0][:, 4] == 0).all()
    assert (ev[ev[:, 3] <= 0][:, 4] == 1).all()
    tr, o = _trace_run(oracle_mod, float("inf"))
    ev = tr[tr[:, 2] == 1]
    assert len(ev) > 100 and (ev[:, 4] == 1).all()
    cnt = o.get_counters()
    refused = int((tr[:, 2] == 2).sum())
    assert cnt["accepted"] == cnt["evaluated"] - refused


# ------------------------------------------------------------------------------------- P4 --
def test_P4_acceptance_frequency_matches_eq2(oracle_mod):
    """Eq 2 (L227): P(accept | dH) = exp(-dH/T) for dH >= 0; 1 for dH < 0.  Binomial 4.5 sigma."""
    T = 20.0
    tr, _ = _trace_run(oracle_mod, T, n_mcs=60, seed=19)
    ev = tr[tr[:, 2] == 1]
    assert (ev[ev[:, 3] <= 0][:, 4] == 1).all()
    tested = 0
    for dh in np.unique(ev[:, 3]):
        if dh <= 0:
            continue
        sel = ev[ev[:, 3] == dh]
        n = len(sel)
        if n < 400:
            continue
        p = math.exp(-dh / T)
        k = int(sel[:, 4].sum())
        sigma = math.sqrt(n * p * (1 - p)) + 1e-9
        assert abs(k - n * p) <= 4.5 * sigma + 1, (dh, n, k, n * p)
        tested += 1
    assert tested >= 5
    # pooled check over everything uphill
    up = ev[(ev[:, 3] > 0)]
    exp_acc = np.exp(-up[:, 3] / T).sum()
    var = (np.exp(-up[:, 3] / T) * (1 - np.exp(-up[:, 3] / T))).sum()
    assert abs(up[:, 4].sum() - exp_acc) <= 4.5 * math.sqrt(var) + 1


# ------------------------------------------------------------------------------------- P6 --
@pytest.mark.parametrize("cfg,dims,act", [("C1", (64, 64), False), ("C3", (32, 32, 32), True)])
def test_P6_order_of_subsections_inside_a_phase_step_is_irrelevant(oracle_mod, cfg, dims, act):
    """Race-freedom of the checkerboard (L49): same-colour subsections never touch the same
    neighbourhood, so any visiting order gives the same lattice, tallies and Act field."""
    import cpm_inputs as ci
    c = ci.make_config(cfg, dims=dims)
    outs = []
    for order in (0, 1, 2):
        o = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], **c["params"])
        o.set_lattice(c["ids"], c["frozen"], c["cell_type"])
        o.set_visit_order(order, 99)
        o.step(5)
        outs.append((o.get_lattice().copy(), o.get_cell_stats(), o.get_act().copy(), o.get_counters()))
    assert (outs[0][0] != c["ids"]).any()
    if act:
        assert outs[0][2].max() > 0
    for other in outs[1:]:
        np.testing.assert_array_equal(outs[0][0], other[0])
        np.testing.assert_array_equal(outs[0][2], other[2])
        for k in outs[0][1]:
            np.testing.assert_array_equal(outs[0][1][k], other[1][k])
        assert outs[0][3] == other[3]


# ------------------------------------------------------------------------------------- P7 --
def test_P7_proposal_statistics_16x16(oracle_mod):
    """The paper's own set-up (L65): 16x16 grid, one MCS = 256 updates.  With one 16x16
    subsection the per-site attempt count per MCS is Binomial(256, 1/256): mean 1, variance
    1 - 1/256; neighbour index uniform over 8; exactly N attempts per MCS, all inside."""
    ob = oracle_mod
    J = np.array([[0, 5], [5, 9]], np.int32)
    o = ob.Oracle((16, 16), J=J, lambda_V=[0, 1], target_V=[0, 20], max_cells=1, subsection=16, seed=5)
    ids = np.zeros((16, 16), np.uint32); ids[4:10, 4:10] = 1
    o.set_lattice(ids, None, np.array([0, 1], np.uint8))
    M = 4000
    buf, cnt = o.trace(256 * M)
    o.step(M)
    tr = buf[: int(cnt[0])]
    assert len(tr) == 256 * M
    per_mcs = np.zeros((M, 256), np.int64)
    np.add.at(per_mcs, (np.repeat(np.arange(M), 256), tr[:, 0]), 1)
    assert (per_mcs.sum(1) == 256).all()
    assert abs(per_mcs.mean() - 1.0) < 1e-12
    var = per_mcs.var()
    assert abs(var - (1 - 1 / 256)) < 0.01, var
    # per-site totals: chi-square against uniform, 255 dof (mean 255, sd 22.6)
    tot = per_mcs.sum(0)
    chi = ((tot - M) ** 2 / M).sum()
    assert 150 < chi < 370, chi
    nb = np.bincount(tr[:, 1], minlength=8)
    chi_nb = ((nb - len(tr) / 8) ** 2 / (len(tr) / 8)).sum()
    assert chi_nb < 30, chi_nb  # 7 dof
    # waiting time between consecutive updates of a site is geometric-like: P(count=0) = (1-1/256)^256
    p0 = (per_mcs == 0).mean()
    assert abs(p0 - (1 - 1 / 256) ** 256) < 0.005


def test_P7_each_subsection_gets_its_own_attempts(oracle_mod):
    """Reading S11: each subsection gets exactly S^d attempts per MCS, all targets inside it,
    colours visited 0..2^d-1, R repetitions of k attempts."""
    import cpm_inputs as ci
    c = ci.make_config("C1", dims=(64, 32))
    p = dict(c["params"]); p["subsection"] = 8; p["attempts_per_activation"] = 16
    o = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], **p)
    o.set_lattice(c["ids"], None, c["cell_type"])
    sch = o.get_schedule()
    assert sch == {"S": 8, "k": 16, "phase_steps_per_mcs": 16}
    buf, cnt = o.trace(64 * 32)
    o.step(1)
    tr = buf[: int(cnt[0])]
    assert len(tr) == 64 * 32
    x = tr[:, 0] % 64; y = tr[:, 0] // 64
    b = (x // 8) + 8 * (y // 8)
    colour = ((x // 8) & 1) | (((y // 8) & 1) << 1)
    assert (np.bincount(b, minlength=32) == 64).all()
    # forward visiting order: within a phase-step, subsections ascending, k attempts each
    n_active = 32 // 4
    blocks = tr.reshape(16, n_active, 16, 6)
    for ps in range(16):
        cols = colour.reshape(16, n_active, 16)[ps]
        assert (cols == ps % 4).all()
        bs = b.reshape(16, n_active, 16)[ps]
        assert (bs == bs[:, :1]).all() and (np.diff(bs[:, 0]) > 0).all()


# ------------------------------------------------------------------------------------- P8 --
def test_P8_philox_known_answers(oracle_mod):
    rows = H.read_kat(os.path.join(GOLDEN, "philox4x32_10_kat.txt"))
    assert len(rows) >= 3
    for ctr, key, out in rows:
        np.testing.assert_array_equal(oracle_mod.philox4x32_10(ctr, key), np.array(out, np.uint32))
        assert H.philox_py(ctr, key) == out
    rng = np.random.default_rng(0)
    for _ in range(200):
        ctr = rng.integers(0, 1 << 32, 4); key = rng.integers(0, 1 << 32, 2)
        assert list(oracle_mod.philox4x32_10(ctr, key)) == H.philox_py(ctr, key)


def test_P8_counter_layout_and_decode(oracle_mod):
    """ctr = (a>>2, b, 2p+stream, mcs), key = seed (lo, hi); word a&3; decode by multiply-shift
    (readings S15, S16) -- recomputed here with the python Philox."""
    import cpm_inputs as ci
    c = ci.make_config("C1", dims=(32, 32))
    seed = (0xABCDEF12 << 32) | 0x00C0FFEE
    p = dict(c["params"]); p["seed"] = seed
    o = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], **p)
    o.set_lattice(c["ids"], None, c["cell_type"])
    o.set_mcs(41)
    buf, cnt = o.trace(32 * 32)
    o.step(1)
    tr = buf[: int(cnt[0])]
    offs = H.moore_offsets(2)
    i = 0
    thr_hmax, thr = oracle_mod.threshold_table(20.0)
    for pstep in range(4):
        for b in range(4):
            bx, by = b % 2, b // 2
            if ((bx & 1) | ((by & 1) << 1)) != pstep:
                continue
            for a in range(256):
                call, word = a >> 2, a & 3
                w = H.philox_py([call, b, 2 * pstep, 41], [seed & 0xFFFFFFFF, seed >> 32])[word]
                prod = w * 256
                l = prod >> 32
                nb = ((prod & 0xFFFFFFFF) * 8) >> 32
                assert oracle_mod.decode_proposal(w, 256, 8) == (l, nb)
                tx, ty = bx * 16 + l % 16, by * 16 + l // 16
                assert tr[i, 0] == tx + 32 * ty and tr[i, 1] == nb, (pstep, b, a)
                if tr[i, 2] == 1 and 0 < tr[i, 3] <= thr_hmax:
                    u = H.philox_py([call, b, 2 * pstep + 1, 41], [seed & 0xFFFFFFFF, seed >> 32])[word]
                    assert tr[i, 5] == u
                    assert tr[i, 4] == int(u < thr[tr[i, 3]])
                i += 1
    assert i == len(tr)


# ------------------------------------------------------------------------------------ P10 --
def test_P10_resume_is_exact(oracle_mod):
    """Counter-based RNG: step(a+b) == step(a), save, restore into a new context, step(b)."""
    import cpm_inputs as ci
    c = ci.make_config("C3", dims=(32, 32, 32))
    o = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], **c["params"])
    o.set_lattice(c["ids"], c["frozen"], c["cell_type"])
    o.step(7)
    ref_l, ref_a, ref_s = o.get_lattice().copy(), o.get_act().copy(), o.get_cell_stats()
    o1 = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], **c["params"])
    o1.set_lattice(c["ids"], c["frozen"], c["cell_type"])
    o1.step(3)
    o2 = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], **c["params"])
    o2.set_lattice(o1.get_lattice(), c["frozen"], c["cell_type"])
    o2.set_act(o1.get_act())
    o2.set_mcs(3)
    o2.step(4)
    np.testing.assert_array_equal(ref_l, o2.get_lattice())
    np.testing.assert_array_equal(ref_a, o2.get_act())
    for k in ref_s:
        np.testing.assert_array_equal(ref_s[k], o2.get_cell_stats()[k])


# ------------------------------------------------------------------------------------ P11 --
def test_P11_fixed_point_geometric_mean(oracle_mod):
    """Reading S8(iv) vs Eq 9 in double: relative error <= 2^(1/1024)-1 (+ rounding), exact for
    equal powers of two, 0 if any activity is 0."""
    gm = oracle_mod.gm_q16
    assert gm([0]) == 0 and gm([5, 0, 9]) == 0
    for p2 in (1, 2, 4, 8, 16, 32, 64, 128):
        for n in (1, 2, 5, 27):
            assert gm([p2] * n) == p2 * 65536
    rng = np.random.default_rng(3)
    worst = 0.0
    for n in list(range(1, 28)) * 40:
        a = rng.integers(1, 256, size=n)
        exact = float(np.exp(np.log(a.astype(np.float64)).mean()))
        got = gm(a) / 65536.0
        worst = max(worst, abs(got - exact) / exact)
    assert worst <= (2 ** (1 / 1024) - 1) + 3e-5, worst
    # all multisets on a small alphabet, n <= 3
    vals = [1, 2, 3, 7, 40, 255]
    for n in (1, 2, 3):
        for combo in np.ndindex(*([len(vals)] * n)):
            a = [vals[i] for i in combo]
            exact = float(np.prod(a)) ** (1.0 / n)
            assert abs(gm(a) / 65536.0 - exact) / exact <= 7.2e-4


def test_P11_act_bias_sign_and_decay(oracle_mod):
    """Eq 8 with reading S8(i): a copy FROM a high-activity area is MORE likely (dH lowered);
    reading S9: Act(t) = Max_act on an accepted copy, decays by 1 per MCS down to 0 (L255)."""
    ob = oracle_mod
    J = np.array([[0, 5], [5, 9]], np.int32)
    o = ob.Oracle((8, 8), J=J, lambda_V=[0, 1], target_V=[0, 12], lambda_act=[0, 200], max_act=[0, 40],
                  max_cells=2, subsection=8, T=20.0)
    ids = np.zeros((8, 8), np.uint32); ids[2:5, 1:4] = 1; ids[2:5, 4:7] = 2
    o.set_lattice(ids, None, np.array([0, 1, 1], np.uint8))
    act = np.zeros((8, 8), np.float32); act[ids == 1] = 40.0; act[ids == 2] = 5.0
    o.set_act(act)
    offs = H.moore_offsets(2); nb_of = {o_: i for i, o_ in enumerate(offs)}
    t = 4 + 8 * 3  # site (4,3) of cell 2; source (3,3) of cell 1, fully active
    st, dH, dA = o.probe(t, nb_of[(-1, 0, 0)])
    assert st == 1
    # GM(source) = 40, |N| = 6 same-cell sites incl. itself; GM(target) = 5
    assert dA == round(200 / 40 * 40 - 200 / 40 * 5)
    # reverse direction: copying the low-activity cell into the high-activity one is penalised
    st2, dH2, dA2 = o.probe(3 + 8 * 3, nb_of[(1, 0, 0)])
    assert st2 == 1 and dA2 == -dA
    o.force_copy(t, nb_of[(-1, 0, 0)])
    a1 = o.get_act()
    assert a1[3, 4] == 40.0
    o2 = ob.Oracle((8, 8), J=J, lambda_V=[0, 1], target_V=[0, 12], lambda_act=[0, 200], max_act=[0, 40],
                   max_cells=2, subsection=8, T=0.0)
    o2.set_lattice(np.zeros((8, 8), np.uint32), None, np.array([0, 1, 1], np.uint8))
    a = np.zeros((8, 8), np.float32); a[0, 0] = 3; a[1, 1] = 255
    o2.set_act(a)
    o2.step(2)
    g = o2.get_act()
    assert g[0, 0] == 1 and g[1, 1] == 253 and g[2, 2] == 0
    o2.step(2)
    assert o2.get_act()[0, 0] == 0


# ------------------------------------------------------------------------------------ P12 --
@pytest.mark.parametrize("T", [20.0, 10.0, 1.0, 0.5, 137.5])
def test_P12_threshold_table(oracle_mod, T):
    """Reading S7: thr[h] = floor(exp(-h/T) 2^32), Hmax = floor(T 32 ln2): monotone, thr[Hmax] >= 1,
    and the next entry would be 0."""
    hmax, thr = oracle_mod.threshold_table(T)
    assert hmax == math.floor(T * 32 * math.log(2))
    assert len(thr) == hmax + 1
    t = thr[1:].astype(np.int64)
    assert (np.diff(t) <= 0).all()
    assert t[-1] >= 1
    assert math.floor(math.exp(-(hmax + 1) / T) * 2 ** 32) == 0
    for h in (1, 2, hmax // 2, hmax):
        exact = math.exp(-h / T) * 2 ** 32
        assert abs(int(thr[h]) - exact) <= 1 + exact * 1e-12


# ------------------------------------------------------------------------------------ P13 --
def test_P13_deterministic_equals_live_while_no_cell_is_shared(oracle_mod):
    """Reading S12: when no cell is touched by two subsections of the same phase-step the
    snapshot+own-deltas reading sees exactly the live values, so both modes agree bit for bit.
    Config C1 starts inside the precondition (8x8 cells centred in 16x16 subsections)."""
    import cpm_inputs as ci
    c = ci.make_config("C1")
    od = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], mode=0, **c["params"])
    ol = oracle_mod.Oracle(c["dims"], max_cells=c["max_cells"], mode=1, **c["params"])
    for o in (od, ol):
        o.set_lattice(c["ids"], c["frozen"], c["cell_type"])
    agreed = 0
    S = 16
    for m in range(40):
        lat = od.get_lattice()
        # sufficient precondition: every cell (plus the 1-voxel halo that can read it) lies in one subsection
        ok = True
        for cell in range(1, c["max_cells"] + 1):
            ys, xs = np.nonzero(lat == cell)
            if len(xs) == 0:
                continue
            if (xs.min() - 1) // S != (xs.max() + 1) // S or (ys.min() - 1) // S != (ys.max() + 1) // S:
                ok = False
                break
        if not ok:
            break
        od.step(1); ol.step(1)
        np.testing.assert_array_equal(od.get_lattice(), ol.get_lattice())
        for k, v in od.get_cell_stats().items():
            np.testing.assert_array_equal(v, ol.get_cell_stats()[k])
        agreed += 1
    assert agreed >= 3, agreed


# ------------------------------------------------------------------------------- misc ------
def test_extinction_rule(oracle_mod):
    """Reading S13: a copy that would erase a cell (V <= 1) is refused; cells are conserved."""
    ob = oracle_mod
    J = np.array([[0, 1], [1, 1]], np.int32)
    o = ob.Oracle((4, 4), J=J, lambda_V=[0, 50], target_V=[0, 0], max_cells=1, subsection=4, T=float("inf"))
    ids = np.zeros((4, 4), np.uint32); ids[1, 1] = 1
    o.set_lattice(ids, None, np.array([0, 1], np.uint8))
    st, _, _ = o.probe(1 + 4 * 1, 0)
    assert st == 2
    o.step(50)
    assert o.get_cell_stats()["volume"][1] >= 1


def test_argument_validation(oracle_mod):
    ob = oracle_mod
    J = np.array([[0, 1], [2, 1]], np.int32)
    with pytest.raises(ob.OracleError):
        ob.Oracle((8, 8), J=J, max_cells=1)                   # non-symmetric J
    Js = np.array([[0, 1], [1, 1]], np.int32)
    with pytest.raises(ob.OracleError):
        ob.Oracle((10, 8), J=Js, max_cells=1, subsection=4)   # S does not divide dims
    with pytest.raises(ob.OracleError):
        ob.Oracle((12, 12), J=Js, max_cells=1, subsection=4, periodic=(1, 0, 0))  # odd count, periodic
    with pytest.raises(ob.OracleError):
        ob.Oracle((8, 8), J=Js, max_cells=1, T=-1.0)
    o = ob.Oracle((8, 8), J=Js, max_cells=1)
    with pytest.raises(ob.OracleError):
        o.set_lattice(np.full((8, 8), 2, np.uint32), None, np.array([0, 1], np.uint8))  # id > max_cells
    with pytest.raises(ob.OracleError):
        o.step(1)                                             # no lattice yet


# ------------------------------------------------ pins added in round 2 --
def _straddling_case(nd, S, n_per_axis, edge, lamP, act):
    """Cells of extent `edge` <= S-2 on pitch S, offset by S/2 + 1 so that every cell STRADDLES a
    subsection border (it is touched by subsections of different colours, i.e. in different
    phase-steps, but never by two subsections of the same phase-step)."""
    dims = (S * n_per_axis,) * nd
    ids = np.zeros(tuple(reversed(dims)), np.uint32)
    off = S // 2 + 1
    n = 0
    rng = range(n_per_axis - 1)
    for idx in np.ndindex(*([n_per_axis - 1] * nd)):       # idx = (z, y, x) / (y, x)
        n += 1
        sl = tuple(slice(off + S * i, off + S * i + edge) for i in idx)
        ids[sl] = n
    ct = np.ones(n + 1, np.uint8); ct[0] = 0
    ct[2::2] = 2
    J = np.array([[0, 8, 11], [8, 14, 19], [11, 19, 9]], np.int32)
    vol = edge ** nd
    per = int(H.recount(ids, n, nd)[1][1])      # Moore-interface count of one seed block
    kw = dict(J=J, lambda_V=[0, 3, 2], target_V=[0, vol, vol + 3], lambda_P=[0, lamP, lamP],
              target_P=[0, per, per - 6], T=20.0, seed=4242, subsection=S, max_cells=n)
    if act:
        kw.update(lambda_act=[0, 150, 60], max_act=[0, 30, 9])
    return dims, ids, ct, kw


def _no_cell_shared_within_a_phase_step(lat, max_cells, S):
    """SURVEY P13's precondition, checked exactly: a subsection TOUCHES a cell that has a voxel inside it
    or in its 1-voxel halo; no cell may be touched by two subsections of the same colour (= of the same
    phase-step)."""
    nd = lat.ndim
    dims = lat.shape[::-1]
    for cell in range(1, max_cells + 1):
        idx = np.nonzero(lat == cell)            # (z, y, x) / (y, x)
        if len(idx[0]) == 0:
            continue
        coords = np.stack(idx[::-1], 1)          # columns x, y(, z)
        touched = set()
        for shift in np.ndindex(*([3] * nd)):
            c = coords + (np.array(shift) - 1)
            ok = np.ones(len(c), bool)
            for a in range(nd):
                ok &= (c[:, a] >= 0) & (c[:, a] < dims[a])
            for b in np.unique(c[ok] // S, axis=0):
                touched.add(tuple(int(v) for v in b))
        colours = [tuple(v & 1 for v in b) for b in touched]
        if len(set(colours)) != len(colours):
            return False
    return True


@pytest.mark.parametrize("nd,S,n_ax,edge,act", [(2, 16, 5, 10, False), (2, 16, 4, 9, True), (3, 8, 4, 4, True)])
def test_P13b_deterministic_equals_live_with_cells_straddling_borders(oracle_mod, nd, S, n_ax, edge, act):
    """Reading S12 under SURVEY P13's ACTUAL precondition (no cell touched by two subsections of the
    SAME phase-step; sufficient: extent <= S-2), with cells that straddle subsection borders and
    lambda_P != 0.  A straddling cell is changed by one subsection in one phase-step and read by its
    neighbour subsection in a later phase-step of the same MCS, so the two modes agree bit for bit
    only if (i) the snapshot is refreshed at EVERY phase-step (reads may be stale
    only within a step) and (ii) the worker's own deltas carry dP as well as dV."""
    dims, ids, ct, kw = _straddling_case(nd, S, n_ax, edge, lamP=1, act=act)
    n = kw["max_cells"]
    od = oracle_mod.Oracle(dims, mode=0, **kw)
    ol = oracle_mod.Oracle(dims, mode=1, **kw)
    for o in (od, ol):
        o.set_lattice(ids, None, ct)
    # the set-up really straddles: every cell has voxels in at least two subsections
    for cell in range(1, n + 1):
        idx = np.nonzero(ids == cell)
        assert any(ax.min() // S != ax.max() // S for ax in idx)
    agreed = 0
    multi = 0
    for m in range(12):
        if not _no_cell_shared_within_a_phase_step(od.get_lattice(), n, S):
            break
        before = od.get_cell_stats()["perimeter"].astype(np.int64)
        od.step(1); ol.step(1)
        np.testing.assert_array_equal(od.get_lattice(), ol.get_lattice(), err_msg="MCS %d" % m)
        sd, sl = od.get_cell_stats(), ol.get_cell_stats()
        for k in sd:
            np.testing.assert_array_equal(sd[k], sl[k], err_msg="%s MCS %d" % (k, m))
        if act:
            np.testing.assert_array_equal(od.get_act(), ol.get_act())
        assert od.get_counters() == ol.get_counters()
        multi += int((sd["perimeter"].astype(np.int64) != before).sum())
        agreed += 1
    assert agreed >= 4, agreed
    assert multi >= 4 * n // 2          # perimeters really move, so a stale P would be seen
    c = od.get_counters()
    assert c["accepted"] > 20 * agreed


def test_P11b_act_bias_uses_each_sides_own_type(oracle_mod):
    """Eq 8-9 with reading S8(iii): the source side uses lambda_act/Max_act of
    the SOURCE cell's type, the target side those of the TARGET cell's type.  Two motile types with
    different (lambda_act, Max_act); expected dH_act recomputed here in double from Eq 8-9."""
    ob = oracle_mod
    J = np.array([[0, 5, 6], [5, 9, 7], [6, 7, 4]], np.int32)
    lam, mx = [0, 200, 96], [0, 40, 12]
    o = ob.Oracle((8, 8), J=J, lambda_V=[0, 1, 1], target_V=[0, 9, 9], lambda_act=lam, max_act=mx,
                  max_cells=2, subsection=8, T=20.0)
    ids = np.zeros((8, 8), np.uint32); ids[2:5, 1:4] = 1; ids[2:5, 4:7] = 2
    ct = np.array([0, 1, 2], np.uint8)
    o.set_lattice(ids, None, ct)
    rng = np.random.default_rng(5)
    act = np.zeros((8, 8), np.float32)
    act[ids == 1] = rng.integers(20, 41, int((ids == 1).sum()))
    act[ids == 2] = rng.integers(3, 13, int((ids == 2).sum()))
    o.set_act(act)
    offs = H.moore_offsets(2); nb_of = {o_: i for i, o_ in enumerate(offs)}

    def gm(x, y):            # Eq 9 over {site} + same-cell Moore neighbours (reading S8(ii)), in double
        vals = [float(act[y, x])]
        for dx, dy, _ in offs:
            xx, yy = x + dx, y + dy
            if 0 <= xx < 8 and 0 <= yy < 8 and ids[yy, xx] == ids[y, x]:
                vals.append(float(act[yy, xx]))
        return float(np.exp(np.mean(np.log(vals))))

    checked = 0
    for (tx, ty), (dx, dy) in [((4, 3), (-1, 0)), ((3, 3), (1, 0)), ((4, 2), (-1, 1)), ((3, 4), (1, -1)), ((4, 4), (-1, 0))]:
        sx, sy = tx + dx, ty + dy
        tA, tB = int(ct[ids[sy, sx]]), int(ct[ids[ty, tx]])
        assert tA != tB and tA and tB
        st, dH, dA = o.probe(tx + 8 * ty, nb_of[(dx, dy, 0)])
        assert st == 1
        exact = lam[tA] / mx[tA] * gm(sx, sy) - lam[tB] / mx[tB] * gm(tx, ty)
        wrong = lam[tA] / mx[tA] * gm(sx, sy) - lam[tA] / mx[tA] * gm(tx, ty)   # target side with the source's type
        tol = 0.5 + 7.2e-4 * (lam[tA] / mx[tA] * gm(sx, sy) + lam[tB] / mx[tB] * gm(tx, ty)) + 1e-3
        assert abs(dA - exact) <= tol, (dA, exact)
        assert abs(dA - wrong) > 5 * tol      # the cases tell the two readings apart
        checked += 1
    assert checked == 5


def test_act_decay_runs_after_the_last_phase_step(oracle_mod):
    """PAPER.md L255 / reading S9: a copied-into site gets Act = Max_act of its new owner, and the field
    decays by 1 once per MCS AFTER the last phase-step.  So after one MCS every site that received its
    last accepted copy in that MCS holds Max_act(new owner) - 1 (0 for medium), and untouched sites hold
    their start value - 1.  (Decay before the phase loop would leave Max_act itself.)"""
    ob = oracle_mod
    J = np.array([[0, 5, 6], [5, 9, 7], [6, 7, 4]], np.int32)
    mx = [0, 40, 17]
    o = ob.Oracle((16, 16), J=J, lambda_V=[0, 1, 1], target_V=[0, 30, 30], lambda_act=[0, 100, 50], max_act=mx,
                  max_cells=4, subsection=4, T=float("inf"), seed=3)
    ids = np.zeros((16, 16), np.uint32)
    ids[2:8, 2:8] = 1; ids[2:8, 8:14] = 2; ids[8:14, 2:8] = 3; ids[8:14, 8:14] = 4
    ct = np.array([0, 1, 2, 2, 1], np.uint8)
    o.set_lattice(ids, None, ct)
    act0 = np.zeros((16, 16), np.float32); act0[ids > 0] = 7.0
    o.set_act(act0)
    buf, cnt = o.trace(16 * 16)
    o.step(1)
    o.stop_trace()
    assert int(cnt[0]) == 256
    lat, act = o.get_lattice(), o.get_act()
    last_owner = {}
    for site, nb, status, dH, acc, u in buf[: int(cnt[0])]:
        if acc:
            last_owner[int(site)] = True
    assert len(last_owner) >= 20
    for y in range(16):
        for x in range(16):
            if (x + 16 * y) in last_owner:
                owner = int(lat[y, x])
                want = max(mx[ct[owner]] - 1, 0) if owner else 0
            else:
                want = max(float(act0[y, x]) - 1, 0)
            assert act[y, x] == want, (x, y, act[y, x], want)
