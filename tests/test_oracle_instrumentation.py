"""Pins of the oracle's instrumentation: interface counts by cell type (the sorting observable of
PAPER.md Fig 4, L69) and the update statistics of the checkerboard schedule (Fig 3, L65-79).

Expected sides: the brute-force Hamiltonian of tests/helpers.py, a direct pair count, closed forms of the serial
limit (geometric waiting times, binomial pick counts -- the paper's own 16x16 / 256-update set-up), and a pure-python
restatement on the python Philox."""
import itertools

import numpy as np
import pytest

import helpers as H


# ------------------------------------------------------------------------------------ P17 --
@pytest.mark.parametrize("dims,periodic,sub", [((6, 4), (0, 0, 0), 2), ((6, 6), (1, 0, 0), 3), ((4, 6, 4), (0, 0, 0), 2), ((4, 4, 4), (1, 1, 1), 2)])
def test_P17_interface_counts(oracle_mod, dims, periodic, sub):
    """sum over type pairs of J(a,b) x count(a,b) == the adhesion part of Eq 1 (brute force over the whole lattice), for
    several J with distinct entries; and the counts equal a direct enumeration of unordered Moore pairs."""
    nd = len(dims)
    rng = np.random.default_rng(7 + sum(dims))
    shape = tuple(reversed(dims))
    n_cells = 6
    ids = rng.integers(0, n_cells + 1, size=shape).astype(np.uint32)
    ct = np.array([0, 1, 2, 1, 2, 3, 3], dtype=np.uint8)
    nT = 4
    o = oracle_mod.Oracle(dims, J=np.zeros((nT, nT), dtype=np.int32), subsection=sub, max_cells=n_cells, periodic=periodic)
    o.set_lattice(ids, None, ct)
    C = o.get_interface_counts().astype(np.int64)
    np.testing.assert_array_equal(C, C.T)
    # direct enumeration
    want = np.zeros((nT, nT), dtype=np.int64)
    ids3 = ids if nd == 3 else ids[None]
    Z, Y, X = ids3.shape
    seen = set()
    for z, y, x in itertools.product(range(Z), range(Y), range(X)):
        for dx, dy, dz in H.moore_offsets(nd):
            c = [x + dx, y + dy, z + dz]
            outside = False
            for a, n in enumerate((X, Y, Z)):
                if c[a] < 0 or c[a] >= n:
                    if periodic[a]:
                        c[a] %= n
                    else:
                        outside = True
            me = int(ids3[z, y, x]); other = 0 if outside else int(ids3[c[2], c[1], c[0]])
            if me == other:
                continue
            if outside:
                key = ((x, y, z), (dx, dy, dz))
            else:   # an inside pair is met from both ends: keep it once
                key = (min((x, y, z), tuple(c)), max((x, y, z), tuple(c)), (dx, dy, dz) if (x, y, z) < tuple(c) else (-dx, -dy, -dz))
            if key in seen:
                continue
            seen.add(key)
            a, b = int(ct[me]), int(ct[other])
            want[a, b] += 1
            if a != b:
                want[b, a] += 1
    np.testing.assert_array_equal(C, want)
    for trial in range(3):
        J = rng.integers(-20, 40, size=(nT, nT)); J = np.triu(J) + np.triu(J, 1).T
        Hadh = H.brute_force_H(ids, ct, J, [0] * nT, [0] * nT, [0] * nT, [0] * nT, nd, periodic)
        assert int((np.triu(C) * J).sum()) == Hadh


# ------------------------------------------------------------------------------------ P18 --
def test_P18_serial_limit_geometric_waits_and_binomial_counts(oracle_mod):
    """The paper's own set-up (L65, Fig 3C left column): a 16x16 grid as ONE region, 256 updates per MCS, 100 MCS.
    A position is picked with probability 1/256 per update: waiting times are geometric, picks per MCS Binomial(256, 1/256)."""
    N = 256
    tot_w = np.zeros(2048, dtype=np.float64); tot_f = np.zeros(10, dtype=np.float64)
    for seed in range(20):
        o = oracle_mod.Oracle((16, 16), J=np.zeros((2, 2), dtype=np.int32), subsection=16, max_cells=1, seed=900 + seed)
        o.set_lattice(np.zeros((16, 16), dtype=np.uint32), None, np.array([0, 1], dtype=np.uint8))
        f, w = o.update_statistics(100, n_freq=10, n_wait=2048, wait_bin=1)
        assert int(f.sum()) == N * 100                      # every (position, MCS) pair is in the histogram
        assert int(w.sum()) + N >= N * 100 - 40             # all picks but the first of each position (a few never picked)
        tot_w += w; tot_f += f
    p = 1.0 / N
    j = np.arange(1, 2049)
    pw = p * (1 - p) ** (j - 1)
    # compare in coarse bins (expected counts large), 5 sigma
    edges = [0, 32, 64, 128, 192, 256, 384, 512, 768, 1024, 1536, 2047]
    n = tot_w.sum()
    for lo, hi in zip(edges[:-1], edges[1:]):
        ex = n * pw[lo:hi].sum(); got = tot_w[lo:hi].sum()
        assert abs(got - ex) < 5 * np.sqrt(ex) + 5, (lo, hi, got, ex)
    from math import comb
    nf = tot_f.sum()
    for k in range(6):
        ex = nf * comb(N, k) * p ** k * (1 - p) ** (N - k)
        assert abs(tot_f[k] - ex) < 5 * np.sqrt(ex) + 5, (k, tot_f[k], ex)


@pytest.mark.parametrize("dims,S,k,mcs0", [((8, 8), 4, 4, 0), ((8, 12), 4, 16, 7), ((4, 4, 4), 2, 8, 3), ((6, 6), 6, 36, 0)])
def test_P18_update_statistics_equal_python_restatement(oracle_mod, dims, S, k, mcs0):
    """Both histograms restated in pure python on the python Philox4x32-10 (itself pinned by the published vectors):
    counter (a>>2, b, 2p, mcs), word a&3, multiply-shift decode (S15, S16), colours in order, lock-step ticks."""
    nd = len(dims)
    seed = 0x1234567855AA
    o = oracle_mod.Oracle(dims, J=np.zeros((2, 2), dtype=np.int32), subsection=S, attempts_per_activation=k, max_cells=1, seed=seed)
    o.set_lattice(np.zeros(tuple(reversed(dims)), dtype=np.uint32), None, np.array([0, 1], dtype=np.uint8))
    o.set_mcs(mcs0)
    n_mcs, n_freq, n_wait, wbin = 6, 5, 40, 3
    f, w = o.update_statistics(n_mcs, n_freq=n_freq, n_wait=n_wait, wait_bin=wbin)
    sites = S ** nd
    R = sites // k
    nsub = [d // S for d in dims] + ([1] if nd == 2 else [])
    ncol = 1 << nd
    nNb = 8 if nd == 2 else 26
    subs = list(itertools.product(range(nsub[2]), range(nsub[1]), range(nsub[0])))
    colour = lambda bx, by, bz: (bx & 1) | ((by & 1) << 1) | ((bz & 1) << 2)
    occurs = sorted({colour(bx, by, bz) for bz, by, bx in subs})
    E = len(occurs) * R
    last = {}; wf = np.zeros(n_freq, dtype=np.int64); ww = np.zeros(n_wait, dtype=np.int64)
    for m in range(n_mcs):
        cnt = {}
        e = 0
        for rep in range(R):
            for col in occurs:
                p = rep * ncol + col
                for bz, by, bx in subs:
                    if colour(bx, by, bz) != col:
                        continue
                    b = bx + nsub[0] * (by + nsub[1] * bz)
                    for a in range(k):
                        wd = H.philox_py((a >> 2, b, 2 * p, mcs0 + m), (seed & 0xFFFFFFFF, seed >> 32))[a & 3]
                        l = (wd * sites) >> 32
                        site = (bx * S + l % S, by * S + (l // S) % S, bz * S + l // (S * S))
                        tick = (m * E + e) * k + a
                        if site in last:
                            ww[min((tick - last[site] - 1) // wbin, n_wait - 1)] += 1
                        last[site] = tick
                        cnt[site] = cnt.get(site, 0) + 1
                e += 1
        for site in itertools.product(range(dims[0]), range(dims[1]), range(dims[2] if nd == 3 else 1)):
            wf[min(cnt.get(site, 0), n_freq - 1)] += 1
    np.testing.assert_array_equal(f.astype(np.int64), wf)
    np.testing.assert_array_equal(w.astype(np.int64), ww)
    # the lattice and the MCS counter were not touched
    assert o.get_counters()["mcs"] == mcs0 and o.get_counters()["attempts"] == 0
