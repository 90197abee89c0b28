"""Pins of the oracle's vector terms: chemotaxis along a vector field (Eq 4)
and persistence along one vector per cell (Eq 5-7), readings S21-S22 of DESIGN.md.

The expected side never comes from the oracle: the direction table and dH are restated in double precision from
Eq 4-5, the recurrence of Eq 6-7 in numpy on the recorded centroids, the sign by the direction a cell drifts in."""
import numpy as np
import pytest

import helpers as H


def _unit(v):
    n = np.linalg.norm(v, axis=-1, keepdims=True)
    return np.where(n > 0, v / np.where(n > 0, n, 1), 0.0)


# ------------------------------------------------------------------------------------ P14 --
@pytest.mark.parametrize("ndim", [2, 3])
def test_P14_direction_table(oracle_mod, ndim):
    """x^_{i->j} of neighbour index nb is the unit vector from the source s = t + OFF[nb] to the target t (Eq 4-5),
    in Q14; nb enumerates the Moore offsets (dz,dy,dx) lexicographically, dx fastest (S16)."""
    off = np.array(H.moore_offsets(ndim), dtype=np.float64)     # independent enumeration in tests/helpers.py
    want = np.rint(16384.0 * (-off) / np.linalg.norm(off, axis=1, keepdims=True)).astype(np.int64)
    got = oracle_mod.direction_table(ndim)
    np.testing.assert_array_equal(got, want)
    assert (np.abs(np.linalg.norm(got / 16384.0, axis=1) - 1.0) < 1e-4).all()


def _vector_case(ob, rng, dims, periodic=(0, 0, 0), sub=None):
    nd = len(dims)
    shape = tuple(reversed(dims))
    n_cells = 5
    ids = rng.integers(0, n_cells + 1, size=shape).astype(np.uint32)
    frozen = (rng.random(shape) < 0.08).astype(np.uint8)
    cell_type = np.zeros(n_cells + 1, dtype=np.uint8)
    cell_type[1:] = [1, 2, 1, 2, 2]
    J = np.array([[0, 7, -3], [7, 11, 16], [-3, 16, 5]], dtype=np.int32)
    lam_pers, lam_chem = [9, 40, 23], [7, 10, 31]     # type 0 entries must be ignored: medium has no terms (S3)
    o = ob.Oracle(dims, J=J, lambda_V=[0, 4, 6], target_V=[0, 9, 14], lambda_P=[0, 3, 2], target_P=[0, 30, 41],
                  T=20.0, seed=5, subsection=sub or dims[0], max_cells=n_cells, periodic=periodic,
                  lambda_pers=lam_pers, mu_pers=[0.0, 0.95, 0.5], dt_pers=3, lambda_chem=lam_chem)
    o.set_lattice(ids, frozen, cell_type)
    field = _unit(rng.normal(size=shape + (nd,))).astype(np.float32)
    o.set_chemotaxis_field(field)
    phat = np.zeros((n_cells + 1, 3))
    v = rng.normal(size=(n_cells, 3))
    if nd == 2:
        v[:, 2] = 0
    phat[1:] = _unit(v)
    phat[3] = 0.0                         # a cell without a direction yet
    phat[0] = [1.0, 0.0, 0.0]             # entry of medium: must be ignored (S3)
    o.set_persistence(phat)
    return o, ids, frozen, cell_type, lam_pers, lam_chem, field, phat


@pytest.mark.parametrize("dims,periodic,sub", [((7, 7), (0, 0, 0), 7), ((6, 6), (1, 1, 0), 3), ((5, 5, 5), (0, 0, 0), 5),
                                               ((4, 6, 4), (1, 0, 1), 2)])
def test_P14_dH_of_vector_terms_equals_eq4_eq5_in_double(oracle_mod, dims, periodic, sub):
    """dH_dir == round(lambda_pers(tau_A) x^.p^_A + lambda_pers(tau_B) x^.p^_B + (lambda_chem(tau_A) + lambda_chem(tau_B)) x^.C_s)
    with x^ = (t - s)/|t - s|, C at the SOURCE site (Eq 4: C_i), each side only for a real cell (S3), the field 0
    outside a closed lattice; the integer result may differ from the double one by the Q14 quantisation only."""
    rng = np.random.default_rng(101 + sum(dims))
    o, ids, frozen, ct, lam_pers, lam_chem, field, phat = _vector_case(oracle_mod, rng, dims, periodic, sub)
    nd = len(dims)
    off = H.moore_offsets(nd)
    N = int(np.prod(dims))
    X, Y = dims[0], dims[1]
    Z = dims[2] if nd == 3 else 1
    seen_outside = seen_medium = checked = 0
    for t in range(N):
        tx, ty, tz = t % X, (t // X) % Y, t // (X * Y)
        for nb in range(len(off)):
            st, _, _ = o.probe(t, nb)
            got = o.probe_dir(t, nb)
            if st != 1:
                assert got == 0
                continue
            d = np.array(off[nb], dtype=np.float64)
            s = [tx + int(d[0]), ty + int(d[1]), tz + int(d[2])]
            inside = True
            for a, (dim, per) in enumerate(zip((X, Y, Z), periodic)):
                if s[a] < 0 or s[a] >= dim:
                    if per:
                        s[a] %= dim
                    else:
                        inside = False
            xhat = -d / np.linalg.norm(d)
            A = int(ids[s[2], s[1], s[0]] if nd == 3 else ids[s[1], s[0]]) if inside else 0
            B = int(ids.reshape(-1)[t])
            C = np.zeros(3)
            if inside:
                C[:nd] = field[s[2], s[1], s[0]] if nd == 3 else field[s[1], s[0]]
            else:
                seen_outside += 1
            want = 0.0
            lam_c = 0
            if A != 0:
                want += lam_pers[ct[A]] * float(xhat @ phat[A]); lam_c += lam_chem[ct[A]]
            else:
                seen_medium += 1
            if B != 0:
                want += lam_pers[ct[B]] * float(xhat @ phat[B]); lam_c += lam_chem[ct[B]]
            want += lam_c * float(xhat @ C)
            # |round(q) - w| <= 1/2 + |q - w|; q - w: Q14 rounding of 3 vectors, < 3 * 2^-14 per unit of lambda
            tol = 0.5 + (abs(lam_pers[ct[A]]) + abs(lam_pers[ct[B]]) + abs(lam_c)) * 3.0 / 16384.0
            assert abs(got - want) <= tol, (t, nb, got, want)
            checked += 1
    assert checked > 200 and seen_medium > 0 and (any(periodic[:nd]) and all(periodic[:nd]) or seen_outside > 0)


def _single_cell_2d(ob, seed, **kw):
    dims = (48, 48)
    ids = np.zeros((48, 48), dtype=np.uint32)
    ids[19:29, 19:29] = 1
    o = ob.Oracle(dims, J=np.array([[0, 10], [10, 20]], dtype=np.int32), lambda_V=[0, 20], target_V=[0, 100],
                  lambda_P=[0, 1], target_P=[0, 110], T=10.0, seed=seed, subsection=48, max_cells=1, **kw)
    o.set_lattice(ids, None, np.array([0, 1], dtype=np.uint8))
    return o


def _centroid(o):
    st = o.get_cell_stats()
    v = st["volume"][1].astype(np.float64)
    return np.array([st["sum_x"][1] / v, st["sum_y"][1] / v])


def test_P14_sign_a_cell_drifts_along_the_field(oracle_mod):
    """Eq 4 is a bias that moves cells ALONG the field (chemotaxis, L95): with a uniform field (+1, 0) the centroid
    of a lone cell moves in +x, with (0, -1) in -y; without the term it stays (control)."""
    moved = []
    for fx, fy in ((1.0, 0.0), (0.0, -1.0)):
        disp = []
        for seed in range(4):
            o = _single_cell_2d(oracle_mod, 100 + seed, lambda_chem=[0, 40])
            f = np.zeros((48, 48, 2), dtype=np.float32); f[..., 0] = fx; f[..., 1] = fy
            o.set_chemotaxis_field(f)
            c0 = _centroid(o); o.step(60); disp.append(_centroid(o) - c0)
        moved.append(np.mean(disp, axis=0))
    assert moved[0][0] > 4.0 and abs(moved[0][1]) < 2.5, moved
    assert moved[1][1] < -4.0 and abs(moved[1][0]) < 2.5, moved
    o = _single_cell_2d(oracle_mod, 100)
    c0 = _centroid(o); o.step(60)
    assert np.abs(_centroid(o) - c0).max() < 2.5


def test_P14_sign_a_cell_drifts_along_its_persistence_vector(oracle_mod):
    """Eq 5: with mu = 1 the persistence vector never turns (Eq 6 keeps p^_{t-1}); a cell whose p^ is (0, +1) moves in +y."""
    disp = []
    for seed in range(4):
        o = _single_cell_2d(oracle_mod, 200 + seed, lambda_pers=[0, 40], mu_pers=[0.0, 1.0], dt_pers=5)
        o.set_persistence(np.array([[0, 0, 0], [0, 1.0, 0]]))
        c0 = _centroid(o); o.step(60); disp.append(_centroid(o) - c0)
        np.testing.assert_allclose(o.get_persistence()[1], [0, 1.0, 0], atol=1e-15)
    m = np.mean(disp, axis=0)
    assert m[1] > 4.0 and abs(m[0]) < 2.5, m


# ------------------------------------------------------------------------------------ P15 --
@pytest.mark.parametrize("dims,dt,sub", [((32, 32), 3, 8), ((16, 16, 16), 2, 4)])
def test_P15_persistence_recurrence_equals_numpy_restatement(oracle_mod, dims, dt, sub):
    """Eq 6-7 restated in numpy on the centroids the oracle reports after every MCS (Eq 10: sums / volume):
    p = (1 - mu) (X_t - X_{t-dt}) / |.| + mu p^_{t-1}, p^ = p / |p|, X_{t-dt} = X_0 while t < dt, first term dropped
    for a cell that has not moved.  Also: the tallies still equal a recount with the vector terms on (P2)."""
    import cpm_inputs as ci
    nd = len(dims)
    rng = np.random.default_rng(3)
    ids, n = ci.jittered_cubes(dims, pitch=8, edge=5, keep=0.9, rng=rng)
    ct = (1 + (rng.random(n + 1) < 0.5)).astype(np.uint8); ct[0] = 0
    mu = np.array([0.0, 0.95, 0.4])
    o = oracle_mod.Oracle(dims, J=np.array([[0, 4, 4], [4, 9, 12], [4, 12, 9]], dtype=np.int32), lambda_V=[0, 5, 5],
                          target_V=[0, 125, 125], lambda_P=[0, 0, 0], target_P=[0, 0, 0], T=20.0, seed=9, subsection=sub,
                          max_cells=n, lambda_pers=[0, 40, 25], mu_pers=mu, dt_pers=dt)
    o.set_lattice(ids, None, ct)

    def cents():
        st = o.get_cell_stats()
        v = st["volume"].astype(np.float64); v[0] = 1
        return np.stack([st["sum_x"] / v, st["sum_y"] / v, st["sum_z"] / v], axis=1)
    hist = [cents()]
    p_prev = np.zeros((n + 1, 3))
    np.testing.assert_array_equal(o.get_persistence(), p_prev)
    turned = 0
    for t in range(1, 9):
        o.step(1)
        hist.append(cents())
        d = hist[t] - hist[max(t - dt, 0)]
        dn = np.linalg.norm(d, axis=1, keepdims=True)
        m = mu[ct][:, None]
        p = np.where(dn > 0, (1 - m) * d / np.where(dn > 0, dn, 1), 0.0) + m * p_prev
        pn = np.linalg.norm(p, axis=1, keepdims=True)
        want = np.where(pn > 0, p / np.where(pn > 0, pn, 1), 0.0)
        want[0] = 0
        got = o.get_persistence()
        np.testing.assert_allclose(got, want, rtol=0, atol=1e-12, err_msg="MCS %d" % t)
        nrm = np.linalg.norm(got[1:], axis=1)
        assert (np.abs(nrm - 1) < 1e-12).sum() + (nrm == 0).sum() == n
        turned += int((np.abs(got - p_prev).max(axis=1) > 1e-6).sum())
        p_prev = got
    assert turned > n          # directions did change over the run
    rc = H.recount(o.get_lattice(), n, nd)
    st = o.get_cell_stats()
    for k, want in zip(("volume", "perimeter", "sum_x", "sum_y", "sum_z"), rc):
        np.testing.assert_array_equal(st[k][1:].astype(np.int64), want[1:], err_msg=k)


def test_vector_term_parameters_are_validated(oracle_mod):
    J = np.array([[0, 1], [1, 2]], dtype=np.int32)
    with pytest.raises(oracle_mod.OracleError):      # persistence needs a look-back
        oracle_mod.Oracle((8, 8), J=J, subsection=4, max_cells=1, lambda_pers=[0, 5], mu_pers=[0, 0.5], dt_pers=0)
    with pytest.raises(oracle_mod.OracleError):      # mu in [0, 1]
        oracle_mod.Oracle((8, 8), J=J, subsection=4, max_cells=1, lambda_pers=[0, 5], mu_pers=[0, 1.5], dt_pers=2)
    o = oracle_mod.Oracle((8, 8), J=J, subsection=4, max_cells=1, lambda_chem=[0, 5])
    with pytest.raises(oracle_mod.OracleError):      # components in [-1, 1]
        o.set_chemotaxis_field(np.full((8, 8, 2), 1.5, dtype=np.float32))


# ------------------------------------------------------------------------------------ P16 --
def _circular_centroids(lat, n_cells, dims, periodic):
    """Centroid of every cell straight from the lattice with the periodic axes unwrapped around one of the cell's own
    sites (valid for cells smaller than half the lattice): returns (centroid mod dim, volume)."""
    nd = len(dims)
    lat3 = lat if lat.ndim == 3 else lat[None]
    out = np.full((n_cells + 1, 3), np.nan)
    vol = np.zeros(n_cells + 1, dtype=np.int64)
    dimv = [dims[0], dims[1], dims[2] if nd == 3 else 1]
    for cell in range(1, n_cells + 1):
        z, y, x = np.nonzero(lat3 == cell)
        vol[cell] = len(x)
        if len(x) == 0:
            continue
        for a, v in enumerate((x, y, z)):
            v = v.astype(np.float64)
            if periodic[a]:
                r = v[0]
                v = r + ((v - r + dimv[a] / 2.0) % dimv[a]) - dimv[a] / 2.0
                out[cell, a] = v.mean() % dimv[a]
            else:
                out[cell, a] = v.mean()
    return out, vol


def _check_tracked_centroids(o, n_cells, dims, periodic, tag):
    st = o.get_cell_stats()
    v = st["volume"].astype(np.float64); v[v == 0] = np.inf     # Eq 10: sums / volume
    np.testing.assert_array_equal(o.get_centroids(), np.stack([st[k].astype(np.int64) / v for k in ("sum_x", "sum_y", "sum_z")], axis=1))
    want, vol = _circular_centroids(o.get_lattice(), n_cells, dims, periodic)
    np.testing.assert_array_equal(st["volume"][1:], vol[1:])
    dimv = [dims[0], dims[1], dims[2] if len(dims) == 3 else 1]
    for a, k in enumerate(("sum_x", "sum_y", "sum_z")):
        got = st[k][1:].astype(np.int64).astype(np.float64) / np.maximum(vol[1:], 1)
        live = vol[1:] > 0
        if periodic[a]:
            assert ((got[live] >= 0) & (got[live] < dimv[a])).all(), (tag, k, got[live].min(), got[live].max())
            diff = (got[live] - want[1:, a][live] + dimv[a] / 2.0) % dimv[a] - dimv[a] / 2.0
        else:
            diff = got[live] - want[1:, a][live]
        assert np.abs(diff).max() < 1e-9, (tag, k, np.abs(diff).max())


@pytest.mark.parametrize("dims,periodic,sub", [((32, 24), (1, 1, 0), 4), ((16, 16, 16), (1, 0, 1), 4)])
def test_P16_periodic_centroids_follow_cells_through_the_border(oracle_mod, dims, periodic, sub):
    """L297 / reading S23: with unwrap_centroids the tracked sums give, after every MCS, the centroid of the cell as a
    connected object on the torus (computed here from the lattice by unwrapping around one of the cell's own sites),
    kept inside [0, dim); cells are seeded ACROSS the periodic borders."""
    nd = len(dims)
    shape = tuple(reversed(dims))
    ids = np.zeros(shape, dtype=np.uint32)
    n = 0
    if nd == 2:
        for j in range(0, dims[1], 8):
            for i in range(0, dims[0], 8):
                n += 1
                yy = (np.arange(j - 2, j + 3) % dims[1])[:, None]; xx = (np.arange(i - 2, i + 3) % dims[0])[None, :]
                ids[yy, xx] = n                      # 5x5 squares centred on the corners of an 8-pitch grid: (0,0) wraps
    else:
        for k in range(0, dims[2], 8):
            for j in range(0, dims[1], 8):
                for i in range(0, dims[0], 8):
                    n += 1
                    zz = (np.arange(k - 2, k + 2) % dims[2])[:, None, None]
                    yy = np.clip(np.arange(j + 1, j + 5), 0, dims[1] - 1)[None, :, None]
                    xx = (np.arange(i - 2, i + 2) % dims[0])[None, None, :]
                    ids[zz, yy, xx] = n
    ct = np.ones(n + 1, dtype=np.uint8); ct[0] = 0
    kw = dict(J=np.array([[0, 6], [6, 12]], dtype=np.int32), lambda_V=[0, 5], target_V=[0, 30 if nd == 2 else 70],
              T=20.0, seed=4, subsection=sub, max_cells=n, periodic=periodic, unwrap_centroids=1)
    o = oracle_mod.Oracle(dims, **kw)
    o.set_lattice(ids, None, ct)
    _check_tracked_centroids(o, n, dims, periodic, "initial")
    for t in range(8):
        o.step(1)
        _check_tracked_centroids(o, n, dims, periodic, "MCS %d" % (t + 1))
    # without the option the sums are the plain coordinate sums (P2)
    kw["unwrap_centroids"] = 0
    o2 = oracle_mod.Oracle(dims, **kw)
    o2.set_lattice(ids, None, ct); o2.step(3)
    rc = H.recount(o2.get_lattice(), n, nd, periodic)
    st = o2.get_cell_stats()
    for k, want in zip(("volume", "perimeter", "sum_x", "sum_y", "sum_z"), rc):
        np.testing.assert_array_equal(st[k][1:].astype(np.int64), want[1:], err_msg=k)


@pytest.mark.parametrize("sgn", [1, -1])
def test_P16_a_cell_driven_across_the_border_keeps_a_continuous_track(oracle_mod, sgn):
    """A lone cell pushed in +x by a uniform field on a periodic 32-wide lattice crosses the border: the tracked centroid
    stays the torus centroid, moves by small steps (shortest image) and re-enters on the other side; the
    persistence direction (Eq 6, shortest displacement through the border) ends up pointing along +x."""
    dims, periodic = (32, 32), (1, 1, 0)
    ids = np.zeros((32, 32), dtype=np.uint32)
    if sgn > 0:
        ids[12:20, 22:30] = 1
    else:
        ids[12:20, 2:10] = 1
    o = oracle_mod.Oracle(dims, J=np.array([[0, 10], [10, 20]], dtype=np.int32), lambda_V=[0, 20], target_V=[0, 64],
                          lambda_P=[0, 1], target_P=[0, 90], T=10.0, seed=3, subsection=8, max_cells=1, periodic=periodic,
                          lambda_chem=[0, 60], lambda_pers=[0, 1], mu_pers=[0, 0.5], dt_pers=4, unwrap_centroids=1)
    o.set_lattice(ids, None, np.array([0, 1], dtype=np.uint8))
    f = np.zeros((32, 32, 2), dtype=np.float32); f[..., 0] = float(sgn)
    o.set_chemotaxis_field(f)
    prev = None; travelled = 0.0; wraps = 0

    def cent():
        st = o.get_cell_stats()
        v = float(st["volume"][1])
        return np.array([st["sum_x"][1] / v, st["sum_y"][1] / v, 0.0])
    hist = [cent()]; p_prev = np.zeros(3); mu, dt = 0.5, 4
    for t in range(150):
        o.step(1)
        _check_tracked_centroids(o, 1, dims, periodic, "MCS %d" % (t + 1))
        # Eq 6-7 restated with the shortest displacement through the periodic border
        hist.append(cent())
        d = hist[-1] - hist[max(len(hist) - 1 - dt, 0)]
        d[:2] = (d[:2] + 16.0) % 32.0 - 16.0
        dn = np.linalg.norm(d)
        pv = ((1 - mu) * d / dn if dn > 0 else 0.0) + mu * p_prev
        pn = np.linalg.norm(pv)
        p_prev = pv / pn if pn > 0 else np.zeros(3)
        np.testing.assert_allclose(o.get_persistence()[1], p_prev, rtol=0, atol=1e-12, err_msg="MCS %d" % (t + 1))
        p_prev = o.get_persistence()[1]
        st = o.get_cell_stats()
        c = float(st["sum_x"][1]) / float(st["volume"][1])
        if prev is not None:
            step = (c - prev + 16.0) % 32.0 - 16.0
            assert abs(step) < 3.0, (t, prev, c)
            travelled += step
            wraps += int(sgn * (prev - c) > 16.0)
        prev = c
    assert sgn * travelled > 14.0 and wraps >= 1, (travelled, wraps)
    assert sgn * o.get_persistence()[1][0] > 0.7
