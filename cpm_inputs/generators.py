"""Seeded generators for the synthetic workloads C1..C5.

Arrays are numpy, C order, shape dims[::-1] (z, y, x) / (y, x); x is the fastest axis.
No Hamiltonian, no acceptance rule, no schedule lives here: only initial conditions and
parameter tables.
"""
import numpy as np

try:  # scipy is in the image; only the obstacle network needs it
    from scipy.spatial import cKDTree
except Exception:  # pragma: no cover
    cKDTree = None


def config_names():
    return ["C1", "C2", "C3", "C4", "C5", "C6", "C7"]


# --------------------------------------------------------------------------- geometry ----
def ball_moore_perimeter(volume, ndim):
    """(n_sites, Moore-interface count) of the digitised disc/ball whose site count is closest
    to `volume`.  Used to set P* "to the sphere surface of V* in neighbour-face units"
    (BASELINE.json C2); SURVEY.md 4 checked the unit against the paper's Tables 1-2."""
    r0 = (volume / np.pi) ** 0.5 if ndim == 2 else (3.0 * volume / (4.0 * np.pi)) ** (1.0 / 3.0)
    best = None
    for r in np.linspace(max(r0 - 1.0, 0.5), r0 + 1.0, 81):
        R = int(np.ceil(r)) + 2
        ax = np.arange(-R, R + 1)
        if ndim == 2:
            yy, xx = np.meshgrid(ax, ax, indexing="ij")
            m = (xx * xx + yy * yy) <= r * r
        else:
            zz, yy, xx = np.meshgrid(ax, ax, ax, indexing="ij")
            m = (xx * xx + yy * yy + zz * zz) <= r * r
        n = int(m.sum())
        if best is None or abs(n - volume) < abs(best[0] - volume):
            best = (n, m)
    n, m = best
    per = 0
    rng3 = (-1, 0, 1)
    if ndim == 2:
        for dy in rng3:
            for dx in rng3:
                if dx == 0 and dy == 0:
                    continue
                sh = np.roll(np.roll(m, dy, 0), dx, 1)
                per += int((m & ~sh).sum())
    else:
        for dz in rng3:
            for dy in rng3:
                for dx in rng3:
                    if dx == 0 and dy == 0 and dz == 0:
                        continue
                    sh = np.roll(np.roll(np.roll(m, dz, 0), dy, 1), dx, 2)
                    per += int((m & ~sh).sum())
    return n, per


def jittered_cubes(dims, pitch, edge, keep, rng, jitter=None, free=None):
    """Paint edge^d cubes, one per kept slot of a pitch grid, each displaced by a random jitter
    in [0, jitter] per axis (default pitch-edge-1, so neighbouring seeds keep a gap >= 1).
    A jittered grid is the usual cheap stand-in for Poisson-disc positions.
    Returns (ids[z,y,x] uint32, n_cells); ids run 1..n_cells in slot order.
    `free` (bool array or None): voxels where cells may be painted."""
    nd = len(dims)
    if jitter is None:
        jitter = max(pitch - edge - 1, 0)
    slots = [d // pitch for d in dims]            # x, y(, z)
    shape_s = tuple(reversed(slots))              # (nk, nj, ni)
    kept = rng.random(shape_s) < keep
    cell_of_slot = np.zeros(shape_s, dtype=np.uint32)
    n_cells = int(kept.sum())
    cell_of_slot[kept] = np.arange(1, n_cells + 1, dtype=np.uint32)
    jit = [rng.integers(0, jitter + 1, size=shape_s, dtype=np.int16) for _ in range(nd)]  # x, y(, z)

    X, Y = dims[0], dims[1]
    ids = np.zeros(tuple(reversed(dims)), dtype=np.uint32)

    def expand2(a2):  # (nj, ni) -> (Y, X), zero outside the slot grid
        out = np.zeros((Y, X), dtype=a2.dtype)
        e = np.repeat(np.repeat(a2, pitch, axis=0), pitch, axis=1)
        out[: e.shape[0], : e.shape[1]] = e
        return out

    lx = (np.arange(X) % pitch).astype(np.int16)[None, :]
    ly = (np.arange(Y) % pitch).astype(np.int16)[:, None]
    in_grid = np.zeros((Y, X), dtype=bool)
    in_grid[: slots[1] * pitch, : slots[0] * pitch] = True
    if nd == 2:
        jx, jy = expand2(jit[0]), expand2(jit[1])
        inside = in_grid & (lx >= jx) & (lx < jx + edge) & (ly >= jy) & (ly < jy + edge)
        ids[:] = np.where(inside, expand2(cell_of_slot), 0)
    else:
        lz = np.arange(pitch, dtype=np.int16)[:, None, None]
        for k in range(slots[2]):
            jx, jy, jz = expand2(jit[0][k]), expand2(jit[1][k]), expand2(jit[2][k])
            inside_xy = in_grid & (lx >= jx) & (lx < jx + edge) & (ly >= jy) & (ly < jy + edge)
            cid = np.where(inside_xy, expand2(cell_of_slot[k]), 0).astype(np.uint32)
            inz = (lz >= jz[None]) & (lz < jz[None] + edge)
            ids[k * pitch:(k + 1) * pitch] = np.where(inz, cid[None], 0)
    if free is not None:
        ids[~free] = 0
    return ids, n_cells


def _paint_capsule(mask, p0, p1, r):
    """OR a capsule (all voxels within r of segment p0-p1) into the periodic bool box `mask`."""
    P = mask.shape[0]
    lo = np.floor(np.minimum(p0, p1) - r).astype(int)
    hi = np.ceil(np.maximum(p0, p1) + r).astype(int)
    xs = np.arange(lo[0], hi[0] + 1); ys = np.arange(lo[1], hi[1] + 1); zs = np.arange(lo[2], hi[2] + 1)
    zz, yy, xx = np.meshgrid(zs, ys, xs, indexing="ij")
    d = p1 - p0
    L2 = float(d @ d)
    px, py, pz = xx - p0[0], yy - p0[1], zz - p0[2]
    t = (px * d[0] + py * d[1] + pz * d[2]) / L2 if L2 > 0 else np.zeros_like(px, dtype=float)
    t = np.clip(t, 0.0, 1.0)
    dist2 = (px - t * d[0]) ** 2 + (py - t * d[1]) ** 2 + (pz - t * d[2]) ** 2
    inside = dist2 <= r * r
    ix = np.ix_(zs % P, ys % P, xs % P)
    mask[ix] |= inside


def obstacle_network(period, frac, rng, rmin=3, rmax=6, max_iter=6):
    """Synthetic sinusoid/reticular-like obstacle network on a periodic period^3 box: nodes on a
    jittered grid, each candidate edge joins a node to one of its nearest neighbours, the
    shortest 1.5*n candidates are kept (mean node degree 3), each edge becomes a capsule of
    radius U{rmin..rmax}.  Node spacing is adjusted until about `frac` of the voxels are covered.
    Stands in for the imaged liver-sinusoid / FRC networks, which are not
    available.  Returns bool[period, period, period]."""
    assert cKDTree is not None, "scipy needed for the obstacle network"
    rbar2 = np.mean([r * r for r in range(rmin, rmax + 1)])
    L = (1.5 * np.pi * rbar2 / frac) ** 0.5   # tube volume 1.5 n L pi r^2 = frac * n L^3
    mask = None
    for _ in range(max_iter):
        g = max(int(round(period / L)), 2)
        pitch = period / g
        base = np.stack(np.meshgrid(np.arange(g), np.arange(g), np.arange(g), indexing="ij"), -1).reshape(-1, 3)
        sub = np.random.default_rng(int(rng.integers(1 << 31)))
        nodes = (base + sub.random(base.shape) * 0.8) * pitch
        nodes %= period
        n = len(nodes)
        tree = cKDTree(nodes, boxsize=period)
        dist, idx = tree.query(nodes, k=min(7, n))
        pairs = {}
        for i in range(n):
            for j, dd in zip(idx[i, 1:], dist[i, 1:]):
                a, b = (i, int(j)) if i < j else (int(j), i)
                if a != b:
                    pairs[(a, b)] = dd
        cand = sorted(pairs.items(), key=lambda kv: kv[1])[: int(1.5 * n)]
        mask = np.zeros((period, period, period), dtype=bool)
        for (a, b), _dd in cand:
            p0 = nodes[a]
            dvec = nodes[b] - p0
            dvec -= period * np.round(dvec / period)      # minimum image
            _paint_capsule(mask, p0, p0 + dvec, float(sub.integers(rmin, rmax + 1)))
        got = mask.mean()
        if abs(got - frac) < 0.01:
            break
        L *= (got / frac) ** 0.5
    return mask


# --------------------------------------------------------------------------- configs ----
def _sym_J(n_types, rng, lo=5, hi=30):
    J = np.zeros((n_types, n_types), dtype=np.int32)
    for i in range(n_types):
        for j in range(i, n_types):
            J[i, j] = J[j, i] = int(rng.integers(lo, hi + 1))
    J[0, 0] = 0  # medium-medium never contributes (same id)
    return J


def _zeros(n):
    return np.zeros(n, dtype=np.int32)


def make_config(name, dims=None, seed=None, subsection=None):
    """Build one of C1..C5.  `dims` overrides the lattice size (scaled copies for parity tests);
    everything else (seed pitch, parameters) keeps the recipe.  Returns a dict with
    dims, ids, frozen (or None), cell_type, max_cells, params (kwargs for the context), n_mcs."""
    name = name.upper()
    if name == "C1":
        dims = tuple(dims or (128, 128))
        rng_seed = 1 if seed is None else seed
        X, Y = dims
        ids = np.zeros((Y, X), dtype=np.uint32)
        n = 0
        for j in range(Y // 16):
            for i in range(X // 16):
                n += 1
                ids[16 * j + 4:16 * j + 12, 16 * i + 4:16 * i + 12] = 1 + i + (X // 16) * j
        cell_type = np.ones(n + 1, dtype=np.uint8); cell_type[0] = 0
        J = np.array([[0, 10], [10, 20]], dtype=np.int32)
        params = dict(J=J, lambda_V=[0, 50], target_V=[0, 64], lambda_P=[0, 0], target_P=[0, 0],
                      lambda_act=None, max_act=None, T=20.0, seed=rng_seed,
                      subsection=subsection if subsection else 16)
        return dict(name="C1", dims=dims, ids=ids, frozen=None, cell_type=cell_type, max_cells=n,
                    params=params, n_mcs=100)

    if name in ("C2", "C3"):
        dims = tuple(dims or (256, 256, 256))
        rng = np.random.default_rng(20231209 + (2 if name == "C2" else 3) if seed is None else seed)
        if name == "C2":
            ids, n = jittered_cubes(dims, pitch=8, edge=6, keep=0.92, rng=rng)
            vt = 500
        else:
            ids, n = jittered_cubes(dims, pitch=20, edge=10, keep=0.95, rng=rng)
            vt = 1800
        cell_type = (1 + (rng.random(n + 1) < 0.5)).astype(np.uint8); cell_type[0] = 0
        J = _sym_J(3, rng)
        _, pt = ball_moore_perimeter(vt, 3)
        params = dict(J=J, lambda_V=[0, 25, 25], target_V=[0, vt, vt], lambda_P=[0, 2, 2], target_P=[0, pt, pt],
                      lambda_act=None, max_act=None, T=20.0, seed=int(rng.integers(1 << 62)),
                      subsection=subsection if subsection else 8)
        if name == "C3":
            params["lambda_act"] = [0, 200, 200]
            params["max_act"] = [0, 40, 40]
        return dict(name=name, dims=dims, ids=ids, frozen=None, cell_type=cell_type, max_cells=n,
                    params=params, n_mcs=200 if name == "C2" else 500)

    if name == "C4":
        dims = tuple(dims or (1024, 1024, 1024))
        rng = np.random.default_rng(20231209 + 4 if seed is None else seed)
        period = min(min(dims), 256)
        net = obstacle_network(period, 0.20, rng)
        reps = tuple(-(-d // period) for d in reversed(dims))
        frozen = np.tile(net, reps)[: dims[2], : dims[1], : dims[0]]
        frozen = np.ascontiguousarray(frozen)
        ids, n = jittered_cubes(dims, pitch=10, edge=7, keep=0.98, rng=rng, free=~frozen)
        stroma = n + 1
        ids[frozen] = stroma
        cell_type = np.ones(stroma + 1, dtype=np.uint8)
        cell_type[1:n + 1][rng.random(n) < 0.10] = 2      # motile type
        cell_type[0] = 0
        cell_type[stroma] = 3
        J = _sym_J(4, rng)
        _, pt = ball_moore_perimeter(500, 3)
        params = dict(J=J, lambda_V=[0, 25, 25, 0], target_V=[0, 500, 500, 0], lambda_P=[0, 2, 2, 0],
                      target_P=[0, pt, pt, 0], lambda_act=[0, 0, 200, 0], max_act=[0, 0, 40, 0], T=20.0,
                      seed=int(rng.integers(1 << 62)), subsection=subsection if subsection else 8)
        return dict(name="C4", dims=dims, ids=ids, frozen=frozen.astype(np.uint8), cell_type=cell_type,
                    max_cells=stroma, params=params, n_mcs=100)

    if name == "C5":
        dims = tuple(dims or (16384, 16384))
        rng = np.random.default_rng(20231209 + 5 if seed is None else seed)
        ids, n = jittered_cubes(dims, pitch=10, edge=8, keep=0.97, rng=rng)
        cell_type = (1 + (rng.random(n + 1) < 0.5)).astype(np.uint8); cell_type[0] = 0
        J = _sym_J(3, rng)
        _, pt = ball_moore_perimeter(100, 2)
        params = dict(J=J, lambda_V=[0, 25, 25], target_V=[0, 100, 100], lambda_P=[0, 2, 2], target_P=[0, pt, pt],
                      lambda_act=None, max_act=None, T=20.0, seed=int(rng.integers(1 << 62)),
                      subsection=subsection if subsection else 16)
        return dict(name="C5", dims=dims, ids=ids, frozen=None, cell_type=cell_type, max_cells=n,
                    params=params, n_mcs=20)
    if name == "C6":
        # the paper's 3D cell collective with the persistence model (Fig 5C / 6D, Table 2):
        # V* = 150, A* = 1500, J(cell,cell) = 10, J(cell,ECM) = 0, T = 20, mu = 0.95, dt = 15, lambda_pers = 40, density
        # about 0.5.  The paper's lambda_perimeter = 0.2 is not an integer: the whole Hamiltonian and T are scaled by 5
        # (same Boltzmann factors): lambda_P = 1, lambda_V = 125, J = 50, lambda_pers = 200, T = 100.
        dims = tuple(dims or (256, 256, 256))
        rng = np.random.default_rng(20231209 + 6 if seed is None else seed)
        ids, n = jittered_cubes(dims, pitch=6, edge=5, keep=0.72, rng=rng)
        cell_type = np.ones(n + 1, dtype=np.uint8); cell_type[0] = 0
        J = np.array([[0, 0], [0, 50]], dtype=np.int32)
        params = dict(J=J, lambda_V=[0, 125], target_V=[0, 150], lambda_P=[0, 1], target_P=[0, 1500],
                      lambda_act=None, max_act=None, T=100.0, seed=int(rng.integers(1 << 62)),
                      subsection=subsection if subsection else 4,
                      lambda_pers=[0, 200], mu_pers=[0.0, 0.95], dt_pers=15)
        return dict(name="C6", dims=dims, ids=ids, frozen=None, cell_type=cell_type, max_cells=n,
                    params=params, n_mcs=100)

    if name == "C7":
        # the paper's 2D circular chemotaxis simulation (Fig 5A / 6E, Table 1): V* = 2500,
        # A* = 600, lambda_P = 2, J(cell,ECM) = 10, T = 10, lambda_V = 20, lambda_chem = 10; the field is tangential
        # to circles around the lattice centre ("at a 90 degree angle to radial vectors"), unit length.
        dims = tuple(dims or (1024, 1024))
        rng = np.random.default_rng(20231209 + 7 if seed is None else seed)
        ids, n = jittered_cubes(dims, pitch=128, edge=48, keep=0.9, rng=rng)
        cell_type = np.ones(n + 1, dtype=np.uint8); cell_type[0] = 0
        J = np.array([[0, 10], [10, 20]], dtype=np.int32)
        params = dict(J=J, lambda_V=[0, 20], target_V=[0, 2500], lambda_P=[0, 2], target_P=[0, 600],
                      lambda_act=None, max_act=None, T=10.0, seed=int(rng.integers(1 << 62)),
                      subsection=subsection if subsection else 8, lambda_chem=[0, 10])
        return dict(name="C7", dims=dims, ids=ids, frozen=None, cell_type=cell_type, max_cells=n,
                    params=params, n_mcs=100, field=circular_field(dims))
    raise ValueError("unknown config " + name)


def circular_field(dims):
    """Unit vectors at 90 degrees to the radial direction from the lattice centre, float32,
    shape dims[::-1] + (ndim,); the z component (3D) is 0.  The centre voxel itself gets (0, ..)."""
    nd = len(dims)
    X, Y = dims[0], dims[1]
    y, x = np.meshgrid(np.arange(Y, dtype=np.float64) - (Y - 1) / 2.0, np.arange(X, dtype=np.float64) - (X - 1) / 2.0, indexing="ij")
    r = np.sqrt(x * x + y * y)
    r[r == 0] = np.inf
    f2 = np.stack([-y / r, x / r], axis=-1).astype(np.float32)
    if nd == 2:
        return np.ascontiguousarray(f2)
    out = np.zeros((dims[2], Y, X, 3), dtype=np.float32)
    out[..., :2] = f2[None]
    return out


def crop_config(cfg, dims):
    """Corner crop of a config (same ids, same tables): the bounded sample the CPU baseline runs."""
    out = dict(cfg)
    sl = tuple(slice(0, d) for d in reversed(dims))
    out["dims"] = tuple(dims)
    out["ids"] = np.ascontiguousarray(cfg["ids"][sl])
    out["frozen"] = None if cfg["frozen"] is None else np.ascontiguousarray(cfg["frozen"][sl])
    if cfg.get("field") is not None:
        out["field"] = np.ascontiguousarray(cfg["field"][sl])
    return out
