"""Independent numpy/python restatements used to PIN the oracle (not shared with it, nor with
the CUDA path): brute-force Hamiltonian from Eq 1 + Eq 3, recount of the per-cell tallies from
the lattice, a pure-python Philox4x32-10 (itself pinned by tests/golden/philox4x32_10_kat.txt).
"""
import itertools

import numpy as np


def moore_offsets(ndim):
    """(dx,dy,dz) in the enumeration order of DESIGN.md reading S16: (dz,dy,dx) lexicographic,
    dx fastest, centre skipped."""
    out = []
    if ndim == 2:
        for dy, dx in itertools.product((-1, 0, 1), repeat=2):
            if (dx, dy) != (0, 0):
                out.append((dx, dy, 0))
    else:
        for dz, dy, dx in itertools.product((-1, 0, 1), repeat=3):
            if (dx, dy, dz) != (0, 0, 0):
                out.append((dx, dy, dz))
    return out


def _lattice3(ids):
    a = np.asarray(ids)
    return a[None] if a.ndim == 2 else a


def neighbour_id(ids3, x, y, z, periodic):
    """id at (x,y,z) with the boundary rule: periodic axes wrap, closed axes read medium (0)."""
    Z, Y, X = ids3.shape
    c = [x, y, z]
    for a, n in enumerate((X, Y, Z)):
        if c[a] < 0 or c[a] >= n:
            if not periodic[a]:
                return 0
            c[a] %= n
    return int(ids3[c[2], c[1], c[0]])


def brute_force_H(ids, cell_type, J, lamV, tgtV, lamP, tgtP, ndim, periodic=(0, 0, 0)):
    """Eq 1 + Eq 3 (L232) over the whole lattice, nothing incremental:
    every unordered Moore pair once (reading S2) -- pairs of two lattice sites are enumerated
    from both ends and halved, pairs whose other end lies outside a closed lattice (immutable
    medium, reading S5) are seen once from their lattice end -- then the volume and perimeter
    constraints of every non-medium cell (reading S3) from a fresh count of V and of A
    (interfaces with sites not of the same cell, L234)."""
    ids3 = _lattice3(ids)
    Z, Y, X = ids3.shape
    offs = moore_offsets(ndim)
    twice_inside = 0
    outside = 0
    V = {}
    P = {}
    for z in range(Z):
        for y in range(Y):
            for x in range(X):
                me = int(ids3[z, y, x])
                if me:
                    V[me] = V.get(me, 0) + 1
                for dx, dy, dz in offs:
                    c = [x + dx, y + dy, z + dz]
                    is_outside = False
                    for a, n in enumerate((X, Y, Z)):
                        if c[a] < 0 or c[a] >= n:
                            if periodic[a]:
                                c[a] %= n
                            else:
                                is_outside = True
                    other = 0 if is_outside else int(ids3[c[2], c[1], c[0]])
                    if other == me:
                        continue
                    if me:
                        P[me] = P.get(me, 0) + 1
                    e = int(J[cell_type[me]][cell_type[other]])
                    if is_outside:
                        outside += e
                    else:
                        twice_inside += e
    assert twice_inside % 2 == 0
    H = twice_inside // 2 + outside
    for cell, v in V.items():
        t = cell_type[cell]
        H += int(lamV[t]) * (v - int(tgtV[t])) ** 2
        H += int(lamP[t]) * (P.get(cell, 0) - int(tgtP[t])) ** 2
    return H


def recount(ids, max_cells, ndim, periodic=(0, 0, 0)):
    """V, P, sum_x, sum_y, sum_z per cell straight from the lattice (vectorised shifts).
    Medium (id 0) is left at 0 (reading S3)."""
    ids3 = _lattice3(np.asarray(ids, dtype=np.int64))
    Z, Y, X = ids3.shape
    n = max_cells + 1
    V = np.bincount(ids3.ravel(), minlength=n).astype(np.int64)
    zz, yy, xx = np.meshgrid(np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    sx = np.bincount(ids3.ravel(), weights=xx.ravel(), minlength=n).astype(np.int64)
    sy = np.bincount(ids3.ravel(), weights=yy.ravel(), minlength=n).astype(np.int64)
    sz = np.bincount(ids3.ravel(), weights=zz.ravel(), minlength=n).astype(np.int64)
    pad = np.zeros((Z + 2, Y + 2, X + 2), dtype=np.int64)
    pad[1:-1, 1:-1, 1:-1] = ids3
    if periodic[0]:
        pad[:, :, 0] = pad[:, :, X]; pad[:, :, X + 1] = pad[:, :, 1]
    if periodic[1]:
        pad[:, 0, :] = pad[:, Y, :]; pad[:, Y + 1, :] = pad[:, 1, :]
    if periodic[2] and ndim == 3:
        pad[0] = pad[Z]; pad[Z + 1] = pad[1]
    foreign = np.zeros((Z, Y, X), dtype=np.int64)
    for dx, dy, dz in moore_offsets(ndim):
        sh = pad[1 + dz:1 + dz + Z, 1 + dy:1 + dy + Y, 1 + dx:1 + dx + X]
        foreign += (sh != ids3)
    P = np.bincount(ids3.ravel(), weights=foreign.ravel(), minlength=n).astype(np.int64)
    for a in (V, P, sx, sy, sz):
        a[0] = 0
    return V, P, sx, sy, sz


# ------------------------------------------------------------- pure-python Philox4x32-10 ----
_M0, _M1 = 0xD2511F53, 0xCD9E8D57
_W0, _W1 = 0x9E3779B9, 0xBB67AE85
_MASK = 0xFFFFFFFF


def philox_py(ctr, key):
    c = [int(v) & _MASK for v in ctr]
    k = [int(v) & _MASK for v in key]
    for r in range(10):
        if r:
            k[0] = (k[0] + _W0) & _MASK
            k[1] = (k[1] + _W1) & _MASK
        p0 = _M0 * c[0]
        p1 = _M1 * c[2]
        c = [((p1 >> 32) ^ c[1] ^ k[0]) & _MASK, p1 & _MASK, ((p0 >> 32) ^ c[3] ^ k[1]) & _MASK, p0 & _MASK]
    return c


def read_kat(path):
    rows = []
    with open(path) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            v = [int(t, 16) for t in line.split()]
            rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def build_toolkit_philox(force=False):
    """Builds tests/cuda/curand_philox_check.cu (the CUDA toolkit's own Philox4x32-10, pin P8(i)) for sm_100a and
    returns the loaded library.  nvcc cross-compiles without a GPU; calling it needs one."""
    import ctypes
    import os
    import subprocess
    here = os.path.dirname(os.path.abspath(__file__))
    src = os.path.join(here, "cuda", "curand_philox_check.cu")
    lib = os.path.join(here, "cuda", "libcurand_philox_check.so")
    if force or not os.path.exists(lib) or os.path.getmtime(lib) < os.path.getmtime(src):
        tmp = lib + ".%d.tmp" % os.getpid()
        subprocess.check_call([os.environ.get("NVCC", "nvcc"), "-gencode", "arch=compute_100a,code=sm_100a", "-O2",
                               "-shared", "-Xcompiler", "-fPIC", "-o", tmp, src])
        os.replace(tmp, lib)
    L = ctypes.CDLL(lib)
    L.toolkit_philox4x32_10.restype = ctypes.c_int
    L.toolkit_philox4x32_10.argtypes = [ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_uint64]
    return L


def toolkit_philox(ctr, key, device=0):
    """curand_Philox4x32_10 on n (ctr[4], key[2]) pairs -> uint32[n, 4]."""
    L = build_toolkit_philox()
    c = np.ascontiguousarray(np.asarray(ctr, dtype=np.uint32)).reshape(-1, 4)
    k = np.ascontiguousarray(np.asarray(key, dtype=np.uint32)).reshape(-1, 2)
    out = np.zeros((len(c), 4), np.uint32)
    rc = L.toolkit_philox4x32_10(device, c.ctypes.data, k.ctypes.data, out.ctypes.data, len(c))
    assert rc == 0, rc
    return out
