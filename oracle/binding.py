"""ctypes binding of the CPU oracle (oracle/cpm_oracle.cpp).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference leg.  Never imported by the product package.
Builds liboracle_cpm.so with g++ on first use (a few seconds).
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cpm_oracle.cpp")
_HDR = os.path.join(_HERE, "cpm_oracle.h")
_LIB = os.path.join(_HERE, "liboracle_cpm.so")

MODE_DETERMINISTIC, MODE_LIVE = 0, 1


def build(force=False):
    """Compile the oracle shared library if it is missing or older than its sources."""
    stale = (not os.path.exists(_LIB)) or any(
        os.path.getmtime(s) > os.path.getmtime(_LIB) for s in (_SRC, _HDR))
    if force or stale:
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wall", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


class _Params(C.Structure):
    _fields_ = [
        ("ndim", C.c_int32), ("dims", C.c_int32 * 3), ("neighbourhood", C.c_int32),
        ("periodic", C.c_int32 * 3), ("n_types", C.c_int32),
        ("J", C.POINTER(C.c_int32)),
        ("lambda_V", C.POINTER(C.c_int32)), ("target_V", C.POINTER(C.c_int32)),
        ("lambda_P", C.POINTER(C.c_int32)), ("target_P", C.POINTER(C.c_int32)),
        ("lambda_act", C.POINTER(C.c_int32)), ("max_act", C.POINTER(C.c_int32)),
        ("T", C.c_double), ("seed", C.c_uint64),
        ("subsection", C.c_int32), ("attempts_per_activation", C.c_int32),
        ("mode", C.c_int32), ("max_cells", C.c_uint32),
        ("device", C.c_int32), ("stream", C.c_void_p),
        ("lambda_pers", C.POINTER(C.c_int32)), ("mu_pers", C.POINTER(C.c_double)), ("dt_pers", C.c_int32),
        ("lambda_chem", C.POINTER(C.c_int32)), ("unwrap_centroids", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp = C.c_void_p
        L.oracle_create.argtypes = [C.POINTER(_Params), C.POINTER(vp)]
        L.oracle_destroy.argtypes = [vp]
        L.oracle_set_lattice.argtypes = [vp, vp, vp, vp]
        L.oracle_set_act.argtypes = [vp, vp]
        L.oracle_set_mcs.argtypes = [vp, C.c_uint32]
        L.oracle_step.argtypes = [vp, C.c_uint32]
        L.oracle_get_lattice.argtypes = [vp, vp]
        L.oracle_get_act.argtypes = [vp, vp]
        L.oracle_get_cell_stats.argtypes = [vp, vp, vp, vp, vp, vp]
        L.oracle_get_counters.argtypes = [vp, vp]
        L.oracle_get_schedule.argtypes = [vp, vp, vp, vp]
        L.oracle_last_error.argtypes = [vp]
        L.oracle_last_error.restype = C.c_char_p
        L.oracle_set_visit_order.argtypes = [vp, C.c_int32, C.c_uint64]
        L.oracle_probe.argtypes = [vp, C.c_uint64, C.c_int32, vp, vp, vp]
        L.oracle_force_copy.argtypes = [vp, C.c_uint64, C.c_int32]
        L.oracle_set_trace.argtypes = [vp, vp, C.c_uint64, vp]
        L.oracle_philox4x32_10.argtypes = [vp, vp, vp]
        L.oracle_philox4x32_10.restype = None
        L.oracle_decode_proposal.argtypes = [C.c_uint32, C.c_uint32, C.c_uint32, vp, vp]
        L.oracle_decode_proposal.restype = None
        L.oracle_threshold_table.argtypes = [C.c_double, vp, C.c_uint64]
        L.oracle_threshold_table.restype = C.c_int64
        L.oracle_gm_q16.argtypes = [vp, C.c_int32]
        L.oracle_gm_q16.restype = C.c_int64
        L.oracle_neighbour_offsets.argtypes = [C.c_int32, vp]
        L.oracle_set_chemotaxis_field.argtypes = [vp, vp]
        L.oracle_set_persistence.argtypes = [vp, vp]
        L.oracle_get_persistence.argtypes = [vp, vp]
        L.oracle_probe_dir.argtypes = [vp, C.c_uint64, C.c_int32, vp]
        L.oracle_get_centroids.argtypes = [vp, vp]
        L.oracle_direction_table.argtypes = [C.c_int32, vp]
        L.oracle_get_interface_counts.argtypes = [vp, vp]
        L.oracle_update_statistics.argtypes = [vp, C.c_uint32, vp, C.c_int32, vp, C.c_int32, C.c_uint32]
        _lib = L
    return _lib


class OracleError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__("oracle error %d %s" % (code, msg))
        self.code = code


def _i32(a, n):
    if a is None:
        return None, None
    arr = np.ascontiguousarray(np.asarray(a, dtype=np.int32))
    assert arr.size == n, (arr.size, n)
    return arr, arr.ctypes.data_as(C.POINTER(C.c_int32))


class Oracle:
    """One oracle context.  Arrays are numpy, C order, shape dims[::-1] (z, y, x)."""

    def __init__(self, dims, J, lambda_V=None, target_V=None, lambda_P=None, target_P=None,
                 lambda_act=None, max_act=None, T=20.0, seed=1, subsection=0,
                 attempts_per_activation=0, mode=MODE_DETERMINISTIC, max_cells=0,
                 periodic=(0, 0, 0), lambda_pers=None, mu_pers=None, dt_pers=0, lambda_chem=None, unwrap_centroids=0):
        L = lib()
        dims = tuple(int(x) for x in dims)
        self.ndim = len(dims)
        self.dims = dims
        self.shape = tuple(reversed(dims))
        self.N = int(np.prod(dims))
        Jm = np.ascontiguousarray(np.asarray(J, dtype=np.int32))
        nT = Jm.shape[0]
        assert Jm.shape == (nT, nT)
        self.n_types = nT
        self.max_cells = int(max_cells)
        p = _Params()
        p.ndim = self.ndim
        for i in range(3):
            p.dims[i] = dims[i] if i < self.ndim else 1
            p.periodic[i] = int(periodic[i]) if i < self.ndim else 0
        p.neighbourhood = 0
        p.n_types = nT
        keep = [Jm]
        p.J = Jm.ctypes.data_as(C.POINTER(C.c_int32))
        for name, val in (("lambda_V", lambda_V), ("target_V", target_V), ("lambda_P", lambda_P),
                          ("target_P", target_P), ("lambda_act", lambda_act), ("max_act", max_act),
                          ("lambda_pers", lambda_pers), ("lambda_chem", lambda_chem)):
            arr, ptr = _i32(val, nT)
            if arr is not None:
                keep.append(arr)
                setattr(p, name, ptr)
        p.T = float(T)
        p.seed = int(seed)
        p.subsection = int(subsection)
        p.attempts_per_activation = int(attempts_per_activation)
        p.mode = int(mode)
        p.max_cells = self.max_cells
        p.device = 0
        p.stream = None
        if mu_pers is not None:
            mu = np.ascontiguousarray(np.asarray(mu_pers, dtype=np.float64))
            assert mu.size == nT
            keep.append(mu)
            p.mu_pers = mu.ctypes.data_as(C.POINTER(C.c_double))
        p.dt_pers = int(dt_pers)
        p.unwrap_centroids = int(unwrap_centroids)
        self.pers_on = lambda_pers is not None and any(int(v) != 0 for v in lambda_pers)
        h = C.c_void_p()
        rc = L.oracle_create(C.byref(p), C.byref(h))
        if rc != 0:
            raise OracleError(rc, "create")
        self._h = h
        self._L = L

    def _chk(self, rc):
        if rc != 0:
            raise OracleError(rc, self._L.oracle_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_lattice(self, ids, frozen=None, cell_type=None):
        ids = np.ascontiguousarray(np.asarray(ids, dtype=np.uint32)).reshape(-1)
        assert ids.size == self.N
        fz = None
        if frozen is not None:
            fz = np.ascontiguousarray(np.asarray(frozen, dtype=np.uint8)).reshape(-1)
            assert fz.size == self.N
        ct = np.ascontiguousarray(np.asarray(cell_type, dtype=np.uint8))
        assert ct.size == self.max_cells + 1
        self._chk(self._L.oracle_set_lattice(self._h, ids.ctypes.data, fz.ctypes.data if fz is not None else None,
                                             ct.ctypes.data))

    def set_act(self, act):
        a = np.ascontiguousarray(np.asarray(act, dtype=np.float32)).reshape(-1)
        assert a.size == self.N
        self._chk(self._L.oracle_set_act(self._h, a.ctypes.data))

    def set_mcs(self, mcs):
        self._chk(self._L.oracle_set_mcs(self._h, int(mcs)))

    def step(self, n=1):
        self._chk(self._L.oracle_step(self._h, int(n)))

    def get_lattice(self):
        out = np.empty(self.N, dtype=np.uint32)
        self._chk(self._L.oracle_get_lattice(self._h, out.ctypes.data))
        return out.reshape(self.shape)

    def get_act(self):
        out = np.empty(self.N, dtype=np.float32)
        self._chk(self._L.oracle_get_act(self._h, out.ctypes.data))
        return out.reshape(self.shape)

    def get_cell_stats(self):
        n = self.max_cells + 1
        V = np.empty(n, np.uint32); P = np.empty(n, np.uint32)
        sx = np.empty(n, np.uint64); sy = np.empty(n, np.uint64); sz = np.empty(n, np.uint64)
        self._chk(self._L.oracle_get_cell_stats(self._h, V.ctypes.data, P.ctypes.data, sx.ctypes.data,
                                                sy.ctypes.data, sz.ctypes.data))
        return {"volume": V, "perimeter": P, "sum_x": sx, "sum_y": sy, "sum_z": sz}

    def get_counters(self):
        out = np.zeros(4, np.uint64)
        self._chk(self._L.oracle_get_counters(self._h, out.ctypes.data))
        return {"attempts": int(out[0]), "evaluated": int(out[1]), "accepted": int(out[2]), "mcs": int(out[3])}

    def get_schedule(self):
        S = C.c_int32(); k = C.c_int32(); n = C.c_int32()
        self._chk(self._L.oracle_get_schedule(self._h, C.addressof(S), C.addressof(k), C.addressof(n)))
        return {"S": S.value, "k": k.value, "phase_steps_per_mcs": n.value}

    # ---- vector terms (Eq 4-7) ----
    def set_chemotaxis_field(self, field):
        """field: shape dims[::-1] + (ndim,), float32, components in [-1, 1]."""
        f = np.ascontiguousarray(np.asarray(field, dtype=np.float32)).reshape(-1)
        assert f.size == self.N * self.ndim
        self._chk(self._L.oracle_set_chemotaxis_field(self._h, f.ctypes.data))

    def set_persistence(self, p):
        a = np.ascontiguousarray(np.asarray(p, dtype=np.float64)).reshape(-1)
        assert a.size == 3 * (self.max_cells + 1)
        self._chk(self._L.oracle_set_persistence(self._h, a.ctypes.data))

    def get_persistence(self):
        out = np.empty((self.max_cells + 1, 3), dtype=np.float64)
        self._chk(self._L.oracle_get_persistence(self._h, out.ctypes.data))
        return out

    def get_centroids(self):
        out = np.empty((self.max_cells + 1, 3), dtype=np.float64)
        self._chk(self._L.oracle_get_centroids(self._h, out.ctypes.data))
        return out

    def probe_dir(self, t_index, nb):
        v = C.c_int64()
        self._chk(self._L.oracle_probe_dir(self._h, int(t_index), int(nb), C.addressof(v)))
        return v.value

    # ---- instrumentation ----
    def get_interface_counts(self):
        out = np.zeros((self.n_types, self.n_types), dtype=np.uint64)
        self._chk(self._L.oracle_get_interface_counts(self._h, out.ctypes.data))
        return out

    def update_statistics(self, n_mcs, n_freq=8, n_wait=64, wait_bin=1):
        freq = np.zeros(n_freq, dtype=np.uint64); wait = np.zeros(n_wait, dtype=np.uint64)
        self._chk(self._L.oracle_update_statistics(self._h, int(n_mcs), freq.ctypes.data, n_freq, wait.ctypes.data, n_wait,
                                                   int(wait_bin)))
        return freq, wait

    # ---- hooks for the pins ----
    def set_visit_order(self, order, seed=0):
        self._chk(self._L.oracle_set_visit_order(self._h, int(order), int(seed)))

    def probe(self, t_index, nb):
        st = C.c_int32(); dh = C.c_int64(); da = C.c_int64()
        self._chk(self._L.oracle_probe(self._h, int(t_index), int(nb), C.addressof(st), C.addressof(dh),
                                       C.addressof(da)))
        return st.value, dh.value, da.value

    def force_copy(self, t_index, nb):
        self._chk(self._L.oracle_force_copy(self._h, int(t_index), int(nb)))

    def trace(self, cap):
        """Start recording per-attempt records; returns (buffer[cap,6], counter)."""
        buf = np.zeros((int(cap), 6), dtype=np.int64)
        cnt = np.zeros(1, dtype=np.uint64)
        self._chk(self._L.oracle_set_trace(self._h, buf.ctypes.data, int(cap), cnt.ctypes.data))
        self._trace_keep = (buf, cnt)
        return buf, cnt

    def stop_trace(self):
        self._chk(self._L.oracle_set_trace(self._h, None, 0, None))


def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32); k = np.asarray(key, dtype=np.uint32)
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(c.ctypes.data, k.ctypes.data, out.ctypes.data)
    return out


def decode_proposal(w, sites, n_nb):
    l = C.c_uint32(); nb = C.c_uint32()
    lib().oracle_decode_proposal(int(w), int(sites), int(n_nb), C.addressof(l), C.addressof(nb))
    return l.value, nb.value


def threshold_table(T):
    hmax = lib().oracle_threshold_table(float(T), None, 0)
    thr = np.zeros(hmax + 1, dtype=np.uint32)
    lib().oracle_threshold_table(float(T), thr.ctypes.data, hmax + 1)
    return hmax, thr


def gm_q16(acts):
    a = np.ascontiguousarray(np.asarray(acts, dtype=np.int32))
    return int(lib().oracle_gm_q16(a.ctypes.data, a.size))


def direction_table(ndim):
    out = np.zeros(26 * 3, dtype=np.int64)
    n = lib().oracle_direction_table(int(ndim), out.ctypes.data)
    return out[: 3 * n].reshape(n, 3)


def neighbour_offsets(ndim):
    out = np.zeros(26 * 3, dtype=np.int32)
    n = lib().oracle_neighbour_offsets(int(ndim), out.ctypes.data)
    return out[: 3 * n].reshape(n, 3)
