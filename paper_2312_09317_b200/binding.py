"""ctypes binding of libcpm_b200.so with the same names as include/cpm.h.

PyTorch is used only for device memory and streams: device tensors are passed by data_ptr(),
the context runs on torch's current CUDA stream.  numpy arrays are passed as host pointers.
"""
import ctypes as C
import os
import re

import numpy as np

from . import build as _build

MODE_DETERMINISTIC, MODE_LIVE_ATOMICS = 0, 1
FLAG_WARP_KERNEL, FLAG_NO_TMA, FLAG_NO_GRAPH = 1, 2, 4

_HEADER = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "cpm.h")


class CPMError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__("cpm error %d: %s" % (code, msg))
        self.code = code


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
        ("flags", C.c_uint32),
        ("lambda_pers", C.POINTER(C.c_int32)), ("mu_pers", C.POINTER(C.c_double)), ("dt_pers", C.c_int32),
        ("lambda_chem", C.POINTER(C.c_int32)), ("unwrap_centroids", C.c_int32),
    ]


def library_path():
    return _build.LIB


def exported_symbols():
    """Names declared in include/cpm.h (every `cpm_*(` prototype)."""
    with open(_HEADER) as f:
        text = f.read()
    return sorted(set(re.findall(r"\b(cpm_[a-z_0-9]+)\s*\(", text)))


_lib = None


def load_library():
    """Load (building first if the sources are newer and nvcc is present).  Raises if the library
    cannot be produced: there is no other implementation to fall back to."""
    global _lib
    if _lib is not None:
        return _lib
    if _build.is_stale():
        try:
            _build.build()
        except Exception as e:  # no nvcc on this box and no prebuilt .so
            if not os.path.exists(_build.LIB):
                raise RuntimeError("libcpm_b200.so is missing and could not be built: %r" % (e,))
    L = C.CDLL(_build.LIB)
    vp = C.c_void_p
    L.cpm_create.argtypes = [C.POINTER(_Params), C.POINTER(vp)]
    L.cpm_destroy.argtypes = [vp]
    L.cpm_set_lattice.argtypes = [vp, vp, vp, vp, C.c_int]
    L.cpm_set_act.argtypes = [vp, vp, C.c_int]
    L.cpm_set_mcs.argtypes = [vp, C.c_uint32]
    L.cpm_set_chemotaxis_field.argtypes = [vp, vp, C.c_int]
    L.cpm_set_persistence.argtypes = [vp, vp, C.c_int]
    L.cpm_get_persistence.argtypes = [vp, vp, C.c_int]
    L.cpm_step.argtypes = [vp, C.c_uint32]
    L.cpm_get_lattice.argtypes = [vp, vp, C.c_int]
    L.cpm_get_act.argtypes = [vp, vp, C.c_int]
    L.cpm_get_cell_stats.argtypes = [vp, vp, vp, vp, vp, vp, C.c_int]
    L.cpm_get_counters.argtypes = [vp, vp]
    L.cpm_get_centroids.argtypes = [vp, vp, C.c_int]
    L.cpm_get_schedule.argtypes = [vp, vp, vp, vp]
    L.cpm_get_interface_counts.argtypes = [vp, vp]
    L.cpm_update_statistics.argtypes = [vp, C.c_uint32, vp, C.c_int32, vp, C.c_int32, C.c_uint32]
    L.cpm_noalloc_setup.argtypes = [C.c_int]
    L.cpm_update_statistics_noalloc.argtypes = [vp, C.c_uint32, vp, C.c_int32, vp, C.c_int32, C.c_uint32, C.c_int]
    L.cpm_get_threshold_table.argtypes = [vp, vp, C.c_uint64]
    L.cpm_get_threshold_table.restype = C.c_int64
    L.cpm_get_launch_info.argtypes = [vp, vp]
    L.cpm_set_kernel_timing.argtypes = [vp, C.c_int]
    L.cpm_get_kernel_timing.argtypes = [vp, vp, vp, C.c_int]
    L.cpm_last_error.argtypes = [vp]
    L.cpm_last_error.restype = C.c_char_p
    L.cpm_debug_philox.argtypes = [C.c_int, vp, vp, vp, C.c_uint64]
    _lib = L
    return L


def _is_tensor(x):
    return hasattr(x, "data_ptr") and hasattr(x, "is_cuda")


def _ptr(x, dtype, n):
    """(pointer, on_device, keepalive) of a numpy array or torch tensor of n elements."""
    if x is None:
        return None, 0, None
    if _is_tensor(x):
        import torch
        want = {np.uint32: (torch.uint32, torch.int32), np.uint8: (torch.uint8,), np.float32: (torch.float32,),
                np.uint64: (torch.uint64, torch.int64), np.float64: (torch.float64,)}[dtype]
        assert x.dtype in want, (x.dtype, want)
        assert x.is_contiguous() and x.numel() == n, (x.shape, n)
        return x.data_ptr(), (1 if x.is_cuda else 0), x
    a = np.ascontiguousarray(np.asarray(x, dtype=dtype))
    assert a.size == n, (a.size, n)
    return a.ctypes.data, 0, a


class CPM:
    """One simulation context (cpm_create .. cpm_destroy).  Lattice arrays have shape dims[::-1]."""

    def __init__(self, dims, J, lambda_V=None, target_V=None, lambda_P=None, target_P=None,
                 lambda_act=None, max_act=None, T=20.0, seed=1, subsection=0,
                 attempts_per_activation=0, mode=MODE_DETERMINISTIC, max_cells=0,
                 periodic=(0, 0, 0), device=None, stream=None, flags=0,
                 lambda_pers=None, mu_pers=None, dt_pers=0, lambda_chem=None, unwrap_centroids=0):
        import torch  # device memory + streams only
        L = load_library()
        if not torch.cuda.is_available():
            raise CPMError(-4, "no CUDA device: the CUDA path is the only implementation")
        if device is None:
            device = torch.cuda.current_device()
        if stream is None:
            stream = torch.cuda.current_stream(device).cuda_stream
        dims = tuple(int(v) for v in dims)
        self.ndim = len(dims)
        self.dims = dims
        self.shape = tuple(reversed(dims))
        self.N = int(np.prod(dims))
        self.device = int(device)
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
            if val is not None:
                arr = np.ascontiguousarray(np.asarray(val, dtype=np.int32))
                assert arr.size == nT
                keep.append(arr)
                setattr(p, name, arr.ctypes.data_as(C.POINTER(C.c_int32)))
        p.T = float(T)
        p.seed = int(seed)
        p.subsection = int(subsection)
        p.attempts_per_activation = int(attempts_per_activation)
        p.mode = int(mode)
        p.max_cells = self.max_cells
        p.device = self.device
        p.stream = C.c_void_p(int(stream))
        p.flags = int(flags)
        if mu_pers is not None:
            mu = np.ascontiguousarray(np.asarray(mu_pers, dtype=np.float64))
            assert mu.size == nT
            keep.append(mu)
            p.mu_pers = mu.ctypes.data_as(C.POINTER(C.c_double))
        p.dt_pers = int(dt_pers)
        p.unwrap_centroids = int(unwrap_centroids)
        h = C.c_void_p()
        rc = L.cpm_create(C.byref(p), C.byref(h))
        if rc != 0:
            raise CPMError(rc, "cpm_create")
        self._h = h
        self._L = L

    def _chk(self, rc):
        if rc != 0:
            raise CPMError(rc, self._L.cpm_last_error(self._h).decode())

    def close(self):
        if getattr(self, "_h", None):
            self._L.cpm_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- the calls of include/cpm.h ----
    def set_lattice(self, ids, frozen=None, cell_type=None):
        pi, di, ki = _ptr(ids, np.uint32, self.N)
        pf, df, kf = _ptr(frozen, np.uint8, self.N)
        pc, dc, kc = _ptr(cell_type, np.uint8, self.max_cells + 1)
        assert frozen is None or df == di, "ids and frozen must live on the same side"
        assert dc == di, "ids and cell_type must live on the same side"
        self._chk(self._L.cpm_set_lattice(self._h, pi, pf, pc, di))

    def set_act(self, act):
        pa, da, ka = _ptr(act, np.float32, self.N)
        self._chk(self._L.cpm_set_act(self._h, pa, da))

    def set_mcs(self, mcs):
        self._chk(self._L.cpm_set_mcs(self._h, int(mcs)))

    def set_chemotaxis_field(self, field):
        """field: shape dims[::-1] + (ndim,), float32 components in [-1, 1] (Eq 4)."""
        pf, df, kf = _ptr(field, np.float32, self.N * self.ndim)
        self._chk(self._L.cpm_set_chemotaxis_field(self._h, pf, df))

    def set_persistence(self, p):
        pp, dp, kp = _ptr(p, np.float64, 3 * (self.max_cells + 1))
        self._chk(self._L.cpm_set_persistence(self._h, pp, dp))

    def get_persistence(self, out=None):
        if out is None:
            out = np.empty(3 * (self.max_cells + 1), dtype=np.float64)
        po, do, ko = _ptr(out, np.float64, 3 * (self.max_cells + 1))
        self._chk(self._L.cpm_get_persistence(self._h, po, do))
        return ko.reshape(self.max_cells + 1, 3)

    def step(self, n=1):
        self._chk(self._L.cpm_step(self._h, int(n)))

    def get_lattice(self, out=None):
        if out is None:
            out = np.empty(self.N, dtype=np.uint32)
        po, do, ko = _ptr(out, np.uint32, self.N)
        self._chk(self._L.cpm_get_lattice(self._h, po, do))
        return ko.reshape(self.shape)

    def get_act(self, out=None):
        if out is None:
            out = np.empty(self.N, dtype=np.float32)
        po, do, ko = _ptr(out, np.float32, self.N)
        self._chk(self._L.cpm_get_act(self._h, po, do))
        return ko.reshape(self.shape)

    def get_cell_stats(self):
        n = self.max_cells + 1
        V = np.empty(n, np.uint32); P = np.empty(n, np.uint32)
        sx = np.empty(n, np.uint64); sy = np.empty(n, np.uint64); sz = np.empty(n, np.uint64)
        self._chk(self._L.cpm_get_cell_stats(self._h, V.ctypes.data, P.ctypes.data, sx.ctypes.data,
                                             sy.ctypes.data, sz.ctypes.data, 0))
        return {"volume": V, "perimeter": P, "sum_x": sx, "sum_y": sy, "sum_z": sz}

    def get_centroids(self, out=None):
        if out is None:
            out = np.empty(3 * (self.max_cells + 1), dtype=np.float64)
        po, do, ko = _ptr(out, np.float64, 3 * (self.max_cells + 1))
        self._chk(self._L.cpm_get_centroids(self._h, po, do))
        return ko.reshape(self.max_cells + 1, 3)

    def get_counters(self):
        out = np.zeros(4, np.uint64)
        self._chk(self._L.cpm_get_counters(self._h, out.ctypes.data))
        return {"attempts": int(out[0]), "evaluated": int(out[1]), "accepted": int(out[2]), "mcs": int(out[3])}

    def get_schedule(self):
        S = C.c_int32(); k = C.c_int32(); n = C.c_int32()
        self._chk(self._L.cpm_get_schedule(self._h, C.addressof(S), C.addressof(k), C.addressof(n)))
        return {"S": S.value, "k": k.value, "phase_steps_per_mcs": n.value}

    def get_interface_counts(self):
        out = np.zeros((self.n_types, self.n_types), dtype=np.uint64)
        self._chk(self._L.cpm_get_interface_counts(self._h, out.ctypes.data))
        return out

    def update_statistics(self, n_mcs, n_freq=8, n_wait=64, wait_bin=1):
        freq = np.zeros(n_freq, dtype=np.uint64); wait = np.zeros(n_wait, dtype=np.uint64)
        self._chk(self._L.cpm_update_statistics(self._h, int(n_mcs), freq.ctypes.data, n_freq, wait.ctypes.data, n_wait,
                                                int(wait_bin)))
        return freq, wait

    def update_statistics_noalloc(self, n_mcs, freq, wait, wait_bin=1):
        """cpm_update_statistics_noalloc: freq / wait are caller-owned uint64 buffers, numpy arrays (host) or CUDA torch
        tensors viewed as int64 (device); nothing is allocated.  Lattices up to NOALLOC_MAX_SITES sites."""
        on_dev = not isinstance(freq, np.ndarray)
        if on_dev != (not isinstance(wait, np.ndarray)):
            raise TypeError("freq and wait must both be numpy arrays or both be device tensors")
        for a in (freq, wait):
            if on_dev:
                if not (a.is_cuda and a.is_contiguous() and a.element_size() == 8):
                    raise TypeError("device outputs must be contiguous 8-byte CUDA tensors")
            elif a.dtype != np.uint64 or not a.flags.c_contiguous:
                raise TypeError("host outputs must be contiguous uint64 arrays")
        n_freq, n_wait = (int(freq.numel()), int(wait.numel())) if on_dev else (freq.size, wait.size)
        pf, pw = (freq.data_ptr(), wait.data_ptr()) if on_dev else (freq.ctypes.data, wait.ctypes.data)
        self._chk(self._L.cpm_update_statistics_noalloc(self._h, int(n_mcs), pf, n_freq, pw, n_wait, int(wait_bin), int(on_dev)))

    def get_threshold_table(self):
        hmax = self._L.cpm_get_threshold_table(self._h, None, 0)
        if hmax < 0:
            raise CPMError(int(hmax), "cpm_get_threshold_table")
        thr = np.zeros(hmax + 1, np.uint32)
        self._L.cpm_get_threshold_table(self._h, thr.ctypes.data, hmax + 1)
        return int(hmax), thr

    def get_launch_info(self):
        out = np.zeros(6, np.uint64)
        self._chk(self._L.cpm_get_launch_info(self._h, out.ctypes.data))
        return {"launches": int(out[0]), "sweep_launches": int(out[1]), "warps_per_cta": int(out[2]),
                "smem_bytes_per_cta": int(out[3]), "uses_tma": bool(out[4]),
                "pooled": bool(out[5])}

    def set_kernel_timing(self, enabled=True):
        self._chk(self._L.cpm_set_kernel_timing(self._h, 1 if enabled else 0))

    def get_kernel_timing(self, reset=True):
        ms = C.c_double(); n = C.c_uint64()
        self._chk(self._L.cpm_get_kernel_timing(self._h, C.addressof(ms), C.addressof(n), 1 if reset else 0))
        return ms.value, int(n.value)


NOALLOC_MAX_SITES = 1 << 20   # CPM_NOALLOC_MAX_SITES of include/cpm.h
NOALLOC_MAX_BINS = 4096       # CPM_NOALLOC_MAX_BINS


def noalloc_setup(device=0):
    """cpm_noalloc_setup: resolve the device address of the library's static scratch array on `device`."""
    rc = load_library().cpm_noalloc_setup(int(device))
    if rc != 0:
        raise CPMError(int(rc), "cpm_noalloc_setup")


def debug_philox(ctr, key, device=0):
    """Run the device Philox4x32-10 on n (ctr[4], key[2]) pairs; returns uint32[n,4]."""
    L = load_library()
    c = np.ascontiguousarray(np.asarray(ctr, dtype=np.uint32)).reshape(-1, 4)
    k = np.ascontiguousarray(np.asarray(key, dtype=np.uint32)).reshape(-1, 2)
    assert len(c) == len(k)
    out = np.zeros((len(c), 4), np.uint32)
    rc = L.cpm_debug_philox(int(device), c.ctypes.data, k.ctypes.data, out.ctypes.data, len(c))
    if rc != 0:
        raise CPMError(rc, "cpm_debug_philox")
    return out
