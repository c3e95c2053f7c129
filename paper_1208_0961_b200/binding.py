"""ctypes binding with the same names as include/cuba.h (marshalling only)."""
from __future__ import annotations

import ctypes
import dataclasses
import os
from ctypes import POINTER, Structure, c_char_p, c_double, c_int, c_int64, c_size_t, c_uint8, c_uint32, c_uint64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

# every symbol include/cuba.h declares
EXPORTS = ("cuba_workspace_bytes", "cuba_init", "cuba_step", "cuba_observables", "cuba_state",
           "cuba_get_particles", "cuba_get_cells", "cuba_step_traced", "cuba_counters", "cuba_run_host", "cuba_destroy",
           "cuba_strerror", "cuba_last_cuda_error", "cuba_launch_count", "cuba_profile_enable",
           "cuba_profile_read", "cuba_profile_name", "cuba_set_option", "cuba_observables_lrf",
           "cuba_step_adaptive", "cuba_step_local_sigma", "cuba_probe_fp64", "cuba_slot_stats",
           "cuba_slab_init", "cuba_slab_owned", "cuba_slab_count", "cuba_slab_buffer_bytes", "cuba_slab_pack", "cuba_slab_unpack",
           "cuba_observables_noalloc", "cuba_slab_layer_index")


# cuba_set_option
OPT_FUSE_HIST, OPT_GRAPH, OPT_SLOTS, OPT_SLOT_MARGIN = 1, 2, 3, 4
PROFILE_GROUPS = 21   # CUBA_PROFILE_GROUPS
NOALLOC_MAX_SLABS = 128   # CUBA_NOALLOC_MAX_SLABS


class CubaError(RuntimeError):
    def __init__(self, code, detail=""):
        self.code = code
        msg = "cuba error %d: %s" % (code, strerror(code))
        if detail:
            msg += " (" + detail + ")"
        super().__init__(msg)


class _Soa(Structure):
    _fields_ = [(k, c_void_p) for k in ("x", "y", "z", "px", "py", "pz", "pid", "cell_start")]


class _Counters(Structure):
    _fields_ = [(k, c_uint64) for k in ("steps", "pairs", "collisions", "rounds", "near_threshold",
                                        "max_occupancy", "overflow_cells", "device_flags")]


class _Trace(Structure):
    _fields_ = [("cell_of_pid", c_void_p), ("pair_capacity", c_int64), ("n_pairs", c_int64),
                ("pair_cell", c_void_p), ("pair_round", c_void_p), ("pid_a", c_void_p), ("pid_b", c_void_p),
                ("P", c_void_p), ("u", c_void_p), ("decided", c_void_p)]


@dataclasses.dataclass
class Counters:
    steps: int
    pairs: int
    collisions: int
    rounds: int
    near_threshold: int
    max_occupancy: int
    overflow_cells: int
    device_flags: int


@dataclasses.dataclass
class Trace:
    cell_of_pid: np.ndarray
    cell: np.ndarray
    round: np.ndarray
    pid_a: np.ndarray
    pid_b: np.ndarray
    P: np.ndarray
    u: np.ndarray
    decided: np.ndarray


def lib_path() -> str:
    """In-tree library; CUBA_LIB_PATH overrides it (used to compare experimental builds)."""
    return os.environ.get("CUBA_LIB_PATH") or os.path.join(_HERE, "libcuba.so")


_lib = None


def lib():
    """Load libcuba.so (built in-tree by `python -m paper_1208_0961_b200.build`)."""
    global _lib
    if _lib is None:
        path = lib_path()
        if not os.path.exists(path):
            raise RuntimeError("%s is missing: build it with `python -m paper_1208_0961_b200.build` "
                               "(there is no CPU fallback)" % path)
        L = ctypes.CDLL(path)
        dp = POINTER(c_double)
        L.cuba_workspace_bytes.argtypes = [c_int64, POINTER(c_int)]
        L.cuba_workspace_bytes.restype = c_size_t
        L.cuba_init.argtypes = [POINTER(c_void_p), dp, POINTER(c_int), c_int64] + [c_void_p] * 6 + \
                               [c_double, c_uint64, c_void_p, c_size_t, c_void_p]
        L.cuba_step.argtypes = [c_void_p, c_int, c_double, c_double]
        L.cuba_observables.argtypes = [c_void_p, dp, c_int, dp]
        L.cuba_state.argtypes = [c_void_p, POINTER(_Soa)]
        L.cuba_get_particles.argtypes = [c_void_p] + [c_void_p] * 7
        L.cuba_get_cells.argtypes = [c_void_p, c_void_p]
        L.cuba_step_traced.argtypes = [c_void_p, c_double, c_double, POINTER(_Trace)]
        L.cuba_counters.argtypes = [c_void_p, POINTER(_Counters)]
        L.cuba_run_host.argtypes = [dp, POINTER(c_int), c_int64] + [c_void_p] * 6 + \
                                   [c_double, c_uint64, c_int, c_double, c_double, dp, c_int, dp, c_void_p, c_int]
        L.cuba_destroy.argtypes = [c_void_p]
        L.cuba_destroy.restype = None
        L.cuba_strerror.argtypes = [c_int]
        L.cuba_strerror.restype = c_char_p
        L.cuba_last_cuda_error.restype = c_char_p
        L.cuba_launch_count.restype = c_uint64
        L.cuba_profile_enable.argtypes = [c_void_p, c_int]
        L.cuba_set_option.argtypes = [c_void_p, c_int, c_int]
        L.cuba_observables_lrf.argtypes = [c_void_p, c_int, dp, dp]
        L.cuba_step_adaptive.argtypes = [c_void_p, c_int, c_double, c_double, dp, dp]
        L.cuba_step_local_sigma.argtypes = [c_void_p, c_int, c_double, c_double]
        L.cuba_profile_read.argtypes = [c_void_p, dp, POINTER(c_uint64)]
        L.cuba_probe_fp64.argtypes = [c_void_p, c_int, dp]
        L.cuba_slot_stats.argtypes = [c_void_p, POINTER(c_uint64)]
        L.cuba_slab_init.argtypes = [POINTER(c_void_p), dp, POINTER(c_int), c_int64, c_int64] + [c_void_p] * 7 + \
                                    [c_double, c_uint64, c_void_p, c_size_t, c_void_p, c_int, c_int]
        L.cuba_slab_owned.argtypes = [c_void_p, POINTER(c_int64)]
        L.cuba_slab_count.argtypes = [c_void_p, c_int, POINTER(c_int64)]
        L.cuba_slab_buffer_bytes.argtypes = [c_int64, POINTER(c_int)]
        L.cuba_slab_buffer_bytes.restype = c_size_t
        L.cuba_slab_pack.argtypes = [c_void_p, c_int, c_void_p, c_size_t]
        L.cuba_slab_unpack.argtypes = [c_void_p, c_void_p, c_int64, c_void_p, c_int64]
        L.cuba_observables_noalloc.argtypes = [c_int64] + [c_void_p] * 4 + [dp, c_double, c_int, c_void_p, c_void_p]
        L.cuba_slab_layer_index.argtypes = [c_double, c_int, c_int64, c_void_p, c_void_p]
        L.cuba_profile_name.argtypes = [c_int]
        L.cuba_profile_name.restype = c_char_p
        _lib = L
    return _lib


def strerror(code: int) -> str:
    try:
        return lib().cuba_strerror(int(code)).decode()
    except Exception:
        return "?"


def _check(rc):
    if rc != 0:
        detail = lib().cuba_last_cuda_error().decode() if rc == -5 else ""
        raise CubaError(rc, detail)


def _c3d(v):
    return (c_double * 3)(*[float(a) for a in v])


def _c3i(v):
    return (c_int * 3)(*[int(a) for a in v])


def workspace_bytes(n, ncell) -> int:
    return int(lib().cuba_workspace_bytes(int(n), _c3i(ncell)))


def launch_count() -> int:
    return int(lib().cuba_launch_count())


def probe_fp64(stream=None, repeats=5) -> float:
    """cuba_probe_fp64: measured thread-level fp64 FMA instructions per second of the device."""
    v = c_double(0.0)
    _check(lib().cuba_probe_fp64(c_void_p(stream) if stream else None, int(repeats), ctypes.byref(v)))
    return float(v.value)


def observables_noalloc(x, px, py, pz, box, n_test, nslab, result, stream=None):
    """cuba_observables_noalloc: sum E, sum p and the energy density per x-slab for a caller that may not
    allocate GPU memory (a plug-in inside another program's memory budget, a hook between the steps of a
    running loop, a service that allocates only at start-up).  Everything is the caller's: x, px, py, pz are
    1-D float64 CUDA tensors of equal length, `result` a float64 CUDA tensor of 4 + nslab entries that
    receives (sum E, sum px, sum py, sum pz, edens[nslab]) in stream order -- nothing is allocated, copied to
    the host or waited for here.  nslab <= NOALLOC_MAX_SLABS (the partial sums live in a fixed array inside
    the library; beyond it CubaError(-2)).  Calls share that array: keep them on one stream, or order them.
    `stream`: a torch.cuda.Stream (default: the current one)."""
    import torch
    for a in (x, px, py, pz, result):
        if not (a.is_cuda and a.dtype == torch.float64 and a.is_contiguous() and a.dim() == 1):
            raise ValueError("x, px, py, pz and result must be contiguous 1-D float64 CUDA tensors")
    n = int(x.shape[0])
    if not (px.shape[0] == n and py.shape[0] == n and pz.shape[0] == n):
        raise ValueError("x, px, py, pz must have the same length")
    if result.shape[0] < 4 + int(nslab):
        raise ValueError("result needs 4 + nslab entries")
    st = stream if stream is not None else torch.cuda.current_stream(x.device)
    with torch.cuda.device(x.device):
        _check(lib().cuba_observables_noalloc(n, *[c_void_p(a.data_ptr()) for a in (x, px, py, pz)], _c3d(box),
                                              float(n_test), int(nslab), c_void_p(result.data_ptr()),
                                              c_void_p(st.cuda_stream)))


def _np_ptr(a):
    return a.ctypes.data_as(c_void_p) if a is not None else None


class Cuba:
    """cuba_init / cuba_step / cuba_observables on torch-allocated device memory."""

    def __init__(self, box, ncell, x, y, z, px, py, pz, n_test, seed, stream=None):
        import torch
        self._h = None
        if not torch.cuda.is_available():
            raise RuntimeError("cuba needs a CUDA device (no CPU fallback)")
        arrs = [x, y, z, px, py, pz]
        for a in arrs:
            if not (a.is_cuda and a.dtype == torch.float64 and a.is_contiguous() and a.dim() == 1):
                raise ValueError("particle arrays must be contiguous 1-D float64 CUDA tensors")
        self.n = int(x.shape[0])
        self.box = tuple(float(v) for v in box)
        self.ncell = tuple(int(v) for v in ncell)
        self.ncells = self.ncell[0] * self.ncell[1] * self.ncell[2]
        self._arrs = arrs                      # keep alive: the library adopts them in place
        wsb = workspace_bytes(self.n, self.ncell)
        if wsb == 0:
            raise CubaError(-2)
        self._ws = torch.empty(wsb + 256, dtype=torch.uint8, device=x.device)
        base = self._ws.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(x.device)
        h = c_void_p()
        rc = lib().cuba_init(ctypes.byref(h), _c3d(box), _c3i(ncell), self.n,
                             *[c_void_p(a.data_ptr()) for a in arrs], float(n_test), int(seed),
                             c_void_p(self._ws_ptr), wsb, c_void_p(self._stream.cuda_stream))
        _check(rc)
        self._h = h

    @classmethod
    def from_workload(cls, w, device="cuda:0", stream=None):
        import torch
        t = [torch.from_numpy(a).to(device) for a in w.arrays()]
        return cls(w.box, w.ncell, *t, w.n_test, w.seed, stream=stream)

    def close(self):
        if self._h:
            lib().cuba_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def step(self, nsteps, dt, sigma):
        _check(lib().cuba_step(self._h, int(nsteps), float(dt), float(sigma)))

    def observables(self, nslab):
        tot = np.zeros(4)
        ed = np.zeros(int(nslab))
        _check(lib().cuba_observables(self._h, tot.ctypes.data_as(POINTER(c_double)), int(nslab),
                                      ed.ctypes.data_as(POINTER(c_double))))
        return tot, ed

    def state(self):
        """Device pointers of the current store (ints), see cuba_state."""
        s = _Soa()
        _check(lib().cuba_state(self._h, ctypes.byref(s)))
        return {k: getattr(s, k) for k, _ in _Soa._fields_}

    def particles(self):
        """(pid, x, y, z, px, py, pz) as host numpy arrays in array order."""
        pid = np.zeros(self.n, dtype=np.uint32)
        a = [np.zeros(self.n) for _ in range(6)]
        _check(lib().cuba_get_particles(self._h, _np_ptr(pid), *[_np_ptr(v) for v in a]))
        return (pid, *a)

    def cell_start(self):
        out = np.zeros(self.ncells + 1, dtype=np.uint32)
        _check(lib().cuba_get_cells(self._h, _np_ptr(out)))
        return out

    def step_traced(self, dt, sigma, pair_capacity=None):
        cap = int(pair_capacity) if pair_capacity is not None else 4 * self.n + 64
        tr = _Trace()
        cell_of_pid = np.zeros(self.n, dtype=np.uint32)
        cell, rnd, pa, pb = (np.zeros(cap, dtype=np.uint32) for _ in range(4))
        P, u = np.zeros(cap), np.zeros(cap)
        dec = np.zeros(cap, dtype=np.uint8)
        tr.cell_of_pid = _np_ptr(cell_of_pid)
        tr.pair_capacity = cap
        tr.pair_cell, tr.pair_round, tr.pid_a, tr.pid_b = _np_ptr(cell), _np_ptr(rnd), _np_ptr(pa), _np_ptr(pb)
        tr.P, tr.u, tr.decided = _np_ptr(P), _np_ptr(u), _np_ptr(dec)
        _check(lib().cuba_step_traced(self._h, float(dt), float(sigma), ctypes.byref(tr)))
        m = int(tr.n_pairs)
        return Trace(cell_of_pid, cell[:m], rnd[:m], pa[:m], pb[:m], P[:m], u[:m], dec[:m])

    def step_local_sigma(self, nsteps, dt, eta_over_s):
        """cuba_step_local_sigma: per-cell cross section for constant eta/s."""
        _check(lib().cuba_step_local_sigma(self._h, int(nsteps), float(dt), float(eta_over_s)))

    def step_adaptive(self, nsteps, dt_max, sigma):
        """cuba_step_adaptive: returns (dt_used[nsteps], elapsed)."""
        used = np.zeros(int(nsteps))
        el = (c_double * 1)()
        _check(lib().cuba_step_adaptive(self._h, int(nsteps), float(dt_max), float(sigma),
                                        used.ctypes.data_as(POINTER(c_double)), el))
        return used, float(el[0])

    def observables_lrf(self, nslab):
        """cuba_observables_lrf: (T[5, nslab] = T00, T0x, Txx, Tyy, Tzz; lrf[4, nslab] = e, v, P_L, P_T)."""
        T = np.zeros((5, int(nslab)))
        lrf = np.zeros((4, int(nslab)))
        _check(lib().cuba_observables_lrf(self._h, int(nslab), T.ctypes.data_as(POINTER(c_double)),
                                          lrf.ctypes.data_as(POINTER(c_double))))
        return T, lrf

    def set_option(self, option: int, value: int):
        """cuba_set_option (OPT_FUSE_HIST, OPT_GRAPH, OPT_SLOTS, OPT_SLOT_MARGIN)."""
        _check(lib().cuba_set_option(self._h, int(option), int(value)))

    def slot_stats(self):
        """cuba_slot_stats: (calls run on the slotted store, of which redone on the compact schedule)."""
        out = (c_uint64 * 2)()
        _check(lib().cuba_slot_stats(self._h, out))
        return int(out[0]), int(out[1])

    def profile_enable(self, mode=1):
        """0 off, 1 per-kernel events (collision classes as one concurrent group), 2 classes serialised."""
        _check(lib().cuba_profile_enable(self._h, int(mode)))

    def profile_read(self):
        """{kernel group: (summed device ms, launches)} since profile_enable."""
        G = PROFILE_GROUPS
        ms = (c_double * G)()
        cnt = (c_uint64 * G)()
        _check(lib().cuba_profile_read(self._h, ms, cnt))
        return {lib().cuba_profile_name(g).decode(): (float(ms[g]), int(cnt[g])) for g in range(G)}

    def counters(self) -> Counters:
        c = _Counters()
        _check(lib().cuba_counters(self._h, ctypes.byref(c)))
        return Counters(*[int(getattr(c, k)) for k, _ in _Counters._fields_])


def run_host(box, ncell, x, y, z, px, py, pz, n_test, seed, nsteps, dt, sigma, nslab, download=False):
    """cuba_run_host: HOST numpy (ideally pinned) arrays in, observables out (end to end)."""
    arrs = [x, y, z, px, py, pz]
    n = int(arrs[0].shape[0])
    tot = np.zeros(4)
    ed = np.zeros(int(nslab))
    pid = np.zeros(n, dtype=np.uint32) if download else None
    ptrs = [c_void_p(a.ctypes.data) if isinstance(a, np.ndarray) else c_void_p(a.data_ptr()) for a in arrs]
    rc = lib().cuba_run_host(_c3d(box), _c3i(ncell), n, *ptrs, float(n_test), int(seed), int(nsteps),
                             float(dt), float(sigma), tot.ctypes.data_as(POINTER(c_double)), int(nslab),
                             ed.ctypes.data_as(POINTER(c_double)), _np_ptr(pid), int(bool(download)))
    _check(rc)
    return tot, ed, pid
