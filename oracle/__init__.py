"""CPU oracle for the CuBA hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

A ctypes front end to `oracle/cuba_oracle.c` (plain single-threaded C, fp64, compiled with
`-ffp-contract=off`).  The arithmetic lives in the C file, each function citing the
PAPER.md passage it follows; this module only builds it and marshals numpy arrays.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` /
`--impl reference` legs may import this package.  It shares no code with, and never
imports, `paper_1208_0961_b200` (the CUDA library); the product never imports it.

Parity unpinned: the paper's Fig. 2-4 curves and the CuBA-vs-BAMPS
overlay -- the images and BAMPS itself are not available.  Every function here is pinned
by tests/test_oracle_*.py.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_int, c_int64, c_uint8, c_uint32, c_uint64, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cuba_oracle.c")
_LIB = os.path.join(_HERE, "libcuba_oracle.so")

# -ffp-contract=off: part of the arithmetic contract (A2).
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c99", "-shared", "-fPIC"]

ERR_NAMES = {0: "ok", -1: "bad argument", -6: "invalid particle state",
             -7: "dt not below the smallest cell edge", -9: "more than 64 rounds needed"}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp.%d" % os.getpid()
        subprocess.check_call(["gcc", *CFLAGS, "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        dp, u32p = POINTER(c_double), POINTER(c_uint32)
        L.oracle_philox4x32_10.argtypes = [u32p, u32p, u32p]
        L.oracle_u53.argtypes = [c_uint32, c_uint32]
        L.oracle_u53.restype = c_double
        L.oracle_stream_reflect.argtypes = [c_int64] + [dp] * 6 + [c_double, dp, dp]
        L.oracle_cell_index.argtypes = [c_int64, dp, dp, dp, dp, POINTER(c_int), u32p]
        L.oracle_counting_sort.argtypes = [c_int64, c_int64, u32p, u32p, POINTER(c_int64)]
        L.oracle_pair_kinematics.argtypes = [dp, dp, dp, dp, dp, dp]
        L.oracle_direction.argtypes = [c_uint64, c_uint32, c_uint32, c_uint32, dp]
        L.oracle_direction.restype = c_int
        L.oracle_scatter.argtypes = [dp, dp, c_double, c_double, c_double, dp, dp, dp]
        L.oracle_init.argtypes = [dp, POINTER(c_int), c_int64] + [dp] * 6 + [c_double, c_uint64, POINTER(c_int)]
        L.oracle_init.restype = c_void_p
        L.oracle_destroy.argtypes = [c_void_p]
        L.oracle_set_trace.argtypes = [c_void_p, c_int]
        L.oracle_set_dirlog.argtypes = [c_void_p, c_int]
        L.oracle_step.argtypes = [c_void_p, c_int, c_double, c_double]
        L.oracle_step.restype = c_int
        L.oracle_observables.argtypes = [c_void_p, dp, c_int, dp]
        L.oracle_step_etas.argtypes = [c_void_p, c_int, c_double, c_double]
        L.oracle_step_etas.restype = c_int
        L.oracle_local_base.argtypes = [c_int64, dp, dp, dp, c_double, c_double]
        L.oracle_local_base.restype = c_double
        L.oracle_step_adaptive.argtypes = [c_void_p, c_int, c_double, c_double, dp, dp]
        L.oracle_step_adaptive.restype = c_int
        L.oracle_observables_lrf.argtypes = [c_void_p, c_int, dp, dp]
        L.oracle_landau_match.argtypes = [c_double] * 5 + [dp]
        L.oracle_get_particles.argtypes = [c_void_p, u32p] + [dp] * 6
        L.oracle_get_cells.argtypes = [c_void_p, u32p, u32p]
        L.oracle_counters.argtypes = [c_void_p, POINTER(c_uint64), dp]
        L.oracle_trace_len.argtypes = [c_void_p]
        L.oracle_trace_len.restype = c_int64
        L.oracle_trace_copy.argtypes = [c_void_p, u32p, u32p, u32p, u32p, dp, dp, POINTER(c_uint8)]
        L.oracle_dirlog_len.argtypes = [c_void_p]
        L.oracle_dirlog_len.restype = c_int64
        L.oracle_dirlog_copy.argtypes = [c_void_p, dp]
        L.oracle_shuffle_order.argtypes = [c_uint64, c_uint32, c_uint32, c_int64, u32p, u32p]
        L.oracle_collide_cells.argtypes = [c_uint64, c_uint32, c_double, c_int64, POINTER(c_int64), POINTER(c_int64),
                                           u32p, u32p, dp, dp, dp, POINTER(c_uint64)]
        L.oracle_collide_cells.restype = c_int
        _lib = L
    return _lib


def _dp(a):
    return a.ctypes.data_as(POINTER(c_double))


def _u32p(a):
    return a.ctypes.data_as(POINTER(c_uint32))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__("oracle error %d: %s" % (code, ERR_NAMES.get(code, "?")))
        self.code = code


# ---- stateless pieces (each pinned on its own) ---------------------------------------

def philox4x32_10(ctr, key):
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().oracle_philox4x32_10(_u32p(c), _u32p(k), _u32p(out))
    return out


def u53(w0, w1):
    return lib().oracle_u53(int(w0), int(w1))


def stream_reflect(x, y, z, px, py, pz, dt, box):
    """S1 + S2 on copies; returns the six new arrays and the wall impulse (3,)."""
    arrs = [_f64(a).copy() for a in (x, y, z, px, py, pz)]
    b = _f64(box)
    wall = np.zeros(3)
    lib().oracle_stream_reflect(arrs[0].shape[0], *[_dp(a) for a in arrs], float(dt), _dp(b), _dp(wall))
    return arrs, wall


def cell_index(x, y, z, box, ncell):
    x, y, z = _f64(x), _f64(y), _f64(z)
    b = _f64(box)
    nc = np.asarray(ncell, dtype=np.int32)
    out = np.zeros(x.shape[0], dtype=np.uint32)
    lib().oracle_cell_index(x.shape[0], _dp(x), _dp(y), _dp(z), _dp(b),
                            nc.ctypes.data_as(POINTER(c_int)), _u32p(out))
    return out


def counting_sort(cell, ncells):
    cell = np.ascontiguousarray(cell, dtype=np.uint32)
    start = np.zeros(ncells + 1, dtype=np.uint32)
    perm = np.zeros(cell.shape[0], dtype=np.int64)
    lib().oracle_counting_sort(cell.shape[0], ncells, _u32p(cell), _u32p(start),
                               perm.ctypes.data_as(POINTER(c_int64)))
    return start, perm


def pair_kinematics(pa, pb):
    pa, pb = _f64(pa), _f64(pb)
    o = [c_double() for _ in range(4)]
    lib().oracle_pair_kinematics(_dp(pa), _dp(pb), *[ctypes.byref(v) for v in o])
    return tuple(v.value for v in o)  # Ea, Eb, s, vrel


def direction(seed, pid, t, rho):
    n = np.zeros(3)
    m = lib().oracle_direction(int(seed), int(pid), int(t), int(rho), _dp(n))
    return n, m


def scatter(pa, pb, Ea, Eb, s, nhat):
    pa, pb, nhat = _f64(pa), _f64(pb), _f64(nhat)
    qa, qb = np.zeros(3), np.zeros(3)
    lib().oracle_scatter(_dp(pa), _dp(pb), Ea, Eb, s, _dp(nhat), _dp(qa), _dp(qb))
    return qa, qb


def local_base(px, py, pz, dt, etas):
    """Eq. 3 without v_rel for one cell with the local cross section (A24)."""
    px, py, pz = _f64(px), _f64(py), _f64(pz)
    return float(lib().oracle_local_base(px.shape[0], _dp(px), _dp(py), _dp(pz), float(dt), float(etas)))


def landau_match(T00, T0x, Txx, Tyy, Tzz):
    """(e, v, P_L, P_T) of one slab's tensor components."""
    o = np.zeros(4)
    lib().oracle_landau_match(float(T00), float(T0x), float(Txx), float(Tyy), float(Tzz), _dp(o))
    return tuple(o)


def shuffle_order(seed, t, rho, pids):
    pids = np.ascontiguousarray(pids, dtype=np.uint32)
    out = np.zeros_like(pids)
    lib().oracle_shuffle_order(int(seed), int(t), int(rho), pids.shape[0], _u32p(pids), _u32p(out))
    return out


def collide_cells(seed, t, base, lo, hi, pid, px, py, pz, cell_id=None):
    """S5 of the oracle on the cells [lo[k], hi[k]) of a cell-sorted state (copies are collided);
    returns (px, py, pz, dict(pairs, collisions, rounds))."""
    lo = np.ascontiguousarray(lo, dtype=np.int64)
    hi = np.ascontiguousarray(hi, dtype=np.int64)
    pid = np.ascontiguousarray(pid, dtype=np.uint32)
    p = [_f64(a).copy() for a in (px, py, pz)]
    cid = None if cell_id is None else np.ascontiguousarray(cell_id, dtype=np.uint32)
    cnt = np.zeros(3, dtype=np.uint64)
    i64p = POINTER(c_int64)
    rc = lib().oracle_collide_cells(int(seed), int(t), float(base), lo.shape[0], lo.ctypes.data_as(i64p),
                                    hi.ctypes.data_as(i64p), None if cid is None else _u32p(cid), _u32p(pid),
                                    _dp(p[0]), _dp(p[1]), _dp(p[2]), cnt.ctypes.data_as(POINTER(c_uint64)))
    if rc != 0:
        raise OracleError(rc)
    return p[0], p[1], p[2], dict(pairs=int(cnt[0]), collisions=int(cnt[1]), rounds=int(cnt[2]))


# ---- a run -----------------------------------------------------------------------------

class Oracle:
    """One simulation state; mirrors cuba_init / cuba_step / cuba_observables."""

    def __init__(self, box, ncell, x, y, z, px, py, pz, n_test, seed):
        self._h = None
        arrs = [_f64(a) for a in (x, y, z, px, py, pz)]
        self.n = arrs[0].shape[0]
        self.box = _f64(box)
        self.ncell = np.asarray(ncell, dtype=np.int32)
        self.ncells = int(np.prod(self.ncell.astype(np.int64)))
        err = c_int(0)
        h = lib().oracle_init(_dp(self.box), self.ncell.ctypes.data_as(POINTER(c_int)), self.n,
                              *[_dp(a) for a in arrs], float(n_test), int(seed), ctypes.byref(err))
        if not h:
            raise OracleError(err.value)
        self._h = c_void_p(h)

    @classmethod
    def from_workload(cls, w):
        return cls(w.box, w.ncell, *w.arrays(), w.n_test, w.seed)

    def close(self):
        if self._h:
            lib().oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def set_trace(self, on=True):
        lib().oracle_set_trace(self._h, int(on))

    def set_dirlog(self, on=True):
        lib().oracle_set_dirlog(self._h, int(on))

    def step(self, nsteps, dt, sigma):
        rc = lib().oracle_step(self._h, int(nsteps), float(dt), float(sigma))
        if rc != 0:
            raise OracleError(rc)

    def step_etas(self, nsteps, dt, etas):
        """Local cross section for constant eta/s (reading A24)."""
        rc = lib().oracle_step_etas(self._h, int(nsteps), float(dt), float(etas))
        if rc != 0:
            raise OracleError(rc)

    def step_adaptive(self, nsteps, dt_max, sigma):
        """Variable dt (reading A23): returns (dt_used[nsteps], elapsed)."""
        used = np.zeros(int(nsteps))
        el = np.zeros(1)
        rc = lib().oracle_step_adaptive(self._h, int(nsteps), float(dt_max), float(sigma), _dp(used), _dp(el))
        if rc != 0:
            raise OracleError(rc)
        return used, float(el[0])

    def observables(self, nslab):
        tot = np.zeros(4)
        ed = np.zeros(nslab)
        lib().oracle_observables(self._h, _dp(tot), int(nslab), _dp(ed))
        return tot, ed

    def observables_lrf(self, nslab):
        """(T, lrf): T[5, nslab] = T00, T0x, Txx, Tyy, Tzz; lrf[4, nslab] = e, v, P_L, P_T."""
        T = np.zeros((5, nslab))
        out = np.zeros((4, nslab))
        lib().oracle_observables_lrf(self._h, int(nslab), _dp(T), _dp(out))
        return T, out

    def particles(self):
        """(pid, x, y, z, px, py, pz) in array order."""
        pid = np.zeros(self.n, dtype=np.uint32)
        a = [np.zeros(self.n) for _ in range(6)]
        lib().oracle_get_particles(self._h, _u32p(pid), *[_dp(v) for v in a])
        return (pid, *a)

    def cells(self):
        """(cell of each slot, cell_start[ncells+1]) after the last binning."""
        c = np.zeros(self.n, dtype=np.uint32)
        s = np.zeros(self.ncells + 1, dtype=np.uint32)
        lib().oracle_get_cells(self._h, _u32p(c), _u32p(s))
        return c, s

    def counters(self):
        out = np.zeros(8, dtype=np.uint64)
        wall = np.zeros(3)
        lib().oracle_counters(self._h, out.ctypes.data_as(POINTER(c_uint64)), _dp(wall))
        keys = ("steps", "pairs", "collisions", "rounds", "near_threshold", "max_occupancy",
                "dir_attempts", "t")
        d = {k: int(v) for k, v in zip(keys, out)}
        d["wall_dp"] = wall
        return d

    def trace(self):
        """Pairs of the last step in (cell, round, k) order."""
        m = lib().oracle_trace_len(self._h)
        cell, rnd, pa, pb = (np.zeros(m, dtype=np.uint32) for _ in range(4))
        P, u = np.zeros(m), np.zeros(m)
        dec = np.zeros(m, dtype=np.uint8)
        if m:
            lib().oracle_trace_copy(self._h, _u32p(cell), _u32p(rnd), _u32p(pa), _u32p(pb),
                                    _dp(P), _dp(u), dec.ctypes.data_as(POINTER(c_uint8)))
        return dict(cell=cell, round=rnd, pid_a=pa, pid_b=pb, P=P, u=u, decided=dec)

    def dirlog(self):
        m = lib().oracle_dirlog_len(self._h)
        out = np.zeros((m, 3))
        if m:
            lib().oracle_dirlog_copy(self._h, _dp(out))
        return out
