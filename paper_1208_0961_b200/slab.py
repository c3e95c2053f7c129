"""x-slab decomposition over several GPUs (include/cuba.h "x-slab decomposition").

Host side only: which cell layers a rank owns, which particles it is given at the start, who sends
which halo buffer to whom, and the marshalling of the cuba_slab_* calls.  Streaming, sorting, pairing
and collisions run in the library's kernels; the bytes of a halo buffer are produced by
cuba_slab_pack on the sender and consumed by cuba_slab_unpack on the receiver.

One process per GPU (`SlabRank` + `exchange_halos` over torch.distributed, NCCL on GPUs); for tests on
one GPU `LocalSlabGroup` steps several ranks' contexts one after the other in one process and hands
the buffers over directly -- the same calls in the same order, no kernel ever waits on another rank.
"""
from __future__ import annotations

import ctypes
from ctypes import c_int64, c_void_p

import numpy as np

from .binding import Cuba, CubaError, _c3d, _c3i, _check, lib, workspace_bytes


def slab_layers(nx: int, world: int, weights=None):
    """[(layer_lo, layer_hi)] per rank: contiguous, whole layers.  Without weights the sizes differ by at most
    one layer; with weights (work per layer, e.g. particles: `layer_weights`) the cuts are put where the running
    sum of the weights crosses k/world of the total, every rank keeping at least one layer."""
    if world < 1 or nx < world:
        raise ValueError("need 1 <= world <= number of cell layers along x")
    if weights is None:
        q, r = divmod(nx, world)
        out, lo = [], 0
        for k in range(world):
            hi = lo + q + (1 if k < r else 0)
            out.append((lo, hi))
            lo = hi
        return out
    wts = np.asarray(weights, dtype=np.float64)
    if wts.shape != (nx,) or np.any(wts < 0) or not np.isfinite(wts).all():
        raise ValueError("one finite non-negative weight per layer")
    cum = np.concatenate([[0.0], np.cumsum(wts)])
    cuts = [0]
    for k in range(1, world):
        target = cum[-1] * k / world
        c = int(np.argmin(np.abs(cum - target)))                 # the layer boundary nearest to the target
        c = max(c, cuts[-1] + 1)                                 # at least one layer for the rank below ...
        c = min(c, nx - (world - k))                             # ... and for every rank above
        cuts.append(c)
    cuts.append(nx)
    return [(cuts[k], cuts[k + 1]) for k in range(world)]


def layer_index(x: np.ndarray, box_x: float, nx: int) -> np.ndarray:
    """cuba_slab_layer_index: the S3 cell layer along x of every particle, computed by the library with the very
    function its kernels bin with (HOST arrays, no device needed).  int32, one per particle."""
    xs = np.ascontiguousarray(x, dtype=np.float64)
    out = np.empty(xs.shape[0], dtype=np.int32)
    _check(lib().cuba_slab_layer_index(float(box_x), int(nx), int(xs.shape[0]), c_void_p(xs.ctypes.data),
                                       c_void_p(out.ctypes.data)))
    return out


def layer_weights(x: np.ndarray, box_x: float, nx: int) -> np.ndarray:
    """Particles per cell layer along x (counts of `layer_index`), to balance the cuts with."""
    return np.bincount(layer_index(x, box_x, nx), minlength=nx).astype(np.float64)


def initial_selection(x: np.ndarray, box_x: float, nx: int, layer_lo: int, layer_hi: int) -> np.ndarray:
    """Ascending global indices of the particles a rank is given at the start: those whose cell layer
    (`layer_index`, the library's S3 index) lies in [layer_lo - 1, layer_hi + 1)."""
    layer = layer_index(x, box_x, nx)
    return np.nonzero((layer >= layer_lo - 1) & (layer < layer_hi + 1))[0]


def neighbours(rank: int, world: int):
    """(lower neighbour, upper neighbour), None at the ends of the box (hard walls, no wrap-around)."""
    return (rank - 1 if rank > 0 else None, rank + 1 if rank + 1 < world else None)


class SlabRank(Cuba):
    """One rank's context: cuba_slab_init and the per-step calls.  The calls of `Cuba` apply to a slab context as
    include/cuba.h says: step (one step at a time), step_local_sigma, counters and the observables (owned
    particles only) work; step_traced and step_adaptive raise CubaError."""

    def __init__(self, w, layer_lo, layer_hi, device="cuda:0", capacity=None, stream=None):
        import torch
        self._h = None
        self.box, self.ncell = tuple(float(v) for v in w.box), tuple(int(v) for v in w.ncell)
        self.layer_lo, self.layer_hi = int(layer_lo), int(layer_hi)
        sel = initial_selection(w.x, self.box[0], self.ncell[0], self.layer_lo, self.layer_hi)
        n = int(sel.shape[0])
        self.capacity = int(capacity) if capacity is not None else int(1.25 * n) + 4096
        if n < 1 or n > self.capacity:
            raise CubaError(-2, "slab of %d particles, capacity %d" % (n, self.capacity))      # CUBA_ERR_SIZE
        self.device = torch.device(device)
        self._arrs = []
        for a in w.arrays():
            t = torch.empty(self.capacity, dtype=torch.float64, device=self.device)
            t[:n] = torch.from_numpy(np.ascontiguousarray(a[sel])).to(self.device)
            self._arrs.append(t)
        self._pid = torch.from_numpy(sel.astype(np.uint32).view(np.int32)).to(self.device)
        wsb = workspace_bytes(self.capacity, self.ncell)
        self._ws = torch.empty(wsb + 256, dtype=torch.uint8, device=self.device)
        ws_ptr = (self._ws.data_ptr() + 255) // 256 * 256
        self._stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        h = c_void_p()
        _check(lib().cuba_slab_init(ctypes.byref(h), _c3d(self.box), _c3i(self.ncell), self.capacity, n,
                                    *[c_void_p(t.data_ptr()) for t in self._arrs], c_void_p(self._pid.data_ptr()),
                                    float(w.n_test), int(w.seed), c_void_p(ws_ptr), wsb,
                                    c_void_p(self._stream.cuda_stream), self.layer_lo, self.layer_hi))
        self._h = h
        self.ncells = self.ncell[0] * self.ncell[1] * self.ncell[2]

    @property
    def n(self):
        """Particles in the local store (owned + ghosts); changes with every halo exchange."""
        return self.owned()[2]

    def owned(self):
        """(first slot, count) of the owned part of the store, particles in the store, capacity."""
        out = (c_int64 * 4)()
        _check(lib().cuba_slab_owned(self._h, out))
        return tuple(int(v) for v in out)

    def count(self, side):
        v = c_int64(0)
        _check(lib().cuba_slab_count(self._h, int(side), ctypes.byref(v)))
        return int(v.value)

    def pack(self, side):
        """(halo buffer as a uint8 CUDA tensor, particle count) of the owned boundary layer on `side`."""
        import torch
        cnt = self.count(side)
        nbytes = int(lib().cuba_slab_buffer_bytes(cnt, _c3i(self.ncell)))
        bufs = self.__dict__.setdefault("_halo", [None, None])      # one buffer per side, grown when needed
        if bufs[side] is None or bufs[side].numel() < nbytes + 16:
            bufs[side] = torch.empty(int(1.25 * nbytes) + 4096, dtype=torch.uint8, device=self.device)
        buf = bufs[side]
        off = (-buf.data_ptr()) % 16
        view = buf[off:off + nbytes]
        _check(lib().cuba_slab_pack(self._h, int(side), c_void_p(view.data_ptr()), nbytes))
        return view, cnt

    def unpack(self, lo, hi):
        """lo / hi: (buffer tensor, count) from the lower / upper neighbour, or None at a wall."""
        def ptr(b):
            if b is None:
                return None, 0
            t, cnt = b
            if t.data_ptr() % 16:
                t = t.clone()        # a received tensor that is not 16-byte aligned (torch allocations are)
            self._keep = getattr(self, "_keep", []) + [t]
            return c_void_p(t.data_ptr()), int(cnt)
        self._keep = []
        lp, lc = ptr(lo)
        hp, hc = ptr(hi)
        _check(lib().cuba_slab_unpack(self._h, lp, lc, hp, hc))

    def owned_particles(self):
        """(pid, x, y, z, px, py, pz) of the owned part as host numpy arrays, in array order."""
        first, cnt, _, _ = self.owned()
        return tuple(v[first:first + cnt] for v in self.particles())


def exchange_halos(dist, rank, world, send_lo, send_hi, device):
    """Halo exchange of one step over torch.distributed (NCCL on GPUs, gloo on CPU tensors).  send_lo / send_hi:
    (uint8 tensor, count) for the lower / upper neighbour or None.  Sizes first (two int64 per message), then
    the payloads, each as one batch of point-to-point operations.  Returns (from_lo, from_hi) like the inputs."""
    import torch
    lo, hi = neighbours(rank, world)
    plan = [(lo, send_lo), (hi, send_hi)]
    meta_out = [torch.tensor([b[0].numel(), b[1]] if b is not None else [0, 0], dtype=torch.int64, device=device)
                for _, b in plan]
    meta_in = [torch.zeros(2, dtype=torch.int64, device=device) for _ in plan]
    ops = []
    for k, (peer, _) in enumerate(plan):
        if peer is not None:
            ops.append(dist.P2POp(dist.isend, meta_out[k], peer))
            ops.append(dist.P2POp(dist.irecv, meta_in[k], peer))
    for r in (dist.batch_isend_irecv(ops) if ops else []):
        r.wait()
    recv = [None, None]
    ops = []
    for k, (peer, b) in enumerate(plan):
        if peer is not None:
            nbytes, cnt = int(meta_in[k][0]), int(meta_in[k][1])
            recv[k] = (torch.empty(nbytes, dtype=torch.uint8, device=device), cnt)
            ops.append(dist.P2POp(dist.isend, b[0], peer))
            ops.append(dist.P2POp(dist.irecv, recv[k][0], peer))
    for r in (dist.batch_isend_irecv(ops) if ops else []):
        r.wait()
    return recv[0], recv[1]


def slab_step(ctx: SlabRank, dist, rank, world, dt, sigma, eta_over_s=None):
    """One step of one rank of a torch.distributed job: step, pack, exchange, unpack.  eta_over_s: the per-cell
    cross section of cuba_step_local_sigma instead of sigma."""
    if eta_over_s is None:
        ctx.step(1, dt, sigma)
    else:
        ctx.step_local_sigma(1, dt, eta_over_s)
    lo, hi = neighbours(rank, world)
    send_lo = ctx.pack(0) if lo is not None else None
    send_hi = ctx.pack(1) if hi is not None else None
    ctx._stream.synchronize()                 # the buffers are complete before the communication library reads them
    from_lo, from_hi = exchange_halos(dist, rank, world, send_lo, send_hi, ctx.device)
    ctx.unpack(from_lo, from_hi)


class LocalSlabGroup:
    """All ranks of a decomposition in ONE process on one device, stepped one after the other: the test vehicle
    where fewer GPUs than ranks are at hand (the calls and their order are those of `slab_step`)."""

    def __init__(self, w, world, device="cuda:0", capacity=None, balance=False):
        self.world = int(world)
        nx = int(w.ncell[0])
        self.layers = slab_layers(nx, self.world, layer_weights(w.x, float(w.box[0]), nx) if balance else None)
        self.ranks = [SlabRank(w, lo, hi, device=device, capacity=capacity) for lo, hi in self.layers]

    def step(self, nsteps, dt, sigma, eta_over_s=None):
        for _ in range(int(nsteps)):
            for r in self.ranks:
                if eta_over_s is None:
                    r.step(1, dt, sigma)
                else:
                    r.step_local_sigma(1, dt, eta_over_s)
            sent = []
            for k, r in enumerate(self.ranks):
                lo, hi = neighbours(k, self.world)
                sent.append((r.pack(0) if lo is not None else None, r.pack(1) if hi is not None else None))
            for k, r in enumerate(self.ranks):
                lo, hi = neighbours(k, self.world)
                r.unpack(sent[lo][1] if lo is not None else None, sent[hi][0] if hi is not None else None)

    def particles(self):
        """The owned parts concatenated in rank order: the array order of the one-GPU store."""
        parts = [r.owned_particles() for r in self.ranks]
        return tuple(np.concatenate([p[k] for p in parts]) for k in range(7))

    def counters(self):
        cs = [r.counters() for r in self.ranks]
        return {k: sum(getattr(c, k) for c in cs) for k in ("pairs", "collisions", "rounds", "near_threshold")}

    def observables(self, nslab):
        res = [r.observables(nslab) for r in self.ranks]
        return sum(t for t, _ in res), sum(e for _, e in res)

    def close(self):
        for r in self.ranks:
            r.close()
