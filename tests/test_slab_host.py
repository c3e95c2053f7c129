"""Host-side logic of the x-slab decomposition on CPU: the partition into whole cell
layers, the initial selection of a rank's particles (owned layers + one ghost layer each side), and the halo
exchange schedule over torch.distributed with the gloo backend, world_size 3 (sizes first, then payloads; no
wrap-around at the walls).  The kernels' side of it is covered on the GPU (tests/test_gpu_slab.py)."""
import os
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def test_slab_layers_cover_the_grid_in_whole_layers():
    from paper_1208_0961_b200.slab import slab_layers, neighbours
    assert slab_layers(32, 1) == [(0, 32)]
    assert slab_layers(32, 2) == [(0, 16), (16, 32)]
    assert slab_layers(8, 3) == [(0, 3), (3, 6), (6, 8)]
    for nx in (8, 13, 64):
        for world in (1, 2, 3, 5, 8):
            parts = slab_layers(nx, world)
            assert parts[0][0] == 0 and parts[-1][1] == nx
            assert all(a[1] == b[0] for a, b in zip(parts, parts[1:]))
            sizes = [hi - lo for lo, hi in parts]
            assert min(sizes) >= 1 and max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        slab_layers(4, 5)
    # weighted cuts: a hot half that holds 8x the particles gets most of the ranks; every rank keeps a layer
    wts = np.array([8.0] * 4 + [1.0] * 4)
    assert slab_layers(8, 2, wts) == [(0, 2), (2, 8)]
    parts = slab_layers(8, 4, wts)
    assert parts[0][0] == 0 and parts[-1][1] == 8 and all(a[1] == b[0] and a[1] > a[0] for a, b in zip(parts, parts[1:]))
    assert max(wts[lo:hi].sum() for lo, hi in parts) <= 16.0
    assert slab_layers(3, 3, np.array([100.0, 0.0, 0.0])) == [(0, 1), (1, 2), (2, 3)]
    with pytest.raises(ValueError):
        slab_layers(8, 2, np.ones(7))
    assert neighbours(0, 1) == (None, None)
    assert neighbours(0, 3) == (None, 1) and neighbours(1, 3) == (0, 2) and neighbours(2, 3) == (1, None)


@pytest.fixture(scope="module", autouse=True)
def built_library():
    from paper_1208_0961_b200 import build
    build.build()          # layer_index goes through the C ABI (host function, no device needed)


def test_layer_index_comes_from_the_library_and_handles_the_faces():
    """the layer index that hands particles to ranks is the library's own S3 function
    (cuba_slab_layer_index), not a numpy copy of it.  Faces: a particle exactly on the face between
    layers k-1 and k belongs to k, one ulp below to k-1; x == L and beyond clamp to the last layer, x < 0 and NaN
    to the first (what cvt.rzi does on the device)."""
    from paper_1208_0961_b200.slab import layer_index, layer_weights
    import paper_1208_0961_b200 as c
    nx, Lx = 8, 8.0                                     # faces at the integers: x * 1.0 is exact
    faces = np.arange(0, nx + 1, dtype=np.float64)
    assert list(layer_index(faces, Lx, nx)) == [0, 1, 2, 3, 4, 5, 6, 7, 7]
    assert list(layer_index(np.nextafter(faces[1:], -np.inf), Lx, nx)) == [0, 1, 2, 3, 4, 5, 6, 7]
    assert list(layer_index(np.array([-0.0, -1e-300, -3.0, 1e300, np.inf, -np.inf, np.nan]), Lx, nx)) == [0, 0, 0, 7, 7, 0, 0]
    # a cell edge that is not a binary fraction: the index is trunc(fl(x * fl(1 / fl(L / nx)))) -- checked in exact
    # rational arithmetic on the three roundings, not by repeating the float expression
    from fractions import Fraction
    nx, Lx = 7, 3.3
    d = Lx / nx
    inv_d = 1.0 / d
    xs = np.concatenate([[k * d for k in range(nx + 1)], np.nextafter([k * d for k in range(1, nx + 1)], -np.inf),
                         np.nextafter([k * d for k in range(nx)], np.inf), np.random.default_rng(5).uniform(0, Lx, 200)])
    got = layer_index(xs, Lx, nx)
    for x, g in zip(xs, got):
        prod = Fraction(float(x)) * Fraction(inv_d)     # exact product of the two doubles
        fl = float(prod)                                # one correct rounding (Fraction -> float rounds to nearest even)
        assert g == min(max(int(fl), 0), nx - 1)
    assert layer_weights(xs, Lx, nx).sum() == xs.size
    assert c.lib().cuba_slab_layer_index(8.0, 0, 1, None, None) == -1          # CUBA_ERR_NULL
    one = np.zeros(1)
    out = np.zeros(1, dtype=np.int32)
    assert c.lib().cuba_slab_layer_index(8.0, 0, 1, one.ctypes.data, out.ctypes.data) == -2   # nx < 1
    assert c.lib().cuba_slab_layer_index(0.0, 4, 1, one.ctypes.data, out.ctypes.data) == -3   # box


def test_initial_selection_is_owned_plus_one_ghost_layer_in_global_order():
    import workloads
    from paper_1208_0961_b200.slab import initial_selection, slab_layers
    w = workloads.riemann_small()
    nx, Lx = w.ncell[0], w.box[0]
    inv_d = 1.0 / (Lx / nx)
    layer = np.minimum((w.x * inv_d).astype(np.int64), nx - 1)
    owned_total = 0
    for lo, hi in slab_layers(nx, 3):
        sel = initial_selection(w.x, Lx, nx, lo, hi)
        assert np.all(np.diff(sel) > 0)                                   # ascending global index: the stable order survives
        assert set(np.unique(layer[sel])) <= set(range(max(lo - 1, 0), min(hi + 1, nx)))
        assert np.count_nonzero((layer >= lo - 1) & (layer < hi + 1)) == sel.size     # nobody missing
        owned_total += np.count_nonzero((layer[sel] >= lo) & (layer[sel] < hi))
    assert owned_total == w.n                                             # every particle is owned exactly once
    # x == L lands in the last layer (A12), as in the library's S3
    x = np.array([0.0, Lx, Lx * (1 - 1e-16), 0.5 * Lx])
    assert list(initial_selection(x, Lx, nx, nx - 1, nx)) == [1, 2]


def _worker(rank, world, port, out_dir):
    import torch
    import torch.distributed as dist
    sys.path.insert(0, ROOT)
    from paper_1208_0961_b200.slab import exchange_halos, neighbours
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ok = True
    for step in range(3):
        lo, hi = neighbours(rank, world)
        # a payload that names its sender, its side and the step, of a size that differs per message
        def payload(side):
            nbytes = 16 + 52 * (10 * rank + 3 * side + step) + 4 * 5
            t = torch.full((nbytes,), (16 * rank + 4 * side + step) % 251, dtype=torch.uint8)
            return t, 10 * rank + 3 * side + step
        send_lo = payload(0) if lo is not None else None
        send_hi = payload(1) if hi is not None else None
        from_lo, from_hi = exchange_halos(dist, rank, world, send_lo, send_hi, torch.device("cpu"))
        if lo is None:
            ok &= from_lo is None
        else:       # what the lower neighbour packed for ITS upper side
            cnt = 10 * lo + 3 * 1 + step
            ok &= from_lo[1] == cnt and from_lo[0].numel() == 16 + 52 * cnt + 20 and bool((from_lo[0] == (16 * lo + 4 + step) % 251).all())
        if hi is None:
            ok &= from_hi is None
        else:
            cnt = 10 * hi + step
            ok &= from_hi[1] == cnt and from_hi[0].numel() == 16 + 52 * cnt + 20 and bool((from_hi[0] == (16 * hi + step) % 251).all())
    dist.barrier()
    dist.destroy_process_group()
    with open(os.path.join(out_dir, "ok%d" % rank), "w") as f:
        f.write("1" if ok else "0")


def test_exchange_halos_gloo_world3(tmp_path):
    import torch.multiprocessing as mp
    mp.spawn(_worker, args=(3, 29753, str(tmp_path)), nprocs=3, join=True)
    assert [open(str(tmp_path / ("ok%d" % r))).read() for r in range(3)] == ["1", "1", "1"]
