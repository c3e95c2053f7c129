"""x-slab decomposition on the GPU: several ranks' contexts stepped in one process on
one device (LocalSlabGroup: the calls of a multi-GPU job in the same order, buffers handed over directly).  The
owned parts concatenated in rank order must be the one-GPU store and the oracle's BIT FOR BIT -- array order,
pids, positions, momenta -- after every step; counters add up; observables add up to 1e-12."""
import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cuba():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1208_0961_b200 import build
    build.build()
    import paper_1208_0961_b200 as c
    return c


@pytest.fixture(scope="module")
def oracle_mod():
    import oracle
    oracle.build()
    return oracle


@pytest.mark.parametrize("world", [2, 3])
def test_slab_ranks_reproduce_the_one_gpu_run_bit_for_bit(cuba, oracle_mod, world):
    w = workloads.riemann_small(seed=51)
    one = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    grp = cuba.LocalSlabGroup(w, world)
    assert [hi - lo for lo, hi in grp.layers] == ([4, 4] if world == 2 else [3, 3, 2])
    for a, b in zip(grp.particles(), one.particles()):          # the initial binning (A19)
        assert np.array_equal(a, b)
    for k in (1, 2, 4):
        grp.step(k, w.dt, w.sigma)
        one.step(k, w.dt, w.sigma)
        o.step(k, w.dt, w.sigma)
        for a, b, c in zip(grp.particles(), one.particles(), o.particles()):
            assert np.array_equal(a, b) and np.array_equal(a, c)
    cg, c1, co = grp.counters(), one.counters(), o.counters()
    assert (cg["pairs"], cg["collisions"], cg["rounds"]) == (c1.pairs, c1.collisions, c1.rounds) == \
           (co["pairs"], co["collisions"], co["rounds"])
    gt, ge = grp.observables(w.nslab)
    ot, oe = o.observables(w.nslab)
    assert np.allclose(ge, oe, rtol=1e-12, atol=0) and np.allclose(gt, ot, rtol=1e-12, atol=1e-9)
    assert all(r.counters().device_flags == 0 for r in grp.ranks)
    assert sum(r.owned()[1] for r in grp.ranks) == w.n         # every particle is owned exactly once
    grp.close()


def test_slab_with_many_rounds_walls_and_thin_layers(cuba, oracle_mod):
    """Dense, strongly interacting gas (several rounds per cell), one-layer slabs at both walls, dt at 90 % of the
    cell edge (every second particle changes cell), 12 steps."""
    w = workloads.riemann(L=(6.0, 2.0, 2.0), ncell=(6, 2, 2), r_test=40.0, sigma_gev2=60.0, dt=0.9, seed=52)
    o = oracle_mod.Oracle.from_workload(w)
    grp = cuba.LocalSlabGroup(w, 6, capacity=w.n)
    for _ in range(3):
        grp.step(4, w.dt, w.sigma)
        o.step(4, w.dt, w.sigma)
        for a, c in zip(grp.particles(), o.particles()):
            assert np.array_equal(a, c)
    cg, co = grp.counters(), o.counters()
    assert (cg["pairs"], cg["collisions"], cg["rounds"]) == (co["pairs"], co["collisions"], co["rounds"])
    grp.close()


def test_slab_with_the_local_cross_section(cuba, oracle_mod):
    """cuba_step_local_sigma (constant eta/s, A24) in a slab context: the per-cell factor needs the cell's own
    particles only, so the decomposition stays exact; mixed with constant-sigma steps."""
    w = workloads.riemann_small(seed=55)
    o = oracle_mod.Oracle.from_workload(w)
    grp = cuba.LocalSlabGroup(w, 3)
    grp.step(3, w.dt, w.sigma, eta_over_s=0.1)
    o.step_etas(3, w.dt, 0.1)
    grp.step(1, w.dt, w.sigma)
    o.step(1, w.dt, w.sigma)
    grp.step(2, w.dt, w.sigma, eta_over_s=0.02)
    o.step_etas(2, w.dt, 0.02)
    for a, c in zip(grp.particles(), o.particles()):
        assert np.array_equal(a, c)
    cg, co = grp.counters(), o.counters()
    assert (cg["pairs"], cg["collisions"], cg["rounds"]) == (co["pairs"], co["collisions"], co["rounds"])
    with pytest.raises(cuba.CubaError):
        grp.ranks[0].step_adaptive(1, w.dt, w.sigma)
    grp.close()


def test_slab_tensor_observables_add_up(cuba, oracle_mod):
    """cuba_observables_lrf in a slab context covers the owned particles: the five tensor components per slab are
    sums over particles, so the ranks' results add up to the oracle's (1e-12); the Landau-matched quantities are
    not additive and are formed from the summed tensor by the caller."""
    w = workloads.riemann_small(seed=56)
    o = oracle_mod.Oracle.from_workload(w)
    grp = cuba.LocalSlabGroup(w, 2)
    grp.step(3, w.dt, w.sigma)
    o.step(3, w.dt, w.sigma)
    T = sum(r.observables_lrf(16)[0] for r in grp.ranks)
    To, _ = o.observables_lrf(16)
    assert np.allclose(T, To, rtol=1e-12, atol=1e-300)
    grp.close()


def test_slab_cuts_balanced_by_particles(cuba, oracle_mod):
    """The cuts follow the particles per layer (the hot half of the Riemann problem gets more ranks); same bits."""
    w = workloads.riemann_small(seed=54)
    o = oracle_mod.Oracle.from_workload(w)
    grp = cuba.LocalSlabGroup(w, 3, balance=True)
    assert grp.layers[0][1] < 3 and grp.layers[-1][1] == 8          # the first rank takes fewer (hot) layers than 8/3
    grp.step(5, w.dt, w.sigma)
    o.step(5, w.dt, w.sigma)
    for a, c in zip(grp.particles(), o.particles()):
        assert np.array_equal(a, c)
    grp.close()


def test_slab_argument_errors(cuba):
    w = workloads.riemann_small(seed=53)
    r = cuba.SlabRank(w, 2, 5)
    with pytest.raises(cuba.CubaError):
        r.step(2, w.dt, w.sigma)                 # a halo exchange belongs between two steps
    with pytest.raises(cuba.CubaError):
        r.unpack(None, None)                     # both neighbours exist
    r.step(1, w.dt, w.sigma)
    first, cnt, n, cap = r.owned()
    assert 0 < first and first + cnt < n <= cap
    assert r.count(0) > 0 and r.count(1) > 0
    # the schedules that are off in a slab context cannot be switched on afterwards (they would
    # collide the ghost cells / bin with a histogram of the owned cells only); switching them off is a no-op
    for opt, val in ((cuba.OPT_SLOTS, 2), (cuba.OPT_SLOTS, 1), (cuba.OPT_FUSE_HIST, 1), (cuba.OPT_GRAPH, 1)):
        with pytest.raises(cuba.CubaError) as e:
            r.set_option(opt, val)
        assert e.value.code == -3                # CUBA_ERR_VALUE
    for opt in (cuba.OPT_SLOTS, cuba.OPT_FUSE_HIST, cuba.OPT_GRAPH):
        r.set_option(opt, 0)
    before = r.counters()
    r.step(1, w.dt, w.sigma)                     # still the compact schedule on the owned cells
    assert r.counters().steps == before.steps + 1 and r.slot_stats() == (0, 0)
    with pytest.raises(cuba.CubaError):
        cuba.SlabRank(w, 5, 5)
    with pytest.raises(cuba.CubaError):
        cuba.SlabRank(w, 0, 4, capacity=10)
    r.close()


def test_slab_unpack_checks_the_buffer_header(cuba):
    """cuba_slab_unpack addresses the sections of a halo buffer with the count the caller passes on.
    The header {count, cells per layer} that cuba_slab_pack wrote is compared with it on the device: a buffer
    paired with the wrong count raises CUBA_ERR_HALO at the next synchronising call, the right pairing does not."""
    w = workloads.riemann_small(seed=54)
    lo, hi = cuba.SlabRank(w, 0, 4), cuba.SlabRank(w, 4, 8)
    for r in (lo, hi):
        r.step(1, w.dt, w.sigma)
    up, down = lo.pack(1), hi.pack(0)             # (buffer, count) for the upper / lower neighbour
    hi.unpack(up, None)
    assert hi.counters().device_flags == 0        # matching header: clean
    lo.unpack(None, (down[0], down[1] - 1))       # one particle short of what the header says
    assert lo.counters().device_flags & 32        # kFlagHalo, sticky
    with pytest.raises(cuba.CubaError) as e:
        lo.observables(4)                         # the next call that synchronises and reports device errors
    assert e.value.code == -11                    # CUBA_ERR_HALO
    assert "halo" in cuba.strerror(-11)
    lo.close()
    hi.close()



def test_layer_index_agrees_with_the_device_binning(cuba):
    """cuba_slab_layer_index (host) against S3 on the device (cuba_init's binning) for particles exactly on the
    layer faces, one ulp to either side, at the walls, and in between -- on a grid whose cell edge (3.3 / 7) is
    not a binary fraction: a particle goes to the ranks that the device will bin it for."""
    nx, ny, nz, Lx = 7, 2, 2, 3.3
    d = Lx / nx
    rng = np.random.default_rng(9)
    xs = np.concatenate([[k * d for k in range(nx + 1)], np.nextafter([k * d for k in range(1, nx + 1)], -np.inf),
                         np.nextafter([k * d for k in range(nx)], np.inf), [Lx, np.nextafter(Lx, 0.0), 0.0],
                         rng.uniform(0, Lx, 3000)])
    xs = np.minimum(xs, Lx)
    n = xs.size
    base = workloads.thermal_box(L=(Lx, 1.0, 1.0), ncell=(nx, ny, nz), count=n, seed=77)
    w = workloads.Workload("faces", (Lx, 1.0, 1.0), (nx, ny, nz), 2.0, 0.1, 0.05, 1, 77, 4,
                           xs.copy(), base.y, base.z, base.px, base.py, base.pz)
    g = cuba.Cuba.from_workload(w)
    pid = g.particles()[0]
    start = g.cell_start()
    cell_of_slot = np.repeat(np.arange(nx * ny * nz), np.diff(start.astype(np.int64)))
    dev_layer = np.empty(n, dtype=np.int64)
    dev_layer[pid] = cell_of_slot // (ny * nz)
    assert np.array_equal(cuba.layer_index(xs, Lx, nx), dev_layer)
    g.close()
