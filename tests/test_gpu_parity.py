"""GPU-vs-oracle parity, through the C ABI (`-m gpu`).  Protocol of SURVEY.md 8(c):
 (i) one traced step from an identical state: cell indices, pair lists, probabilities,
     uniforms and decisions equal bit for bit (decisions within 1e-12 of the threshold are
     counted -- there are none), state within 1e-12 relative (in fact identical bits);
 (ii) many steps: state still identical, energy-density profiles within 1e-12."""
import math
import os

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

REL = 1e-12   # north_star: "positions and momenta within 1e-12 relative in fp64"


@pytest.fixture(scope="module")
def cuba():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1208_0961_b200 as c
    c.lib()   # fails loudly if the extension was not built
    return c


def assert_state_equal(gpu_particles, ora_particles, exact=True):
    assert np.array_equal(gpu_particles[0], ora_particles[0]), "pid / array order differs"
    for name, g, o in zip("x y z px py pz".split(), gpu_particles[1:], ora_particles[1:]):
        scale = np.maximum(np.abs(o), 1e-300)
        assert np.all(np.abs(g - o) <= REL * scale), name
        if exact:
            assert np.array_equal(g, o), name + " bits differ"


def run_traced_step(cuba, oracle_mod, w):
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    assert_state_equal(g.particles(), o.particles())           # A19: init sort
    assert np.array_equal(g.cell_start(), o.cells()[1])
    o.set_trace(True)
    o.step(1, w.dt, w.sigma)
    tg = g.step_traced(w.dt, w.sigma)
    to = o.trace()
    # cell indices by pid
    ocell, ostart = o.cells()
    opid = o.particles()[0]
    ocell_of_pid = np.empty(w.n, dtype=np.uint32)
    ocell_of_pid[opid] = ocell
    assert np.array_equal(tg.cell_of_pid, ocell_of_pid)
    # pair lists in (cell, round, k) order, probabilities, uniforms, decisions
    assert tg.cell.shape[0] == to["cell"].shape[0]
    assert np.array_equal(tg.cell, to["cell"]) and np.array_equal(tg.round, to["round"])
    assert np.array_equal(tg.pid_a, to["pid_a"]) and np.array_equal(tg.pid_b, to["pid_b"])
    near = np.abs(to["u"] - to["P"]) <= 1e-12
    assert near.sum() == 0
    assert np.array_equal(tg.u, to["u"])
    assert np.array_equal(tg.P, to["P"])
    assert np.array_equal(tg.decided[~near], to["decided"][~near])
    # state
    assert_state_equal(g.particles(), o.particles())
    assert np.array_equal(g.cell_start(), ostart)
    gc, oc = g.counters(), o.counters()
    assert (gc.pairs, gc.collisions, gc.rounds, gc.near_threshold, gc.max_occupancy) == \
           (oc["pairs"], oc["collisions"], oc["rounds"], oc["near_threshold"], oc["max_occupancy"])
    assert gc.device_flags == 0
    return g, o


def test_one_step_bit_exact_thermal_box(cuba, oracle_mod):
    run_traced_step(cuba, oracle_mod, workloads.make(0))


def test_one_step_bit_exact_riemann_small(cuba, oracle_mod):
    g, o = run_traced_step(cuba, oracle_mod, workloads.riemann_small())
    # keep going untraced: 9 more steps, still identical
    w = workloads.riemann_small()
    g.step(9, w.dt, w.sigma)
    o.step(9, w.dt, w.sigma)
    assert_state_equal(g.particles(), o.particles())


def test_one_step_bit_exact_many_rounds_and_size_classes(cuba, oracle_mod):
    """sigma = 50 GeV^-2 on half-width cells (the configs[3] regime: R up to 3), with cells in
    the 32- and 512-thread classes (riemann_small covers the 128-thread one) and a ragged last tile."""
    w = workloads.riemann(L=(6.0, 3.0, 2.0), ncell=(12, 3, 2), r_test=90.0, sigma_gev2=50.0, dt=0.05, seed=13)
    assert w.n % 1024 != 0
    g, o = run_traced_step(cuba, oracle_mod, w)
    assert o.counters()["rounds"] > 1.5 * (np.diff(o.cells()[1].astype(np.int64)) >= 2).sum()
    assert o.counters()["max_occupancy"] > 512


@pytest.mark.parametrize("n", [128, 129, 256, 257, 512, 513, 896, 897, 1536, 1537, 2048, 2049, 4544, 4545])
def test_one_step_bit_exact_at_every_size_class_boundary(cuba, oracle_mod, n):
    """One cell holding exactly n particles (the capacities of the collision classes and one more,
    up to the global-memory overflow kernel) next to a small one; three rounds (A6)."""
    base_w = workloads.thermal_box(L=(2.0, 1.0, 1.0), ncell=(2, 1, 1), count=n + 77, seed=100 + n)
    rng = np.random.default_rng(n)
    pos = rng.uniform(0.3, 0.7, (3, n + 77))          # dt = 0.1 moves nobody across a face
    pos[0, n:] += 1.0
    r_test, dt = 2.0, 0.1
    cn = n if n % 2 else n - 1
    sigma = (2.5 / (2.0 * cn)) * r_test * 1.0 / dt    # pmax = 2.5 in the big cell: R = 3
    w = workloads.Workload("class_boundary_%d" % n, (2.0, 1.0, 1.0), (2, 1, 1), r_test, sigma, dt, 1, 100 + n, 2,
                           pos[0].copy(), pos[1].copy(), pos[2].copy(), base_w.px, base_w.py, base_w.pz)
    g, o = run_traced_step(cuba, oracle_mod, w)
    base = (sigma * dt) / (r_test * 1.0)
    assert o.counters()["max_occupancy"] == n
    assert o.counters()["rounds"] == 3 + max(1, math.ceil((2.0 * 77) * base))
    assert g.counters().overflow_cells == (1 if n > 4544 else 0)
    g.step(2, w.dt, w.sigma)                           # fused schedule on the same cells
    o.step(2, w.dt, w.sigma)
    assert_state_equal(g.particles(), o.particles())


def test_config0_full_run_matches_oracle(cuba, oracle_mod):
    """BASELINE.json:configs[0]: 50 steps, state bit-identical, totals and profile to 1e-12."""
    w = workloads.make(0)
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    tot0, _ = g.observables(8)
    g.step(w.steps, w.dt, w.sigma)
    o.step(w.steps, w.dt, w.sigma)
    assert_state_equal(g.particles(), o.particles())
    gt, ge = g.observables(8)
    ot, oe = o.observables(8)
    assert np.allclose(ge, oe, rtol=REL, atol=0)
    assert gt[0] == pytest.approx(ot[0], rel=REL)
    assert np.allclose(gt[1:], ot[1:], rtol=0, atol=REL * ot[0])
    assert abs(gt[0] - tot0[0]) / tot0[0] < 1e-10        # PAPER.md:66 energy conservation
    gc, oc = g.counters(), o.counters()
    assert (gc.steps, gc.pairs, gc.collisions, gc.rounds) == (50, oc["pairs"], oc["collisions"], oc["rounds"])
    assert gc.near_threshold == 0 and gc.device_flags == 0 and gc.overflow_cells == 0


def test_riemann_profiles_over_many_steps(cuba, oracle_mod):
    """Protocol (ii) at a size the oracle finishes in seconds: 64-slab profiles every 10 steps."""
    w = workloads.riemann(L=(16.0, 4.0, 4.0), ncell=(16, 4, 4), r_test=10.0, seed=14)
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    for _ in range(4):
        g.step(10, w.dt, w.sigma)
        o.step(10, w.dt, w.sigma)
        gt, ge = g.observables(64)
        ot, oe = o.observables(64)
        assert np.allclose(ge, oe, rtol=REL, atol=0)
        assert np.allclose(gt, ot, rtol=REL, atol=REL * ot[0])
    assert_state_equal(g.particles(), o.particles())


def assert_lrf_equal(got, ref):
    """Tensor sums differ from the oracle's only by summation order (1e-12);
    the Landau-matched quantities go through a square root of a difference: 1e-10."""
    (gT, gl), (oT, ol) = got, ref
    scale = np.maximum(oT[0], 1e-300)                   # T00 of the slab sets the scale of every component
    assert np.all(np.abs(gT - oT) <= REL * scale), "tensor components"
    assert np.all(np.abs(gl[0] - ol[0]) <= 1e-10 * scale), "e"
    assert np.all(np.abs(gl[1] - ol[1]) <= 1e-10), "v"
    assert np.all(np.abs(gl[2:] - ol[2:]) <= 1e-10 * scale), "P_L, P_T"


def test_observables_with_many_slabs_per_cell_layer(cuba, oracle_mod):
    """nslab > 2 nx: a layer of cells touches more than two slabs and the running sums live in per-lane
    shared-memory columns over a window of slabs (observe.cuh, WIDE), beyond the window the peel loop:
    energy density and tensor within 1e-12 / 1e-10 of the oracle, and bit-reproducible from call to call."""
    w = workloads.riemann(L=(16.0, 4.0, 4.0), ncell=(16, 4, 4), r_test=10.0, seed=16)
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    g.step(5, w.dt, w.sigma)
    o.step(5, w.dt, w.sigma)
    for nslab in (33, 40, 128, 500, 1024):          # windows of 4, 4, 9, 32 + peel, 32 + peel
        gt, ge = g.observables(nslab)
        ot, oe = o.observables(nslab)
        assert np.allclose(ge, oe, rtol=REL, atol=0) and np.allclose(gt, ot, rtol=REL, atol=1e-9)
        gt2, ge2 = g.observables(nslab)
        assert np.array_equal(ge, ge2) and np.array_equal(gt, gt2)
    for nslab in (33, 40, 100, 144, 256):           # tensor: windows of 4, 4, 8, 9 + peel, 9 + peel
        a = g.observables_lrf(nslab)
        assert_lrf_equal(a, o.observables_lrf(nslab))
        b = g.observables_lrf(nslab)
        assert np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1])


def test_lrf_observables_match_oracle(cuba, oracle_mod):
    """T00, T0x, Txx, Tyy, Tzz per slab and the Landau matching, on an evolving
    Riemann problem (a flow develops at the discontinuity), for several slab counts incl. the
    limits, slabs that cut through cell layers, and empty slabs."""
    w = workloads.riemann(L=(16.0, 4.0, 4.0), ncell=(16, 4, 4), r_test=10.0, seed=15)
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    for nslab in (1, 16, 37, 256):
        assert_lrf_equal(g.observables_lrf(nslab), o.observables_lrf(nslab))
    g.step(25, w.dt, w.sigma)
    o.step(25, w.dt, w.sigma)
    for nslab in (1, 16, 37, 256):
        assert_lrf_equal(g.observables_lrf(nslab), o.observables_lrf(nslab))
    T, lrf = g.observables_lrf(16)
    assert np.array_equal(np.isfinite(lrf), np.ones_like(lrf, dtype=bool))
    assert lrf[1].max() > 0.05                          # matter flows from the hot to the cold side
    assert np.allclose(T[0], g.observables(16)[1], rtol=REL)       # T00 is the energy density of Fig. 2
    # empty slabs: particles only in x < 4 of a 16 fm box
    w2 = workloads.thermal_box(L=(16.0, 2.0, 2.0), ncell=(16, 2, 2), count=5000, seed=8, r_test=3.0)
    w2.x[:] = 4.0 * np.random.default_rng(2).random(w2.n)
    g2, o2 = cuba.Cuba.from_workload(w2), oracle_mod.Oracle.from_workload(w2)
    T2, l2 = g2.observables_lrf(8)
    assert_lrf_equal((T2, l2), o2.observables_lrf(8))
    assert np.all(T2[:, 2:] == 0.0) and np.all(l2[:, 2:] == 0.0)
    for bad in (0, 257):
        with pytest.raises(cuba.CubaError):
            g.observables_lrf(bad)


def test_cuda_graph_replay_is_bit_identical(cuba, oracle_mod):
    """CUBA_OPT_GRAPH: on a capturable stream, small problems replay a two-step CUDA graph (step
    index in device memory).  Same bits as plain launches and as the oracle: even and odd step
    counts, a start from either copy of the store, a change of dt (re-capture), single steps in
    between, and the launch counter keeps counting the kernels a replay stands for."""
    import torch
    w = workloads.riemann(L=(6.0, 3.0, 2.0), ncell=(12, 3, 2), r_test=90.0, sigma_gev2=50.0, dt=0.05, seed=23)
    st = torch.cuda.Stream()
    graph = cuba.Cuba.from_workload(w, stream=st)
    plain = cuba.Cuba.from_workload(w, stream=torch.cuda.Stream())
    plain.set_option(2, 0)
    plain.set_option(3, 0)      # plain launches of the compact schedule: the graph is a capture of exactly those
    o = oracle_mod.Oracle.from_workload(w)
    l0 = cuba.launch_count()
    graph.step(8, w.dt, w.sigma)
    lg = cuba.launch_count() - l0
    l0 = cuba.launch_count()
    plain.step(8, w.dt, w.sigma)
    lp = cuba.launch_count() - l0
    assert lp - 8 <= lg <= lp + 8                        # + k_set_t / k_bump_t, - nothing hidden
    o.step(8, w.dt, w.sigma)
    for k, dt in ((7, w.dt), (1, w.dt), (5, 0.5 * w.dt), (6, 0.5 * w.dt), (3, w.dt), (9, w.dt)):
        graph.step(k, dt, w.sigma)
        plain.step(k, dt, w.sigma)
        o.step(k, dt, w.sigma)
        for a, b, c in zip(graph.particles(), plain.particles(), o.particles()):
            assert np.array_equal(a, b) and np.array_equal(a, c)
    cg, co = graph.counters(), o.counters()
    assert (cg.steps, cg.pairs, cg.collisions, cg.rounds) == (39, co["pairs"], co["collisions"], co["rounds"])
    assert cg.device_flags == 0
    # configs[0], the PR1 reference config, through the graph: 50 steps in one call
    w0 = workloads.make(0)
    g0 = cuba.Cuba.from_workload(w0, stream=st)
    o0 = oracle_mod.Oracle.from_workload(w0)
    g0.step(w0.steps, w0.dt, w0.sigma)
    o0.step(w0.steps, w0.dt, w0.sigma)
    assert_state_equal(g0.particles(), o0.particles())


def test_local_cross_section_matches_oracle(cuba, oracle_mod):
    """sigma per cell from the cell's n and <E> for constant eta/s.  The
    per-cell factor comes from an order-free fixed-point energy sum, so rounds, decisions and the
    state are the oracle's bit for bit: several size classes, many rounds (small eta/s), the
    overflow kernel, both schedules, mixed with constant-sigma steps."""
    cases = [(workloads.riemann_small(), 0.4), (workloads.riemann_small(), 0.02),
             (workloads.riemann(L=(6.0, 3.0, 2.0), ncell=(12, 3, 2), r_test=90.0, dt=0.05, seed=13), 0.1),
             (workloads.thermal_box(L=(1.0, 1.0, 1.0), ncell=(1, 1, 1), count=6000, seed=4, r_test=2000.0), 0.5)]
    for w, etas in cases:
        for fuse in (1, 0):
            g = cuba.Cuba.from_workload(w)
            g.set_option(1, fuse)
            o = oracle_mod.Oracle.from_workload(w)
            g.step_local_sigma(3, w.dt, etas)
            o.step_etas(3, w.dt, etas)
            assert_state_equal(g.particles(), o.particles())
            g.step(1, w.dt, w.sigma)
            o.step(1, w.dt, w.sigma)
            g.step_local_sigma(2, w.dt, etas)
            o.step_etas(2, w.dt, etas)
            assert_state_equal(g.particles(), o.particles())
            gc, oc = g.counters(), o.counters()
            assert (gc.pairs, gc.collisions, gc.rounds) == (oc["pairs"], oc["collisions"], oc["rounds"])
            assert gc.device_flags == 0 and oc["collisions"] > 0
    assert oracle_mod.Oracle.from_workload(cases[1][0]) is not None
    g = cuba.Cuba.from_workload(cases[0][0])
    with pytest.raises(cuba.CubaError):
        g.step_local_sigma(1, 0.1, 0.0)


def test_adaptive_time_step_matches_oracle(cuba, oracle_mod):
    """the dt sequence (a function of the integer occupancy of the fullest
    cell), the elapsed time and the state are the oracle's bit for bit -- where the rule binds
    (dense box: dt far below dt_max), where it does not (riemann_small), with fixed steps in
    between (the device-side occupancy must be fetched), with and without the fused histogram."""
    dense = workloads.thermal_box(L=(3.0, 3.0, 3.0), ncell=(3, 3, 3), count=6000, seed=5, r_test=1.2,
                                  sigma_gev2=10.0, dt=0.1)
    loose = workloads.riemann_small()
    loose.sigma *= 0.1                                  # the limit is ~0.75 fm/c: dt_max = 0.1 always wins
    for w, binds in ((dense, True), (workloads.riemann_small(), True), (loose, False)):
        for fuse in (1, 0):
            g = cuba.Cuba.from_workload(w)
            g.set_option(1, fuse)
            o = oracle_mod.Oracle.from_workload(w)
            ug, eg = g.step_adaptive(5, w.dt, w.sigma)
            uo, eo = o.step_adaptive(5, w.dt, w.sigma)
            assert np.array_equal(ug, uo) and eg == eo
            assert bool(np.all(ug < w.dt)) == binds and bool(np.all(ug == w.dt)) == (not binds)
            assert_state_equal(g.particles(), o.particles())
            g.step(2, 0.5 * ug[-1], w.sigma)            # fixed steps: no occupancy read-back
            o.step(2, 0.5 * uo[-1], w.sigma)
            ug, eg = g.step_adaptive(3, w.dt, w.sigma)
            uo, eo = o.step_adaptive(3, w.dt, w.sigma)
            assert np.array_equal(ug, uo) and eg == eo
            assert_state_equal(g.particles(), o.particles())
            gc, oc = g.counters(), o.counters()
            assert (gc.steps, gc.pairs, gc.collisions, gc.rounds) == (10, oc["pairs"], oc["collisions"], oc["rounds"])
            assert gc.device_flags == 0
    g = cuba.Cuba.from_workload(dense)
    with pytest.raises(cuba.CubaError):
        g.step_adaptive(1, -0.1, dense.sigma)
    with pytest.raises(cuba.CubaError):
        g.step_adaptive(1, 5.0, 0.0)                    # sigma = 0: dt = dt_max beyond the cell edge


def test_k_steps_equal_k_single_steps_and_determinism(cuba):
    w = workloads.riemann_small()
    a, b, c = (cuba.Cuba.from_workload(w) for _ in range(3))
    a.step(4, w.dt, w.sigma)
    for _ in range(4):
        b.step(1, w.dt, w.sigma)
    c.step(4, w.dt, w.sigma)
    pa, pb, pc = a.particles(), b.particles(), c.particles()
    for u, v, x in zip(pa, pb, pc):
        assert np.array_equal(u, v) and np.array_equal(u, x)
    assert np.array_equal(a.observables(16)[1], c.observables(16)[1])   # reductions are order-fixed


def test_fused_histogram_schedule_is_bit_identical(cuba, oracle_mod):
    """CUBA_OPT_FUSE_HIST: the collision kernel of step t writes the counting-sort histogram
    of step t+1.  Same results as the separate pass and as the oracle, also when dt changes
    between calls (the prepared histogram is for the wrong dt and must be discarded), after a
    traced step, and for all size classes incl. the overflow kernel and single-particle cells."""
    w = workloads.riemann(L=(6.0, 3.0, 2.0), ncell=(12, 3, 2), r_test=90.0, sigma_gev2=50.0, dt=0.05, seed=21)
    fused, plain = cuba.Cuba.from_workload(w), cuba.Cuba.from_workload(w)
    plain.set_option(1, 0)
    o = oracle_mod.Oracle.from_workload(w)
    schedule = [(3, w.dt), (1, w.dt), (2, 0.5 * w.dt), (1, w.dt), (2, w.dt)]
    for k, dt in schedule:
        fused.step(k, dt, w.sigma)
        plain.step(k, dt, w.sigma)
        o.step(k, dt, w.sigma)
        for a, b, c in zip(fused.particles(), plain.particles(), o.particles()):
            assert np.array_equal(a, b) and np.array_equal(a, c)
        assert np.array_equal(fused.cell_start(), o.cells()[1])
    fused.step_traced(w.dt, w.sigma)
    plain.step_traced(w.dt, w.sigma)
    fused.step(2, w.dt, w.sigma)
    plain.step(2, w.dt, w.sigma)
    o.step(3, w.dt, w.sigma)
    for a, b, c in zip(fused.particles(), plain.particles(), o.particles()):
        assert np.array_equal(a, b) and np.array_equal(a, c)
    cf, cp, co = fused.counters(), plain.counters(), o.counters()
    assert (cf.pairs, cf.collisions, cf.rounds) == (cp.pairs, cp.collisions, cp.rounds) == \
           (co["pairs"], co["collisions"], co["rounds"])
    assert cf.device_flags == 0 and cp.device_flags == 0
    with pytest.raises(cuba.CubaError):
        fused.set_option(99, 1)


def test_slotted_schedule_is_bit_identical(cuba, oracle_mod):
    """CUBA_OPT_SLOTS (opt-in): every cell owns a fixed region of 27 inbox segments and a call of n steps is
    n + 1 passes of one kernel per size class.  Same bits as the compact schedule and the oracle: calls of
    every length, a change of dt, a traced step in between, observables read from the packed result,
    counters; the library reports that the slotted store really ran and that nothing had to be redone."""
    w = workloads.riemann(L=(6.0, 3.0, 2.0), ncell=(12, 3, 2), r_test=90.0, sigma_gev2=50.0, dt=0.05, seed=31)
    slots, compact = cuba.Cuba.from_workload(w), cuba.Cuba.from_workload(w)
    slots.set_option(3, 2)
    compact.set_option(3, 0)
    o = oracle_mod.Oracle.from_workload(w)
    for k, dt in [(1, w.dt), (4, w.dt), (2, 0.5 * w.dt), (7, w.dt), (3, w.dt)]:
        slots.step(k, dt, w.sigma)
        compact.step(k, dt, w.sigma)
        o.step(k, dt, w.sigma)
        for a, b, c in zip(slots.particles(), compact.particles(), o.particles()):
            assert np.array_equal(a, b) and np.array_equal(a, c)
        assert np.array_equal(slots.cell_start(), o.cells()[1])
    slots.step_traced(w.dt, w.sigma)
    o.step(1, w.dt, w.sigma)
    slots.step(5, w.dt, w.sigma)
    o.step(5, w.dt, w.sigma)
    for a, c in zip(slots.particles(), o.particles()):
        assert np.array_equal(a, c)
    gt, ge = slots.observables(w.nslab)
    ot, oe = o.observables(w.nslab)
    assert np.allclose(ge, oe, rtol=1e-12, atol=0) and abs(gt[0] - ot[0]) <= 1e-12 * ot[0]
    cs, co = slots.counters(), o.counters()
    assert (cs.pairs, cs.collisions, cs.rounds) == (co["pairs"], co["collisions"], co["rounds"])
    assert cs.device_flags == 0
    runs, replays = slots.slot_stats()
    assert runs >= 6 and replays == 0
    assert compact.slot_stats() == (0, 0)
    # mode 1: only calls of at least 4 steps go to the slotted store
    m1 = cuba.Cuba.from_workload(w)
    m1.set_option(3, 1)
    m1.step(3, w.dt, w.sigma)
    assert m1.slot_stats()[0] == 0
    m1.step(4, w.dt, w.sigma)
    assert m1.slot_stats() == (1, 0)


def test_slotted_run_that_outgrows_a_segment_is_redone_on_the_compact_schedule(cuba, oracle_mod):
    """CUBA_OPT_SLOT_MARGIN: with the segment capacities cut to a fraction, a run overflows an inbox segment;
    that is detected at the next synchronising call and the run is redone on the compact schedule from the
    untouched copy it started from -- the result never depends on the capacities."""
    w = workloads.riemann(L=(6.0, 3.0, 2.0), ncell=(12, 3, 2), r_test=90.0, sigma_gev2=50.0, dt=0.05, seed=32)
    g = cuba.Cuba.from_workload(w)
    g.set_option(3, 2)
    g.set_option(4, 5)          # 5 % of the usual capacities
    o = oracle_mod.Oracle.from_workload(w)
    for k in (3, 6):
        g.step(k, w.dt, w.sigma)
        o.step(k, w.dt, w.sigma)
        for a, c in zip(g.particles(), o.particles()):
            assert np.array_equal(a, c)
    runs, replays = g.slot_stats()
    assert runs >= 1 and replays >= 1
    cg, co = g.counters(), o.counters()
    assert (cg.pairs, cg.collisions, cg.rounds) == (co["pairs"], co["collisions"], co["rounds"])
    assert cg.device_flags == 0


def test_slotted_store_grows_after_an_overflow(cuba, oracle_mod):
    """after a run outgrew a segment the next call must lay the slotted store out with a larger
    margin (x 1.5 per overflow) instead of reusing the undersized one and being redone on the compact schedule
    every time.  From 20 % of the usual capacities at most a handful of calls are redone; after that the
    slotted store runs without replays, and the state equals the oracle's all along."""
    w = workloads.riemann(L=(6.0, 3.0, 2.0), ncell=(12, 3, 2), r_test=90.0, sigma_gev2=50.0, dt=0.05, seed=33)
    g = cuba.Cuba.from_workload(w)
    g.set_option(3, 2)
    g.set_option(4, 20)
    o = oracle_mod.Oracle.from_workload(w)
    history = []
    for _ in range(9):
        g.step(3, w.dt, w.sigma)
        o.step(3, w.dt, w.sigma)
        history.append(g.slot_stats())
    for a, c in zip(g.particles(), o.particles()):
        assert np.array_equal(a, c)
    runs, replays = zip(*history)
    assert replays[0] >= 1, "20 % of the capacities was meant to overflow"
    assert replays[-1] == replays[-2] == replays[-3], history       # the last calls were not redone ...
    assert runs[-1] == runs[-3] + 2, history                        # ... and did run on the slotted store
    assert replays[-1] <= 6, history                                # 0.2 * 1.5^k passes 1 at k = 4
    assert g.counters().device_flags == 0


@pytest.mark.parametrize("n", [129, 513, 897, 1537, 2049, 4545])
def test_slotted_schedule_in_every_size_class(cuba, oracle_mod, n):
    """CUBA_OPT_SLOTS with one cell of n particles next to a thin one, particles spread over the whole cells so
    that movers cross the face both ways; two rounds in the big cell.  n = 4545 is beyond the largest
    shared-memory class: the slotted store declines (or flags) it and the compact schedule does the run."""
    base_w = workloads.thermal_box(L=(2.0, 1.0, 1.0), ncell=(2, 1, 1), count=n + 77, seed=200 + n)
    rng = np.random.default_rng(n)
    pos = rng.uniform(0.0, 1.0, (3, n + 77))
    pos[0, n:] += 1.0
    r_test, dt = 2.0, 0.1
    cn = n if n % 2 else n - 1
    sigma = (1.5 / (2.0 * cn)) * r_test * 1.0 / dt    # pmax = 1.5 in the big cell: R = 2
    w = workloads.Workload("slots_class_%d" % n, (2.0, 1.0, 1.0), (2, 1, 1), r_test, sigma, dt, 1, 200 + n, 2,
                           pos[0].copy(), pos[1].copy(), pos[2].copy(), base_w.px, base_w.py, base_w.pz)
    g = cuba.Cuba.from_workload(w)
    g.set_option(3, 2)
    o = oracle_mod.Oracle.from_workload(w)
    for k in (2, 3):
        g.step(k, w.dt, w.sigma)
        o.step(k, w.dt, w.sigma)
        assert_state_equal(g.particles(), o.particles())
    cg, co = g.counters(), o.counters()
    assert (cg.pairs, cg.collisions, cg.rounds) == (co["pairs"], co["collisions"], co["rounds"])
    assert cg.device_flags == 0
    runs, replays = g.slot_stats()
    assert (runs >= 1) if n < 4000 else (runs == 0 or replays == runs)


@pytest.mark.parametrize("case", ["single", "two", "one_cell_overflow", "flat_grid", "empty_cells"])
def test_edge_cases_match_oracle(cuba, oracle_mod, case):
    rng = np.random.default_rng(77)
    if case == "single":          # n = 1: nothing to pair
        w = workloads.thermal_box(L=(2.0, 2.0, 2.0), ncell=(2, 2, 2), count=1, seed=3)
    elif case == "two":
        w = workloads.thermal_box(L=(1.0, 1.0, 1.0), ncell=(1, 1, 1), count=2, seed=3, r_test=0.05)
    elif case == "one_cell_overflow":   # one cell far beyond the largest shared-memory class
        w = workloads.thermal_box(L=(1.0, 1.0, 1.0), ncell=(1, 1, 1), count=6000, seed=4, r_test=2000.0)
    elif case == "flat_grid":     # a single layer of cells in y and z, odd sizes
        w = workloads.thermal_box(L=(7.0, 1.0, 3.0), ncell=(7, 1, 3), count=3001, seed=5, r_test=1.0)
    else:                         # most cells empty: particles only in two far-apart blobs
        w = workloads.thermal_box(L=(16.0, 16.0, 16.0), ncell=(16, 16, 16), count=4000, seed=6, r_test=2.0)
        w.x[:] = np.where(rng.random(w.n) < 0.5, 0.5, 15.2) + 0.3 * rng.random(w.n)
        w.y[:] = 7.0 + 2.0 * rng.random(w.n)
        w.z[:] = 0.1 + 0.5 * rng.random(w.n)
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    for _ in range(3):
        g.step(1, w.dt, w.sigma)
        o.step(1, w.dt, w.sigma)
        assert_state_equal(g.particles(), o.particles())
        assert np.array_equal(g.cell_start(), o.cells()[1])
    gc, oc = g.counters(), o.counters()
    assert (gc.pairs, gc.collisions, gc.rounds) == (oc["pairs"], oc["collisions"], oc["rounds"])
    if case == "one_cell_overflow":
        assert gc.overflow_cells == 3 and oc["collisions"] > 100
    if case == "single":
        assert gc.pairs == 0


@pytest.mark.parametrize("case", ["cfl_limit", "thin_axis", "anisotropic_cells", "sparse_grid", "odd_box"])
def test_stress_geometries_match_oracle(cuba, oracle_mod, case):
    """Geometries that stress the direction logic of the fused histogram and the placement:
    dt just below the smallest cell edge (about half of the particles change cell,
    many through edges and corners, reflections combined with cell changes), an axis one cell
    thick (both faces of every cell are walls), strongly anisotropic cells, a grid where most
    cells hold no or one particle, and a box with non-representable cell edges."""
    if case == "cfl_limit":
        w = workloads.thermal_box(L=(6.0, 5.0, 4.0), ncell=(6, 5, 4), count=40000, seed=61, r_test=30.0, dt=0.999)
    elif case == "thin_axis":
        w = workloads.thermal_box(L=(9.0, 1.0, 7.0), ncell=(9, 1, 7), count=30000, seed=62, r_test=40.0, dt=0.6)
    elif case == "anisotropic_cells":
        w = workloads.thermal_box(L=(4.0, 8.0, 2.0), ncell=(16, 4, 2), count=50000, seed=63, r_test=60.0, dt=0.24)
    elif case == "sparse_grid":
        w = workloads.thermal_box(L=(20.0, 20.0, 20.0), ncell=(40, 40, 40), count=30000, seed=64, r_test=2.0, dt=0.3)
    else:
        w = workloads.thermal_box(L=(3.3, 2.7, 1.9), ncell=(7, 3, 5), count=20000, seed=65, r_test=25.0, dt=0.3)
    for fuse in (1, 0):
        g = cuba.Cuba.from_workload(w)
        g.set_option(1, fuse)
        o = oracle_mod.Oracle.from_workload(w)
        for _ in range(4):
            g.step(2, w.dt, w.sigma)
            o.step(2, w.dt, w.sigma)
            assert_state_equal(g.particles(), o.particles())
            assert np.array_equal(g.cell_start(), o.cells()[1])
        gc, oc = g.counters(), o.counters()
        assert (gc.pairs, gc.collisions, gc.rounds) == (oc["pairs"], oc["collisions"], oc["rounds"])
        assert gc.device_flags == 0
        if case != "sparse_grid":
            assert oc["collisions"] > 100


@pytest.mark.parametrize("seed", range(int(os.environ.get("CUBA_FUZZ_SEEDS", "16"))))
def test_random_configurations_match_oracle(cuba, oracle_mod, seed):
    """Seeded fuzz over the parameter space: box shape, grid, density, cross section (from no
    collisions to several rounds), dt up to the CFL limit, step mix (fixed / traced / adaptive /
    local cross section), schedule options, capturable or default stream.  State, cell table and
    counters must be the oracle's bit for bit after every call."""
    import torch
    rng = np.random.default_rng(1000 + seed)
    ncell = tuple(int(v) for v in rng.integers(1, 9, 3))
    d = rng.uniform(0.3, 1.5, 3)
    L = tuple(float(a * b) for a, b in zip(ncell, d))
    ncells = ncell[0] * ncell[1] * ncell[2]
    per_cell = float(rng.choice([0.3, 3.0, 30.0, 300.0]))
    count = int(min(60000, max(2, per_cell * ncells)))
    dmin = float(d.min())
    dt = float(rng.uniform(0.05, 0.98)) * dmin
    V = float(np.prod(d))
    target = float(rng.choice([0.0, 0.2, 0.9, 2.5, 6.0]))              # 2 cn base in a typical cell
    mean_n = max(count / ncells, 2.0)
    sigma_fm2 = 0.389379
    r_test = max(2.0 * mean_n * sigma_fm2 * dt / V / target, 1e-3) if target > 0 else 1.0
    w = workloads.thermal_box(L=L, ncell=ncell, count=count, seed=500 + seed, r_test=r_test,
                              sigma_gev2=(10.0 if target > 0 else 0.0), dt=dt, T=float(rng.uniform(0.1, 0.6)))
    stream = torch.cuda.Stream() if seed % 2 else None
    g = cuba.Cuba.from_workload(w, stream=stream)
    g.set_option(1, int(rng.integers(0, 2)))
    g.set_option(2, int(rng.integers(0, 2)))
    g.set_option(3, int(np.random.default_rng(7000 + seed).integers(0, 3)))      # compact or slotted schedule
    o = oracle_mod.Oracle.from_workload(w)

    def check():
        assert_state_equal(g.particles(), o.particles())
        assert np.array_equal(g.cell_start(), o.cells()[1])
        gc, oc = g.counters(), o.counters()
        assert (gc.steps, gc.pairs, gc.collisions, gc.rounds) == (oc["steps"], oc["pairs"], oc["collisions"], oc["rounds"])
        assert gc.device_flags == 0

    check()
    for _ in range(5):
        kind = rng.choice(["fixed", "fixed", "traced", "adaptive", "local", "halfdt"])
        k = int(rng.integers(1, 8))
        if kind == "fixed":
            g.step(k, w.dt, w.sigma); o.step(k, w.dt, w.sigma)
        elif kind == "halfdt":
            g.step(k, 0.5 * w.dt, w.sigma); o.step(k, 0.5 * w.dt, w.sigma)
        elif kind == "traced":
            g.step_traced(w.dt, w.sigma); o.step(1, w.dt, w.sigma)
        elif kind == "adaptive":
            ug, eg = g.step_adaptive(k, w.dt, w.sigma)
            uo, eo = o.step_adaptive(k, w.dt, w.sigma)
            assert np.array_equal(ug, uo) and eg == eo
        else:
            etas = float(rng.uniform(0.05, 1.0)) * max(1.0, 40.0 / mean_n)   # keeps the rounds below the cap of 64
            g.step_local_sigma(k, w.dt, etas); o.step_etas(k, w.dt, etas)
        check()
    gt, ge = g.observables(7)
    ot, oe = o.observables(7)
    assert np.allclose(ge, oe, rtol=REL, atol=0) and gt[0] == pytest.approx(ot[0], rel=REL)


def test_config1_full_run_profiles_match_oracle(cuba, oracle_mod):
    """Protocol (ii) of SURVEY 8(c) at BASELINE.json:configs[1] itself: 2.49M testparticles, 100
    steps, 64-slab energy-density profiles every 10 steps.  Under the arithmetic contract A2 the
    trajectories are identical, so the profiles agree to the summation-order tolerance and the
    final store bit for bit (the oracle needs about a minute of one host core)."""
    w = workloads.make(1)
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    tot0, _ = g.observables(64)
    for _ in range(10):
        g.step(10, w.dt, w.sigma)
        o.step(10, w.dt, w.sigma)
        gt, ge = g.observables(64)
        ot, oe = o.observables(64)
        assert np.allclose(ge, oe, rtol=REL, atol=0)
        assert gt[0] == pytest.approx(ot[0], rel=REL)
    assert_state_equal(g.particles(), o.particles())
    assert abs(gt[0] - tot0[0]) / tot0[0] < 1e-10
    T, lrf = g.observables_lrf(64)
    assert_lrf_equal((T, lrf), o.observables_lrf(64))
    # two waves leave the initial discontinuity at x = 16: the far ends are still
    # at their initial energy densities, the middle lies in between, matter flows to the right
    assert lrf[0, :8].mean() == pytest.approx(16.204, rel=0.02) and lrf[0, -8:].mean() == pytest.approx(1.0127, rel=0.03)
    assert 1.5 < lrf[0, 30:36].mean() < 15.0 and lrf[1, 28:40].max() > 0.2
    gc, oc = g.counters(), o.counters()
    assert (gc.steps, gc.pairs, gc.collisions) == (100, oc["pairs"], oc["collisions"])


def test_wall_reflection_on_device_preserves_energy_bits(cuba):
    """PAPER.md:44 with sigma = 0: after many wall hits every |p| is bit-identical."""
    import torch
    w = workloads.thermal_box(L=(2.0, 2.0, 2.0), ncell=(2, 2, 2), count=50000, seed=9)
    g = cuba.Cuba.from_workload(w)
    E0 = np.sqrt((w.px * w.px + w.py * w.py) + w.pz * w.pz)
    g.step(30, 0.9, 0.0)
    pid, x, y, z, px, py, pz = g.particles()
    E1 = np.sqrt((px * px + py * py) + pz * pz)
    assert np.array_equal(E1, E0[pid])
    for a, L in zip((x, y, z), w.box):
        assert a.min() >= 0.0 and a.max() <= L
    assert (np.sign(px) != np.sign(w.px[pid])).sum() > 1000


def test_errors_are_codes_not_crashes(cuba):
    import torch
    w = workloads.thermal_box(L=(2.0, 2.0, 2.0), ncell=(2, 2, 2), count=500, seed=1)
    g = cuba.Cuba.from_workload(w)
    with pytest.raises(cuba.CubaError) as e:
        g.step(1, 1.0, 0.1)                      # dt == cell edge
    assert e.value.code == -7
    with pytest.raises(cuba.CubaError) as e:
        g.step(1, -0.1, 0.1)
    assert e.value.code == -3
    with pytest.raises(cuba.CubaError) as e:
        g.observables(0)
    assert e.value.code == -2
    g.step(1, 0.1, 1e9)                          # needs > 64 rounds: reported at the next sync
    with pytest.raises(cuba.CubaError) as e:
        g.observables(4)
    assert e.value.code == -9
    bad = [torch.from_numpy(a.copy()).cuda() for a in w.arrays()]
    bad[0][7] = 2.5                              # outside the box
    with pytest.raises(cuba.CubaError) as e:
        cuba.Cuba(w.box, w.ncell, *bad, 1.0, 1)
    assert e.value.code == -6
    bad = [torch.from_numpy(a.copy()).cuda() for a in w.arrays()]
    bad[3][7] = bad[4][7] = bad[5][7] = 0.0      # p = 0
    with pytest.raises(cuba.CubaError) as e:
        cuba.Cuba(w.box, w.ncell, *bad, 1.0, 1)
    assert e.value.code == -6


def test_run_host_end_to_end_matches_oracle(cuba, oracle_mod):
    w = workloads.riemann_small()
    host = [a.copy() for a in w.arrays()]
    tot, ed, pid = cuba.run_host(w.box, w.ncell, *host, w.n_test, w.seed, 5, w.dt, w.sigma, 16, download=True)
    o = oracle_mod.Oracle.from_workload(w)
    o.step(5, w.dt, w.sigma)
    ot, oe = o.observables(16)
    assert np.allclose(ed, oe, rtol=REL, atol=0) and tot[0] == pytest.approx(ot[0], rel=REL)
    assert_state_equal((pid, *host), o.particles())
    assert cuba.launch_count() > 0


def test_short_trace_capacity_completes_the_step(cuba, oracle_mod):
    """cuba_step_traced with too little room reports CUBA_ERR_TRACE but still takes the step (untraced):
    the context is never left streamed-but-not-collided, and a retry traces the next step."""
    w = workloads.riemann_small()
    g = cuba.Cuba.from_workload(w)
    o = oracle_mod.Oracle.from_workload(w)
    with pytest.raises(cuba.CubaError) as e:
        g.step_traced(w.dt, w.sigma, pair_capacity=5)
    assert e.value.code == -10
    o.step(1, w.dt, w.sigma)
    assert_state_equal(g.particles(), o.particles())
    assert g.counters().steps == 1
    o.set_trace(True)
    o.step(1, w.dt, w.sigma)
    tg = g.step_traced(w.dt, w.sigma)
    to = o.trace()
    assert np.array_equal(tg.pid_a, to["pid_a"]) and np.array_equal(tg.decided, to["decided"])
    g.step(3, w.dt, w.sigma)
    o.step(3, w.dt, w.sigma)
    assert_state_equal(g.particles(), o.particles())


def test_fp64_probe_reports_a_plausible_peak(cuba):
    """cuba_probe_fp64 (the measured fp64 leg of the roofline): a B200 does tens of TFLOP/s in fp64; argument errors."""
    rate = cuba.probe_fp64(repeats=2)
    assert 2e12 < rate < 4e13                       # thread-level DFMA per second (x 2 = FLOP/s)
    with pytest.raises(cuba.CubaError):
        cuba.probe_fp64(repeats=0)

