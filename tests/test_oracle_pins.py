"""Pins for the CPU oracle: each test ties one part of oracle/cuba_oracle.c to something
other than itself -- a library routine, a closed form, an invariant, brute force on tiny
inputs -- chosen so that a dropped term, a wrong sign or index, or a transposed operand
fails at least one of them.  All CPU (`-m "not gpu"`).  P-numbers refer to SURVEY.md 8(c).
"""
import ctypes
import math
import os
import subprocess
from fractions import Fraction

import numpy as np
import pytest
from scipy import stats

import workloads

HERE = os.path.dirname(os.path.abspath(__file__))


def golden():
    out = {}
    with open(os.path.join(HERE, "golden", "paper_closed_forms.txt")) as f:
        for line in f:
            line = line.split("#")[0].strip()
            if line:
                k, v = line.split()
                out[k] = float(v)
    return out


# ---------------------------------------------------------------------------- P1: Philox

@pytest.fixture(scope="session")
def curand_ref(tmp_path_factory):
    """cuRAND's own Philox4x32-10 block function, compiled for the host from the toolkit
    header (library routine; tests/helpers/curand_philox_ref.cu)."""
    out = str(tmp_path_factory.mktemp("curand") / "libcurand_ref.so")
    src = os.path.join(HERE, "helpers", "curand_philox_ref.cu")
    subprocess.check_call(["nvcc", "-O1", "-shared", "-Xcompiler", "-fPIC",
                           "-Wno-deprecated-gpu-targets", "-o", out, src])
    L = ctypes.CDLL(out)

    def f(ctr, key):
        c = np.asarray(ctr, dtype=np.uint32).copy()
        k = np.asarray(key, dtype=np.uint32).copy()
        o = np.zeros(4, dtype=np.uint32)
        L.curand_ref_philox4x32_10(c.ctypes.data_as(ctypes.c_void_p), k.ctypes.data_as(ctypes.c_void_p),
                                   o.ctypes.data_as(ctypes.c_void_p))
        return o
    return f


def test_philox_matches_curand_block_function(oracle_mod, curand_ref):
    rng = np.random.default_rng(123)
    cases = [([0, 0, 0, 0], [0, 0]), ([0xFFFFFFFF] * 4, [0xFFFFFFFF] * 2),
             ([1, 0, 0, 0], [0, 0]), ([0, 1, 0, 0], [0, 0]), ([0, 0, 1, 0], [0, 0]),
             ([0, 0, 0, 1], [0, 0]), ([0, 0, 0, 0], [1, 0]), ([0, 0, 0, 0], [0, 1])]
    for _ in range(500):
        cases.append((rng.integers(0, 2 ** 32, 4, dtype=np.uint64), rng.integers(0, 2 ** 32, 2, dtype=np.uint64)))
    seen = set()
    for ctr, key in cases:
        got = oracle_mod.philox4x32_10(ctr, key)
        ref = curand_ref(ctr, key)
        assert np.array_equal(got, ref), (ctr, key)
        seen.add(tuple(got))
    assert len(seen) == len(cases)  # every single-word change moved the output


def test_philox_matches_curand_host_generator(oracle_mod):
    """The cuRAND HOST generator CURAND_RNG_PHILOX4_32_10 (runs on the CPU): with seed s and
    offset 4g it emits Philox(ctr = (g >> 16, 0, g & 0xffff, 0), key = (s_lo, s_hi)) --
    mapping found empirically, as SURVEY.md P1 asks."""
    try:
        lib = ctypes.CDLL("libcurand.so.10")
    except OSError:
        lib = ctypes.CDLL("/usr/local/cuda/lib64/libcurand.so.10")

    def curand(seed, n, offset):
        gen = ctypes.c_void_p()
        assert lib.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0
        assert lib.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
        assert lib.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(offset)) == 0
        out = np.zeros(n, dtype=np.uint32)
        assert lib.curandGenerate(gen, out.ctypes.data_as(ctypes.c_void_p), ctypes.c_size_t(n)) == 0
        lib.curandDestroyGenerator(gen)
        return out.reshape(-1, 4)

    for seed in (1, 0x0123456789ABCDEF, 2 ** 64 - 1):
        key = [seed & 0xFFFFFFFF, seed >> 32]
        for g0 in (0, 65535, 65536 * 7 + 3):
            blocks = curand(seed, 16, 4 * g0)
            for j, blk in enumerate(blocks):
                g = g0 + j
                assert np.array_equal(blk, oracle_mod.philox4x32_10([g >> 16, 0, g & 0xFFFF, 0], key))


def test_u53_is_the_exact_53_bit_fraction(oracle_mod):
    assert oracle_mod.u53(0, 0) == 0.0
    assert oracle_mod.u53(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    rng = np.random.default_rng(5)
    for w0, w1 in rng.integers(0, 2 ** 32, (200, 2)):
        exact = Fraction(((int(w0) >> 5) << 26) | (int(w1) >> 6), 2 ** 53)
        assert Fraction(oracle_mod.u53(w0, w1)) == exact


# ------------------------------------------------------------- P2: streaming and the walls

def test_streaming_moves_at_light_speed_along_p(oracle_mod):
    """Eq. 2 with c = 1 and E = |p|: displacement = dt * p/|p|."""
    rng = np.random.default_rng(7)
    n = 1000
    pos = rng.uniform(10, 20, (3, n))
    mom = rng.normal(size=(3, n)) * rng.uniform(0.01, 5.0, n)
    (x, y, z, px, py, pz), wall = oracle_mod.stream_reflect(*pos, *mom, 0.1, [30.0, 30.0, 30.0])
    d = np.array([x, y, z]) - pos
    assert np.allclose(np.linalg.norm(d, axis=0), 0.1, rtol=0, atol=1e-14)
    unit = mom / np.linalg.norm(mom, axis=0)
    assert np.allclose(d / 0.1, unit, rtol=0, atol=1e-13)
    assert np.array_equal(np.array([px, py, pz]), mom) and np.all(wall == 0)


def test_each_of_the_six_walls_mirrors(oracle_mod):
    """one particle aimed at each wall comes back mirrored, |p| bit-identical."""
    L = [4.0, 6.0, 8.0]
    dt = 0.5
    for axis in range(3):
        for side in (0, 1):
            pos = np.array([2.0, 3.0, 4.0])
            mom = np.array([0.3, -0.2, 0.1])
            sign = -1.0 if side == 0 else 1.0
            mom[axis] = sign * 2.0
            pos[axis] = 0.1 if side == 0 else L[axis] - 0.1
            (x, y, z, px, py, pz), wall = oracle_mod.stream_reflect(
                *[np.array([v]) for v in pos], *[np.array([v]) for v in mom], dt, L)
            new_pos = np.array([x[0], y[0], z[0]])
            new_mom = np.array([px[0], py[0], pz[0]])
            free = pos + dt * mom / np.linalg.norm(mom)
            wallpos = 0.0 if side == 0 else L[axis]
            expect = free.copy()
            expect[axis] = 2 * wallpos - free[axis]      # mirror image in the wall plane
            assert np.allclose(new_pos, expect, atol=1e-14)
            assert 0.0 <= new_pos[axis] <= L[axis]
            flipped = mom.copy()
            flipped[axis] = -flipped[axis]
            assert np.array_equal(new_mom, flipped)      # bits, not just values
            assert wall[axis] == -2.0 * mom[axis] and np.all(np.delete(wall, axis) == 0)


def test_reflection_preserves_energy_bits_and_keeps_positions_inside(oracle_mod):
    w = workloads.thermal_box(L=(2.0, 2.0, 2.0), ncell=(2, 2, 2), count=20000, seed=9)
    E0 = np.sqrt((w.px * w.px + w.py * w.py) + w.pz * w.pz)
    (x, y, z, px, py, pz), wall = oracle_mod.stream_reflect(*w.arrays(), 0.9, w.box)
    E1 = np.sqrt((px * px + py * py) + pz * pz)
    assert np.array_equal(E0, E1)
    for a, L in zip((x, y, z), w.box):
        assert a.min() >= 0.0 and a.max() <= L
    assert (px != w.px).sum() > 1000  # the walls were actually hit
    # impulse bookkeeping: change of total momentum == what the walls handed over
    assert np.allclose([px.sum() - w.px.sum(), py.sum() - w.py.sum(), pz.sum() - w.pz.sum()], wall, atol=1e-9)


# ------------------------------------------------------------------- S3 / P11: cells, sort

def test_cell_index_layout_and_boundaries(oracle_mod):
    box, ncell = [4.0, 3.0, 10.0], [4, 6, 5]      # d = 1, 0.5, 2 ; x slowest
    pts = np.array([
        [0.0, 0.0, 0.0], [-0.0, 0.0, 0.0], [3.999, 2.999, 9.999], [4.0, 3.0, 10.0],
        [1.0, 0.0, 0.0], [0.0, 0.5, 0.0], [0.0, 0.0, 2.0], [0.999999, 0.49999, 1.99999],
        [2.5, 1.75, 7.0]])
    c = oracle_mod.cell_index(pts[:, 0], pts[:, 1], pts[:, 2], box, ncell)
    ny, nz = 6, 5
    expect = [0, 0, (3 * ny + 5) * nz + 4, (3 * ny + 5) * nz + 4,
              (1 * ny + 0) * nz + 0, (0 * ny + 1) * nz + 0, 1, 0,
              (2 * ny + 3) * nz + 3]
    assert list(c) == expect


def test_cell_index_against_floor_division(oracle_mod):
    rng = np.random.default_rng(3)
    box, ncell = [32.0, 16.0, 8.0], [32, 8, 16]
    p = rng.random((3, 5000)) * np.array(box)[:, None]
    c = oracle_mod.cell_index(*p, box, ncell)
    d = np.array(box) / np.array(ncell)
    ii = np.minimum(np.floor(p / d[:, None]).astype(np.int64), np.array(ncell)[:, None] - 1)
    assert np.array_equal(c, (ii[0] * ncell[1] + ii[1]) * ncell[2] + ii[2])


def test_counting_sort_is_the_stable_sort(oracle_mod):
    """P11 brute force: numpy's stable argsort is the definition of 'stable'."""
    rng = np.random.default_rng(4)
    for n, ncells in ((1, 1), (17, 5), (5000, 64), (5000, 20000)):
        cell = rng.integers(0, ncells, n).astype(np.uint32)
        start, perm = oracle_mod.counting_sort(cell, ncells)
        assert np.array_equal(perm, np.argsort(cell, kind="stable"))
        assert np.array_equal(start, np.searchsorted(np.sort(cell), np.arange(ncells + 1), side="left"))


def test_init_and_step_keep_a_stable_cell_sorted_permutation(oracle_mod):
    w = workloads.riemann_small()
    o = oracle_mod.Oracle.from_workload(w)
    pid, x, y, z, px, py, pz = o.particles()
    cell, start = o.cells()
    assert np.array_equal(np.sort(pid), np.arange(w.n))          # a permutation
    assert np.all(np.diff(cell.astype(np.int64)) >= 0)           # cells non-decreasing
    for c in np.unique(cell)[:50]:                               # A19: init order = original index
        seg = pid[start[c]:start[c + 1]]
        assert np.all(np.diff(seg.astype(np.int64)) > 0)
    assert np.array_equal(x, w.x[pid]) and np.array_equal(pz, w.pz[pid])
    prev_slot_of_pid = np.empty(w.n, dtype=np.int64)
    prev_slot_of_pid[pid] = np.arange(w.n)
    o.step(1, w.dt, 0.0)
    pid2, x2, *_ = o.particles()
    cell2, start2 = o.cells()
    assert np.array_equal(np.sort(pid2), np.arange(w.n))
    assert np.array_equal(cell2, oracle_mod.cell_index(*o.particles()[1:4], w.box, w.ncell))
    assert np.all(np.diff(cell2.astype(np.int64)) >= 0)
    assert np.array_equal(start2, np.searchsorted(cell2, np.arange(o.ncells + 1), side="left"))
    prev = prev_slot_of_pid[pid2]
    same = cell2[1:] == cell2[:-1]
    assert np.all(prev[1:][same] > prev[:-1][same])              # A8: ascending previous index


# -------------------------------------------------------------- P3: collision kinematics

def lorentz_boost_matrix(beta):
    """Textbook 4x4 boost taking rest-frame components to the frame where the rest frame
    moves with velocity beta."""
    b2 = float(beta @ beta)
    g = 1.0 / math.sqrt(1.0 - b2)
    Lm = np.eye(4)
    Lm[0, 0] = g
    Lm[0, 1:] = g * beta
    Lm[1:, 0] = g * beta
    Lm[1:, 1:] += (g - 1.0) * np.outer(beta, beta) / b2
    return Lm


def thermal_pairs(rng, n, T=0.4):
    def mom():
        mag = rng.gamma(3.0, T, n)
        v = rng.normal(size=(n, 3))
        return mag[:, None] * v / np.linalg.norm(v, axis=1)[:, None]
    return mom(), mom()


def test_pair_kinematics_is_mandelstam_s_and_vrel(oracle_mod):
    """s = (p1+p2)^2, v_rel = s/(2 E1 E2) (= 1 - cos theta for massless)."""
    rng = np.random.default_rng(11)
    A, B = thermal_pairs(rng, 2000)
    for pa, pb in zip(A, B):
        Ea, Eb, s, vrel = oracle_mod.pair_kinematics(pa, pb)
        Et, P = np.linalg.norm(pa) + np.linalg.norm(pb), pa + pb
        assert Ea == pytest.approx(np.linalg.norm(pa), rel=1e-15)
        assert Eb == pytest.approx(np.linalg.norm(pb), rel=1e-15)
        assert s == pytest.approx(Et * Et - P @ P, rel=1e-9, abs=1e-13)
        cos = (pa @ pb) / (np.linalg.norm(pa) * np.linalg.norm(pb))
        assert vrel == pytest.approx(1.0 - cos, rel=1e-9, abs=1e-13)
    # collinear pair: s = 0 exactly, never negative (A9)
    Ea, Eb, s, vrel = oracle_mod.pair_kinematics([0.3, 0.4, 1.2], [0.6, 0.8, 2.4])
    assert s >= 0.0 and s < 1e-28 and vrel >= 0.0
    # a swap of the two particles must not change s
    s1 = oracle_mod.pair_kinematics(A[0], B[0])[2]
    s2 = oracle_mod.pair_kinematics(B[0], A[0])[2]
    assert s1 == pytest.approx(s2, rel=1e-15)


def test_scatter_conserves_four_momentum_and_matches_matrix_boost(oracle_mod):
    """P3 (north_star: per-collision four-momentum conservation to 1e-12 relative); the
    closed form of A10 against the explicit Lorentz-matrix boost of (sqrt(s)/2)(1, +-n)."""
    rng = np.random.default_rng(12)
    A, B = thermal_pairs(rng, 3000)
    # add near-collinear pairs (tiny v_rel)
    for k in range(200):
        B[k] = A[k] * rng.uniform(0.2, 3.0) + rng.normal(size=3) * 10.0 ** rng.uniform(-7, -2)
    worst = 0.0
    for pa, pb in zip(A, B):
        Ea, Eb, s, vrel = oracle_mod.pair_kinematics(pa, pb)
        v = rng.normal(size=3)
        nhat = v / np.linalg.norm(v)
        qa, qb = oracle_mod.scatter(pa, pb, Ea, Eb, s, nhat)
        Et = Ea + Eb
        dP = np.abs((qa + qb) - (pa + pb)).max() / Et
        dE = abs((np.linalg.norm(qa) + np.linalg.norm(qb)) - Et) / Et
        worst = max(worst, dP, dE)
        assert dP <= 1e-12 and dE <= 1e-12
        s_new = oracle_mod.pair_kinematics(qa, qb)[2]
        assert s_new == pytest.approx(s, rel=1e-7, abs=1e-18)
        if vrel > 1e-6:                                   # matrix boost loses digits as gamma -> inf
            Lm = lorentz_boost_matrix((pa + pb) / Et)
            rs = math.sqrt(s)
            ref_a = Lm @ np.concatenate([[rs / 2], rs / 2 * nhat])
            ref_b = Lm @ np.concatenate([[rs / 2], -rs / 2 * nhat])
            assert np.allclose(qa, ref_a[1:], rtol=0, atol=1e-9 * Et / max(vrel, 1e-3) * 1e-3)
            assert np.allclose(qb, ref_b[1:], rtol=0, atol=1e-9 * Et / max(vrel, 1e-3) * 1e-3)
    assert worst < 5e-15


def test_scatter_in_the_cm_frame_is_back_to_back_along_n(oracle_mod):
    """Special case with P = 0 (already the CM frame): p_a' = E n, p_b' = -E n."""
    pa, pb = np.array([0.0, 0.0, 0.7]), np.array([0.0, 0.0, -0.7])
    Ea, Eb, s, vrel = oracle_mod.pair_kinematics(pa, pb)
    assert s == pytest.approx(4 * 0.49) and vrel == pytest.approx(2.0)
    nhat = np.array([0.6, 0.0, 0.8])
    qa, qb = oracle_mod.scatter(pa, pb, Ea, Eb, s, nhat)
    assert np.allclose(qa, 0.7 * nhat, atol=1e-15) and np.allclose(qb, -0.7 * nhat, atol=1e-15)


# --------------------------------------------------------------------- P6: isotropy

def test_direction_is_a_unit_vector_uniform_on_the_sphere(oracle_mod):
    n = 40000
    dirs = np.empty((n, 3))
    attempts = 0
    for i in range(n):
        dirs[i], m = oracle_mod.direction(99, i, 3, 0)
        attempts += m
    assert np.abs(np.linalg.norm(dirs, axis=1) - 1.0).max() < 1e-15 * 8
    assert stats.kstest(dirs[:, 2], stats.uniform(-1, 2).cdf).pvalue > 1e-3
    assert stats.kstest(dirs[:, 0], stats.uniform(-1, 2).cdf).pvalue > 1e-3
    assert stats.kstest(np.arctan2(dirs[:, 1], dirs[:, 0]), stats.uniform(-math.pi, 2 * math.pi).cdf).pvalue > 1e-3
    # Marsaglia's rejection accepts with probability pi/4
    assert n / attempts == pytest.approx(math.pi / 4, abs=4 * math.sqrt(0.785 * 0.215 / attempts))


# ----------------------------------------------------------------- P12: shuffle and pairs

def matching_id(order):
    pairs = sorted(tuple(sorted((int(order[2 * k]), int(order[2 * k + 1])))) for k in range(len(order) // 2))
    return tuple(pairs)


@pytest.mark.parametrize("n,count", [(4, 3), (5, 15), (6, 15)])
def test_pairings_are_uniform_over_perfect_matchings(oracle_mod, n, count):
    """P12: on tiny cells the pairing (order[2k], order[2k+1]) is uniform over the (n-1)!!
    perfect matchings (n even) or the n (n-2)!! matchings that leave one out (n odd)."""
    pids = np.array([17, 3, 250, 9, 1000003, 42][:n], dtype=np.uint32)
    hist = {}
    trials = 6000
    for t in range(trials):
        order = oracle_mod.shuffle_order(1234, t, t % 8, pids)   # all four words of both Philox calls
        assert sorted(order) == sorted(pids)
        hist[matching_id(order)] = hist.get(matching_id(order), 0) + 1
    assert len(hist) == count
    chi2 = sum((v - trials / count) ** 2 / (trials / count) for v in hist.values())
    assert stats.chi2.sf(chi2, count - 1) > 1e-3



def _keys_from_philox(oracle_mod, seed, t, rho, pids):
    """A7 assembled in the test from the cuRAND-pinned Philox routine: key = word (rho mod 4) of the
    call with counter {pid, t, rho div 4, SHUF << 16 | 0}, key {seed lo, seed hi}; << 32 | pid."""
    key = [seed & 0xFFFFFFFF, seed >> 32]
    out = []
    for pid in pids:
        w = oracle_mod.philox4x32_10([int(pid), t, rho >> 2, 0], key)
        out.append((int(w[rho & 3]) << 32) | int(pid))
    return out


def test_shuffle_key_is_word_rho_mod_4_of_call_rho_div_4(oracle_mod):
    """A7 for every round of two Philox calls (rho = 0..7) and beyond: the order is the argsort of
    keys assembled here; the eight orders differ pairwise (a dropped `>> 2` would repeat rounds
    0-3 in 4-7, a dropped `& 3` would read the wrong word)."""
    pids = np.array([5, 900001, 17, 3, 250, 9, 1000003, 42, 77, 123456, 31, 64, 65, 66, 4000000000], dtype=np.uint32)
    seed, t = (0x9ABCDEF0 << 32) | 0x12345678, 11
    orders = []
    for rho in list(range(8)) + [8, 13, 63]:
        keys = _keys_from_philox(oracle_mod, seed, t, rho, pids)
        expect = pids[np.argsort(np.array(keys, dtype=np.uint64), kind="stable")]
        got = oracle_mod.shuffle_order(seed, t, rho, pids)
        assert np.array_equal(got, expect), rho
        orders.append(tuple(int(v) for v in got))
    assert len(set(orders)) == len(orders)


def test_step_pairs_follow_the_key_layout_in_every_round(oracle_mod):
    """The same pin on the step itself (collide_cell, not the stand-alone shuffle): a dense
    single-layer box that needs R = 7 rounds; in every round the traced (pid_a, pid_b) list of a
    cell is its pids ordered by the keys assembled in the test from Philox, paired 2k with 2k+1."""
    n_per_cell, A = 23, 3
    arrs = one_cell_ensemble(n_per_cell, A, seed=7)
    dt, r, seed = 1e-9, 2.0, 0xDEADBEEF12345
    base = 6.5 / (2.0 * n_per_cell)          # pmax = 6.5 -> R = 7 (uses words 0-3 of call 0, 0-2 of call 1)
    sigma = base * r / dt
    o = oracle_mod.Oracle([A, A, A], [A, A, A], *arrs, r, seed)
    o.set_trace(True)
    o.step(2, dt, sigma)                     # the traced step is the second one: t = 1
    tr = o.trace()
    assert int(tr["round"].max()) == 6 and o.counters()["rounds"] == 2 * 7 * A ** 3
    cell, start = o.cells()
    pid = o.particles()[0]
    seen = set()
    for c in range(A ** 3):
        ids = pid[start[c]:start[c + 1]]
        for rho in range(7):
            keys = _keys_from_philox(oracle_mod, seed, 1, rho, ids)
            order = ids[np.argsort(np.array(keys, dtype=np.uint64), kind="stable")]
            m = (tr["cell"] == c) & (tr["round"] == rho)
            assert np.array_equal(tr["pid_a"][m], order[0:2 * (n_per_cell // 2):2]), (c, rho)
            assert np.array_equal(tr["pid_b"][m], order[1:2 * (n_per_cell // 2):2]), (c, rho)
            if c == 0:
                seen.add(tuple(int(v) for v in order))
    assert len(seen) == 7                    # no round repeats another round's pairing
    # the decision uniform of round rho is keyed by rho itself (not rho div 4): A20
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for i in np.random.default_rng(3).integers(0, tr["u"].size, 40):
        w = oracle_mod.philox4x32_10([int(tr["pid_a"][i]), 1, int(tr["round"][i]), 1 << 16], key)
        assert tr["u"][i] == oracle_mod.u53(w[0], w[1])


def test_shuffle_does_not_depend_on_arrival_order(oracle_mod):
    """A7: the order is a function of the set of pids, not of how the cell was filled."""
    pids = np.arange(100, 160, dtype=np.uint32)
    a = oracle_mod.shuffle_order(5, 7, 1, pids)
    b = oracle_mod.shuffle_order(5, 7, 1, pids[::-1].copy())
    assert np.array_equal(a, b) and not np.array_equal(a, pids)
    assert not np.array_equal(a, oracle_mod.shuffle_order(5, 8, 1, pids))   # step enters the key
    assert not np.array_equal(a, oracle_mod.shuffle_order(5, 7, 2, pids))   # round enters the key
    assert not np.array_equal(a, oracle_mod.shuffle_order(6, 7, 1, pids))   # seed enters the key


def test_step_trace_pairs_every_particle_at_most_once_per_round(oracle_mod):
    w = workloads.riemann_small()
    o = oracle_mod.Oracle.from_workload(w)
    o.set_trace(True)
    o.step(1, w.dt, w.sigma)
    tr = o.trace()
    cell, start = o.cells()
    pid = o.particles()[0]
    cell_of_pid = np.empty(w.n, dtype=np.uint32)
    cell_of_pid[pid] = cell
    counts = np.diff(start.astype(np.int64))
    assert np.all(cell_of_pid[tr["pid_a"]] == tr["cell"]) and np.all(cell_of_pid[tr["pid_b"]] == tr["cell"])
    for rho in range(int(tr["round"].max()) + 1):
        m = tr["round"] == rho
        both = np.concatenate([tr["pid_a"][m], tr["pid_b"][m]])
        assert np.unique(both).size == both.size
    r0 = tr["round"] == 0
    per_cell = np.bincount(tr["cell"][r0], minlength=o.ncells)
    assert np.array_equal(per_cell, counts // 2)                 # exactly floor(n/2) pairs
    assert np.all(np.diff(tr["cell"].astype(np.int64)) >= 0)     # (cell, round, k) order
    assert np.array_equal(tr["decided"], (tr["u"] < tr["P"]).astype(np.uint8))
    assert stats.kstest(tr["u"], "uniform").pvalue > 1e-3


def test_traced_probability_is_eq3_with_the_pair_count_scaling(oracle_mod):
    """PAPER.md:40 Eq. 3 assembled independently: P = v_rel * sigma/r_test * dt/V_cell * cn/R with
    v_rel from E_t^2 - P^2, cn = n(n-1)/(2 floor(n/2)) (A5) -- checked on round 0 of every cell
    that needs a single round (momenta there are still the streamed ones)."""
    w = workloads.riemann_small()
    o = oracle_mod.Oracle.from_workload(w)
    o.set_trace(True)
    o.step(1, w.dt, w.sigma)
    tr = o.trace()
    (x, y, z, px, py, pz), _ = oracle_mod.stream_reflect(*w.arrays(), w.dt, w.box)   # indexed by pid
    _, start = o.cells()
    counts = np.diff(start.astype(np.int64))
    V = np.prod(np.array(w.box) / np.array(w.ncell))
    rounds_of_cell = np.bincount(tr["cell"], weights=None, minlength=o.ncells) // np.maximum(counts // 2, 1)
    m = (tr["round"] == 0) & (rounds_of_cell[tr["cell"]] == 1)
    assert m.sum() > 500
    a, b = tr["pid_a"][m], tr["pid_b"][m]
    Ea = np.sqrt(px[a] ** 2 + py[a] ** 2 + pz[a] ** 2)
    Eb = np.sqrt(px[b] ** 2 + py[b] ** 2 + pz[b] ** 2)
    s = (Ea + Eb) ** 2 - ((px[a] + px[b]) ** 2 + (py[a] + py[b]) ** 2 + (pz[a] + pz[b]) ** 2)
    n = counts[tr["cell"][m]]
    cn = n * (n - 1) / (2.0 * (n // 2))
    P = s / (2 * Ea * Eb) * (w.sigma / w.n_test) * (w.dt / V) * cn
    assert np.allclose(tr["P"][m], P, rtol=1e-9, atol=1e-15)
    # cells that were split into R rounds carry P/R with R = ceil(2 cn base)
    multi = np.unique(tr["cell"][rounds_of_cell[tr["cell"]] > 1])
    base = w.sigma * w.dt / (w.n_test * V)
    for c in multi[:20]:
        nn = counts[c]
        cnn = nn * (nn - 1) / (2.0 * (nn // 2))
        assert rounds_of_cell[c] == math.ceil(2 * cnn * base)


# ------------------------------------------------------------ P5: rate (A5, A6 readings)

def one_cell_ensemble(n_per_cell, ncell_axis, seed):
    """ncell_axis^3 unit cells each holding exactly n_per_cell isotropic thermal particles,
    parked near the cell centre so a tiny dt moves nobody across a face."""
    rng = np.random.default_rng(seed)
    nc = ncell_axis ** 3
    idx = np.repeat(np.arange(nc), n_per_cell)
    ix, iy, iz = idx // (ncell_axis * ncell_axis), (idx // ncell_axis) % ncell_axis, idx % ncell_axis
    jitter = rng.uniform(0.3, 0.7, (3, idx.size))
    pa, _ = thermal_pairs(rng, idx.size)
    return (ix + jitter[0], iy + jitter[1], iz + jitter[2], pa[:, 0].copy(), pa[:, 1].copy(), pa[:, 2].copy())


@pytest.mark.parametrize("n_per_cell,target_pmax", [(2, 0.5), (3, 0.6), (4, 0.6), (5, 0.8), (27, 0.9),
                                                     (40, 2.6), (41, 3.3), (26, 5.4), (31, 7.7)])
def test_collision_rate_matches_all_pairs_expectation(oracle_mod, n_per_cell, target_pmax):
    """north_star: rate = n^2 <v_rel> sigma / (2 N_test).  Exactly: sum over all n(n-1)/2 pairs of
    Eq. 3 with <v_rel> = 1 for an isotropic massless gas, i.e. n(n-1)/2 * base per cell per step,
    whatever the parity of n (A5) and however many rounds the step is split into (A6)."""
    A = 12
    arrs = one_cell_ensemble(n_per_cell, A, seed=100 + n_per_cell)
    dt, r = 1e-9, 3.0
    cn = n_per_cell if n_per_cell % 2 else n_per_cell - 1
    base = target_pmax / (2.0 * cn)
    sigma = base * r * 1.0 / dt
    o = oracle_mod.Oracle([A, A, A], [A, A, A], *arrs, r, 42)
    steps = 12
    o.step(steps, dt, sigma)
    c = o.counters()
    expect = steps * A ** 3 * n_per_cell * (n_per_cell - 1) / 2.0 * base
    assert c["max_occupancy"] == n_per_cell
    assert c["rounds"] == steps * A ** 3 * max(1, math.ceil(target_pmax))
    assert abs(c["collisions"] - expect) < 3.5 * math.sqrt(expect), (c["collisions"], expect)


def test_collision_rate_config0_closed_form(oracle_mod):
    """P5 on BASELINE.json:configs[0]: 3634.7 collisions per step, 181.7k in 50 steps, 3 sigma."""
    g = golden()
    w = workloads.make(0)
    assert w.n == g["N_config0"]
    o = oracle_mod.Oracle.from_workload(w)
    E0 = o.observables(1)[0]
    o.set_dirlog(True)
    o.step(50, w.dt, w.sigma)
    c = o.counters()
    expect = 50 * g["rate_config0_per_step"]
    assert abs(c["collisions"] - expect) < 3 * math.sqrt(expect)
    assert c["near_threshold"] == 0
    # P4: energy conserved to 1e-10 over the run; momentum changes only through the walls
    E1 = o.observables(1)[0]
    assert abs(E1[0] - E0[0]) / E0[0] < 1e-10
    assert np.allclose(E1[1:] - E0[1:], c["wall_dp"], atol=1e-8)
    # P6 on the directions actually used in the run
    d = o.dirlog()
    assert d.shape[0] == c["collisions"]
    assert stats.kstest(d[:, 2], stats.uniform(-1, 2).cdf).pvalue > 1e-3
    assert stats.kstest(np.arctan2(d[:, 1], d[:, 0]), stats.uniform(-math.pi, 2 * math.pi).cdf).pvalue > 1e-3
    # P7: the thermal box stays Boltzmann: E/T ~ Gamma(3,1)
    p = o.particles()
    E = np.sqrt(p[4] ** 2 + p[5] ** 2 + p[6] ** 2)
    assert stats.kstest(E / 0.4, stats.gamma(3).cdf).pvalue > 1e-3
    cz = p[6] / E
    assert stats.kstest(cz, stats.uniform(-1, 2).cdf).pvalue > 1e-3


def test_monoenergetic_gas_relaxes_to_boltzmann(oracle_mod):
    """P7, strong form: start with |p| = 3T for everybody; isotropic 2->2 scattering must
    drive the energy spectrum to Gamma(3, T) at the same energy per particle."""
    T = 0.4
    w = workloads.thermal_box(seed=21)
    mag = np.sqrt(w.px ** 2 + w.py ** 2 + w.pz ** 2)
    f = 3 * T / mag
    o = oracle_mod.Oracle(w.box, w.ncell, w.x, w.y, w.z, w.px * f, w.py * f, w.pz * f, w.n_test, 21)
    E = lambda p: np.sqrt(p[4] ** 2 + p[5] ** 2 + p[6] ** 2)
    assert stats.kstest(E(o.particles()) / T, stats.gamma(3).cdf).pvalue < 1e-10
    o.step(60, w.dt, w.sigma)
    e = E(o.particles())
    assert e.mean() == pytest.approx(3 * T, rel=1e-9)
    assert stats.kstest(e / T, stats.gamma(3).cdf).pvalue > 1e-3


# ----------------------------------------------------------------- P8 / P9: observables

def test_observables_against_exactly_rounded_sums(oracle_mod):
    w = workloads.riemann_small()
    o = oracle_mod.Oracle.from_workload(w)
    nslab = 16
    tot, ed = o.observables(nslab)
    E = np.sqrt((w.px * w.px + w.py * w.py) + w.pz * w.pz)
    assert tot[0] == pytest.approx(math.fsum(E), rel=1e-15)
    for k, a in enumerate((w.px, w.py, w.pz)):
        assert tot[k + 1] == pytest.approx(math.fsum(a), rel=1e-12, abs=1e-11)
    slab = np.minimum((w.x / (w.box[0] / nslab)).astype(int), nslab - 1)
    vol = w.n_test * (w.box[0] / nslab) * w.box[1] * w.box[2]
    for j in range(nslab):
        assert ed[j] == pytest.approx(math.fsum(E[slab == j]) / vol, rel=1e-14)
    assert ed.sum() * vol == pytest.approx(tot[0], rel=1e-14)


def test_initial_energy_density_is_3nT(oracle_mod):
    """P8: e = 3 n T = 16.204 GeV/fm^3 at T = 0.4 and 1.0127 at T = 0.2."""
    g = golden()
    w = workloads.riemann(L=(16.0, 8.0, 8.0), ncell=(16, 8, 8), r_test=20.0, seed=31)
    o = oracle_mod.Oracle.from_workload(w)
    _, ed = o.observables(16)
    nl = w.n * g["n_T0.4"] / (g["n_T0.4"] + g["n_T0.2"])
    for side, key, npart in ((ed[:8], "e_T0.4", nl), (ed[8:], "e_T0.2", w.n - nl)):
        rel_sigma = math.sqrt(1.0 / 3.0) / math.sqrt(npart)      # fixed counts: only E fluctuates
        assert side.mean() == pytest.approx(g[key], rel=4 * rel_sigma + 2e-5)


def test_free_streaming_riemann_profile_closed_form(oracle_mod):
    """P9 (sigma = 0): v_x = cos(theta) is uniform on [-1,1] and independent of E, so
    e(x,t) = e_L (1-xi)/2 + e_R (1+xi)/2, xi = clamp((x-x0)/t, -1, 1), until the fan reaches a
    wall.  Pins streaming, binning-free transport, the slab observable and the units."""
    g = golden()
    w = workloads.riemann(L=(16.0, 3.0, 3.0), ncell=(16, 3, 3), r_test=120.0, seed=32)
    o = oracle_mod.Oracle.from_workload(w)
    nslab, t_end = 32, 4.0
    o.step(int(round(t_end / w.dt)), w.dt, 0.0)
    _, ed = o.observables(nslab)
    eL, eR, x0 = g["e_T0.4"], g["e_T0.2"], 8.0
    edges = np.linspace(0, 16.0, nslab + 1)

    def cum(x):       # integral of e(x', t) dx' from x0 - t, piecewise quadratic inside the fan
        xi = np.clip((x - x0) / t_end, -1.0, 1.0)
        inside = t_end * (0.5 * (eL + eR) * (xi + 1) + 0.25 * (eR - eL) * (xi * xi - 1))
        return inside + eL * np.minimum(x - (x0 - t_end), 0.0) + eR * np.maximum(x - (x0 + t_end), 0.0)
    expect = np.diff(cum(edges)) / np.diff(edges)
    V_slab = 0.5 * 9.0 * w.n_test
    n_j = np.maximum(expect * V_slab / (3 * 0.3), 50)             # rough particle count per slab
    zscore = (ed - expect) / (expect * 1.155 / np.sqrt(n_j))
    # the walls are never touched (fan edge at 4 and 12) but particles near them reflect:
    # the profile stays flat there, so all slabs are comparable
    assert np.abs(zscore).max() < 4.5, zscore
    chi2 = float((zscore ** 2).sum())
    assert stats.chi2.sf(chi2, nslab) > 1e-4
    # and the discontinuity really moved: centre slabs are between the two plateaus
    assert eR * 1.5 < ed[nslab // 2] < eL * 0.75


# ------------------------------------------------------------------ argument validation

def test_oracle_rejects_bad_arguments(oracle_mod):
    w = workloads.thermal_box(L=(2.0, 2.0, 2.0), ncell=(2, 2, 2), count=100, seed=1)
    o = oracle_mod.Oracle.from_workload(w)
    with pytest.raises(oracle_mod.OracleError) as e:
        o.step(1, 1.0, 0.1)          # dt == cell edge: PAPER.md:62 wants dt < dx
    assert e.value.code == -7
    with pytest.raises(oracle_mod.OracleError):
        o.step(1, 0.1, 1e9)          # needs more than 64 rounds
    bad = [a.copy() for a in w.arrays()]
    bad[0][3] = 2.5                   # outside the box
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(w.box, w.ncell, *bad, 1.0, 1)
    bad = [a.copy() for a in w.arrays()]
    bad[3][5] = bad[4][5] = bad[5][5] = 0.0   # p = 0: a massless particle without a velocity
    with pytest.raises(oracle_mod.OracleError):
        oracle_mod.Oracle(w.box, w.ncell, *bad, 1.0, 1)


def test_k_steps_equal_k_single_steps(oracle_mod):
    """cuba_step(k) == k x cuba_step(1) bit for bit: the step counter is the only RNG state."""
    w = workloads.riemann_small()
    a = oracle_mod.Oracle.from_workload(w)
    b = oracle_mod.Oracle.from_workload(w)
    a.step(4, w.dt, w.sigma)
    for _ in range(4):
        b.step(1, w.dt, w.sigma)
    for u, v in zip(a.particles(), b.particles()):
        assert np.array_equal(u, v)


def test_collide_cells_entry_point_is_the_steps_s5(oracle_mod):
    """oracle_collide_cells (used by the full-size GPU checks) is S5 of oracle_step: colliding every
    cell of the streamed, binned state reproduces the step's momenta and counters bit for bit."""
    w = workloads.riemann_small()
    a = oracle_mod.Oracle.from_workload(w)
    a.step(2, w.dt, w.sigma)                       # t = 2 afterwards
    b = oracle_mod.Oracle.from_workload(w)
    b.step(2, w.dt, w.sigma)
    b.step(1, w.dt, 0.0)                           # S1-S4 of the third step only
    cb = a.counters()
    a.step(1, w.dt, w.sigma)
    pid, x, y, z, px, py, pz = b.particles()
    _, start = b.cells()
    V = float(np.prod(np.array(w.box) / np.array(w.ncell)))
    base = (w.sigma * w.dt) / (w.n_test * V)
    lo, hi = start[:-1].astype(np.int64), start[1:].astype(np.int64)
    qx, qy, qz, cnt = oracle_mod.collide_cells(w.seed, 2, base, lo, hi, pid, px, py, pz)
    ref = a.particles()
    assert np.array_equal(ref[0], pid)
    assert np.array_equal(qx, ref[4]) and np.array_equal(qy, ref[5]) and np.array_equal(qz, ref[6])
    ca = a.counters()
    assert cnt["collisions"] == ca["collisions"] - cb["collisions"] > 100
    assert cnt["pairs"] == ca["pairs"] - cb["pairs"] and cnt["rounds"] == ca["rounds"] - cb["rounds"]
