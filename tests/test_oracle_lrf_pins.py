"""Pins of the oracle's local-rest-frame observables (A22) against
things other than itself: numpy's eigen-decomposition, hand-built slabs with results known by
inspection, exactly rounded sums, the massless trace identity, a thermal box at rest and a
boosted thermal ensemble (textbook: e = 3 n* T, v = beta, isotropic pressure e/3)."""
import math

import numpy as np
import pytest

import workloads


def make_oracle(oracle_mod, box, ncell, x, y, z, px, py, pz, r_test):
    f = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    return oracle_mod.Oracle(box, ncell, f(x), f(y), f(z), f(px), f(py), f(pz), r_test, 1)


def test_landau_match_is_the_timelike_eigenpair_of_the_mixed_tensor(oracle_mod):
    """T^mu_nu u^nu = e u^mu on the (t, x) block; numpy.linalg.eig is the independent route."""
    rng = np.random.default_rng(3)
    for _ in range(200):
        m = int(rng.integers(2, 40))
        p = rng.normal(size=(3, m)) * rng.uniform(0.1, 3.0)
        p[0] += rng.uniform(-2.0, 2.0)                       # a net flow along x
        E = np.sqrt((p * p).sum(axis=0))
        T00, T0x = E.sum(), p[0].sum()
        Txx, Tyy, Tzz = (p[0] ** 2 / E).sum(), (p[1] ** 2 / E).sum(), (p[2] ** 2 / E).sum()
        e, v, PL, PT = oracle_mod.landau_match(T00, T0x, Txx, Tyy, Tzz)
        lam, vec = np.linalg.eig(np.array([[T00, -T0x], [T0x, -Txx]]))
        k = int(np.argmax(np.abs(vec[0]) - np.abs(vec[1])))  # timelike eigenvector: |u^0| > |u^x|
        assert abs(vec[0, k]) > abs(vec[1, k])
        assert e == pytest.approx(lam[k].real, rel=1e-10)
        assert v == pytest.approx((vec[1, k] / vec[0, k]).real, rel=1e-9, abs=1e-12)
        assert PL == pytest.approx(-lam[1 - k].real, rel=1e-9, abs=1e-12 * T00)
        assert PT == pytest.approx(0.5 * (Tyy + Tzz), rel=1e-15)
        assert abs(v) < 1.0 and e > 0.0
        assert e == pytest.approx(PL + 2.0 * PT, rel=1e-9)   # massless: the tensor is traceless


def test_hand_built_slabs(oracle_mod):
    """Slab 0: one particle along +x (no rest frame: e = 0, v = 1).  Slab 1: back to back along x
    (e = T00, v = 0, P_L = e, P_T = 0).  Slab 2: back to back along y (P_L = 0, P_T = e/2).
    Slab 3: empty.  Normalisation 1/(r_test V_slab) with V_slab = 1 x 2 x 3 fm^3, r_test = 4."""
    box, r = (4.0, 2.0, 3.0), 4.0
    x = [0.5, 1.25, 1.75, 2.5, 2.6]
    px = [2.0, 1.5, -1.5, 0.0, 0.0]
    py = [0.0, 0.0, 0.0, 0.7, -0.7]
    o = make_oracle(oracle_mod, box, (4, 1, 1), x, [1.0] * 5, [1.0] * 5, px, py, [0.0] * 5, r)
    T, lrf = o.observables_lrf(4)
    vol = r * 1.0 * 2.0 * 3.0
    assert np.allclose(T[:, 0], [2.0 / vol, 2.0 / vol, 2.0 / vol, 0.0, 0.0], rtol=1e-15)
    assert lrf[0, 0] == 0.0 and lrf[1, 0] == 1.0
    assert np.allclose(T[:, 1], [3.0 / vol, 0.0, 3.0 / vol, 0.0, 0.0], rtol=1e-15)
    assert np.allclose(lrf[:, 1], [3.0 / vol, 0.0, 3.0 / vol, 0.0], rtol=1e-15)
    assert np.allclose(T[:, 2], [1.4 / vol, 0.0, 0.0, 1.4 / vol, 0.0], rtol=1e-15)
    assert np.allclose(lrf[:, 2], [1.4 / vol, 0.0, 0.0, 0.7 / vol], rtol=1e-15)
    assert np.all(T[:, 3] == 0.0) and np.all(lrf[:, 3] == 0.0)


def test_tensor_components_are_the_exactly_rounded_sums_and_traceless(oracle_mod):
    w = workloads.riemann_small()
    o = oracle_mod.Oracle.from_workload(w)
    pid, x, y, z, px, py, pz = o.particles()
    nslab = 16
    T, lrf = o.observables_lrf(nslab)
    _, ed = o.observables(nslab)
    assert np.array_equal(T[0], ed)                               # T00 is the energy density of Fig. 2 (A15)
    E = np.sqrt((px * px + py * py) + pz * pz)
    slab = np.minimum((x / (w.box[0] / nslab)).astype(int), nslab - 1)
    vol = w.n_test * (w.box[0] / nslab) * w.box[1] * w.box[2]
    for j in range(nslab):
        m = slab == j
        for k, contrib in enumerate((E, px, px * px / E, py * py / E, pz * pz / E)):
            assert T[k, j] == pytest.approx(math.fsum(contrib[m]) / vol, rel=1e-13, abs=1e-13)
    assert np.allclose(T[0], T[2] + T[3] + T[4], rtol=1e-13)      # E^2 = p^2
    # the derived quantities are the stand-alone matching of the same components
    for j in range(nslab):
        assert tuple(lrf[:, j]) == oracle_mod.landau_match(*T[:, j])


def test_thermal_box_at_rest_is_isotropic(oracle_mod):
    """e = 3 n T (16.204 GeV/fm^3 at T = 0.4, tests/golden/paper_closed_forms.txt), P_L = P_T = e/3,
    v = 0, all within the statistical error of the sample."""
    w = workloads.thermal_box(L=(8.0, 8.0, 8.0), ncell=(8, 8, 8), T=0.4, r_test=8.0, seed=41)
    o = oracle_mod.Oracle.from_workload(w)
    T, lrf = o.observables_lrf(1)
    e_exact = 3.0 * workloads.gluon_density(0.4) * 0.4
    sig = 1.0 / math.sqrt(w.n)
    assert lrf[0, 0] == pytest.approx(e_exact, rel=4 * sig)
    assert abs(lrf[1, 0]) < 4 * sig
    assert lrf[2, 0] == pytest.approx(e_exact / 3.0, rel=6 * sig)
    assert lrf[3, 0] == pytest.approx(e_exact / 3.0, rel=6 * sig)


@pytest.mark.parametrize("beta", [0.5, -0.8])
def test_boosted_thermal_ensemble(oracle_mod, beta):
    """A fluid element at temperature T moving with velocity beta along x: f(p) = exp(-p.u/T).
    Rest-frame thermal momenta boosted to the lab and accepted with probability proportional to
    E/E* (d^3p = (E/E*) d^3p*) sample f in the lab.  Then n_lab = gamma n*, and Landau matching
    must return e = 3 n* T, v = beta, P_L = P_T = e/3 within the statistical error."""
    T_fluid, gamma = 0.3, 1.0 / math.sqrt(1.0 - beta * beta)
    rng = np.random.default_rng(17)
    m = 1_500_000
    u = 1.0 - rng.random((3, m))
    Es = -T_fluid * np.log(u).sum(axis=0)
    cz = 2.0 * rng.random(m) - 1.0
    phi = 2.0 * math.pi * rng.random(m)
    st = np.sqrt(1.0 - cz * cz)
    pxs, pys, pzs = Es * cz, Es * st * np.cos(phi), Es * st * np.sin(phi)
    E = gamma * (Es + beta * pxs)
    px = gamma * (pxs + beta * Es)
    keep = rng.random(m) < (E / Es) / (gamma * (1.0 + abs(beta)))
    px, py, pz = px[keep], pys[keep], pzs[keep]
    n = int(keep.sum())
    assert n > 300_000
    box, r = (2.0, 2.0, 2.0), 50.0
    pos = [2.0 * rng.random(n) for _ in range(3)]
    o = make_oracle(oracle_mod, box, (2, 2, 2), *pos, px, py, pz, r)
    Tt, lrf = o.observables_lrf(1)
    n_lab = n / (r * 8.0)
    e_expect = 3.0 * (n_lab / gamma) * T_fluid
    sig = 1.0 / math.sqrt(n)
    assert lrf[0, 0] == pytest.approx(e_expect, rel=6 * sig)
    assert lrf[1, 0] == pytest.approx(beta, abs=6 * sig)
    assert lrf[2, 0] == pytest.approx(e_expect / 3.0, rel=12 * sig)
    assert lrf[3, 0] == pytest.approx(e_expect / 3.0, rel=12 * sig)
