"""Seeded synthetic input generators for the CuBA hot path (harness-side data only).

This module holds NONE of the method's arithmetic (no streaming, binning, pairing,
collision or Philox code).  It only draws initial conditions with numpy and is the one
module that both the CPU oracle (`oracle/`) and the CUDA library
(`paper_1208_0961_b200/`) are fed from, so that they see identical bits.

The paper's workload is a parametrised initial condition, not a dataset
(section 5: box 32^3 fm^3, sigma = 10 GeV^-2, dt = 0.1 fm/c, "equal particle
distribution", T_left = 0.4 GeV / T_right = 0.2 GeV).  The five configurations of
BASELINE.json:configs are reproduced here (sizes as derived in SURVEY.md section 8(d)):

  * massless Boltzmann gluons, degeneracy 16: n(T) = 16 T^3 / (pi^2 (hbar c)^3) fm^-3,
    hbar c = 0.197327 GeV fm (BASELINE.json:configs[0]);
  * fixed (not Poisson) counts  N_region = round(n(T) V_region r_test)  (A17);
  * |p| = -T ln(u1 u2 u3)  (a Gamma(3, T) variate), direction isotropic,
    positions uniform inside the region, array order shuffled.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Callable, Optional

import numpy as np

HBARC = 0.197327  # GeV fm, BASELINE.json:configs[0]
GEV2_TO_FM2 = HBARC * HBARC  # 1 GeV^-2 in fm^2 (10 GeV^-2 -> 0.389379 fm^2)


def gluon_density(T: float) -> float:
    """Physical number density of a massless Boltzmann gluon gas, fm^-3 (T in GeV)."""
    return 16.0 * T ** 3 / (math.pi ** 2 * HBARC ** 3)


@dataclasses.dataclass
class Workload:
    """One initial condition plus the run parameters the config names."""
    name: str
    box: tuple            # (Lx, Ly, Lz) fm
    ncell: tuple          # (nx, ny, nz)
    n_test: float         # r_test of PAPER.md:44
    sigma: float          # fm^2
    dt: float             # fm/c
    steps: int
    seed: int             # Philox seed handed to cuba_init / oracle_init
    nslab: int
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    px: np.ndarray
    py: np.ndarray
    pz: np.ndarray
    note: str = ""

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    @property
    def ncells(self) -> int:
        return int(self.ncell[0] * self.ncell[1] * self.ncell[2])

    def arrays(self):
        return (self.x, self.y, self.z, self.px, self.py, self.pz)


def _thermal_momenta(rng: np.random.Generator, T, count: int):
    """|p| ~ Gamma(3, T) via -T ln(u1 u2 u3); direction uniform on the sphere.

    `T` may be a scalar or an array of per-particle temperatures."""
    u = 1.0 - rng.random((3, count))            # (0, 1]
    mag = -T * (np.log(u[0]) + np.log(u[1]) + np.log(u[2]))
    # a zero magnitude needs u1=u2=u3=1 exactly; guard anyway (massless p=0 has no velocity)
    mag = np.maximum(mag, 1e-300)
    cz = 2.0 * rng.random(count) - 1.0
    phi = 2.0 * math.pi * rng.random(count)
    st = np.sqrt(np.maximum(0.0, 1.0 - cz * cz))
    return mag * st * np.cos(phi), mag * st * np.sin(phi), mag * cz


def _uniform_region(rng, count, lo, hi):
    return [lo[k] + (hi[k] - lo[k]) * rng.random(count) for k in range(3)]


def _assemble(rng, parts):
    """Concatenate regions and shuffle the array order (so the first binning is not a no-op)."""
    cols = [np.concatenate([p[k] for p in parts]) for k in range(6)]
    perm = rng.permutation(cols[0].shape[0])
    return [np.ascontiguousarray(c[perm], dtype=np.float64) for c in cols]


def thermal_box(L=(8.0, 8.0, 8.0), ncell=(8, 8, 8), T=0.4, r_test=2.0,
                sigma_gev2=10.0, dt=0.1, steps=50, seed=1, name="thermal_box",
                nslab=8, count: Optional[int] = None) -> Workload:
    """Homogeneous thermal box (BASELINE.json:configs[0])."""
    rng = np.random.Generator(np.random.Philox(seed))
    V = L[0] * L[1] * L[2]
    n = int(round(gluon_density(T) * V * r_test)) if count is None else int(count)
    pos = _uniform_region(rng, n, (0.0, 0.0, 0.0), L)
    mom = _thermal_momenta(rng, T, n)
    cols = _assemble(rng, [pos + list(mom)])
    return Workload(name, tuple(L), tuple(ncell), float(r_test), sigma_gev2 * GEV2_TO_FM2,
                    dt, steps, seed, nslab, *cols)


def riemann(L=(32.0, 32.0, 32.0), ncell=(32, 32, 32), T_left=0.4, T_right=0.2,
            r_test=10.0, sigma_gev2=10.0, dt=0.1, steps=100, seed=2, name="riemann",
            nslab=64, x_split: Optional[float] = None) -> Workload:
    """Riemann problem: T_left for x < x_split, T_right beyond; transversely
    homogeneous; fixed counts per side (BASELINE.json:configs[1..3])."""
    rng = np.random.Generator(np.random.Philox(seed))
    xs = 0.5 * L[0] if x_split is None else x_split
    parts = []
    for (lo, hi, T) in (((0.0, 0.0, 0.0), (xs, L[1], L[2]), T_left),
                        ((xs, 0.0, 0.0), (L[0], L[1], L[2]), T_right)):
        V = (hi[0] - lo[0]) * (hi[1] - lo[1]) * (hi[2] - lo[2])
        n = int(round(gluon_density(T) * V * r_test))
        pos = _uniform_region(rng, n, lo, hi)
        mom = _thermal_momenta(rng, T, n)
        parts.append(pos + list(mom))
    cols = _assemble(rng, parts)
    return Workload(name, tuple(L), tuple(ncell), float(r_test), sigma_gev2 * GEV2_TO_FM2,
                    dt, steps, seed, nslab, *cols)


def skewed(L=(64.0, 32.0, 32.0), ncell=(64, 32, 32), T0=0.5, T1=0.1, r_test=100.0,
           sigma_gev2=10.0, dt=0.1, steps=50, seed=5, name="skewed", nslab=64) -> Workload:
    """Temperature linear in x from T0 (x=0) to T1 (x=Lx); density ~ T(x)^3, so x is drawn by
    inverting the CDF of T(x)^3 and |p| uses the local T (BASELINE.json:configs[4])."""
    rng = np.random.Generator(np.random.Philox(seed))
    Lx, Ly, Lz = L
    # N = r * Ly Lz * int_0^Lx n(T(x)) dx ;  int T^3 dx = Lx (T0^4 - T1^4) / (4 (T0 - T1))
    integral = Lx * (T0 ** 4 - T1 ** 4) / (4.0 * (T0 - T1))
    n = int(round(16.0 / (math.pi ** 2 * HBARC ** 3) * integral * Ly * Lz * r_test))
    u = rng.random(n)
    # CDF(x) = (T0^4 - T(x)^4) / (T0^4 - T1^4)  ->  T(x) = (T0^4 - u (T0^4 - T1^4))^(1/4)
    Tx = (T0 ** 4 - u * (T0 ** 4 - T1 ** 4)) ** 0.25
    x = (T0 - Tx) * (Lx / (T0 - T1))
    x = np.minimum(np.maximum(x, 0.0), np.nextafter(Lx, 0.0))
    y = Ly * rng.random(n)
    z = Lz * rng.random(n)
    mom = _thermal_momenta(rng, Tx, n)
    cols = _assemble(rng, [[x, y, z] + list(mom)])
    return Workload(name, tuple(L), tuple(ncell), float(r_test), sigma_gev2 * GEV2_TO_FM2,
                    dt, steps, seed, nslab, *cols)


# BASELINE.json:configs, 0-indexed as in the JSON (SURVEY.md numbers them 1..5).
CONFIGS: dict = {
    0: lambda: thermal_box(name="configs[0] thermal box 8^3, r_test=2"),
    1: lambda: riemann(r_test=10.0, seed=2, steps=100, name="configs[1] Riemann r_test=10"),
    2: lambda: riemann(r_test=100.0, seed=3, steps=100, name="configs[2] Riemann hi-stat r_test=100"),
    3: lambda: riemann(ncell=(64, 32, 32), r_test=40.0, sigma_gev2=50.0, dt=0.05, steps=200,
                       seed=4, name="configs[3] Riemann fine cells sigma=50"),
    4: lambda: skewed(r_test=100.0, seed=5, steps=50, name="configs[4] skewed occupancy r_test=100"),
    # the ~100M-particle variant of configs[4] (BASELINE.json says "~100M"; r_test = 100 gives 53.9M)
    5: lambda: skewed(r_test=185.5, seed=5, steps=50, name="configs[4] skewed occupancy r_test=185.5 (~100M)"),
}


def make(config: int) -> Workload:
    """Build BASELINE.json:configs[config] (0-indexed)."""
    return CONFIGS[config]()


def riemann_small(seed=11, r_test=6.0, L=(8.0, 4.0, 4.0), ncell=(8, 4, 4), **kw) -> Workload:
    """A scaled-down Riemann problem with the same temperatures, sigma, dt and cell size as
    configs[1] (parity-test size: the oracle finishes in well under a second per step)."""
    return riemann(L=L, ncell=ncell, r_test=r_test, seed=seed, steps=10,
                   name="riemann_small", nslab=16, **kw)
