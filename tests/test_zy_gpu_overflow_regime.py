"""The ~100M-particle variant of BASELINE.json:configs[4] (workloads index 5, r_test = 185.5) at full size
(`-m gpu`, parity gap a).  Its hottest cells hold more than 4544 particles, beyond the largest
shared-memory class, so `k_collide_overflow` (global-memory scratch, momenta in place) works in its real
regime: the sampled check of tests/test_gpu_large.py with the eight fullest cells re-collided by the oracle
bit for bit, the streaming / binning / stability checks on all 100M particles, counters and energy.

Heavy on host memory (several copies of 6 x 100M doubles) and a few minutes long, hence a file of its own that
is collected after the other parity tests: should the box be too small for it, `pytest -x` has run them all."""
import pytest

from test_gpu_large import check_full_size_step, cuba  # noqa: F401  (the fixture)

pytestmark = pytest.mark.gpu


def test_100m_particle_step_sampled_against_oracle(cuba, oracle_mod):  # noqa: F811
    import psutil
    if psutil.virtual_memory().available < 70e9:
        pytest.skip("needs ~60 GB of host memory for the 100M-particle arrays and their oracle copies")
    check_full_size_step(cuba, oracle_mod, 5, n_hot=8, n_random=12, expect_overflow=True)
