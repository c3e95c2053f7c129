"""cuba_observables_noalloc against cuba_observables (`-m gpu`).

Who needs this entry point: code that may not allocate GPU memory at the moment it wants the observables -- a
plug-in running inside another program's memory budget, an analysis hook called between the steps of a loop
that must not stall, a service that allocates once at start-up and never again.  cuba_observables wants a
context (pinned host memory, streams, events, a workspace); the no-alloc call wants only the caller's input
and output arrays and keeps its per-block partial sums in a fixed array inside the library.

What is checked: the same sums as the existing path, within the tolerance the observables tests use (1e-12
relative; identical bits where both run the same kernel on the same array order), on two calls in a row that
share the fixed array (different data and slab counts, so stale contents would show), the size limit, and that
the call leaves the amount of free device memory alone.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  It runs alone in a fresh process (the no-alloc call is then the first thing the library does on
the device) as well as after the rest of the suite."""
import ctypes

import numpy as np
import pytest

import workloads

pytestmark = pytest.mark.gpu

REL = 1e-12   # as tests/test_gpu_parity.py: sums within 1e-12 relative


@pytest.fixture(scope="module")
def cuba():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_1208_0961_b200 as c
    c.lib()   # fails loudly if the extension was not built
    return c


def assert_sums_close(res, tot, ed):
    assert np.allclose(res[4:], ed, rtol=REL, atol=0)
    assert np.allclose(res[:4], tot, rtol=REL, atol=1e-9)   # sum p is ~0: absolute, as in the parity tests


def test_no_alloc_observables_match_the_context_path_on_consecutive_calls(cuba):
    import torch
    # ~14.6k particles: 14 tiles of 1024 and a ragged tail, 12 cell layers along x
    w = workloads.riemann(L=(12.0, 4.0, 4.0), ncell=(12, 4, 4), r_test=10.0, seed=23)
    assert w.n % 1024 != 0 and w.n > 8 * 1024
    dev = torch.device("cuda:0")
    x, y, z, px, py, pz = (torch.from_numpy(a).to(dev) for a in w.arrays())
    res_a = torch.full((4 + 24,), float("nan"), dtype=torch.float64, device=dev)
    res_b = torch.full((4 + 7,), float("nan"), dtype=torch.float64, device=dev)
    res_c = torch.full((4 + cuba.NOALLOC_MAX_SLABS,), float("nan"), dtype=torch.float64, device=dev)
    torch.cuda.synchronize()

    # call 1 -- before any context exists (alone in a fresh process this is the library's first call on the
    # device: the one that looks up the address of the fixed array).  The caller's arrays are still in their
    # shuffled input order here, so the sums are taken in another order than the context path will: 1e-12.
    cuba.observables_noalloc(x, px, py, pz, w.box, w.n_test, 24, res_a)
    torch.cuda.synchronize()
    first = res_a.cpu().numpy()

    g = cuba.Cuba(w.box, w.ncell, x, y, z, px, py, pz, w.n_test, w.seed)   # sorts the caller's arrays in place
    tot, ed = g.observables(24)
    assert_sums_close(first, tot, ed)

    # call 2 -- right after call 1 on the same fixed array, other data (five steps later), other slab count,
    # straight on the device pointers of the context's current store (the in-situ hook use).  Same kernel,
    # same array order as cuba_observables: the bits agree.  Free device memory does not move.
    g.step(5, w.dt, w.sigma)
    st = g.state()
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(dev)[0]
    launches = cuba.launch_count()
    box = (ctypes.c_double * 3)(*w.box)
    rc = cuba.lib().cuba_observables_noalloc(w.n, *[ctypes.c_void_p(st[k]) for k in ("x", "px", "py", "pz")], box,
                                             float(w.n_test), 7, ctypes.c_void_p(res_b.data_ptr()),
                                             ctypes.c_void_p(torch.cuda.current_stream(dev).cuda_stream))
    assert rc == 0
    torch.cuda.synchronize()
    assert cuba.launch_count() == launches + 2
    assert torch.cuda.mem_get_info(dev)[0] == free_before
    second = res_b.cpu().numpy()
    tot, ed = g.observables(7)
    assert_sums_close(second, tot, ed)
    assert np.array_equal(second[4:], ed) and np.array_equal(second[:4], tot)

    # call 3 -- the largest slab count the fixed array holds; the context path switches to its wide-window
    # kernel there (128 > 2 nx), another summation order: 1e-12
    host = g.particles()            # (pid, x, y, z, px, py, pz) in array order
    x_c, px_c, py_c, pz_c = (torch.from_numpy(host[k]).to(dev) for k in (1, 4, 5, 6))
    cuba.observables_noalloc(x_c, px_c, py_c, pz_c, w.box, w.n_test, cuba.NOALLOC_MAX_SLABS, res_c)
    torch.cuda.synchronize()
    tot, ed = g.observables(cuba.NOALLOC_MAX_SLABS)
    assert_sums_close(res_c.cpu().numpy(), tot, ed)
    g.close()


def test_no_alloc_observables_reject_what_the_fixed_array_cannot_hold(cuba):
    import torch
    dev = torch.device("cuda:0")
    a = torch.full((1000,), 0.5, dtype=torch.float64, device=dev)
    res = torch.zeros(4 + 2 * cuba.NOALLOC_MAX_SLABS, dtype=torch.float64, device=dev)
    launches = cuba.launch_count()
    for nslab in (cuba.NOALLOC_MAX_SLABS + 1, 0, -3):
        with pytest.raises(cuba.CubaError) as e:
            cuba.observables_noalloc(a, a, a, a, (1.0, 1.0, 1.0), 1.0, nslab, res)
        assert e.value.code == -2                              # CUBA_ERR_SIZE
    with pytest.raises(cuba.CubaError) as e:
        cuba.observables_noalloc(a, a, a, a, (1.0, 0.0, 1.0), 1.0, 4, res)
    assert e.value.code == -3                                  # CUBA_ERR_VALUE
    assert cuba.launch_count() == launches                     # nothing was launched
    torch.cuda.synchronize()
    assert float(res.abs().sum()) == 0.0                       # and nothing written
    # a valid call still works afterwards: 1000 particles of |p| = sqrt(0.75) in a unit box, one slab
    cuba.observables_noalloc(a, a, a, a, (1.0, 1.0, 1.0), 2.0, 1, res)
    torch.cuda.synchronize()
    r = res.cpu().numpy()
    assert np.isclose(r[0], 1000 * np.sqrt(0.75), rtol=REL) and np.isclose(r[4], r[0] / 2.0, rtol=REL)
    assert np.allclose(r[1:4], 500.0, rtol=REL)
