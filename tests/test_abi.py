"""CPU checks of the boundary: the C-ABI library loads and exports every symbol that
include/cuba.h declares, and argument validation that needs no device works."""
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def cuba():
    from paper_1208_0961_b200 import build
    build.build()
    import paper_1208_0961_b200 as c
    return c


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "cuba.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(cuba_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(cuba):
    syms = declared_symbols()
    assert len(syms) >= 13
    L = cuba.lib()
    for s in syms:
        assert hasattr(L, s), s
    assert sorted(cuba.EXPORTS) == syms


def test_workspace_bytes_and_strerror(cuba):
    assert cuba.workspace_bytes(0, (8, 8, 8)) == 0
    assert cuba.workspace_bytes(100, (0, 8, 8)) == 0
    assert cuba.workspace_bytes(100, (1 << 10, 1 << 10, 1 << 10)) == 0
    small, big = cuba.workspace_bytes(1000, (8, 8, 8)), cuba.workspace_bytes(2000000, (32, 32, 32))
    assert 0 < small < big
    assert big >= 2000000 * 56                      # the second copy of the store fits
    assert cuba.strerror(0) == "ok" and "cell edge" in cuba.strerror(-7)
    assert cuba.launch_count() == 0                 # nothing ran


def test_product_does_not_import_the_oracle():
    """The oracle is test infrastructure: nothing under the package may reference it."""
    pkg = os.path.join(ROOT, "paper_1208_0961_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "cuba_oracle" not in text, f
    otext = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "cuba_oracle.c")).read()
    assert "import paper_1208_0961_b200" not in otext and "cuba.h" not in otext and "csrc" not in otext


def test_compute_calls_fail_loudly_without_a_device(cuba):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    import numpy as np
    with pytest.raises(RuntimeError):
        cuba.Cuba((1, 1, 1), (1, 1, 1), *[torch.zeros(4, dtype=torch.float64)] * 6, 1.0, 1)
    a = [np.full(4, 0.5) for _ in range(6)]
    with pytest.raises(cuba.CubaError) as e:
        cuba.run_host((1.0, 1.0, 1.0), (1, 1, 1), *a, 1.0, 1, 1, 0.1, 0.1, 4)
    assert e.value.code == -5                       # CUBA_ERR_CUDA: no fallback
