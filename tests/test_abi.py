"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/tm.h declares; host-side logic."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def tm():
    from paper_1309_2256_b200 import build
    build.build()
    import paper_1309_2256_b200 as tm
    return tm


def test_every_declared_symbol_is_exported(tm):
    hdr = open(os.path.join(ROOT, "include", "tm.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(tm_[A-Za-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 20
    lib = ctypes.CDLL(tm.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name
    assert declared == set(tm.ABI_SYMBOLS)


def test_version_and_errors(tm):
    assert tm.tm_version() == 100
    for s in range(0, -7, -1):
        assert tm.tm_strerror(s) != "unknown status"
    assert tm.tm_strerror(-99) == "unknown status"


def test_lattice_and_sizes(tm):
    for bad in ((3, 4, 4, 4), (4, 4, 4, 2), (4, 5, 4, 4)):
        with pytest.raises(tm.TmError):
            tm.tm_lattice_create(bad)
    L = tm.tm_lattice_create((32, 32, 32, 64))
    V = 32 ** 3 * 64
    # SURVEY.md 8 size table
    assert tm.tm_gauge_bytes(L, 4, 18) == 4 * V * 18 * 4 == 603979776
    assert tm.tm_gauge_bytes(L, 4, 12) == 4 * V * 12 * 4
    assert tm.tm_gauge_bytes(L, 2, 12) == 4 * V * 12 * 2
    assert tm.tm_spinor_bytes(L, 8, 0, 1) == V // 2 * 24 * 8
    assert tm.tm_spinor_bytes(L, 2, 0, 1) == V // 2 * (24 * 2 + 4)
    assert tm.tm_spinor_bytes(L, 2, 1, 12) == 12 * V * (24 * 2 + 4)
    assert tm.tm_cg_workspace_bytes(L, 8, 2, tm.TM_CG_LP_TRUNCATED, 12) > 6 * 12 * tm.tm_spinor_bytes(L, 2, 0, 1)
    assert tm.tm_gauge_bytes(L, 3, 18) == 0 and tm.tm_gauge_bytes(L, 4, 9) == 0 and tm.tm_gauge_bytes(L, 4, 8) * 18 == tm.tm_gauge_bytes(L, 4, 18) * 8


def test_no_cpu_fallback(tm):
    """Compute calls fail loudly without a device (or with bad pointers) instead of routing anywhere else."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    L = tm.tm_lattice_create((4, 4, 4, 4))
    import numpy as np
    a = np.zeros(1 << 16, dtype=np.uint8)
    with pytest.raises(tm.TmError):
        tm.tm_dslash(L, a.ctypes.data // 256 * 256 + 256, 4, 18, a.ctypes.data // 256 * 256 + 512, a.ctypes.data // 256 * 256 + 1024,
                     None, 0, 0, 0, 0.1, 0.0, 1, stream=0)
