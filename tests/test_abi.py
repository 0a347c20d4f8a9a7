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
    for s in range(0, -10, -1):
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
    assert tm.tm_gauge_bytes(L, 2, tm.TM_RECON_12_FIX16) == 4 * V * 12 * 2 and tm.tm_gauge_bytes(L, 2, tm.TM_RECON_18_FIX16) == 4 * V * 18 * 2
    assert tm.tm_gauge_bytes(L, 4, tm.TM_RECON_12_FIX16) == 4 * V * 12 * 4 and tm.tm_gauge_bytes(L, 2, 108) == 0  # flag ignored above 16 bits
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


def test_every_wrapper_reaches_the_library(tm):
    """Each Python wrapper marshals its arguments into the C call and turns the status into TmError: called with NULL for a
    required pointer the LIBRARY must answer TM_ERR_ARG (no device needed); a TypeError here would be a wrapper bug."""
    import numpy as np
    import torch
    L = tm.tm_lattice_create((4, 4, 4, 4))
    buf = torch.zeros(1 << 12, dtype=torch.uint8)  # host memory: never dereferenced, the NULL argument is rejected first
    prm = tm.make_cg_params(0.16, 0.005, 1e-2, 10, tm.TM_CG_LP_TRUNCATED)
    mom = np.zeros((1, 3), dtype=np.int32)
    calls = [
        lambda: tm.tm_gauge_pack(L, None, 4, 18, buf, 1e-10, stream=0),
        lambda: tm.tm_spinor_pack(L, None, 4, 1, buf, stream=0),
        lambda: tm.tm_spinor_unpack(L, None, 4, 1, buf, stream=0),
        lambda: tm.tm_spinor_pack_z4(L, None, 4, 1, buf, stream=0),
        lambda: tm.tm_spinor_pack_z4_bits(L, None, 4, 1, buf, stream=0),
        lambda: tm.tm_noise_z4(L, 1, 1, 4, 1, None, stream=0),
        lambda: tm.tm_gauge_synthetic(L, 1, 1.0, 0.5, None, stream=0),
        lambda: tm.tm_dslash(L, None, 4, 18, buf, buf, None, 0, 0, 0, 0.1, 0.0, 1, stream=0),
        lambda: tm.tm_dslash_general(L, None, 4, 18, buf, buf, None, 0, 0, (0, 0, 1, 0), 1, stream=0),
        lambda: tm.tm_MdagM(L, None, 4, 18, buf, buf, buf, 0, 0.1, 0.0, 1, stream=0),
        lambda: tm.tm_M(L, None, 4, 18, buf, buf, 0.1, 0.0, 0, 1, stream=0),
        lambda: tm.tm_cg_multi(L, None, 8, None, 4, 18, buf, buf, prm, 2, buf, stream=0),
        lambda: tm.tm_cg(L, None, 8, None, 4, 18, buf, buf, prm, buf, stream=0),
        lambda: tm.tm_loop_contract(L, None, buf, 4, 1, buf, buf, stream=0),
        lambda: tm.tm_loop_contract_static(L, None, buf, 4, 1, buf, stream=0),
        lambda: tm.tm_loop_contract_ex(L, None, buf, 4, 1, 1, 0, 2j, buf, buf, stream=0),
        lambda: tm.tm_loop_contract_slice(L, None, buf, 4, 1, 0, buf, buf, stream=0),
        lambda: tm.tm_loop_momentum(L, None, buf, 4, 1, mom, buf, buf, stream=0),
        lambda: tm.tm_contract_field(L, None, buf, 4, 1, buf, stream=0),
        lambda: tm.tm_covdev(L, None, 4, 18, buf, buf, 0, 1, stream=0),
        lambda: tm.tm_time_dilute(L, None, 4, 1, [1, 0, 0, 0], buf, stream=0),
        lambda: tm.tm_hpe_remainder(L, None, 4, 18, buf, buf, buf, 0.1, 0.0, 1, stream=0),
        lambda: tm.tm_oneend_loops(L, None, 4, 18, None, tm.TM_ONEEND_TAU3, 0.1, 0.0, 1, buf, buf, stream=0),
        lambda: tm.tm_tsm_combine(4, None, None, 1, None, 0, buf, stream=0),
        lambda: tm.tm_tsm_batch_host(L, None, 2, 12, buf, prm, 2, buf, buf, stream=0),
        lambda: tm.tm_tsm_batch_host_bits(L, None, 2, 12, buf, prm, 2, buf, buf, stream=0),
    ]
    for k, call in enumerate(calls):
        with pytest.raises(tm.TmError) as e:
            call()
        assert e.value.status == tm.TM_ERR_ARG, (k, e.value.status)
    assert tm.tm_hpe_local_traces(0.16, 0.005).shape == (16,)
    assert tm.tm_loop_momentum_workspace_bytes(L, 1, 1, 0) > 0 and tm.tm_oneend_workspace_bytes(L, 4, 1) > 0
    assert tm.tm_tsm_workspace_bytes(L, 2, 2) > 0 and tm.tm_loop_workspace_bytes(L, 1) > 0
    assert isinstance(tm.tm_launch_count(), int)
