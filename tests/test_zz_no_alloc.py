"""-m gpu: tm_loop_contract_static, the loop contraction for callers that cannot allocate device memory (tm.h).

Collected last on purpose (file name): the suite runs with `pytest -x`, a failure here must not hide other tests.  The entry
point keeps its scratch in a file-scope device array that all calls share and that keeps the last call's contents, so the
checks run twice in a row with different inputs and shapes: against the existing path (tm_loop_contract with a caller
workspace; same kernels, so far inside the tolerance of the other tests) and against the oracle."""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel

pytestmark = pytest.mark.gpu


def _both_paths(F, a, b, prec, nrhs):
    pa, pb = F.pack(a, prec), F.pack(b, prec)
    T = F.dims[3]
    ref = torch.zeros((nrhs, 16, T, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, nrhs))
    tm.tm_loop_contract(F.L, pa, pb, prec, nrhs, ref, ws)
    got = torch.full((nrhs, 16, T, 2), float("nan"), dtype=torch.float64, device="cuda")
    tm.tm_loop_contract_static(F.L, pa, pb, prec, nrhs, got)
    torch.cuda.synchronize()
    return got.cpu().numpy().view(np.complex128)[..., 0], ref.cpu().numpy().view(np.complex128)[..., 0]


@pytest.mark.parametrize("prec", [8, 4, 2])
def test_static_scratch_equals_workspace_path_two_calls_in_a_row(prec):
    # call 1: 12 sources on 8^3 x 16 (several blocks per time slice); call 2: other fields, another lattice and source count,
    # so that stale partials of call 1 lie under and beside the ones call 2 uses
    for call, (dims, nrhs, seed) in enumerate((((8, 8, 8, 16), 12, 40), ((4, 6, 4, 8), 3, 60))):
        U = ti.gauge(dims)
        F = Fields(dims, U, True)
        a = np.stack([ti.z4(dims, seed=seed + r) for r in range(nrhs)])
        b = np.stack([ti.gauss_spinor(dims, seed + 100 + r) for r in range(nrhs)])
        got, ref = _both_paths(F, a, b, prec, nrhs)
        assert np.isfinite(got).all()
        assert rel(got, ref) < TOL[8], (call, prec)           # same kernels, same summation order
        for r in (0, nrhs - 1):
            assert rel(got[r], oracle.loop(a[r], b[r])) < TOL[prec], (call, prec, r)


def test_static_scratch_limit_is_enforced_without_a_launch():
    """64^3 x 128 with 16 sources needs 16 MiB of partials: refused with TM_ERR_STATIC_LIMIT before anything is touched (the
    buffers here are dummies); the same lattice with 8 sources is within the limit by size."""
    L = tm.tm_lattice_create((64, 64, 64, 128), True)
    assert tm.tm_loop_workspace_bytes(L, 16) > tm.TM_LOOP_STATIC_BYTES >= tm.tm_loop_workspace_bytes(L, 8)
    dummy = tm.device_buffer(1024)
    n0 = tm.tm_launch_count()
    with pytest.raises(tm.TmError) as e:
        tm.tm_loop_contract_static(L, dummy, dummy, 2, 16, dummy)
    assert e.value.status == tm.TM_ERR_STATIC_LIMIT and "TM_LOOP_STATIC_BYTES" in str(e.value)
    assert tm.tm_launch_count() == n0
    L32 = tm.tm_lattice_create((32, 32, 32, 64), True)
    assert tm.tm_loop_workspace_bytes(L32, 16) <= tm.TM_LOOP_STATIC_BYTES   # the benchmark lattice: up to 16 sources per call
