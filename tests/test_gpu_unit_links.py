"""-m gpu: special gauge fields -- the temporal-gauge copy of the synthetic field (unit temporal links on all slices but the last, where
the Polyakov loop meets the antiperiodic sign) and the free field -- through the batched solver, and the gauge invariance of the loops
through the GPU.  (Skipping the SU(3) product of unit links in the 12-rhs kernel was measured and not kept; these
fields stay as parity cases: 12-real reconstruction of exact unit links, a boundary slice that differs from all others.)"""
import numpy as np
import pytest

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, rel
from test_gpu_cg import solve

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU


@pytest.mark.parametrize("prec", [2, 4])
def test_temporal_gauge_batched_solve(prec):
    """12 truncated solves on the temporal-gauge copy of the synthetic field (unit temporal links on 15 of 16 slices, the Polyakov
    loop on the last, antiperiodic sign on top): against the oracle's CG on the same field, and bit-equal to the unbatched solve."""
    dims = (8, 8, 8, 16)
    U, g = oracle.temporal_gauge(ti.gauge(dims))
    F = Fields(dims, U, True)
    nrhs = 12
    eta = np.stack([ti.z4(dims, seed=ti.NOISE_SEED + r) for r in range(nrhs)])
    rc, info, s = solve(F, eta, 8, prec, 12, tm.TM_CG_LP_TRUNCATED, 1e-2, 500, nrhs=nrhs)
    assert rc == tm.TM_OK
    for r in (0, 5, 11):
        s_ref, iref = oracle.cg_solve(U, eta[r], KAPPA, MU, 1e-2, 500)
        assert info[r].status == tm.TM_OK and abs(info[r].iters - iref["iters"]) <= 2
        assert rel(s[r], s_ref) < (2e-2 if prec == 2 else 1e-4)
    rc1, info1, s1 = solve(F, eta[5], 8, prec, 12, tm.TM_CG_LP_TRUNCATED, 1e-2, 500)
    assert info1[0].iters == info[5].iters and np.array_equal(s1, s[5])


def test_loops_are_gauge_invariant_through_the_gpu():
    """eta' = g eta solved on the temporal-gauge field gives the loops of eta on the original field (the reason the gauge may be
    fixed at all): both solved to 1e-9 on the GPU, loops contracted on the GPU."""
    dims = (4, 4, 4, 8)
    U0 = ti.gauge(dims)
    U1, g = oracle.temporal_gauge(U0)
    eta0 = ti.z4(dims, seed=77)
    eta1 = np.einsum("tzyxab,tzyxsb->tzyxsa", g, eta0)
    loops = []
    for U, eta in ((U0, eta0), (U1, eta1)):
        F = Fields(dims, U, True)
        rc, info, s = solve(F, eta, 8, 4, 12, tm.TM_CG_HP_MIXED, 1e-9, 5000)
        assert rc == tm.TM_OK
        loops.append(oracle.loop(eta, s))
    assert rel(loops[1], loops[0]) < 1e-7


def test_free_field_batched_solve():
    """U = 1, periodic in time, 18-real links, a lattice with four different extents: 12 solves against the oracle."""
    dims = (8, 4, 6, 4)
    U = ti.unit_gauge(dims)
    F = Fields(dims, U, False)
    nrhs = 12
    eta = np.stack([ti.z4(dims, seed=300 + r) for r in range(nrhs)])
    pe = F.pack(eta, 2)
    s = F.zeros_full(2, nrhs)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 2, tm.TM_CG_LP_TRUNCATED, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 4)
    rc, info = tm.tm_cg_multi(F.L, None, 8, F.gauge(2, 18), 2, 18, s, pe, prm, nrhs, ws)
    assert rc == tm.TM_OK
    got = F.unpack(s, 2, nrhs=nrhs)
    for r in (0, 11):
        s_ref, iref = oracle.cg_solve(U, eta[r], KAPPA, MU, 1e-2, 500, ap=False)
        assert abs(info[r].iters - iref["iters"]) <= 2 and rel(got[r], s_ref) < 2e-2
