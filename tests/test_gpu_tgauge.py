"""-m gpu: fields DECLARED in temporal gauge (TM_RECON_18_TG / TM_RECON_12_TG, include/tm.h): the single-rhs fp32 / fp16 hopping-term
kernels load no link and multiply by none on temporal hops inside the lattice; everything else reads the stored unit links."""
import numpy as np
import pytest

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel
from test_gpu_parity import oracle_dslash, run_dslash
from test_gpu_cg import solve

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU
TG = {18: tm.TM_RECON_18_TG, 12: tm.TM_RECON_12_TG}
_cache = {}


def tg_fields(dims, ap=True):
    key = (tuple(dims), ap)
    if key not in _cache:
        U = oracle.temporal_gauge(ti.gauge(dims))[0]
        _cache[key] = (Fields(dims, U, ap), U)
    return _cache[key]


@pytest.mark.parametrize("dims", [(4, 6, 8, 10), (8, 8, 8, 16), (6, 6, 6, 6)])
@pytest.mark.parametrize("prec", [8, 4, 2])
@pytest.mark.parametrize("reals", [18, 12])
def test_tg_dslash_all_kinds(dims, prec, reals):
    """Every kind x parity x dagger against the oracle on the gauge-fixed field (fp64 ignores the declaration), and bit-equal to the
    plain code on the same field: skipping a unit link is what multiplying by it gives."""
    F, U = tg_fields(dims)
    psi, x = ti.gauss_spinor(dims, 3), ti.gauss_spinor(dims, 4)
    for out_parity in (0, 1):
        for dagger in (0, 1):
            for kind in (0, 1, 2):
                got = run_dslash(F, prec, TG[reals], psi, x, out_parity, dagger, kind)
                ref = oracle_dslash(U, psi, x, out_parity, dagger, kind)
                assert rel(got, ref) < TOL[prec], (dims, prec, reals, out_parity, dagger, kind)
                assert np.array_equal(got, run_dslash(F, prec, reals, psi, x, out_parity, dagger, kind))


def test_tg_periodic_time_and_free_field():
    """Periodic time direction (no boundary sign) and the unit field, where the wrapping hop crosses a unit link too."""
    dims = (4, 4, 4, 8)
    F, U = tg_fields(dims, ap=False)
    psi = ti.gauss_spinor(dims, 9)
    for prec in (4, 2):
        got = run_dslash(F, prec, TG[12], psi, psi, 1, 0, 1)
        assert rel(got, oracle_dslash(U, psi, psi, 1, 0, 1, ap=False)) < TOL[prec]
    U1 = ti.unit_gauge(dims)
    F1 = Fields(dims, U1, True)
    got = run_dslash(F1, 4, TG[18], psi, psi, 0, 1, 2)
    assert rel(got, oracle_dslash(U1, psi, psi, 0, 1, 2)) < TOL[4]


def test_tg_pack_refuses_a_field_that_is_not_gauge_fixed():
    dims = (4, 4, 4, 4)
    F = Fields(dims, ti.gauge(dims), True)
    for prec in (8, 4, 2):
        buf = tm.device_buffer(tm.tm_gauge_bytes(F.L, prec, TG[12]))
        assert tm.tm_gauge_bytes(F.L, prec, TG[12]) == tm.tm_gauge_bytes(F.L, prec, 12)
        with pytest.raises(tm.TmError) as e:
            tm.tm_gauge_pack(F.L, F.U_dev, prec, TG[12], buf, 1e-10)
        assert e.value.status == tm.TM_ERR_NOT_TGAUGE


@pytest.mark.parametrize("prec", [4, 2])
def test_tg_multi_rhs_MdagM_and_solves(prec):
    """Multi-rhs launches, MdagM and the solvers accept the declaration (multi-rhs kernels read the stored unit links)."""
    dims = (8, 8, 8, 16)
    F, U = tg_fields(dims)
    psi = ti.gauss_spinor(dims, 31)
    p1, o1 = F.pack(psi, prec), F.zeros_full(prec)
    tmp = tm.device_buffer(2 * F.pb(prec))
    tm.tm_MdagM(F.L, F.gauge(prec, TG[12]), prec, TG[12], F.half(o1, prec, 0), F.half(p1, prec, 0), tmp, 0, KAPPA, MU)
    assert rel(F.unpack(o1, prec), oracle.MdagM(U, oracle.project(psi, 0), KAPPA, MU, parity=0)) < TOL[prec]
    nrhs = 12
    eta = np.stack([ti.z4(dims, seed=ti.NOISE_SEED + r) for r in range(nrhs)])
    rc, info, s = solve(F, eta, 8, prec, TG[12], tm.TM_CG_LP_TRUNCATED, 1e-2, 500, nrhs=nrhs)
    assert rc == tm.TM_OK
    s_ref, iref = oracle.cg_solve(U, eta[3], KAPPA, MU, 1e-2, 500)
    assert abs(info[3].iters - iref["iters"]) <= 2 and rel(s[3], s_ref) < (2e-2 if prec == 2 else 1e-4)
    rc, info1, s1 = solve(F, eta[3], 8, prec, TG[12], tm.TM_CG_LP_TRUNCATED, 1e-2, 500)  # unbatched: the kernels that skip
    assert rc == tm.TM_OK and info1[0].iters == info[3].iters and np.array_equal(s1, s[3])
    rc, infoh, sh = solve(F, eta[0], 8, prec, TG[12], tm.TM_CG_HP_MIXED, 1e-9, 3000)
    assert rc == tm.TM_OK and infoh[0].true_resid < 1e-9


@pytest.mark.parametrize("dims", [(4, 6, 8, 10), (8, 8, 8, 16)])
def test_gauge_fix_temporal_on_the_device(dims):
    """tm_gauge_fix_temporal against the input-preparation routine pinned by P25 (oracle.temporal_gauge): the transformed field and
    the transformation to rounding, exact unit links where they belong, and the result is accepted under the temporal-gauge code."""
    import torch
    from tm_harness import to_dev
    U0 = ti.gauge(dims)
    U_ref, g_ref = oracle.temporal_gauge(U0)
    L = tm.tm_lattice_create(dims, True)
    U_dev = to_dev(U0)
    g_dev = torch.empty(L.V * 18, dtype=torch.float64, device="cuda")
    tm.tm_gauge_fix_temporal(L, U_dev, g_dev)
    torch.cuda.synchronize()
    U_got = U_dev.cpu().numpy().view(np.complex128).reshape(U0.shape)
    g_got = g_dev.cpu().numpy().view(np.complex128).reshape(g_ref.shape)
    assert np.abs(g_got - g_ref).max() < 1e-13
    assert np.abs(U_got - U_ref).max() < 1e-13
    assert np.array_equal(U_got[:-1, ..., 3, :, :], U_ref[:-1, ..., 3, :, :])  # exactly 1
    buf = tm.device_buffer(tm.tm_gauge_bytes(L, 4, TG[12]))
    tm.tm_gauge_pack(L, U_dev, 4, TG[12], buf, 1e-10)  # raises on TM_ERR_NOT_TGAUGE / TM_ERR_NOT_SU3
