"""-m gpu: full-size parity for every remaining configuration bench.py times (SURVEY.md section 4 T2, round-1 verdict item 5).

* 32^3x64: the fp32-STORAGE 12-rhs truncated solve through the link cache (the one kernel short of L2), the temporal-gauge
  codes TM_RECON_*_TG on the whole field, tm_MdagM on the whole field, and TM_CG_HP_DEFECT x 12 with the residual recomputed by
  the oracle's full operator.
* 64^3x128: XPAY_TWIST (and its dagger) on sampled sites against the single-site oracle.
"""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel, to_dev, gather_site_inputs
from test_gpu_large import _sample_sites

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU
A = 2 * KAPPA * MU
DIMS = (32, 32, 32, 64)


def test_32x64_tsm_step_fp32_storage_through_the_link_cache():
    """bench.py `lp_batched_fp32_recon12`: 12 sources, fp32 storage, 12-real links, batched truncated CG (tol 1e-2) fed from the
    fp32 link cache, 16-Gamma loops.  Against the oracle's CG (iteration count, truncated solution), the oracle's full operator
    (residual of the returned solution), the oracle's loops, and bit-equal to the unbatched solve."""
    nrhs, prec, recon = 12, 4, 12
    U = ti.gauge(DIMS)
    F = Fields(DIMS, U, True)
    codes = np.stack([ti.z4_codes(DIMS, seed=ti.NOISE_SEED + r) for r in range(nrhs)])
    pe = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, nrhs))
    tm.tm_spinor_pack_z4(F.L, to_dev(codes), prec, nrhs, pe)
    del codes
    g = F.gauge(prec, recon)
    F.drop_canonical()
    s = F.zeros_full(prec, nrhs)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 0, 1)
    rc, info = tm.tm_cg_multi(F.L, None, 8, g, prec, recon, s, pe, prm, nrhs, ws)
    assert rc == tm.TM_OK
    T = DIMS[3]
    loops = torch.zeros((nrhs, 16, T, 2), dtype=torch.float64, device="cuda")
    lws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, nrhs))
    tm.tm_loop_contract(F.L, pe, s, prec, nrhs, loops, lws)
    loops = loops.cpu().numpy().view(np.complex128)[..., 0]
    fb = tm.tm_spinor_bytes(F.L, prec, 1, 1)
    r = 7
    eta = ti.z4(DIMS, seed=ti.NOISE_SEED + r)
    s_ref, iref = oracle.cg_solve(U, eta, KAPPA, MU, 1e-2, 500)
    s_r = F.unpack(s[r * fb:(r + 1) * fb], prec)
    assert info[r].status == tm.TM_OK and info[r].iterated_resid <= 1e-2
    assert abs(info[r].iters - iref["iters"]) <= 1
    assert rel(oracle.M(U, s_r, KAPPA, MU), eta) < 1.1 * iref["true_resid_full"]
    if info[r].iters == iref["iters"]:
        assert rel(s_r, s_ref) < 1e-4   # the same steps from x0 = 0 in fp32 storage
    assert rel(loops[r], oracle.loop(eta, s_r)) < TOL[prec]
    for q in (0, 11):  # the unbatched solve (single-rhs kernels, no link cache) gives the same bits
        s1 = F.zeros_full(prec, 1)
        ws1 = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, 1))
        rc1, info1 = tm.tm_cg_multi(F.L, None, 8, g, prec, recon, s1, pe[q * fb:(q + 1) * fb], prm, 1, ws1)
        assert rc1 == tm.TM_OK and info1[0].iters == info[q].iters
        assert torch.equal(s1, s[q * fb:(q + 1) * fb])


@pytest.mark.parametrize("prec,reals", [(2, 12), (4, 18)])
def test_32x64_temporal_gauge_codes_whole_field(prec, reals):
    """bench.py `dslash_temporal_gauge`: the field is gauge-fixed on the device by tm_gauge_fix_temporal (checked against the
    oracle's time-ordered product), packed under TM_RECON_*_TG, and the single-rhs kernel that skips the unit links is compared
    with the oracle's hop on the oracle's gauge-fixed field, whole field, both epilogue kinds."""
    code = 200 + reals
    U0 = ti.gauge(DIMS)
    U_ref, g_ref = oracle.temporal_gauge(U0)
    del g_ref
    L = tm.tm_lattice_create(DIMS, True)
    Ud = to_dev(U0)
    del U0
    gd = torch.empty(L.V * 18, dtype=torch.float64, device="cuda")
    tm.tm_gauge_fix_temporal(L, Ud, gd)
    del gd
    got_U = Ud.cpu().numpy().view(np.complex128).reshape(U_ref.shape)
    assert np.abs(got_U - U_ref).max() < 1e-12
    del got_U
    F = Fields.__new__(Fields)
    F.dims, F.L, F.V, F.U_dev, F._gauge = DIMS, L, L.V, Ud, {}
    eta = ti.z4(DIMS, seed=778)
    pin = F.pack(eta, prec)
    g = F.gauge(prec, code)
    out = F.zeros_full(prec)
    d = oracle.hop(U_ref, oracle.project(eta, 0), ap=True)
    tm.tm_dslash(F.L, g, prec, code, F.half(out, prec, 1), F.half(pin, prec, 0), None, 1, 0, tm.TM_KIND_TWIST_INV, KAPPA, MU)
    assert rel(F.unpack(out, prec), oracle.project(oracle.twist(d, A, inverse=True), 1)) < TOL[prec]
    out.zero_()
    tm.tm_dslash(F.L, g, prec, code, F.half(out, prec, 1), F.half(pin, prec, 0), F.half(pin, prec, 1), 1, 0, tm.TM_KIND_XPAY_TWIST, KAPPA, MU)
    ref = oracle.project(oracle.twist(oracle.project(eta, 1), A) - KAPPA ** 2 * d, 1)
    assert rel(F.unpack(out, prec), ref) < TOL[prec]


@pytest.mark.parametrize("prec,recon", [(4, 12), (2, 12), (8, 12)])
def test_32x64_MdagM_whole_field(prec, recon):
    """bench.py `MdagM_fp*_recon12`: four fused launches with the library's temporaries, whole field against oracle.MdagM."""
    U = ti.gauge(DIMS)
    F = Fields(DIMS, U, True)
    psi = ti.gauss_spinor(DIMS, 31)
    pin = F.pack(psi, prec)
    out = F.zeros_full(prec)
    tmp = tm.device_buffer(2 * F.pb(prec))
    tm.tm_MdagM(F.L, F.gauge(prec, recon), prec, recon, F.half(out, prec, 0), F.half(pin, prec, 0), tmp, 0, KAPPA, MU)
    ref = oracle.MdagM(U, oracle.project(psi, 0), KAPPA, MU, parity=0)
    assert rel(F.unpack(out, prec), ref) < TOL[prec]


def test_32x64_hp_defect_twelve_sources():
    """bench.py `cg_mixed_1e-8.defect_x12_fp64+fp16`: 12 sources to 1e-8 by batched defect correction (fp64 outer residual,
    fp16-storage truncated inner solves through the link cache).  The stopping rule is the FULL-system residual; it is recomputed
    here for two of the sources with the oracle's unpreconditioned operator."""
    nrhs, tol = 12, 1e-8
    U = ti.gauge(DIMS)
    F = Fields(DIMS, U, True)
    pb8 = tm.tm_spinor_bytes(F.L, 8, 1, 1)
    eta = tm.device_buffer(pb8 * nrhs)
    c1 = tm.device_buffer(F.L.V * 12)
    for r in range(nrhs):
        c1.copy_(torch.from_numpy(ti.z4_codes(DIMS, seed=ti.NOISE_SEED + 900 + r).reshape(-1)))
        tm.tm_spinor_pack_z4(F.L, c1, 8, 1, eta[r * pb8:(r + 1) * pb8])
    g8, g2 = F.gauge(8, 12), F.gauge(2, 12)
    F.drop_canonical()
    s = tm.device_buffer(pb8 * nrhs)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 2, tm.TM_CG_HP_DEFECT, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, tol, 5000, tm.TM_CG_HP_DEFECT, 0.0)
    rc, info = tm.tm_cg_multi(F.L, g8, 8, g2, 2, 12, s, eta, prm, nrhs, ws)
    assert rc == tm.TM_OK
    for r in range(nrhs):
        assert info[r].status == tm.TM_OK and 0 < info[r].true_resid <= tol and 2 <= info[r].reliable_updates <= 8
    for r in (0, 11):
        e = ti.z4(DIMS, seed=ti.NOISE_SEED + 900 + r)
        s_r = F.unpack(s[r * pb8:(r + 1) * pb8], 8)
        res = np.linalg.norm((e - oracle.M(U, s_r, KAPPA, MU)).ravel()) / np.linalg.norm(e.ravel())
        assert res <= 1.05 * tol and abs(res - info[r].true_resid) <= 0.05 * tol


def test_32x64_hp_defect_one_source():
    """bench.py `cg_mixed_1e-8.defect_x1_fp64+fp16` (configs[2]: mixed-precision CG to 1e-8 on ONE source): nrhs = 1 runs the fused
    single-rhs iteration without a link cache; full-system residual recomputed with the oracle's operator."""
    tol = 1e-8
    U = ti.gauge(DIMS)
    F = Fields(DIMS, U, True)
    e = ti.z4(DIMS, seed=ti.NOISE_SEED + 77)
    eta = F.pack(e, 8)
    g8, g2 = F.gauge(8, 12), F.gauge(2, 12)
    F.drop_canonical()
    s = F.zeros_full(8)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 2, tm.TM_CG_HP_DEFECT, 1))
    prm = tm.make_cg_params(KAPPA, MU, tol, 5000, tm.TM_CG_HP_DEFECT, 0.0)
    rc, info = tm.tm_cg_multi(F.L, g8, 8, g2, 2, 12, s, eta, prm, 1, ws)
    assert rc == tm.TM_OK and info[0].status == tm.TM_OK and 0 < info[0].true_resid <= tol
    res = np.linalg.norm((e - oracle.M(U, F.unpack(s, 8), KAPPA, MU)).ravel()) / np.linalg.norm(e.ravel())
    assert res <= 1.05 * tol and abs(res - info[0].true_resid) <= 0.05 * tol


def test_64x128_xpay_twist_sampled_sites():
    """configs[4] `xpay_twist_*` rows: out = R(+-a) x - kappa^2 D in (dagger too), fp32 and fp16 storage, 18- and 12-real links,
    on ~3e4 sampled sites per case (random + two planes that touch every wrap-around) against the single-site oracle."""
    dims = (64, 64, 64, 128)
    X, Y, Z, T = dims
    seed = ti.NOISE_SEED
    F = Fields.from_slabs(dims, True)
    gauges = {(p, r): F.gauge(p, r) for p in (4, 2) for r in (18, 12)}
    F.drop_canonical()
    codes = torch.empty((T, Z, Y, X, 4, 3), dtype=torch.uint8, device="cuda")
    for t0 in range(0, T, 16):
        codes[t0:t0 + 16].copy_(torch.from_numpy(ti.z4_codes(dims, seed=seed, t0=t0, t1=t0 + 16)))
    parity = 0
    sites = _sample_sites(dims, parity, 15000, 21)
    Uf, Ub, nf, nb, sf, sb = gather_site_inputs(dims, sites, seed, ap=True)
    xs = ti.z4_sites(sites, seed=seed).reshape(-1, 1, 1, 1, 4, 3)
    refs = {}
    for dagger in (0, 1):
        d = np.stack([oracle.hop_gathered(Uf[k], Ub[k], nf[k], nb[k], sf[k], sb[k], dagger=bool(dagger)) for k in range(sites.size)])
        a = -A if dagger else A
        refs[dagger] = (oracle.twist(xs, a) - KAPPA ** 2 * d.reshape(-1, 1, 1, 1, 4, 3)).reshape(-1, 4, 3)
    canon = torch.empty((T * Z * Y * X, 4, 3, 2), dtype=torch.float64, device="cuda")
    idx = torch.from_numpy(sites).cuda()
    for prec in (4, 2):
        pin = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, 1))
        tm.tm_spinor_pack_z4(F.L, codes, prec, 1, pin)
        out = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, 1))
        for recon in (18, 12):
            for dagger in (0, 1):
                out.zero_()
                tm.tm_dslash(F.L, gauges[(prec, recon)], prec, recon, F.half(out, prec, parity), F.half(pin, prec, 1 - parity),
                             F.half(pin, prec, parity), parity, dagger, tm.TM_KIND_XPAY_TWIST, KAPPA, MU)
                tm.tm_spinor_unpack(F.L, out, prec, 1, canon)
                torch.cuda.synchronize()
                got = canon[idx].cpu().numpy().view(np.complex128)[..., 0]
                assert rel(got, refs[dagger]) < TOL[prec], (prec, recon, dagger)
                worst = np.abs(got - refs[dagger]).reshape(sites.size, -1).max(axis=1).max() / np.abs(refs[dagger]).max()
                assert worst < 20 * TOL[prec], (prec, recon, dagger, worst)
