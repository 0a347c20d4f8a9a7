"""-m gpu: tm_cg / tm_cg_multi / tm_tsm_batch_host against the oracle CG (an iteration: pinned by residuals, iteration
counts and sqrt(cond)*tol bounds, never bit-equality -- DESIGN.md readings 9-12, 23)."""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, rel, to_dev

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU

_cache = {}


def fields(dims):
    if dims not in _cache:
        U = ti.gauge(dims)
        _cache[dims] = (Fields(dims, U, True), U)
    return _cache[dims]


def solve(F, eta, prec_hp, prec_lp, recon, mode, tol, max_iter, nrhs=None, check_every=4):
    n = 1 if nrhs is None else nrhs
    prec_io = prec_hp if mode == tm.TM_CG_HP_MIXED else prec_lp
    pe = F.pack(eta, prec_io)
    s = F.zeros_full(prec_io, n)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, prec_hp, prec_lp, mode, n))
    prm = tm.make_cg_params(KAPPA, MU, tol, max_iter, mode, 0.1, check_every)
    rc, info = tm.tm_cg_multi(F.L, F.gauge(prec_hp, recon), prec_hp, F.gauge(prec_lp, recon), prec_lp, recon, s, pe, prm, n, ws)
    return rc, info, F.unpack(s, prec_io, nrhs=nrhs)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10)])
def test_cg_fp64_matches_oracle_cg(dims):
    """configs[0]: CG to 1e-12 in pure fp64 (LP_TRUNCATED mode with prec_lp = fp64 is plain CG in one precision)."""
    F, U = fields(dims)
    eta = ti.z4(dims)
    s_ref, iref = oracle.cg_solve(U, eta, KAPPA, MU, 1e-12, 2000)
    rc, info, s = solve(F, eta, 8, 8, 18, tm.TM_CG_LP_TRUNCATED, 1e-12, 2000, check_every=1)
    assert rc == tm.TM_OK and info[0].status == tm.TM_OK
    assert abs(info[0].iters - iref["iters"]) <= 1           # P15
    assert info[0].iterated_resid <= 1e-12 and info[0].true_resid < 3e-12
    res_full = rel(oracle.M(U, s, KAPPA, MU), eta)            # P8 with the full unpreconditioned oracle operator
    assert res_full < 1e-10
    assert rel(s, s_ref) < 1e-9
    # fixed-iteration truncation (reading 12): tol = 0 runs exactly max_iter
    rc, info, s5 = solve(F, eta, 8, 8, 18, tm.TM_CG_LP_TRUNCATED, 0.0, 5)
    s5_ref, i5 = oracle.cg_solve(U, eta, KAPPA, MU, 0.0, 5)
    assert rc == tm.TM_OK and info[0].iters == 5 and i5["iters"] == 5
    assert rel(s5, s5_ref) < 1e-11                            # same x0 = 0, same 5 steps
    # max_iter reached before tol
    rc, info, _ = solve(F, eta, 8, 8, 18, tm.TM_CG_LP_TRUNCATED, 1e-12, 3)
    assert rc == tm.TM_ERR_MAXITER and info[0].iters == 3


@pytest.mark.parametrize("prec_lp,recon", [(4, 18), (4, 12), (2, 12), (2, 18)])
def test_cg_hp_mixed(prec_lp, recon):
    """configs[2]: mixed-precision CG to relative residual 1e-8 (fp64 outer, fp32 or fp16-storage inner)."""
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    eta = ti.z4(dims)
    rc, info, s = solve(F, eta, 8, prec_lp, recon, tm.TM_CG_HP_MIXED, 1e-8, 4000)
    s_ref, iref = oracle.cg_solve(U, eta, KAPPA, MU, 1e-8, 2000)
    assert rc == tm.TM_OK, (rc, info[0].iters, info[0].true_resid)
    assert info[0].true_resid <= 1e-8 and info[0].reliable_updates >= 1
    assert rel(oracle.M(U, s, KAPPA, MU), eta) < 2e-7        # c * tol, c = O(sqrt(cond)) (reading 9)
    assert rel(s, s_ref) < 1e-6
    assert info[0].iters <= (2 if prec_lp == 4 else 4) * iref["iters"] + 10


@pytest.mark.parametrize("prec,recon", [(2, 12), (2, 18), (4, 12), (2, 8), (4, 8)])
def test_cg_lp_truncated_batched(prec, recon):
    """configs[3] in small: 12 truncated solves (tol 1e-2) sharing every gauge load; batched == unbatched bit for bit."""
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    nrhs = 12
    eta = np.stack([ti.z4(dims, seed=ti.NOISE_SEED + r) for r in range(nrhs)])
    rc, info, s = solve(F, eta, 8, prec, recon, tm.TM_CG_LP_TRUNCATED, 1e-2, 500, nrhs=nrhs)
    assert rc == tm.TM_OK
    for r in range(nrhs):
        s_ref, iref = oracle.cg_solve(U, eta[r], KAPPA, MU, 1e-2, 500)
        assert info[r].status == tm.TM_OK and info[r].iterated_resid <= 1e-2
        assert abs(info[r].iters - iref["iters"]) <= 2       # P15
        assert info[r].true_resid < 1.3e-2
        # truncated solution: same x0 = 0 and (nearly) the same steps -> close to the oracle's truncated solution
        assert rel(s[r], s_ref) < (2e-2 if prec == 2 else 1e-4)
    for r in (0, 7):
        rc1, info1, s1 = solve(F, eta[r], 8, prec, recon, tm.TM_CG_LP_TRUNCATED, 1e-2, 500)
        assert info1[0].iters == info[r].iters
        assert np.array_equal(s1, s[r])


def test_cg_zero_source_and_mixed_convergence_times():
    dims = (4, 4, 4, 4)
    F, U = fields(dims)
    eta = np.stack([ti.z4(dims, seed=1), np.zeros_like(ti.z4(dims)), 1e-3 * ti.gauss_spinor(dims, 2)])
    rc, info, s = solve(F, eta, 8, 4, 18, tm.TM_CG_LP_TRUNCATED, 1e-5, 500, nrhs=3, check_every=3)
    assert rc == tm.TM_OK and info[1].iters == 0 and not s[1].any()
    for r in (0, 2):
        assert rel(oracle.M(U, s[r], KAPPA, MU), eta[r]) < 1e-4
    # x_0 = 0 is the solver's own business (written by the first iteration's vector kernel, or by a memset when max_iter = 0): a
    # solution buffer full of garbage changes nothing, and the zero source still gets an all-zero solution
    for prec, max_iter in ((4, 500), (2, 500), (4, 0)):
        pe = F.pack(eta, prec)
        sd = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, 3))
        sd.fill_(0x3C)
        ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, 3))
        prm = tm.make_cg_params(KAPPA, MU, 1e-2, max_iter, tm.TM_CG_LP_TRUNCATED)
        rc2, info2 = tm.tm_cg_multi(F.L, None, 8, F.gauge(prec, 18), prec, 18, sd, pe, prm, 3, ws)
        got = F.unpack(sd, prec, nrhs=3)
        assert not got[1].any() and np.isfinite(got).all()
        if max_iter == 0:
            assert not oracle.project(got[0], 0).any()   # no iteration: s_e = x_0 = 0, s_o = R^-1 eta_o
        else:
            assert rc2 == tm.TM_OK and rel(oracle.M(U, got[0], KAPPA, MU), eta[0]) < 3e-2


def test_skip_true_resid_changes_nothing_but_the_report():
    """tm_cg_params.skip_true_resid drops the diagnostic M^dag M after a truncated solve: same solution bit for bit."""
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    nrhs, prec, recon = 5, 2, 12  # 5: also covers a right-hand-side count that does not fill the CTA's rhs rows
    eta = np.stack([ti.z4(dims, seed=800 + r) for r in range(nrhs)])
    pe = F.pack(eta, prec)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, nrhs))
    sols = []
    for skip in (0, 1):
        s = F.zeros_full(prec, nrhs)
        prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 4, skip)
        rc, info = tm.tm_cg_multi(F.L, None, 8, F.gauge(prec, recon), prec, recon, s, pe, prm, nrhs, ws)
        assert rc == tm.TM_OK
        for r in range(nrhs):
            assert info[r].iterated_resid <= 1e-2
            assert (info[r].true_resid == -1.0) if skip else (0 < info[r].true_resid < 1.3e-2)
        sols.append(s.clone())
    assert torch.equal(sols[0], sols[1])


def test_tsm_batch_host_end_to_end():
    """H2D of Z2xiZ2 codes -> pack -> batched truncated CG -> 16-Gamma loop per time slice -> D2H, one call."""
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    nrhs, prec, recon = 4, 2, 12
    codes = np.stack([ti.z4_codes(dims, seed=300 + r) for r in range(nrhs)])
    codes_host = torch.from_numpy(codes).pin_memory()
    loops_host = torch.zeros((nrhs, 16, dims[3], 2), dtype=torch.float64).pin_memory()
    ws = tm.device_buffer(tm.tm_tsm_workspace_bytes(F.L, prec, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED)
    rc, info = tm.tm_tsm_batch_host(F.L, F.gauge(prec, recon), prec, recon, codes_host, prm, nrhs, loops_host, ws)
    assert rc == tm.TM_OK
    got = loops_host.numpy().view(np.complex128)[..., 0]
    for r in range(nrhs):
        eta = ti.z4(dims, seed=300 + r)
        s_ref, iref = oracle.cg_solve(U, eta, KAPPA, MU, 1e-2, 500)
        assert abs(info[r].iters - iref["iters"]) <= 2
        ref = oracle.loop(eta, s_ref)
        assert rel(got[r], ref) < 3e-2  # LP solution differs from the oracle's at the truncation level
    # bit-packed noise (3 bytes per site over PCIe): identical field, identical loops
    bits = np.stack([ti.z4_bits(dims, seed=300 + r) for r in range(nrhs)])
    a, b = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, nrhs)), tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, nrhs))
    tm.tm_spinor_pack_z4(F.L, torch.from_numpy(codes).cuda(), prec, nrhs, a)
    tm.tm_spinor_pack_z4_bits(F.L, torch.from_numpy(bits).cuda(), prec, nrhs, b)
    assert torch.equal(a, b)
    loops2 = torch.zeros_like(loops_host).pin_memory()
    rc2, info2 = tm.tm_tsm_batch_host_bits(F.L, F.gauge(prec, recon), prec, recon, torch.from_numpy(bits).pin_memory(), prm, nrhs, loops2, ws)
    assert rc2 == tm.TM_OK and torch.equal(loops2, loops_host)


def test_full_dilution_exact_trace_4x4():
    """north_star pin through the GPU: unit sources on one time slice of 4^4 -> Tr_t[Gamma M^-1] from the dense inverse."""
    from oracle import dense
    dims = (4, 4, 4, 4)
    F, U = fields(dims)
    Minv = np.linalg.inv(dense.dense_M(U, KAPPA, MU, ap=True))
    ref = dense.timeslice_traces(Minv, dims)
    t = 3
    nrhs = 12
    acc = np.zeros((16, 4), dtype=np.complex128)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 8, tm.TM_CG_LP_TRUNCATED, nrhs))
    lws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, nrhs))
    out = torch.zeros((nrhs, 16, 4, 2), dtype=torch.float64, device="cuda")
    prm = tm.make_cg_params(KAPPA, MU, 1e-11, 2000, tm.TM_CG_LP_TRUNCATED, 0.1, 8)
    g = F.gauge(8, 18)
    for site in range(64):
        e = np.zeros((nrhs, 4, 4, 4, 4, 4, 3), dtype=np.complex128)
        for k in range(12):
            e[k].reshape(-1)[(t * 64 + site) * 12 + k] = 1
        pe = F.pack(e, 8)
        s = F.zeros_full(8, nrhs)
        rc, info = tm.tm_cg_multi(F.L, g, 8, g, 8, 18, s, pe, prm, nrhs, ws)
        assert rc == tm.TM_OK
        tm.tm_loop_contract(F.L, pe, s, 8, nrhs, out, lws)
        acc += out.cpu().numpy().view(np.complex128)[..., 0].sum(axis=0)
    assert np.abs(acc[:, :3]).max() < 1e-12
    assert rel(acc[:, t], ref[:, t]) < 1e-9


@pytest.mark.parametrize("prec_lp,recon", [(2, 12), (4, 12), (4, 18)])
def test_cg_hp_defect_batched(prec_lp, recon):
    """TM_CG_HP_DEFECT: fp64 outer residual, batched truncated inner solves (reading 10, second scheme).  The stopping
    rule is the FULL-system residual |eta - M s| <= tol |eta|, checked here with the oracle's unpreconditioned operator (P8)."""
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    nrhs, tol = 3, 1e-9
    eta = np.stack([ti.z4(dims, seed=400 + r) for r in range(nrhs)])
    pe = F.pack(eta, 8)
    s = F.zeros_full(8, nrhs)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec_lp, tm.TM_CG_HP_DEFECT, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, tol, 2000, tm.TM_CG_HP_DEFECT, 0.0)
    rc, info = tm.tm_cg_multi(F.L, F.gauge(8, recon), 8, F.gauge(prec_lp, recon), prec_lp, recon, s, pe, prm, nrhs, ws)
    assert rc == tm.TM_OK
    got = F.unpack(s, 8, nrhs=nrhs)
    for r in range(nrhs):
        assert info[r].status == tm.TM_OK and 0 < info[r].true_resid <= tol
        res = np.linalg.norm((eta[r] - oracle.M(U, got[r], KAPPA, MU)).ravel()) / np.linalg.norm(eta[r].ravel())
        assert res <= 1.05 * tol and abs(res - info[r].true_resid) <= 0.05 * tol
        s_ref, iref = oracle.cg_solve(U, eta[r], KAPPA, MU, 1e-12, 4000)
        assert rel(got[r], s_ref) < 20 * tol
        assert 2 <= info[r].reliable_updates <= 8 and info[r].iters >= iref["iters"] // 3


def test_cg_lp_truncated_ragged_6x6x6x6():
    """Vh = 648: the last 32-site tile of the link-cache kernel holds 8 sites and the fp16 parity block (33 696 B) is not a
    multiple of 256 B; 12 right-hand sides, iteration counts against the oracle CG, batched == unbatched bit for bit."""
    dims = (6, 6, 6, 6)
    F, U = fields(dims)
    nrhs, prec, recon = 12, 2, 12
    eta = np.stack([ti.z4(dims, seed=800 + r) for r in range(nrhs)])
    pe = F.pack(eta, prec)
    s = F.zeros_full(prec, nrhs)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED)
    rc, info = tm.tm_cg_multi(F.L, None, 8, F.gauge(prec, recon), prec, recon, s, pe, prm, nrhs, ws)
    assert rc == tm.TM_OK
    got = F.unpack(s, prec, nrhs=nrhs)
    for r in (0, 11):
        s_ref, iref = oracle.cg_solve(U, eta[r], KAPPA, MU, 1e-2, 500)
        assert abs(info[r].iters - iref["iters"]) <= 2
        assert rel(got[r], s_ref) < 3e-2
    s1 = F.zeros_full(prec, 1)
    ws1 = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, 1))
    fb = tm.tm_spinor_bytes(F.L, prec, 1, 1)
    e1 = tm.device_buffer(fb)  # the slice of the batch is only 16-byte aligned on this lattice: copy to an aligned buffer
    e1.copy_(pe[5 * fb:6 * fb])
    rc1, info1 = tm.tm_cg(F.L, None, 8, F.gauge(prec, recon), prec, recon, s1, e1, prm, ws1)
    assert rc1 == tm.TM_OK and info1.iters == info[5].iters
    assert torch.equal(s1, s[5 * fb:6 * fb])


@pytest.mark.parametrize("nrhs", [7, 8, 9])
@pytest.mark.parametrize("prec", [2, 4])
def test_cg_lp_truncated_seven_to_nine_rhs(nrhs, prec):
    """7 and 8 right-hand sides take the 8-rhs launch shape of the link-cache kernel (the last batch of 200 sources, N_HP = 8), 9 the
    12-rhs shape with three idle rows: oracle iteration counts, and every source bit-equal to its unbatched solve."""
    dims = (6, 6, 6, 6)
    F, U = fields(dims)
    recon = 12
    eta = np.stack([ti.z4(dims, seed=820 + r) for r in range(nrhs)])
    pe = F.pack(eta, prec)
    s = F.zeros_full(prec, nrhs)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED)
    rc, info = tm.tm_cg_multi(F.L, None, 8, F.gauge(prec, recon), prec, recon, s, pe, prm, nrhs, ws)
    assert rc == tm.TM_OK
    got = F.unpack(s, prec, nrhs=nrhs)
    s_ref, iref = oracle.cg_solve(U, eta[nrhs - 1], KAPPA, MU, 1e-2, 500)
    assert abs(info[nrhs - 1].iters - iref["iters"]) <= 2 and rel(got[nrhs - 1], s_ref) < 3e-2
    fb = tm.tm_spinor_bytes(F.L, prec, 1, 1)
    ws1 = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, 1))
    e1, s1 = tm.device_buffer(fb), tm.device_buffer(fb)
    for r in (0, nrhs - 1):
        e1.copy_(pe[r * fb:(r + 1) * fb])
        s1.zero_()
        rc1, info1 = tm.tm_cg(F.L, None, 8, F.gauge(prec, recon), prec, recon, s1, e1, prm, ws1)
        assert rc1 == tm.TM_OK and info1.iters == info[r].iters
        assert torch.equal(s1, s[r * fb:(r + 1) * fb])


def test_cg_breakdown_is_per_rhs():
    """A NaN source makes <p,Ap> NaN: that right-hand side stops with TM_ERR_BREAKDOWN, the others of the batch converge."""
    dims = (4, 4, 4, 8)
    F, U = fields(dims)
    nrhs = 3
    eta = np.stack([ti.z4(dims, seed=950 + r) for r in range(nrhs)])
    eta[1, 2, 1, 3, 0, 1, 2] = np.nan
    for prec in (4, 2):
        pe = F.pack(eta, prec)
        s = F.zeros_full(prec, nrhs)
        ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, nrhs))
        prm = tm.make_cg_params(KAPPA, MU, 1e-2, 200, tm.TM_CG_LP_TRUNCATED)
        rc, info = tm.tm_cg_multi(F.L, None, 8, F.gauge(prec, 12), prec, 12, s, pe, prm, nrhs, ws)
        assert rc == tm.TM_ERR_BREAKDOWN
        assert [i.status for i in info] == [tm.TM_OK, tm.TM_ERR_BREAKDOWN, tm.TM_OK]
        got = F.unpack(s, prec, nrhs=nrhs)
        for r in (0, 2):
            s_ref, _ = oracle.cg_solve(U, eta[r], KAPPA, MU, 1e-2, 200)
            assert rel(got[r], s_ref) < 3e-2
