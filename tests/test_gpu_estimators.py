"""-m gpu: NEXT-1 entry points (tm_M, tm_loop_contract_ex, tm_oneend_loops, tm_tsm_combine) against the oracle."""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel, to_dev

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU

_cache = {}


def fields(dims):
    if dims not in _cache:
        U = ti.gauge(dims)
        _cache[dims] = (Fields(dims, U, True), U)
    return _cache[dims]


def loops_of(t):
    return t.cpu().numpy().view(np.complex128)[..., 0]


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 18), (4, 12), (2, 12), (2, 18)])
@pytest.mark.parametrize("dagger", [0, 1])
def test_full_operator(prec, recon, dagger):
    """tm_M = M(kappa, mu) on both parities, its dagger, and D_W = M(kappa, 0) (Eq. 14); 3 right-hand sides."""
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    psi = np.stack([ti.gauss_spinor(dims, 21), ti.z4(dims, seed=22), ti.gauss_spinor(dims, 23)])
    pin = F.pack(psi, prec)
    for mu in (MU, 0.0, -0.3):
        out = F.zeros_full(prec, 3)
        tm.tm_M(F.L, F.gauge(prec, recon), prec, recon, out, pin, KAPPA, mu, dagger, 3)
        got = F.unpack(out, prec, nrhs=3)
        for r in range(3):
            assert rel(got[r], oracle.M(U, psi[r], KAPPA, mu, ap=True, dagger=bool(dagger))) < TOL[prec], (mu, r)


@pytest.mark.parametrize("prec", [8, 4, 2])
def test_loop_contract_ex_gamma5_and_scale(prec):
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    a = np.stack([ti.gauss_spinor(dims, 31), ti.z4(dims, seed=32)])
    b = np.stack([ti.gauss_spinor(dims, 33), ti.gauss_spinor(dims, 34)])
    pa, pb_ = F.pack(a, prec), F.pack(b, prec)
    out = torch.zeros((2, 16, dims[3], 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, 2))
    tol = {8: 1e-12, 4: 1e-5, 2: 5e-3}[prec]
    for gl, gr, sc in ((0, 0, 1.0), (1, 0, 2j), (0, 1, -0.5), (1, 1, 3 - 1j)):
        tm.tm_loop_contract_ex(F.L, pa, pb_, prec, 2, gl, gr, sc, out, ws)
        got = loops_of(out)
        for r in range(2):
            ref = sc * oracle.loop(oracle.gamma5(a[r]) if gl else a[r], oracle.gamma5(b[r]) if gr else b[r])
            assert rel(got[r], ref) < tol, (gl, gr, sc, r)


@pytest.mark.parametrize("prec,recon", [(8, 18), (4, 12), (2, 12)])
def test_oneend_loops(prec, recon):
    """Eq. (13) and Eq. (15) loops of given solution vectors (any spinor serves as s for the bilinear itself)."""
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    nrhs = 3
    s = np.stack([ti.gauss_spinor(dims, 41 + r) for r in range(nrhs)])
    ps = F.pack(s, prec)
    out = torch.zeros((nrhs, 16, dims[3], 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_oneend_workspace_bytes(F.L, prec, nrhs))
    tm.tm_oneend_loops(F.L, None, prec, recon, ps, tm.TM_ONEEND_TAU3, KAPPA, MU, nrhs, out, ws)
    got3 = loops_of(out).copy()
    tm.tm_oneend_loops(F.L, F.gauge(prec, recon), prec, recon, ps, tm.TM_ONEEND_GENERAL, KAPPA, MU, nrhs, out, ws)
    gotg = loops_of(out).copy()
    for r in range(nrhs):
        assert rel(got3[r], oracle.loop_oneend_tau3(s[r], KAPPA, MU)) < TOL[prec]
        assert rel(gotg[r], oracle.loop_oneend_general(U, s[r], KAPPA)) < TOL[prec]


def test_oneend_full_dilution_exact_traces_4x4():
    """PAPER.md:127-141 through the GPU: all 3072 unit sources on 4^4 solved with tm_cg_multi (fp64), one-end loops summed:
    tau3 form -> Tr_t[(M_d^-1 - M_u^-1) Gamma_n], generalised form -> Tr_t[(M_u^-1 + M_d^-1) Gamma_n] from dense inverses."""
    from oracle import dense
    dims = (4, 4, 4, 4)
    F, U = fields(dims)
    tr_u = dense.timeslice_traces(np.linalg.inv(dense.dense_M(U, KAPPA, MU, ap=True)), dims)
    tr_d = dense.timeslice_traces(np.linalg.inv(dense.dense_M(U, KAPPA, -MU, ap=True)), dims)
    nrhs = 12
    g = F.gauge(8, 18)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 8, tm.TM_CG_LP_TRUNCATED, nrhs))
    ows = tm.device_buffer(tm.tm_oneend_workspace_bytes(F.L, 8, nrhs))
    out = torch.zeros((nrhs, 16, 4, 2), dtype=torch.float64, device="cuda")
    prm = tm.make_cg_params(KAPPA, MU, 1e-12, 3000, tm.TM_CG_LP_TRUNCATED, 0.1, 8, 1)
    acc3 = torch.zeros((16, 4, 2), dtype=torch.float64, device="cuda")
    accg = torch.zeros_like(acc3)
    e = torch.zeros((nrhs, 256, 12, 2), dtype=torch.float64, device="cuda")
    pe = tm.device_buffer(tm.tm_spinor_bytes(F.L, 8, 1, nrhs))
    s = F.zeros_full(8, nrhs)
    for site in range(256):
        e.zero_()
        for k in range(12):
            e[k, site, k, 0] = 1.0
        tm.tm_spinor_pack(F.L, e, 8, nrhs, pe)
        rc, info = tm.tm_cg_multi(F.L, g, 8, g, 8, 18, s, pe, prm, nrhs, ws)
        assert rc == tm.TM_OK
        tm.tm_oneend_loops(F.L, g, 8, 18, s, tm.TM_ONEEND_TAU3, KAPPA, MU, nrhs, out, ows)
        acc3 += out.sum(dim=0)
        tm.tm_oneend_loops(F.L, g, 8, 18, s, tm.TM_ONEEND_GENERAL, KAPPA, MU, nrhs, out, ows)
        accg += out.sum(dim=0)
    got3, gotg = loops_of(acc3), loops_of(accg)
    assert np.abs(got3 - (tr_d - tr_u)).max() < 1e-8 * np.abs(tr_u).max()
    assert rel(gotg, tr_u + tr_d) < 1e-9


def test_tsm_combine_matches_eq8():
    T = 10
    rng = np.random.default_rng(5)
    hp = rng.normal(size=(3, 16, T)) + 1j * rng.normal(size=(3, 16, T))
    lps = rng.normal(size=(3, 16, T)) + 1j * rng.normal(size=(3, 16, T))
    lp = rng.normal(size=(7, 16, T)) + 1j * rng.normal(size=(7, 16, T))
    out = torch.zeros((16, T, 2), dtype=torch.float64, device="cuda")
    tm.tm_tsm_combine(T, to_dev(hp), to_dev(lps), 3, to_dev(lp), 7, out)
    assert np.abs(loops_of(out) - oracle.tsm_combine(hp, lps, lp)).max() < 1e-14
    tm.tm_tsm_combine(T, to_dev(hp), to_dev(lps), 3, None, 0, out)
    assert np.abs(loops_of(out) - oracle.tsm_combine(hp, lps, lp[:0])).max() < 1e-14
    tm.tm_tsm_combine(T, None, None, 0, to_dev(lp), 7, out)
    assert np.abs(loops_of(out) - oracle.tsm_combine(hp[:0], lps[:0], lp)).max() < 1e-14


def test_tsm_estimator_end_to_end_8x16():
    """Eq. (8) with the library end to end: N_HP = 2 sources solved to 1e-9 (HP_MIXED) and to 1e-2 (LP), N_LP = 6 more LP
    sources, standard loops eta^dag Gamma s, combined on the device; same chain through the oracle."""
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    T = dims[3]
    n_hp, n_lp = 2, 6
    etas = np.stack([ti.z4(dims, seed=900 + r) for r in range(n_hp + n_lp)])
    lws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, n_lp))
    # LP: fp16 storage, all 8 sources in one batch
    pe2 = F.pack(etas, 2)
    s2 = F.zeros_full(2, n_hp + n_lp)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 2, tm.TM_CG_LP_TRUNCATED, n_hp + n_lp))
    prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 4, 1)
    rc, _ = tm.tm_cg_multi(F.L, None, 8, F.gauge(2, 12), 2, 12, s2, pe2, prm, n_hp + n_lp, ws)
    assert rc == tm.TM_OK
    l_lp = torch.zeros((n_hp + n_lp, 16, T, 2), dtype=torch.float64, device="cuda")
    lws8 = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, n_hp + n_lp))
    tm.tm_loop_contract(F.L, pe2, s2, 2, n_hp + n_lp, l_lp, lws8)
    # HP: fp64 with fp32 inner iterations, one source at a time
    l_hp = torch.zeros((n_hp, 16, T, 2), dtype=torch.float64, device="cuda")
    wsh = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 4, tm.TM_CG_HP_MIXED, 1))
    prmh = tm.make_cg_params(KAPPA, MU, 1e-9, 5000, tm.TM_CG_HP_MIXED, 0.1, 1)
    for r in range(n_hp):
        pe8 = F.pack(etas[r], 8)
        s8 = F.zeros_full(8)
        rc, info = tm.tm_cg(F.L, F.gauge(8, 12), 8, F.gauge(4, 12), 4, 12, s8, pe8, prmh, wsh)
        assert rc == tm.TM_OK
        tm.tm_loop_contract(F.L, pe8, s8, 8, 1, l_hp[r:r + 1], lws)
    out = torch.zeros((16, T, 2), dtype=torch.float64, device="cuda")
    tm.tm_tsm_combine(T, l_hp, l_lp[:n_hp], n_hp, l_lp[n_hp:], n_lp, out)
    # oracle chain
    o_hp, o_lp = [], []
    for r in range(n_hp + n_lp):
        s_lp, _ = oracle.cg_solve(U, etas[r], KAPPA, MU, 1e-2, 500)
        o_lp.append(oracle.loop(etas[r], s_lp))
        if r < n_hp:
            s_hp, _ = oracle.cg_solve(U, etas[r], KAPPA, MU, 1e-9, 5000)
            o_hp.append(oracle.loop(etas[r], s_hp))
    ref = oracle.tsm_combine(np.array(o_hp), np.array(o_lp[:n_hp]), np.array(o_lp[n_hp:]))
    # the LP solutions differ from the oracle's at the truncation level (fp16 storage), the HP part at 1e-9
    assert rel(loops_of(out), ref) < 3e-2
    assert rel(loops_of(l_hp), np.array(o_hp)) < 1e-6
