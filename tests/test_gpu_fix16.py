"""-m gpu: 16-bit fixed-point links (TM_RECON_18_FIX16 / TM_RECON_12_FIX16; Fig. 4 names only "16-bit (half)" precision, reading 32).

The stored words are integers, so the pack is checked bit for bit against the format include/tm.h states; every kernel that reads
links is then checked against the oracle at the fp16-storage tolerance, and the links' share of the error against the binary16 links.
"""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel
from test_gpu_parity import fields, oracle_dslash, run_dslash

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU
FIX = {18: tm.TM_RECON_18_FIX16, 12: tm.TM_RECON_12_FIX16}


def expected_words(U, dims, reals):
    """Format of include/tm.h written out: word = 32768 + rint(32767 u) per stored real, [parity][mu][16-byte chunk][cb][8 words]
    followed by the tail array [cb][reals - 8 * chunks]; cb = site >> 1 of the parity's sites in lexicographic order."""
    X, Y, Z, T = dims
    Vh = X * Y * Z * T // 2
    u = U.reshape(T, Z, Y, X, 4, 9).view(np.float64).reshape(T * Z * Y * X, 4, 18)[:, :, :reals]
    q = (32768 + np.rint(np.clip(u, -1.0, 1.0) * 32767.0)).astype(np.uint16)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    par = ((x + y + z + t) & 1).reshape(-1)
    out = []
    nfull = reals // 8
    for parity in (0, 1):
        sites = np.nonzero(par == parity)[0]  # ascending site index == ascending cb
        assert sites.size == Vh
        for mu in range(4):
            w = q[sites, mu]  # [cb][reals]
            for k in range(nfull):
                out.append(w[:, 8 * k:8 * k + 8].reshape(-1))
            out.append(w[:, 8 * nfull:].reshape(-1))
    return np.concatenate(out)


@pytest.mark.parametrize("reals", [18, 12])
def test_fix16_pack_words_are_the_documented_format(reals):
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    buf = F.gauge(2, FIX[reals])
    assert tm.tm_gauge_bytes(F.L, 2, FIX[reals]) == tm.tm_gauge_bytes(F.L, 2, reals)
    torch.cuda.synchronize()
    got = buf.cpu().numpy().view(np.uint16)
    want = expected_words(U, dims, reals)
    assert np.array_equal(got[:want.size], want)


def test_fix16_unit_links_are_exact():
    """+-1 are representable (value = q / 32767): the free-field plane wave keeps the fp16-storage accuracy of the spinors alone."""
    dims = (4, 4, 4, 8)
    F, U = fields(dims, unit=True)
    psi = ti.z4(dims, seed=7)  # +-1/sqrt(2): exact in fp16 storage up to the fp32 site norm
    for reals in (18, 12):
        got = run_dslash(F, 2, FIX[reals], psi, psi, 0, 0, 0)
        ref = oracle_dslash(U, psi, psi, 0, 0, 0)
        assert rel(got, ref) < 3e-4  # the output's own binary16 rounding only


@pytest.mark.parametrize("dims", [(4, 6, 8, 10), (8, 8, 8, 16)])
@pytest.mark.parametrize("reals", [18, 12])
def test_fix16_dslash_all_kinds(dims, reals):
    F, U = fields(dims)
    psi, x = ti.gauss_spinor(dims, 3), ti.gauss_spinor(dims, 4)
    for out_parity in (0, 1):
        for dagger in (0, 1):
            for kind in (0, 1, 2):
                got = run_dslash(F, 2, FIX[reals], psi, x, out_parity, dagger, kind)
                ref = oracle_dslash(U, psi, x, out_parity, dagger, kind)
                assert rel(got, ref) < TOL[2], (dims, reals, out_parity, dagger, kind)


@pytest.mark.parametrize("reals", [18, 12])
def test_fix16_links_are_more_accurate_than_binary16_links(reals):
    """Z2 x iZ2 input (exact in fp16 storage): what is left is the links' rounding and the output's.  Fixed point halves it."""
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    psi = ti.z4(dims, seed=11)
    ref = oracle_dslash(U, psi, psi, 0, 0, 0)
    e_half = rel(run_dslash(F, 2, reals, psi, psi, 0, 0, 0), ref)
    e_fix = rel(run_dslash(F, 2, FIX[reals], psi, psi, 0, 0, 0), ref)
    print("recon %d: binary16 links %.3e, fixed-point links %.3e" % (reals, e_half, e_fix))
    assert e_fix < 0.9 * e_half


def test_fix16_flag_is_ignored_above_16_bits():
    """One `recon` serves a mixed-precision solve: with fp64 / fp32 the FIX16 codes mean the plain 12 / 18-real field."""
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    psi = ti.gauss_spinor(dims, 5)
    for prec in (8, 4):
        assert tm.tm_gauge_bytes(F.L, prec, 112) == tm.tm_gauge_bytes(F.L, prec, 12)
        a = run_dslash(F, prec, 112, psi, psi, 0, 0, 1)
        b = run_dslash(F, prec, 12, psi, psi, 0, 0, 1)
        assert np.array_equal(a, b)


@pytest.mark.parametrize("reals", [12, 18])
def test_fix16_multi_rhs_and_MdagM(reals):
    """12 right-hand sides through the shared-memory link tiles == one at a time; MdagM against the oracle."""
    dims = (8, 4, 6, 4)
    F, U = fields(dims)
    nrhs = 12
    recon = FIX[reals]
    psi = np.stack([ti.gauss_spinor(dims, 20 + r) for r in range(nrhs)])
    pin = F.pack(psi, 2)
    ostack = tm.device_buffer(F.pb(2) * nrhs)
    tm.tm_dslash(F.L, F.gauge(2, recon), 2, recon, ostack, F.half(pin, 2, 1, nrhs), None, 0, 0, 1, KAPPA, MU, nrhs)
    out = F.zeros_full(2, nrhs)
    F.put_half(out, ostack, 2, 0, nrhs)
    got = F.unpack(out, 2, nrhs=nrhs)
    for r in (0, 5, 11):
        assert np.array_equal(got[r], run_dslash(F, 2, recon, psi[r], psi[r], 0, 0, 1))
    p1 = F.pack(psi[0], 2)
    o1 = F.zeros_full(2)
    tmp = tm.device_buffer(2 * F.pb(2))
    tm.tm_MdagM(F.L, F.gauge(2, recon), 2, recon, F.half(o1, 2, 0), F.half(p1, 2, 0), tmp, 0, KAPPA, MU)
    assert rel(F.unpack(o1, 2), oracle.MdagM(U, oracle.project(psi[0], 0), KAPPA, MU, parity=0)) < TOL[2]


def test_fix16_truncated_batched_solve_and_mixed_cg():
    """The TSM solve (link cache built from the fixed-point field) and a mixed fp64 + fp16 solve with ONE recon code."""
    from test_gpu_cg import solve
    dims = (8, 8, 8, 16)
    F, U = fields(dims)
    nrhs = 12
    eta = np.stack([ti.z4(dims, seed=ti.NOISE_SEED + r) for r in range(nrhs)])
    rc, info, s = solve(F, eta, 8, 2, 112, tm.TM_CG_LP_TRUNCATED, 1e-2, 500, nrhs=nrhs)
    assert rc == tm.TM_OK
    for r in (0, 6, 11):
        s_ref, iref = oracle.cg_solve(U, eta[r], KAPPA, MU, 1e-2, 500)
        assert info[r].status == tm.TM_OK and abs(info[r].iters - iref["iters"]) <= 2
        assert rel(s[r], s_ref) < 2e-2
    rc1, info1, s1 = solve(F, eta[6], 8, 2, 112, tm.TM_CG_LP_TRUNCATED, 1e-2, 500)
    assert np.array_equal(s1, s[6])  # batched == unbatched, as for the binary16 links
    rc, info, sh = solve(F, eta[0], 8, 2, 112, tm.TM_CG_HP_MIXED, 1e-10, 2000)
    assert rc == tm.TM_OK and info[0].true_resid < 1e-10
    assert rel(sh, oracle.cg_solve(U, eta[0], KAPPA, MU, 1e-12, 5000)[0]) < 1e-7


def test_fix16_covdev():
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    psi = np.stack([ti.gauss_spinor(dims, 51), ti.z4(dims, seed=52)])
    pin = F.pack(psi, 2)
    for reals in (18, 12):
        for mu in range(4):
            out = F.zeros_full(2, 2)
            tm.tm_covdev(F.L, F.gauge(2, FIX[reals]), 2, FIX[reals], out, pin, mu, 2)
            got = F.unpack(out, 2, nrhs=2)
            for r in range(2):
                assert rel(got[r], oracle.covdev(U, psi[r], mu)) < TOL[2], (reals, mu, r)
