"""-m gpu: NEXT-2 / NEXT-3 entry points (tm_covdev, tm_contract_field, tm_loop_momentum, tm_time_dilute,
tm_loop_contract_slice, tm_hpe_remainder, tm_hpe_local_traces) against oracle/insertions.py, element by element."""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU

_cache = {}


def fields(dims):
    if dims not in _cache:
        U = ti.gauge(dims)
        _cache[dims] = (Fields(dims, U, True), U)
    return _cache[dims]


def cplx(t):
    return t.cpu().numpy().view(np.complex128)[..., 0]


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 18), (4, 12), (2, 12), (2, 18), (8, 8), (4, 8), (2, 8)])
def test_covdev(prec, recon):
    """D_mu on an antiperiodic lattice with four different extents (every wrap-around, the temporal sign), 2 right-hand sides."""
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    psi = np.stack([ti.gauss_spinor(dims, 51), ti.z4(dims, seed=52)])
    pin = F.pack(psi, prec)
    for mu in range(4):
        out = F.zeros_full(prec, 2)
        tm.tm_covdev(F.L, F.gauge(prec, recon), prec, recon, out, pin, mu, 2)
        got = F.unpack(out, prec, nrhs=2)
        for r in range(2):
            assert rel(got[r], oracle.covdev(U, psi[r], mu)) < TOL[prec], (mu, r)


@pytest.mark.parametrize("prec", [8, 4, 2])
def test_derivative_loops(prec):
    """One-derivative insertion a^dag Gamma_n D_mu b = tm_loop_contract(a, tm_covdev(b))."""
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    a, b = ti.z4(dims, seed=61), ti.gauss_spinor(dims, 62)
    pa, pb_ = F.pack(a, prec), F.pack(b, prec)
    d = F.zeros_full(prec)
    out = torch.zeros((1, 16, dims[3], 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, 1))
    for mu in range(4):
        tm.tm_covdev(F.L, F.gauge(prec, 12), prec, 12, d, pb_, mu, 1)
        tm.tm_loop_contract(F.L, pa, d, prec, 1, out, ws)
        assert rel(cplx(out)[0], oracle.loop_derivative(U, a, b, mu)) < TOL[prec], mu


@pytest.mark.parametrize("prec", [8, 4, 2])
def test_contract_field(prec):
    dims = (4, 6, 8, 10)
    X, Y, Z, T = dims
    F, U = fields(dims)
    a = np.stack([ti.gauss_spinor(dims, 71), ti.z4(dims, seed=72)])
    b = np.stack([ti.gauss_spinor(dims, 73), ti.gauss_spinor(dims, 74)])
    pa, pb_ = F.pack(a, prec), F.pack(b, prec)
    out = torch.zeros((2, T, Z, Y, X, 4, 4, 2), dtype=torch.float64, device="cuda")
    tm.tm_contract_field(F.L, pa, pb_, prec, 2, out)
    got = cplx(out)
    for r in range(2):
        assert rel(got[r], oracle.contract_field(a[r], b[r])) < TOL[prec]


@pytest.mark.parametrize("prec", [8, 4, 2])
@pytest.mark.parametrize("dims,p2max", [((4, 6, 8, 10), 9), ((8, 8, 8, 4), 14), ((16, 16, 16, 4), 9),
                                        # the row kernel's other shapes: two sites per lane (X = 64), X / 2 odd and more than four
                                        # row-warps per plane (Y = 40), the unrolled X = 32 form with a single warp and a ragged row count
                                        ((64, 4, 4, 4), 9), ((12, 40, 4, 4), 9), ((32, 6, 4, 4), 5)])
def test_loop_momentum(prec, dims, p2max):
    """Fused contraction + partial DFT against the plain nested sums; the p^2 <= 9 list of PAPER.md:427 (123 momenta), and a
    larger list reaching |m_i| = 3 with several y-row passes and a ragged last pass (Y = 6)."""
    F, U = fields(dims)
    T = dims[3]
    a = np.stack([ti.z4(dims, seed=81), ti.gauss_spinor(dims, 82)])
    b = np.stack([ti.gauss_spinor(dims, 83), ti.gauss_spinor(dims, 84)])
    pa, pb_ = F.pack(a, prec), F.pack(b, prec)
    mom = oracle.momenta_p2_max(p2max)
    K = len(mom)
    pmax = int(np.abs(mom).max())
    out = torch.zeros((2, 16, T, K, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_momentum_workspace_bytes(F.L, 2, K, pmax))
    tm.tm_loop_momentum(F.L, pa, pb_, prec, 2, mom, out, ws)
    got = cplx(out)
    for r in range(2):
        ref = oracle.loop_momentum(a[r], b[r], mom)
        assert rel(got[r], ref) < TOL[prec]
    # zero momentum == the time-slice loop kernel (same arithmetic per site, different summation tree)
    k0 = [i for i, p in enumerate(mom) if tuple(p) == (0, 0, 0)][0]
    o2 = torch.zeros((2, 16, T, 2), dtype=torch.float64, device="cuda")
    ws2 = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, 2))
    tm.tm_loop_contract(F.L, pa, pb_, prec, 2, o2, ws2)
    assert rel(got[:, :, :, k0], cplx(o2)) < (1e-13 if prec == 8 else 1e-6)


def test_loop_momentum_rejects_large_momenta():
    dims = (4, 4, 4, 4)
    F, U = fields(dims)
    pa = F.pack(ti.z4(dims, seed=1), 4)
    out = torch.zeros((1, 16, 4, 1, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(1 << 20)
    with pytest.raises(tm.TmError):
        tm.tm_loop_momentum(F.L, pa, pa, 4, 1, np.array([[5, 0, 0]]), out, ws)


@pytest.mark.parametrize("prec", [8, 4, 2])
def test_time_dilution_and_slice_contraction(prec):
    dims = (4, 4, 6, 8)
    T = dims[3]
    F, U = fields(dims)
    eta = np.stack([ti.z4(dims, seed=91), ti.z4(dims, seed=92)])
    b = np.stack([ti.gauss_spinor(dims, 93), ti.gauss_spinor(dims, 94)])
    pe, pb_ = F.pack(eta, prec), F.pack(b, prec)
    dil = F.zeros_full(prec, 2)
    for slices in ([3], [0, 4], [7]):
        keep = [1 if t in slices else 0 for t in range(T)]
        tm.tm_time_dilute(F.L, pe, prec, 2, keep, dil)
        got = F.unpack(dil, prec, nrhs=2)
        for r in range(2):
            ref = oracle.time_dilute(eta[r], slices)
            assert np.array_equal(got[r] == 0, ref == 0)  # support is exact
            assert rel(got[r], ref) < TOL[prec]
    out = torch.zeros((2, 16, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, 2))
    for t0 in (0, 3, T - 1):
        tm.tm_loop_contract_slice(F.L, pe, pb_, prec, 2, t0, out, ws)
        got = cplx(out)
        for r in range(2):
            assert rel(got[r], oracle.loop_slice(eta[r], b[r], t0)) < TOL[prec]


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 12), (2, 12)])
def test_hpe_remainder(prec, recon):
    """(B H)^4 s against the oracle; fp16 rounds after each of the 4 applications, hence 4x the one-hop tolerance."""
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    s = np.stack([ti.gauss_spinor(dims, 101), ti.z4(dims, seed=102)])
    ps = F.pack(s, prec)
    out, tmp = F.zeros_full(prec, 2), F.zeros_full(prec, 2)
    tm.tm_hpe_remainder(F.L, F.gauge(prec, recon), prec, recon, out, ps, tmp, KAPPA, MU, 2)
    got = F.unpack(out, prec, nrhs=2)
    for r in range(2):
        assert rel(got[r], oracle.hpe_remainder(U, s[r], KAPPA, MU)) < TOL[prec]  # measured 5.6e-4 (fp16) / 2.0e-7 (fp32) at 32^3x64: DESIGN.md reading 34


def test_hpe_estimator_exact_on_4x4():
    """Eq. (16)/(17) end to end on 4^4 in fp64 through the GPU: for EVERY unit source e_i (complete set, no noise),
    sum_i e_i^dag Gamma_n (BH)^4 M^-1 e_i + V3 * local terms = Tr_t[Gamma_n M^-1] from the dense inverse."""
    from oracle import dense
    dims = (4, 4, 4, 4)
    F, U = fields(dims)
    Minv = np.linalg.inv(dense.dense_M(U, KAPPA, MU, ap=True))
    ref = dense.timeslice_traces(Minv, dims)
    loc = tm.tm_hpe_local_traces(KAPPA, MU)
    assert np.allclose(loc, oracle.hpe_local_traces(KAPPA, MU), atol=1e-13)
    N = 12 * 256
    nb = 16
    acc = np.zeros((16, 4), dtype=np.complex128)
    out = torch.zeros((nb, 16, 4, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, nb))
    rem, tmp = F.zeros_full(8, nb), F.zeros_full(8, nb)
    for i0 in range(0, N, nb):
        e = np.zeros((nb, N), dtype=np.complex128)
        e[np.arange(nb), i0 + np.arange(nb)] = 1.0
        s = np.ascontiguousarray(Minv[:, i0:i0 + nb].T)
        pe = F.pack(e.reshape(nb, 4, 4, 4, 4, 4, 3), 8)
        ps = F.pack(s.reshape(nb, 4, 4, 4, 4, 4, 3), 8)
        tm.tm_hpe_remainder(F.L, F.gauge(8, 18), 8, 18, rem, ps, tmp, KAPPA, MU, nb)
        tm.tm_loop_contract(F.L, pe, rem, 8, nb, out, ws)
        acc += cplx(out).sum(axis=0)
    assert np.allclose(acc + 64 * loc[:, None], ref, atol=1e-9)
