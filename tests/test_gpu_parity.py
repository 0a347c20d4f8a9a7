"""-m gpu: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by element on the same seeded inputs.

Tolerances (north_star): relative L2 per field 1e-12 (fp64), 1e-5 (fp32), 5e-3 (fp16 storage).
"""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel, to_dev

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU
A = 2 * KAPPA * MU

_cache = {}


def fields(dims, ap=True, unit=False):
    key = (tuple(dims), ap, unit)
    if key not in _cache:
        U = ti.unit_gauge(dims) if unit else ti.gauge(dims)
        _cache[key] = (Fields(dims, U, ap), U)
    return _cache[key]


# ---- a0 / a1: layouts ------------------------------------------------------------------------------------
@pytest.mark.parametrize("prec", [8, 4, 2])
def test_spinor_pack_roundtrip(prec):
    dims = (4, 6, 8, 10)
    F, _ = fields(dims)
    psi = np.stack([ti.gauss_spinor(dims, 5), ti.z4(dims)])
    back = F.unpack(F.pack(psi, prec), prec, nrhs=2)
    if prec == 8:
        assert np.array_equal(back, psi)  # bit-exact
    elif prec == 4:
        assert np.array_equal(back, psi.astype(np.complex64).astype(np.complex128))
    else:
        # per-site fp32 max-norm, components RN to binary16 (reading 13)
        flat = psi.reshape(-1, 12).astype(np.complex64)
        nrm = np.maximum(np.abs(flat.real), np.abs(flat.imag)).max(axis=1, keepdims=True).astype(np.float32)
        q = ((flat.real / nrm).astype(np.float16).astype(np.float32) * nrm) + 1j * ((flat.imag / nrm).astype(np.float16).astype(np.float32) * nrm)
        assert rel(back.reshape(-1, 12), q.astype(np.complex128)) < 2e-4  # 1/norm vs division differ by an ulp at most
        assert rel(back, psi) < 6e-4


def test_z4_code_pack_matches_spinor_pack():
    dims = (4, 6, 8, 10)
    F, _ = fields(dims)
    codes = np.stack([ti.z4_codes(dims, seed=7), ti.z4_codes(dims, seed=8)])
    ref = np.stack([ti.z4(dims, seed=7), ti.z4(dims, seed=8)])
    for prec in (8, 4, 2):
        buf = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, 2))
        tm.tm_spinor_pack_z4(F.L, to_dev(codes), prec, 2, buf)
        assert rel(F.unpack(buf, prec, nrhs=2), ref) < (1e-15 if prec == 8 else 1e-7 if prec == 4 else 6e-4)


@pytest.mark.parametrize("prec", [8, 4, 2])
def test_device_noise_is_the_host_generator(prec):
    """tm_noise_z4 (sources made on the GPU) == the host generator's codes through tm_spinor_pack_z4, bit for bit."""
    dims = (4, 6, 8, 10)
    F, _ = fields(dims)
    nrhs, seed, stride = 3, 4242, 7
    codes = np.stack([ti.z4_codes(dims, seed=seed + r * stride) for r in range(nrhs)])
    a = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, nrhs))
    b = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, nrhs))
    tm.tm_spinor_pack_z4(F.L, to_dev(codes), prec, nrhs, a)
    tm.tm_noise_z4(F.L, seed, stride, prec, nrhs, b)
    assert torch.equal(a, b)


def test_gauge_pack_rejects_non_su3_for_recon12():
    dims = (4, 4, 4, 4)
    U = ti.gauge(dims).copy()
    U[1, 2, 3, 0, 2, 1, 1] *= 1.01
    L = tm.tm_lattice_create(dims)
    Ud = to_dev(U)
    buf = tm.device_buffer(tm.tm_gauge_bytes(L, 4, 12))
    with pytest.raises(tm.TmError) as e:
        tm.tm_gauge_pack(L, Ud, 4, 12, buf, 1e-10)
    assert e.value.status == tm.TM_ERR_NOT_SU3
    buf18 = tm.device_buffer(tm.tm_gauge_bytes(L, 4, 18))
    tm.tm_gauge_pack(L, Ud, 4, 18, buf18, 1e-10)  # 18 reals accept any 3x3


def test_argument_errors():
    dims = (4, 4, 4, 4)
    F, _ = fields(dims)
    g = F.gauge(4, 18)
    s = F.zeros_full(4)
    half = F.half(s, 4, 0)
    for call in (lambda: tm.tm_dslash(F.L, g, 4, 18, half, half, None, 0, 0, 0, KAPPA, MU),           # out aliases in
                 lambda: tm.tm_dslash(F.L, g, 4, 18, F.half(s, 4, 1), half, None, 0, 0, 2, KAPPA, MU),  # XPAY without x
                 lambda: tm.tm_dslash(F.L, g, 4, 18, F.half(s, 4, 1), half, None, 0, 0, 0, KAPPA, MU, nrhs=17),
                 lambda: tm.tm_dslash(F.L, g, 5, 18, F.half(s, 4, 1), half, None, 0, 0, 0, KAPPA, MU)):
        with pytest.raises(tm.TmError) as e:
            call()
        assert e.value.status == tm.TM_ERR_ARG
    with pytest.raises(tm.TmError) as e:
        tm.tm_dslash(F.L, g, 4, 18, F.half(s, 4, 1)[8:], half, None, 0, 0, 0, KAPPA, MU)  # not 16-byte aligned
    assert e.value.status == tm.TM_ERR_LAYOUT


# ---- a2 / a3: dslash -------------------------------------------------------------------------------------
def oracle_dslash(U, psi, x, out_parity, dagger, kind, ap=True):
    """Reference for tm_dslash from the oracle's plain operators (full-lattice arrays, zero on the other parity)."""
    d = oracle.project(oracle.hop(U, oracle.project(psi, 1 - out_parity), ap=ap, dagger=dagger), out_parity)
    a = -A if dagger else A
    if kind == tm.TM_KIND_PLAIN:
        return d
    if kind == tm.TM_KIND_TWIST_INV:
        return oracle.twist(d, a, inverse=True)
    return oracle.twist(oracle.project(x, out_parity), a) - KAPPA ** 2 * d


def run_dslash(F, prec, recon, psi, x, out_parity, dagger, kind):
    pin, px = F.pack(psi, prec), F.pack(x, prec)
    out = F.zeros_full(prec)
    tm.tm_dslash(F.L, F.gauge(prec, recon), prec, recon, F.half(out, prec, out_parity), F.half(pin, prec, 1 - out_parity),
                 F.half(px, prec, out_parity) if kind == tm.TM_KIND_XPAY_TWIST else None, out_parity, dagger, kind, KAPPA, MU)
    return F.unpack(out, prec)


@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10), (8, 4, 6, 4)])
@pytest.mark.parametrize("prec", [8, 4, 2])
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_dslash_all_kinds(dims, prec, recon):
    F, U = fields(dims)
    psi, x = ti.gauss_spinor(dims, 3), ti.gauss_spinor(dims, 4)
    for out_parity in (0, 1):
        for dagger in (0, 1):
            for kind in (0, 1, 2):
                got = run_dslash(F, prec, recon, psi, x, out_parity, dagger, kind)
                ref = oracle_dslash(U, psi, x, out_parity, dagger, kind)
                assert rel(got, ref) < TOL[prec], (dims, prec, recon, out_parity, dagger, kind)
                assert not oracle.project(got, 1 - out_parity).any()


def test_gauge_pack_recon8_refuses_the_singular_chart():
    """The stored matrix is V = U P (columns shifted cyclically, reading 31): the chart is singular where V01 = V02 = 0,
    i.e. |U02| = 1 -- not at the unit link, which packs (free fields, temporal-gauge fields)."""
    dims = (4, 4, 4, 4)
    L = tm.tm_lattice_create(dims)
    buf = tm.device_buffer(tm.tm_gauge_bytes(L, 4, 8))
    tm.tm_gauge_pack(L, to_dev(ti.unit_gauge(dims)), 4, 8, buf, 1e-10)
    bad = ti.unit_gauge(dims).copy()
    bad[2, 1, 0, 3, 1] = np.array([[0, 0, 1], [1, 0, 0], [0, 1, 0]], dtype=np.complex128)  # an SU(3) link with |U02| = 1
    with pytest.raises(tm.TmError) as e:
        tm.tm_gauge_pack(L, to_dev(bad), 4, 8, buf, 1e-10)
    assert e.value.status == tm.TM_ERR_RECON8
    U = ti.gauge(dims).copy()
    U[1, 2, 3, 0, 2, 1, 1] *= 1.01
    with pytest.raises(tm.TmError) as e:
        tm.tm_gauge_pack(L, to_dev(U), 4, 8, buf, 1e-10)
    assert e.value.status == tm.TM_ERR_NOT_SU3
    tm.tm_gauge_pack(L, to_dev(ti.gauge(dims)), 4, 8, buf, 1e-10)
    assert tm.tm_gauge_bytes(L, 4, 8) * 18 == tm.tm_gauge_bytes(L, 4, 18) * 8


@pytest.mark.parametrize("prec,recon", [(8, 18), (8, 12), (4, 12), (2, 12), (2, 18), (8, 8), (4, 8), (2, 8)])
def test_dslash_free_field_plane_wave(prec, recon):
    """P2 through the GPU: U = 1, odd temporal momentum across the antiperiodic boundary, all three reconstructs (the unit link is a
    regular point of the 8-real chart since the stored matrix is U P)."""
    dims = (4, 6, 4, 8)
    F, U = fields(dims, unit=True)
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    n = (1, 2, 3, 3)
    p = np.array([2 * np.pi * n[0] / X, 2 * np.pi * n[1] / Y, 2 * np.pi * n[2] / Z, (2 * n[3] + 1) * np.pi / T])
    u = np.random.default_rng(1).normal(size=(4, 3)) + 1j * np.random.default_rng(2).normal(size=(4, 3))
    psi = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))[..., None, None] * u
    from oracle import dense
    H = sum(2 * np.cos(p[m]) * np.eye(4) - 2j * dense.GAMMA[m] * np.sin(p[m]) for m in range(4))
    ref = np.einsum("ab,...bc->...ac", H, psi)
    for par in (0, 1):
        got = run_dslash(F, prec, recon, psi, psi, par, 0, 0)
        assert rel(got, oracle.project(ref, par)) < TOL[prec]


@pytest.mark.parametrize("prec", [4, 2])
def test_dslash_16x32_and_general_epilogue(prec):
    dims = (16, 16, 16, 32)
    F, U = fields(dims)
    psi, x = ti.z4(dims), ti.gauss_spinor(dims, 9)
    for recon in (18, 12):
        got = run_dslash(F, prec, recon, psi, x, 0, 0, 1)
        assert rel(got, oracle_dslash(U, psi, x, 0, 0, 1)) < TOL[prec]
    # general epilogue with arbitrary coefficients
    pq = (0.7, -0.3, 0.2, 1.1)
    pin, px = F.pack(psi, prec), F.pack(x, prec)
    out = F.zeros_full(prec)
    tm.tm_dslash_general(F.L, F.gauge(prec, 12), prec, 12, F.half(out, prec, 1), F.half(pin, prec, 0), F.half(px, prec, 1), 1, 1, pq)
    g5 = np.array([1, 1, -1, -1.0])[:, None]
    d = oracle.project(oracle.hop(U, oracle.project(psi, 0), dagger=True), 1)
    xo = oracle.project(x, 1)
    ref = pq[0] * xo + 1j * pq[1] * g5 * xo + pq[2] * d + 1j * pq[3] * g5 * d
    assert rel(F.unpack(out, prec), ref) < TOL[prec]


@pytest.mark.parametrize("prec,recon,nrhs", [(8, 18, 2), (8, 12, 3), (4, 18, 12), (4, 12, 5), (2, 12, 12), (2, 18, 8), (2, 12, 16), (4, 8, 12),
                                             (2, 8, 5), (8, 8, 2)])
def test_dslash_multi_rhs_equals_single(prec, recon, nrhs):
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    psi = np.stack([ti.gauss_spinor(dims, 100 + r) for r in range(nrhs)])
    x = np.stack([ti.gauss_spinor(dims, 200 + r) for r in range(nrhs)])
    pin, px = F.pack(psi, prec), F.pack(x, prec)
    out = F.zeros_full(prec, nrhs)
    ostack = tm.device_buffer(F.pb(prec) * nrhs)
    tm.tm_dslash(F.L, F.gauge(prec, recon), prec, recon, ostack, F.half(pin, prec, 1, nrhs), F.half(px, prec, 0, nrhs), 0, 0, 2, KAPPA, MU,
                 nrhs=nrhs)
    F.put_half(out, ostack, prec, 0, nrhs)
    got = F.unpack(out, prec, nrhs=nrhs)
    for r in range(nrhs):
        single = run_dslash(F, prec, recon, psi[r], x[r], 0, 0, 2)
        assert np.array_equal(got[r], single)  # batched == unbatched bit for bit
        assert rel(got[r], oracle_dslash(U, psi[r], x[r], 0, 0, 2)) < TOL[prec]


# ---- a4: MdagM -------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10)])
@pytest.mark.parametrize("prec", [8, 4, 2])
@pytest.mark.parametrize("recon", [18, 12, 8])
def test_MdagM(dims, prec, recon):
    F, U = fields(dims)
    psi = ti.gauss_spinor(dims, 17)
    pin = F.pack(psi, prec)
    for parity in (0, 1):
        out = F.zeros_full(prec)
        tmp = tm.device_buffer(2 * F.pb(prec))
        tm.tm_MdagM(F.L, F.gauge(prec, recon), prec, recon, F.half(out, prec, parity), F.half(pin, prec, parity), tmp, parity, KAPPA, MU)
        ref = oracle.MdagM(U, oracle.project(psi, parity), KAPPA, MU, parity=parity)
        assert rel(F.unpack(out, prec), ref) < TOL[prec]


# ---- a8: loop contraction --------------------------------------------------------------------------------
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 8, 10), (16, 16, 16, 32)])
@pytest.mark.parametrize("prec", [8, 4, 2])
def test_loop_contract(dims, prec):
    F, U = fields(dims)
    nrhs = 3 if dims[0] == 4 else 1
    a = np.stack([ti.z4(dims, seed=50 + r) for r in range(nrhs)])
    b = np.stack([ti.gauss_spinor(dims, 60 + r) for r in range(nrhs)])
    pa, pb_ = F.pack(a, prec), F.pack(b, prec)
    T = dims[3]
    out = torch.zeros((nrhs, 16, T, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, nrhs))
    tm.tm_loop_contract(F.L, pa, pb_, prec, nrhs, out, ws)
    got = out.cpu().numpy().view(np.complex128)[..., 0]
    for r in range(nrhs):
        ref = oracle.loop(a[r], b[r])
        # loop sums cancel heavily: relative L2 over the whole [16][T] array (reading 22)
        assert rel(got[r], ref) < TOL[prec]
    # P13 closed form through the GPU: a = b = eta -> L[0][t] = 12 V3
    tm.tm_loop_contract(F.L, pa, pa, prec, nrhs, out, ws)
    got = out.cpu().numpy().view(np.complex128)[..., 0]
    assert np.allclose(got[:, 0, :], 12 * dims[0] * dims[1] * dims[2], rtol=2 * TOL[prec])
    # run-to-run bit reproducibility
    out2 = torch.zeros_like(out)
    tm.tm_loop_contract(F.L, pa, pa, prec, nrhs, out2, ws)
    assert torch.equal(out, out2)


# ---- ragged tails: Vh = 648 is not a multiple of the 32-site tiles / 128-site CTAs, X/2 = 3 is odd -------------------
@pytest.mark.parametrize("prec,recon", [(8, 12), (4, 18), (4, 12), (2, 12), (2, 8)])
def test_ragged_lattice_6x6x6x6(prec, recon):
    dims = (6, 6, 6, 6)
    F, U = fields(dims)
    nrhs = 12
    psi = np.stack([ti.gauss_spinor(dims, 700 + r) for r in range(nrhs)])
    x = np.stack([ti.z4(dims, seed=720 + r) for r in range(nrhs)])
    # single rhs, every kind
    for out_parity, dagger, kind in ((0, 0, 1), (1, 1, 2), (1, 0, 0)):
        got = run_dslash(F, prec, recon, psi[0], x[0], out_parity, dagger, kind)
        assert rel(got, oracle_dslash(U, psi[0], x[0], out_parity, dagger, kind)) < TOL[prec]
    # 12 right-hand sides through the multi-rhs tile kernels (last tile has 8 of 32 sites)
    pin, px = F.pack(psi, prec), F.pack(x, prec)
    pb = F.pb(prec)
    ostack = tm.device_buffer(pb * nrhs)
    tm.tm_dslash(F.L, F.gauge(prec, recon), prec, recon, ostack, F.half(pin, prec, 1, nrhs), F.half(px, prec, 0, nrhs), 0, 0, 2, KAPPA, MU,
                 nrhs)
    full = F.zeros_full(prec, nrhs)
    F.put_half(full, ostack, prec, 0, nrhs)
    got = F.unpack(full, prec, nrhs=nrhs)
    for r in (0, 5, 11):
        assert rel(got[r], oracle_dslash(U, psi[r], x[r], 0, 0, 2)) < TOL[prec]
    # loops of 3 right-hand sides
    T = dims[3]
    out = torch.zeros((nrhs, 16, T, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, nrhs))
    tm.tm_loop_contract(F.L, px, pin, prec, nrhs, out, ws)
    got = out.cpu().numpy().view(np.complex128)[..., 0]
    for r in (0, 7):
        assert rel(got[r], oracle.loop(x[r], psi[r])) < TOL[prec]


@pytest.mark.parametrize("prec", [8, 4, 2])
def test_symmetric_preconditioned_operator_from_the_general_epilogue(prec):
    """PAPER.md:376 Eq. (A3): M_sym = 1 - kappa^2 R^-1 Dslash R^-1 Dslash is two launches of the same kernels (TWIST_INV, then the
    general epilogue with p = 1, q = -kappa^2 R^-1); its normal operator is M_pc^dag M_pc / (1 + a^2) (pin P24), so CG needs
    no separate symmetric mode."""
    dims = (4, 6, 8, 10)
    F, U = fields(dims)
    v = ti.gauss_spinor(dims, 333)
    pin = F.pack(v, prec)
    t1, out = F.zeros_full(prec), F.zeros_full(prec)
    a = 2 * KAPPA * MU
    d = 1.0 / (1.0 + a * a)
    g = F.gauge(prec, 12)
    tm.tm_dslash(F.L, g, prec, 12, F.half(t1, prec, 1), F.half(pin, prec, 0), None, 1, 0, tm.TM_KIND_TWIST_INV, KAPPA, MU)
    tm.tm_dslash_general(F.L, g, prec, 12, F.half(out, prec, 0), F.half(t1, prec, 1), F.half(pin, prec, 0), 0, 0,
                         (1.0, 0.0, -KAPPA ** 2 * d, KAPPA ** 2 * a * d))
    assert rel(F.unpack(out, prec), oracle.Mpc_sym(U, v, KAPPA, MU)) < TOL[prec]
