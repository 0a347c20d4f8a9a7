"""-m gpu: parity at BASELINE.json's full sizes, in the launch configurations bench.py times.

* 32^3x64 (configs[2], [3]): the 12-right-hand-side fp16 / 12-real tile kernel and the single-rhs kernels, whole fields
  against the oracle stencil.
* 64^3x128 (configs[4]): sampled output sites (random + every site of two boundary-touching 2-D planes) against the
  single-site oracle `hop_gathered`, whose inputs are regenerated from the counter-based generators.
"""
import numpy as np
import pytest
import torch

import oracle
import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import Fields, TOL, rel, to_dev, gather_site_inputs

pytestmark = pytest.mark.gpu
KAPPA, MU = ti.KAPPA, ti.MU
A = 2 * KAPPA * MU


def test_32x64_twelve_rhs_dslash_whole_field():
    """configs[3] launch shape: fp16 storage, 12-real links, 12 right-hand sides per gauge load, both epilogue kinds."""
    dims = (32, 32, 32, 64)
    nrhs, prec, recon = 12, 2, 12
    U = ti.gauge(dims)
    F = Fields(dims, U, True)
    codes = np.stack([ti.z4_codes(dims, seed=ti.NOISE_SEED + r) for r in range(nrhs)])
    pin = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, nrhs))
    tm.tm_spinor_pack_z4(F.L, to_dev(codes), prec, nrhs, pin)
    del codes
    out = F.zeros_full(prec, nrhs)
    src_o = F.half(pin, prec, 1, nrhs)
    x_e = F.half(pin, prec, 0, nrhs)
    for kind, dagger in ((tm.TM_KIND_TWIST_INV, 0), (tm.TM_KIND_XPAY_TWIST, 1)):
        res = tm.device_buffer(F.pb(prec) * nrhs)
        tm.tm_dslash(F.L, F.gauge(prec, recon), prec, recon, res, src_o, x_e if kind == tm.TM_KIND_XPAY_TWIST else None, 0, dagger,
                     kind, KAPPA, MU, nrhs)
        out.zero_()
        F.put_half(out, res, prec, 0, nrhs)
        got = F.unpack(out, prec, nrhs=nrhs)
        for r in (0, 5, 11):
            eta = ti.z4(dims, seed=ti.NOISE_SEED + r)
            d = oracle.hop(U, oracle.project(eta, 1), ap=True, dagger=bool(dagger))
            a = -A if dagger else A
            if kind == tm.TM_KIND_TWIST_INV:
                ref = oracle.twist(d, a, inverse=True)
            else:
                ref = oracle.twist(oracle.project(eta, 0), a) - KAPPA ** 2 * d
            ref = oracle.project(ref, 0)
            assert rel(got[r], ref) < TOL[prec], (kind, dagger, r)


def test_32x64_tsm_step_through_the_link_cache():
    """configs[3], the step bench.py times: 12 Z2xiZ2 sources from their codes -> batched truncated CG (tol 1e-2, fp16 storage,
    12-real links: the 12-rhs kernel fed from the per-solve link cache by cp.async.bulk) -> 16-Gamma loops, at 32^3x64.
    Checked against the oracle's CG on one source, the oracle's full operator and loop on the solutions, and the unbatched solve."""
    dims = (32, 32, 32, 64)
    nrhs, prec, recon = 12, 2, 12
    U = ti.gauge(dims)
    F = Fields(dims, U, True)
    codes = np.stack([ti.z4_codes(dims, seed=ti.NOISE_SEED + r) for r in range(nrhs)])
    pe = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, nrhs))
    tm.tm_spinor_pack_z4(F.L, to_dev(codes), prec, nrhs, pe)
    del codes
    g = F.gauge(prec, recon)
    F.drop_canonical()
    s = F.zeros_full(prec, nrhs)
    ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, nrhs))
    prm = tm.make_cg_params(KAPPA, MU, 1e-2, 500, tm.TM_CG_LP_TRUNCATED, 0.1, 0, 1)  # bench.py's parameters
    rc, info = tm.tm_cg_multi(F.L, None, 8, g, prec, recon, s, pe, prm, nrhs, ws)
    assert rc == tm.TM_OK
    T = dims[3]
    loops = torch.zeros((nrhs, 16, T, 2), dtype=torch.float64, device="cuda")
    lws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, nrhs))
    tm.tm_loop_contract(F.L, pe, s, prec, nrhs, loops, lws)
    loops = loops.cpu().numpy().view(np.complex128)[..., 0]
    fb = tm.tm_spinor_bytes(F.L, prec, 1, 1)
    s_ref, iref = oracle.cg_solve(U, ti.z4(dims, seed=ti.NOISE_SEED), KAPPA, MU, 1e-2, 500)
    for r in (0, 11):
        eta = ti.z4(dims, seed=ti.NOISE_SEED + r)
        s_r = F.unpack(s[r * fb:(r + 1) * fb], prec)
        assert info[r].status == tm.TM_OK and info[r].iterated_resid <= 1e-2
        assert abs(info[r].iters - iref["iters"]) <= 1                               # P15
        assert rel(oracle.M(U, s_r, KAPPA, MU), eta) < 1.3 * iref["true_resid_full"]  # the truncated residual, by the oracle's operator
        assert rel(loops[r], oracle.loop(eta, s_r)) < TOL[prec]
        if r == 0:
            assert rel(s_r, s_ref) < 2e-2   # same x0 = 0 and the same steps up to storage rounding (as test_cg_lp_truncated_batched)
        # the unbatched solve (single-rhs kernels, no link cache) gives the same bits
        s1 = F.zeros_full(prec, 1)
        ws1 = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, prec, tm.TM_CG_LP_TRUNCATED, 1))
        rc1, info1 = tm.tm_cg_multi(F.L, None, 8, g, prec, recon, s1, pe[r * fb:(r + 1) * fb], prm, 1, ws1)
        assert rc1 == tm.TM_OK and info1[0].iters == info[r].iters
        assert torch.equal(s1, s[r * fb:(r + 1) * fb])


@pytest.mark.parametrize("prec,recon", [(4, 18), (4, 12), (2, 18), (2, 12)])
def test_32x64_single_rhs_dslash_whole_field(prec, recon):
    """configs[2]: the single-rhs kernels bench.py's dslash table times."""
    dims = (32, 32, 32, 64)
    U = ti.gauge(dims)
    F = Fields(dims, U, True)
    eta = ti.z4(dims, seed=777)
    pin = F.pack(eta, prec)
    out = F.zeros_full(prec)
    tm.tm_dslash(F.L, F.gauge(prec, recon), prec, recon, F.half(out, prec, 1), F.half(pin, prec, 0), None, 1, 0, tm.TM_KIND_TWIST_INV,
                 KAPPA, MU)
    ref = oracle.project(oracle.twist(oracle.hop(U, oracle.project(eta, 0), ap=True), A, inverse=True), 1)
    assert rel(F.unpack(out, prec), ref) < TOL[prec]


def _sample_sites(dims, parity, n_random, seed):
    """Global indices of output sites of `parity`: random ones plus all sites of the planes (x, t) at y = z = 0 and
    (y, z) at x = X-1, t = T-1, which touch every wrap-around of the lattice."""
    X, Y, Z, T = dims
    rng = np.random.default_rng(seed)
    s = rng.integers(0, X * Y * Z * T, size=2 * n_random)
    xs, ts = np.meshgrid(np.arange(X), np.arange(T), indexing="ij")
    ys, zs = np.meshgrid(np.arange(Y), np.arange(Z), indexing="ij")
    plane1 = ti.site_index(dims, xs.ravel(), 0, 0, ts.ravel())
    plane2 = ti.site_index(dims, X - 1, ys.ravel(), zs.ravel(), T - 1)
    s = np.unique(np.concatenate([s, plane1, plane2]))
    c = (s % X) + ((s // X) % Y) + ((s // (X * Y)) % Z) + (s // (X * Y * Z))
    return s[(c & 1) == parity]


def test_64x128_dslash_sampled_sites():
    """configs[4]: 33.5 M sites.  TWIST_INV hop, fp32 and fp16 storage, 18- and 12-real links, both output parities,
    checked on ~6e4 sampled sites per case against the single-site oracle."""
    dims = (64, 64, 64, 128)
    X, Y, Z, T = dims
    seed = ti.NOISE_SEED
    F = Fields.from_slabs(dims, True)
    gauges = {(p, r): F.gauge(p, r) for p in (4, 2) for r in (18, 12)}
    F.drop_canonical()
    codes = torch.empty((T, Z, Y, X, 4, 3), dtype=torch.uint8, device="cuda")
    for t0 in range(0, T, 16):
        codes[t0:t0 + 16].copy_(torch.from_numpy(ti.z4_codes(dims, seed=seed, t0=t0, t1=t0 + 16)))
    refs = {}
    for parity in (0, 1):
        sites = _sample_sites(dims, parity, 30000, 11 + parity)
        Uf, Ub, nf, nb, sf, sb = gather_site_inputs(dims, sites, seed, ap=True)
        d = np.stack([oracle.hop_gathered(Uf[k], Ub[k], nf[k], nb[k], sf[k], sb[k]) for k in range(sites.size)])
        refs[parity] = (sites, oracle.twist(d.reshape(-1, 1, 1, 1, 4, 3), A, inverse=True).reshape(-1, 4, 3))
    canon = torch.empty((T * Z * Y * X, 4, 3, 2), dtype=torch.float64, device="cuda")
    for prec in (4, 2):
        pin = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, 1))
        tm.tm_spinor_pack_z4(F.L, codes, prec, 1, pin)
        out = tm.device_buffer(tm.tm_spinor_bytes(F.L, prec, 1, 1))
        for recon in (18, 12):
            out.zero_()
            for parity in (0, 1):
                tm.tm_dslash(F.L, gauges[(prec, recon)], prec, recon, F.half(out, prec, parity), F.half(pin, prec, 1 - parity), None,
                             parity, 0, tm.TM_KIND_TWIST_INV, KAPPA, MU)
            tm.tm_spinor_unpack(F.L, out, prec, 1, canon)
            torch.cuda.synchronize()
            for parity in (0, 1):
                sites, ref = refs[parity]
                got = canon[torch.from_numpy(sites).cuda()].cpu().numpy().view(np.complex128)[..., 0]
                assert rel(got, ref) < TOL[prec], (prec, recon, parity)
                # per-site bound as well: no single sampled site may be off by more than 20x the field tolerance
                worst = np.abs(got - ref).reshape(sites.size, -1).max(axis=1).max() / np.abs(ref).max()
                assert worst < 20 * TOL[prec], (prec, recon, parity, worst)


_REF = {}


@pytest.mark.parametrize("prec", [4, 2])
def test_32x64_insertions_full_size(prec):
    """NEXT-2 / NEXT-3 kernels at the bench size (32^3x64, the launch shapes bench.py times): the covariant derivative on the
    whole field, momentum-projected loops at all 123 momenta of p^2 <= 9 against the plain phase sums, the zero
    momentum against the time-slice loop kernel, the single-slice contraction, and (BH)^4 on the whole field."""
    dims = (32, 32, 32, 64)
    X, Y, Z, T = dims
    U = ti.gauge(dims)
    F = Fields(dims, U, True)
    a, b = ti.z4(dims, seed=1201), ti.gauss_spinor(dims, 1202)
    pa, pb_ = F.pack(a, prec), F.pack(b, prec)
    # covariant derivative, mu = t (antiperiodic boundary) and mu = x (checkerboard shifts)
    d = F.zeros_full(prec)
    for mu in (3, 0):
        tm.tm_covdev(F.L, F.gauge(prec, 12), prec, 12, d, pb_, mu, 1)
        assert rel(F.unpack(d, prec), oracle.covdev(U, b, mu)) < TOL[prec]
    # momentum-projected loops
    mom = oracle.momenta_p2_max(9)
    K = len(mom)
    out = torch.zeros((1, 16, T, K, 2), dtype=torch.float64, device="cuda")
    ws = tm.device_buffer(tm.tm_loop_momentum_workspace_bytes(F.L, 1, K, 3))
    tm.tm_loop_momentum(F.L, pa, pb_, prec, 1, mom, out, ws)
    got = out.cpu().numpy().view(np.complex128)[0, ..., 0]
    if "mom" not in _REF:  # every one of the 123 momenta (the plain phase sums of the oracle: about a minute, shared by both precisions)
        _REF["mom"] = oracle.loop_momentum(a, b, mom)
    ref = _REF["mom"]
    for k in range(K):
        assert rel(got[:, :, k], ref[:, :, k]) < TOL[prec], mom[k]
    o2 = torch.zeros((1, 16, T, 2), dtype=torch.float64, device="cuda")
    lws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, 1))
    tm.tm_loop_contract(F.L, pa, pb_, prec, 1, o2, lws)
    k0 = [i for i, p in enumerate(mom) if tuple(p) == (0, 0, 0)][0]
    assert rel(got[:, :, k0], o2.cpu().numpy().view(np.complex128)[0, ..., 0]) < 1e-6
    # single-slice contraction
    o3 = torch.zeros((1, 16, 2), dtype=torch.float64, device="cuda")
    tm.tm_loop_contract_slice(F.L, pa, pb_, prec, 1, 37, o3, lws)
    assert rel(o3.cpu().numpy().view(np.complex128)[0, ..., 0], oracle.loop_slice(a, b, 37)) < TOL[prec]
    # hopping-parameter remainder
    tmp = F.zeros_full(prec)
    tm.tm_hpe_remainder(F.L, F.gauge(prec, 12), prec, 12, d, pb_, tmp, KAPPA, MU, 1)
    err = rel(F.unpack(d, prec), oracle.hpe_remainder(U, b, KAPPA, MU))
    print("(BH)^4 relative L2 error at 32^3x64, storage bytes %d: %.3e" % (prec, err))
    # eight launches in a row, each rounding its result to the storage format; measured 5.6e-4 (fp16 storage) and 2.0e-7 (fp32)
    # on this field: the single-launch bound holds with room to spare (reading 34)
    assert err < TOL[prec]
