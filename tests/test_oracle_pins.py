"""Pins for the CPU oracle (no GPU): what the paper and the mathematics fix, independent of the oracle's own code.

P-numbers follow SURVEY.md section 8(c-3); readings are listed in DESIGN.md.
"""
import numpy as np
import pytest

import oracle
import tm_inputs as ti
from oracle import dense

KAPPA, MU = ti.KAPPA, ti.MU
A = 2 * KAPPA * MU
D4 = (4, 4, 4, 4)


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


@pytest.fixture(scope="module")
def U4():
    return ti.gauge(D4)


@pytest.fixture(scope="module")
def dense4(U4):
    Mat = dense.dense_M(U4, KAPPA, MU, ap=True)
    return Mat, np.linalg.inv(Mat)


# ---- P1 Clifford algebra ---------------------------------------------------------------------------------
def test_P1_clifford():
    g = [oracle.gamma(m) for m in range(4)]
    for m in range(4):
        assert np.allclose(g[m], g[m].conj().T)
        assert np.allclose(g[m], dense.GAMMA[m])  # C++ table vs the independently typed numpy table
        for n in range(4):
            assert np.allclose(g[m] @ g[n] + g[n] @ g[m], 2 * np.eye(4) * (m == n))
    g5 = oracle.gamma(4)
    assert np.allclose(g5, g[0] @ g[1] @ g[2] @ g[3])
    assert np.allclose(g5, np.diag([1, 1, -1, -1]))
    for n in range(16):
        G = oracle.Gamma(n)
        assert np.allclose(G, dense.Gamma_n(n))
        pc = bin(n).count("1")
        sign = 1 if pc in (0, 1, 4) else -1
        assert np.allclose(G.conj().T, sign * G)
        assert np.count_nonzero(np.abs(G) > 1e-14) == 4 and np.allclose(np.abs(G[np.abs(G) > 1e-14]), 1)
    assert np.allclose(oracle.Gamma(0), np.eye(4)) and np.allclose(oracle.Gamma(8), g[3])
    assert np.allclose(oracle.Gamma(15), g5)


# ---- P2 free field closed form ---------------------------------------------------------------------------
def plane_wave(dims, n, u):
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    p = np.array([2 * np.pi * n[0] / X, 2 * np.pi * n[1] / Y, 2 * np.pi * n[2] / Z, (2 * n[3] + 1) * np.pi / T])
    ph = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return p, ph[..., None, None] * u


@pytest.mark.parametrize("dims,n", [((4, 4, 4, 4), (1, 0, 3, 0)), ((4, 6, 8, 10), (1, 2, 3, 4)),
                                    ((6, 4, 4, 8), (5, 1, 2, 7)), ((4, 4, 4, 8), (0, 0, 0, 3))])
def test_P2_free_field(dims, n):
    rng = np.random.default_rng(7)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    U = ti.unit_gauge(dims)
    p, psi = plane_wave(dims, n, u)
    g = dense.GAMMA
    Mp = (1 - 2 * KAPPA * np.sum(np.cos(p))) * np.eye(4) + 2j * KAPPA * sum(g[m] * np.sin(p[m]) for m in range(4)) \
        + 1j * A * dense.GAMMA5
    ref = np.einsum("ab,...bc->...ac", Mp, psi)
    out = oracle.M(U, psi, KAPPA, MU, ap=True)
    assert rel(out, ref) < 1e-13
    # M^dag M psi = lambda(p) psi, lambda = A^2 + B^2 + (2 kappa mu)^2
    lam = (1 - 2 * KAPPA * np.sum(np.cos(p))) ** 2 + 4 * KAPPA ** 2 * np.sum(np.sin(p) ** 2) + A ** 2
    out2 = oracle.M(U, out, KAPPA, MU, ap=True, dagger=True)
    assert rel(out2, lam * psi) < 1e-13
    # even-odd: M_pc psi_e = [R - kappa^2 H R^-1 H] u e^{ipx} on even sites, H(p) = sum_mu (2 cos p - 2 i g_mu sin p)
    H = sum(2 * np.cos(p[m]) * np.eye(4) - 2j * g[m] * np.sin(p[m]) for m in range(4))
    R = np.eye(4) + 1j * A * dense.GAMMA5
    Mpc_p = R - KAPPA ** 2 * H @ np.linalg.inv(R) @ H
    ref_pc = oracle.project(np.einsum("ab,...bc->...ac", Mpc_p, psi), 0)
    assert rel(oracle.Mpc(U, psi, KAPPA, MU, parity=0), ref_pc) < 1e-13
    # the hop itself: Dslash psi = H(p) psi
    assert rel(oracle.hop(U, psi), np.einsum("ab,...bc->...ac", H, psi)) < 1e-13


# ---- P3 adjointness / gamma5-hermiticity -----------------------------------------------------------------
@pytest.mark.parametrize("dims", [(4, 4, 4, 4), (4, 6, 4, 8)])
def test_P3_gamma5_hermiticity(dims):
    U = ti.gauge(dims)
    phi, psi = ti.gauss_spinor(dims, 11), ti.gauss_spinor(dims, 12)
    g5 = np.array([1, 1, -1, -1.0])[:, None]
    # <phi, D psi> = <D^dag phi, psi>, and D^dag = g5 D g5
    assert abs(vdot(phi, oracle.hop(U, psi)) - vdot(oracle.hop(U, phi, dagger=True), psi)) < 1e-10
    assert rel(oracle.hop(U, phi, dagger=True), g5 * oracle.hop(U, g5 * phi)) < 1e-14
    # <phi, M(mu) psi> = <g5 M(-mu) g5 phi, psi>
    lhs = vdot(phi, oracle.M(U, psi, KAPPA, MU))
    assert abs(lhs - vdot(g5 * oracle.M(U, g5 * phi, KAPPA, -MU), psi)) < 1e-10
    assert abs(lhs - vdot(oracle.M(U, phi, KAPPA, MU, dagger=True), psi)) < 1e-10
    for par in (0, 1):
        pe, qe = oracle.project(phi, par), oracle.project(psi, par)
        lhs = vdot(pe, oracle.Mpc(U, qe, KAPPA, MU, parity=par))
        assert abs(lhs - vdot(oracle.Mpc(U, pe, KAPPA, MU, parity=par, dagger=True), qe)) < 1e-10
        assert abs(lhs - vdot(g5 * oracle.Mpc(U, g5 * pe, KAPPA, -MU, parity=par), qe)) < 1e-10
        q = vdot(qe, oracle.MdagM(U, qe, KAPPA, MU, parity=par))
        assert abs(q.imag) < 1e-10 and q.real > 0
        assert abs(q.real - np.linalg.norm(oracle.Mpc(U, qe, KAPPA, MU, parity=par)) ** 2) < 1e-9


# ---- P4 gauge covariance ---------------------------------------------------------------------------------
def test_P4_gauge_covariance():
    dims = (4, 6, 4, 8)
    U = ti.gauge(dims)
    g = ti.su3_field(dims, 99)
    psi, phi = ti.gauss_spinor(dims, 5), ti.gauss_spinor(dims, 6)
    Ug = np.empty_like(U)
    for m, ax in enumerate((3, 2, 1, 0)):  # mu = x,y,z,t <-> array axes 3,2,1,0
        gf = np.roll(g, -1, axis=ax)  # g(x+mu)
        Ug[..., m, :, :] = np.einsum("...ab,...bc,...dc->...ad", g, U[..., m, :, :], gf.conj())
    psig = np.einsum("...ab,...sb->...sa", g, psi)
    phig = np.einsum("...ab,...sb->...sa", g, phi)
    out = oracle.M(U, psi, KAPPA, MU)
    outg = oracle.M(Ug, psig, KAPPA, MU)
    assert rel(outg, np.einsum("...ab,...sb->...sa", g, out)) < 1e-13
    assert np.allclose(oracle.loop(phig, outg), oracle.loop(phi, out), atol=1e-9)


# ---- P5 dense brute force on 4^4 -------------------------------------------------------------------------
def test_P5_dense_matvec(U4, dense4):
    Mat, _ = dense4
    psi = ti.gauss_spinor(D4, 21)
    assert rel(oracle.M(U4, psi, KAPPA, MU), (Mat @ psi.ravel()).reshape(psi.shape)) < 1e-13
    assert rel(oracle.M(U4, psi, KAPPA, MU, dagger=True), (Mat.conj().T @ psi.ravel()).reshape(psi.shape)) < 1e-13
    # hop = (1 + i a g5 - M)/kappa
    Mat0 = dense.dense_M(U4, KAPPA, 0.0)
    assert rel(oracle.hop(U4, psi), ((psi.ravel() - Mat0 @ psi.ravel()) / KAPPA).reshape(psi.shape)) < 1e-12
    # Schur complement from dense blocks vs oracle Mpc
    par = ti.parity_mask(D4).ravel()
    e = np.repeat(par == 0, 12)
    o = ~e
    Mee, Meo, Moe, Moo = Mat[np.ix_(e, e)], Mat[np.ix_(e, o)], Mat[np.ix_(o, e)], Mat[np.ix_(o, o)]
    S = Mee - Meo @ np.linalg.inv(Moo) @ Moe
    v = psi.ravel()[e]
    out = oracle.Mpc(U4, oracle.project(psi, 0), KAPPA, MU, parity=0).ravel()
    assert rel(out[e], S @ v) < 1e-13 and np.abs(out[o]).max() == 0


def test_P5_P8_cg_vs_dense_solve(U4, dense4):
    Mat, Minv = dense4
    eta = ti.z4(D4)
    s, info = oracle.cg_solve(U4, eta, KAPPA, MU, 1e-12, 2000)
    ref = (Minv @ eta.ravel()).reshape(eta.shape)
    assert info["iterated_resid"] <= 1e-12 and info["true_resid_normal"] < 2e-12
    assert info["true_resid_full"] < 1e-11  # P8: full unpreconditioned residual
    assert rel(s, ref) < 1e-10
    assert rel((Mat @ s.ravel()), eta.ravel()) < 1e-11
    # truncated LP mode: ~1/10 of the HP iteration count as a sanity band
    s2, info2 = oracle.cg_solve(U4, eta, KAPPA, MU, 1e-2, 2000)
    assert info2["iterated_resid"] <= 1e-2 and 3 <= info2["iters"] <= info["iters"] // 3
    # fixed-iteration truncation
    s3, info3 = oracle.cg_solve(U4, eta, KAPPA, MU, 0.0, 5)
    assert info3["iters"] == 5


# ---- P6 Eq. (11), (14) -----------------------------------------------------------------------------------
def test_P6_flavour_identities(U4):
    psi = ti.gauss_spinor(D4, 31)
    g5 = np.array([1, 1, -1, -1.0])[:, None]
    Mu, Md = oracle.M(U4, psi, KAPPA, MU), oracle.M(U4, psi, KAPPA, -MU)
    assert rel(Mu - Md, 2j * A * g5 * psi) < 1e-13               # Eq. (11), kappa-normalised
    assert rel(Mu + Md, 2 * oracle.M(U4, psi, KAPPA, 0.0)) < 1e-14  # Eq. (14)


# ---- P7 HPE identity Eq. (16) ----------------------------------------------------------------------------
def test_P7_hpe_identity(U4, dense4):
    _, Minv = dense4
    eta = ti.z4(D4, seed=77)
    B = lambda v: oracle.twist(v, A, inverse=True)
    H = lambda v: -KAPPA * oracle.hop(U4, v)
    BH = lambda v: B(H(v))
    s = (Minv @ eta.ravel()).reshape(eta.shape)
    t0 = B(eta)
    t1 = BH(t0)
    t2 = BH(t1)
    t3 = BH(t2)
    rhs = t0 - t1 + t2 - t3 + BH(BH(BH(BH(s))))
    assert rel(rhs, s) < 1e-12
    # with the oracle's own CG solution
    s_cg, _ = oracle.cg_solve(U4, eta, KAPPA, MU, 1e-12, 2000)
    assert rel(t0 - t1 + t2 - t3 + BH(BH(BH(BH(s_cg)))), s_cg) < 1e-10
    # Tr H = 0 (the hopping matrix is traceless): unit sources never return to their own site
    e = np.zeros_like(eta)
    e[1, 2, 3, 0, 2, 1] = 1
    assert oracle.hop(U4, e)[1, 2, 3, 0].any() == False  # noqa: E712


# ---- P9 spectral bound -----------------------------------------------------------------------------------
def test_P9_spectral_bound(U4, dense4):
    Mat, _ = dense4
    w = np.linalg.eigvalsh(Mat.conj().T @ Mat)
    assert w.min() >= A ** 2 * (1 - 1e-9)
    for seed in range(3):
        v = ti.gauss_spinor(D4, 40 + seed)
        q = np.linalg.norm(oracle.M(U4, v, KAPPA, MU)) ** 2 / np.linalg.norm(v) ** 2
        assert q >= A ** 2


# ---- P10 locality ----------------------------------------------------------------------------------------
def test_P10_locality():
    dims = (4, 6, 4, 8)
    X, Y, Z, T = dims
    U = ti.gauge(dims)
    e = np.zeros((T, Z, Y, X, 4, 3), dtype=np.complex128)
    c = (0, 3, 5, 3)  # t,z,y,x
    e[c][1, 2] = 1
    out = oracle.hop(U, e)
    nz = set(map(tuple, np.argwhere(np.abs(out).sum(axis=(4, 5)) > 0)))
    exp = set()
    for ax, L in zip(range(4), (T, Z, Y, X)):
        for d in (-1, 1):
            cc = list(c)
            cc[ax] = (cc[ax] + d) % L
            exp.add(tuple(cc))
    assert nz == exp
    out2 = oracle.Mpc(U, e, KAPPA, MU, parity=sum(c) & 1)
    for idx in np.argwhere(np.abs(out2).sum(axis=(4, 5)) > 0):
        dist = sum(min((a - b) % L, (b - a) % L) for a, b, L in zip(idx, c, (T, Z, Y, X)))
        assert dist in (0, 2)


# ---- P11 translation covariance --------------------------------------------------------------------------
@pytest.mark.parametrize("ax", [0, 1, 2, 3])
def test_P11_translation(ax):
    dims = (4, 6, 4, 8)
    U = ti.gauge(dims)
    psi = ti.gauss_spinor(dims, 3)
    ap = ax != 0  # for a time shift use periodic b.c. (the boundary sign would have to move with the shift)
    out = oracle.M(U, psi, KAPPA, MU, ap=ap)
    out_s = oracle.M(np.roll(U, 1, axis=ax), np.roll(psi, 1, axis=ax), KAPPA, MU, ap=ap)
    assert rel(out_s, np.roll(out, 1, axis=ax)) < 1e-14


# ---- P13 noise closed forms ------------------------------------------------------------------------------
def test_P13_noise_closed_forms():
    dims = (4, 6, 4, 8)
    X, Y, Z, T = dims
    eta = ti.z4(dims)
    L = oracle.loop(eta, eta)
    assert np.allclose(L[0], 12 * X * Y * Z)
    for n in range(16):
        herm = bin(n).count("1") in (0, 1, 4)
        assert np.allclose(L[n].imag if herm else L[n].real, 0, atol=1e-10)
    a, b = ti.gauss_spinor(dims, 1), ti.gauss_spinor(dims, 2)
    L = oracle.loop(a, b)
    assert abs(L[0].sum() - vdot(a, b)) < 1e-9
    # against a direct numpy evaluation with the independently typed Gamma table
    for n in (1, 6, 9, 15):
        ref = np.einsum("tzyxac,ab,tzyxbc->t", a.conj(), dense.Gamma_n(n), b)
        assert np.allclose(L[n], ref)


# ---- P14 exact trace ------------------------------------------------------------------------------------
def test_P14_loop_of_exact_columns_is_exact_trace(U4, dense4):
    """sum_i e_i^dag Gamma_n (M^-1 e_i) over all 3072 unit sources = Tr_t[Gamma_n M^-1]; columns from the dense inverse."""
    _, Minv = dense4
    ref = dense.timeslice_traces(Minv, D4)
    acc = np.zeros((16, 4), dtype=np.complex128)
    V = 256
    for i in range(0, 12 * V, 97):  # a strided subset through the loop routine, the rest through linearity below
        e = np.zeros(12 * V, dtype=np.complex128)
        e[i] = 1
        acc += oracle.loop(e.reshape(4, 4, 4, 4, 4, 3), Minv[:, i].reshape(4, 4, 4, 4, 4, 3))
    sub = np.zeros_like(acc)
    blocks = Minv.reshape(V, 4, 3, V, 4, 3)
    for i in range(0, 12 * V, 97):
        x, al, c = i // 12, (i // 3) % 4, i % 3
        for n in range(16):
            sub[n, x // 64] += (dense.Gamma_n(n)[al, :] * blocks[x, :, c, x, al, c]).sum()
    assert np.allclose(acc, sub, atol=1e-12)
    assert np.abs(ref).max() > 1  # Tr[1 M^-1] is O(V)


@pytest.mark.slow
def test_P14_fully_diluted_cg_loop_timeslice(U4, dense4):
    """north_star: fully spin-colour-site-diluted loop on 4^4 = exact Tr[Gamma M^-1] per time slice (slice t=3, which
    touches the antiperiodic boundary), every solve by the oracle CG."""
    from concurrent.futures import ThreadPoolExecutor
    _, Minv = dense4
    ref = dense.timeslice_traces(Minv, D4)
    t = 3

    def one(i):
        e = np.zeros((4, 4, 4, 4, 4, 3), dtype=np.complex128)
        e.reshape(-1)[t * 64 * 12 + i] = 1
        s, info = oracle.cg_solve(U4, e, KAPPA, MU, 1e-11, 2000)
        return oracle.loop(e, s)

    with ThreadPoolExecutor(8) as ex:
        acc = sum(ex.map(one, range(64 * 12)))
    assert np.abs(acc[:, [0, 1, 2]]).max() < 1e-12
    assert rel(acc[:, t], ref[:, t]) < 1e-9


def test_P14_stochastic_estimate_converges(U4, dense4):
    """Eq. (10): (1/N_r) sum_r eta_r^dag Gamma s_r -> Tr[Gamma M^-1] as 1/sqrt(N_r) (here with exact columns)."""
    _, Minv = dense4
    ref = dense.timeslice_traces(Minv, D4)
    errs = []
    for nr in (4, 64):
        acc = np.zeros((16, 4), dtype=np.complex128)
        for r in range(nr):
            eta = ti.z4(D4, seed=1000 + r)
            acc += oracle.loop(eta, (Minv @ eta.ravel()).reshape(eta.shape))
        errs.append(np.linalg.norm(acc / nr - ref))
    assert errs[1] < 0.6 * errs[0]
    assert errs[1] / np.linalg.norm(ref) < 0.05


@pytest.mark.parametrize("dagger", [False, True])
def test_hop_gathered_is_the_stencil_at_one_site(dagger):
    """orc_hop_gathered (single-site evaluation used for sampled parity at 64^3x128) against the pinned full-lattice
    stencil on every site of an antiperiodic 4x4x6x8 lattice, inputs regenerated site by site from the counter-based
    generators -- and against the free-field closed form H(p) u e^{ipx} of P2 at one site."""
    import sys, os
    sys.path.insert(0, os.path.dirname(__file__))
    from tm_harness import gather_site_inputs
    dims = (4, 4, 6, 8)
    X, Y, Z, T = dims
    U = ti.gauge(dims)
    psi = ti.z4(dims, seed=91)
    ref = oracle.hop(U, psi, ap=True, dagger=dagger).reshape(-1, 4, 3)
    sites = np.arange(X * Y * Z * T)
    Uf, Ub, nf, nb, sf, sb = gather_site_inputs(dims, sites, 91, ap=True)
    got = np.stack([oracle.hop_gathered(Uf[k], Ub[k], nf[k], nb[k], sf[k], sb[k], dagger=dagger) for k in sites])
    assert np.abs(got - ref).max() < 1e-13
    # free field: U = 1, psi = u e^{ipx}: (Dslash psi)(x) = sum_mu (2 cos p_mu - 2 i E gamma_mu sin p_mu) u e^{ipx}
    rng = np.random.default_rng(3)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    p = np.array([2 * np.pi * 1 / X, 2 * np.pi * 3 / Y, 0.0, 2 * np.pi * 2 / T])
    x = np.array([1, 2, 5, 3])
    one = np.broadcast_to(np.eye(3, dtype=np.complex128), (4, 3, 3)).copy()
    nfw = np.stack([u * np.exp(1j * (p @ x + p[mu])) for mu in range(4)])
    nbw = np.stack([u * np.exp(1j * (p @ x - p[mu])) for mu in range(4)])
    got1 = oracle.hop_gathered(one, one, nfw, nbw, np.ones(4), np.ones(4), dagger=dagger)
    E = -1.0 if dagger else 1.0
    H = sum(2 * np.cos(p[mu]) * np.eye(4) - 2j * E * np.sin(p[mu]) * oracle.gamma(mu) for mu in range(4))
    assert np.abs(got1 - np.exp(1j * (p @ x)) * (H @ u)).max() < 1e-13


def test_P17_one_end_trick_exact_traces(U4, dense4):
    """PAPER.md:120-141 Eq. (11)-(15) as exact identities on 4^4: summing the one-end loops over ALL 3072 unit sources
    (s_i = column i of the dense inverse) gives Tr_t[(M_d^-1 - M_u^-1) Gamma_n] (tau3 form, s = M_u^-1 eta; DESIGN.md
    reading 25 on the sign) and Tr_t[(M_u^-1 + M_d^-1) Gamma_n] (generalised form)."""
    dims = (4, 4, 4, 4)
    _, Su = dense4
    Sd = np.linalg.inv(dense.dense_M(U4, KAPPA, -MU, ap=True))
    tr_u, tr_d = dense.timeslice_traces(Su, dims), dense.timeslice_traces(Sd, dims)
    acc3 = np.zeros((16, 4), dtype=np.complex128)
    accg = np.zeros((16, 4), dtype=np.complex128)
    for i in range(Su.shape[1]):
        s = Su[:, i].reshape(4, 4, 4, 4, 4, 3)
        acc3 += oracle.loop_oneend_tau3(s, KAPPA, MU)
        accg += oracle.loop_oneend_general(U4, s, KAPPA)
    assert np.abs(acc3 - (tr_d - tr_u)).max() < 1e-11 * max(1.0, np.abs(tr_u).max())
    assert np.abs(accg - (tr_u + tr_d)).max() < 1e-10 * np.abs(tr_u).max()
    # gamma5 of the oracle is the diagonal (1,1,-1,-1) of the declared basis and squares to one
    psi = ti.gauss_spinor(dims, 4)
    assert np.array_equal(oracle.gamma5(psi), psi * np.array([1, 1, -1, -1])[:, None])


def test_P18_tsm_combination_closed_forms():
    """PAPER.md:75-77 Eq. (8): constants c1, c2, c3 give c1 - c2 + c3; identical HP/LP pairs leave the LP mean; N_LP = 0
    leaves the mean correction; the combination is linear."""
    rng = np.random.default_rng(8)
    shp = (16, 6)
    c1, c2, c3 = (rng.normal(size=shp) + 1j * rng.normal(size=shp) for _ in range(3))
    out = oracle.tsm_combine([c1] * 3, [c2] * 3, [c3] * 5)
    assert np.abs(out - (c1 - c2 + c3)).max() < 1e-14
    hp = rng.normal(size=(4,) + shp) + 0j
    lp = rng.normal(size=(7,) + shp) + 0j
    assert np.abs(oracle.tsm_combine(hp, hp, lp) - lp.mean(axis=0)).max() < 1e-14
    lps = rng.normal(size=(4,) + shp) + 0j
    assert np.abs(oracle.tsm_combine(hp, lps, lp[:0]) - (hp - lps).mean(axis=0)).max() < 1e-14
    assert np.abs(oracle.tsm_combine(2 * hp, 2 * lps, 2 * lp) - 2 * oracle.tsm_combine(hp, lps, lp)).max() < 1e-13
