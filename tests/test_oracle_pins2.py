"""Pins for oracle/insertions.py, CPU only.

P19 covariant derivative, P20 contraction field and momentum projection, P21 one-derivative loops,
P22 time dilution / single-slice contraction, P23 hopping-parameter expansion (Eq. 16-17).
Every pin ties the numpy definitions to something outside them: the pinned C++ stencil, closed forms, np.fft, the
dense 4^4 matrices of oracle/dense.py.
"""
import numpy as np
import pytest

import oracle
import tm_inputs as ti
from oracle import dense

KAPPA, MU = ti.KAPPA, ti.MU
A = 2 * KAPPA * MU
D4 = (4, 4, 4, 4)
AXIS = (3, 2, 1, 0)


def rel(a, b):
    return np.linalg.norm((a - b).ravel()) / np.linalg.norm(b.ravel())


def vdot(a, b):
    return np.vdot(a.ravel(), b.ravel())


def plane_wave(dims, n, u, ap=True):
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    p = np.array([2 * np.pi * n[0] / X, 2 * np.pi * n[1] / Y, 2 * np.pi * n[2] / Z,
                  ((2 * n[3] + 1) if ap else 2 * n[3]) * np.pi / T])
    ph = np.exp(1j * (p[0] * x + p[1] * y + p[2] * z + p[3] * t))
    return p, ph[..., None, None] * u


def gauge_transform(U, g):
    """U'_mu(x) = g(x) U_mu(x) g(x+mu)^dag."""
    Up = np.empty_like(U)
    for m in range(4):
        gup = np.roll(g, -1, axis=AXIS[m])
        Up[..., m, :, :] = np.einsum("...ab,...bc,...dc->...ad", g, U[..., m, :, :], gup.conj())
    return Up


# ---- P19 covariant derivative ---------------------------------------------------------------------------------
def test_P19_covdev_against_the_pinned_stencil():
    """Dslash = sum_mu [U psi(x+mu) + U^dag psi(x-mu)] - 2 sum_mu g_mu D_mu and Dslash^dag flips the g_mu sign, hence
    sum_mu g_mu D_mu psi = (Dslash^dag - Dslash) psi / 4 with the C++ stencil (pinned by P2-P5): fixes the link orientation,
    the sign of the backward term, the factor 1/2 and the antiperiodic sign for the four directions together."""
    dims = (4, 6, 4, 8)
    U = ti.gauge(dims)
    psi = ti.gauss_spinor(dims, 11)
    for ap in (True, False):
        lhs = sum(np.einsum("ab,...bc->...ac", oracle.gamma(m), oracle.covdev(U, psi, m, ap=ap)) for m in range(4))
        rhs = (oracle.hop(U, psi, ap=ap, dagger=True) - oracle.hop(U, psi, ap=ap)) / 4
        assert rel(lhs, rhs) < 1e-14


@pytest.mark.parametrize("dims,n", [((4, 4, 4, 4), (1, 0, 3, 0)), ((4, 6, 8, 10), (1, 2, 3, 4)), ((4, 4, 4, 8), (0, 3, 1, 7))])
def test_P19_covdev_free_field_each_direction(dims, n):
    """U = 1: D_mu u e^{ipx} = i sin(p_mu) u e^{ipx}, per direction (the stencil pin only fixes the gamma-weighted sum);
    p_4 is an odd multiple of pi/T so the wave crosses the antiperiodic boundary."""
    rng = np.random.default_rng(5)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    p, psi = plane_wave(dims, n, u)
    U = ti.unit_gauge(dims)
    for m in range(4):
        d = oracle.covdev(U, psi, m)
        assert np.linalg.norm(d - 1j * np.sin(p[m]) * psi) < 1e-13 * np.linalg.norm(psi)


def test_P19_covdev_antihermitian_gauge_covariant_local():
    dims = (4, 4, 6, 4)
    U = ti.gauge(dims)
    phi, psi = ti.gauss_spinor(dims, 1), ti.gauss_spinor(dims, 2)
    g = ti.su3_field(dims, 77)
    Up = gauge_transform(U, g)
    for m in range(4):
        d = oracle.covdev(U, psi, m)
        assert abs(vdot(phi, d) + vdot(oracle.covdev(U, phi, m), psi)) < 1e-12 * abs(vdot(phi, phi))
        dp = oracle.covdev(Up, np.einsum("...ab,...sb->...sa", g, psi), m, ap=True)
        assert rel(dp, np.einsum("...ab,...sb->...sa", g, d)) < 1e-13
    # unit source at x0: D_mu e is non-zero only at x0 -+ mu, with -+(1/2) the link (locality, orientation)
    X, Y, Z, T = dims
    e = np.zeros((T, Z, Y, X, 4, 3), dtype=np.complex128)
    x0 = (1, 2, 3, 0)  # x,y,z,t ; t = 0 so that the backward neighbour in time sits across the antiperiodic boundary
    e[x0[3], x0[2], x0[1], x0[0], 2, 1] = 1.0
    for m in range(4):
        d = oracle.covdev(U, e, m)
        nz = np.argwhere(np.abs(d).sum(axis=(4, 5)) > 0)
        assert len(nz) == 2
        c = list(x0)
        c[m] = (x0[m] - 1) % dims[m]  # site x0 - mu sees e through its forward link: +1/2 s U_mu(x0 - mu)
        s = -1.0 if (m == 3) else 1.0
        got = d[c[3], c[2], c[1], c[0], 2, :]
        assert np.allclose(got, 0.5 * s * U[c[3], c[2], c[1], c[0], m][:, 1])
        c[m] = (x0[m] + 1) % dims[m]  # site x0 + mu sees e through U_mu(x0)^dag: -1/2 conj(U_mu(x0)[1, :])
        got = d[c[3], c[2], c[1], c[0], 2, :]
        assert np.allclose(got, -0.5 * U[x0[3], x0[2], x0[1], x0[0], m][1, :].conj())


# ---- P20 contraction field, momentum projection -----------------------------------------------------------------
def test_P20_momentum_zero_is_the_timeslice_loop_and_fft():
    dims = (4, 6, 8, 4)
    X, Y, Z, T = dims
    a, b = ti.gauss_spinor(dims, 21), ti.gauss_spinor(dims, 22)
    mom = oracle.momenta_p2_max(9)
    L = oracle.loop_momentum(a, b, mom)
    k0 = [i for i, p in enumerate(mom) if tuple(p) == (0, 0, 0)][0]
    assert rel(L[:, :, k0], oracle.loop(a, b)) < 1e-13  # the pinned C++ routine
    # library route (the paper's own: FFT of the contraction field): np.fft over z, y, x
    C = oracle.contract_field(a, b)
    F = np.fft.fftn(C, axes=(1, 2, 3))
    for k, (nx, ny, nz) in enumerate(mom):
        if abs(nx) >= X // 2 + 1 or abs(ny) >= Y // 2 + 1 or abs(nz) >= Z // 2 + 1:
            continue
        Ct = F[:, nz % Z, ny % Y, nx % X]
        ref = np.array([[np.sum(oracle.Gamma(n) * Ct[t]) for t in range(T)] for n in range(16)])
        assert rel(L[:, :, k], ref) < 1e-12


def test_P20_momentum_plane_wave_delta_and_list():
    """b = a e^{iqx} with |a_i| = 1 (Z2xiZ2 noise): sum_x e^{-ipx} a^dag b = 12 V3 delta_{p,q} for Gamma_0."""
    dims = (8, 8, 8, 4)
    X, Y, Z, T = dims
    a = ti.z4(dims, seed=5)
    q = (2, -1, 3)
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    b = a * np.exp(2j * np.pi * (q[0] * x / X + q[1] * y / Y + q[2] * z / Z))[..., None, None]
    mom = oracle.momenta_p2_max(14)
    L = oracle.loop_momentum(a, b, mom)
    for k, p in enumerate(mom):
        expect = 12.0 * X * Y * Z if tuple(p) == q else 0.0
        assert np.allclose(L[0, :, k], expect, atol=1e-9)
    # the p^2 <= 9 list of PAPER.md:427: 123 vectors, closed under p -> -p, sorted by p^2
    m9 = oracle.momenta_p2_max(9)
    assert len(m9) == 123 and len(oracle.momenta_p2_max(0)) == 1 and len(oracle.momenta_p2_max(1)) == 7
    s = {tuple(p) for p in m9}
    assert all((-p[0], -p[1], -p[2]) in s for p in s) and all(p[0] ** 2 + p[1] ** 2 + p[2] ** 2 <= 9 for p in s)
    p2 = (m9 ** 2).sum(axis=1)
    assert np.all(np.diff(p2) >= 0)


# ---- P21 one-derivative loops -----------------------------------------------------------------------------------
def test_P21_derivative_loop_gauge_invariant_and_free_field():
    dims = (4, 4, 4, 6)
    U = ti.gauge(dims)
    a, b = ti.gauss_spinor(dims, 31), ti.gauss_spinor(dims, 32)
    g = ti.su3_field(dims, 78)
    Up = gauge_transform(U, g)
    ga, gb = np.einsum("...ab,...sb->...sa", g, a), np.einsum("...ab,...sb->...sa", g, b)
    for m in range(4):
        assert rel(oracle.loop_derivative(Up, ga, gb, m), oracle.loop_derivative(U, a, b, m)) < 1e-12
    # free field, a = b = plane wave u e^{ipx}: L[n][t] = i sin(p_mu) V3 u^dag Gamma_n u
    rng = np.random.default_rng(9)
    u = rng.normal(size=(4, 3)) + 1j * rng.normal(size=(4, 3))
    p, psi = plane_wave(dims, (1, 3, 2, 4), u)
    U1 = ti.unit_gauge(dims)
    for m in range(4):
        L = oracle.loop_derivative(U1, psi, psi, m)
        for n in range(16):
            expect = 1j * np.sin(p[m]) * 64 * np.einsum("ac,ab,bc->", u.conj(), oracle.Gamma(n), u)
            assert np.allclose(L[n], expect, atol=1e-10)


# ---- P22 time dilution ------------------------------------------------------------------------------------------
def test_P22_time_dilution_partition_and_slice_contraction():
    dims = (4, 4, 4, 8)
    eta = ti.z4(dims, seed=3)
    parts = [oracle.time_dilute(eta, [t]) for t in range(8)]
    assert np.array_equal(sum(parts), eta)  # the m = T sub-spaces partition the source
    coh = oracle.time_dilute(eta, [1, 5])     # coherent source: two well separated slices
    assert np.array_equal(coh, parts[1] + parts[5])
    assert np.count_nonzero(np.abs(coh).sum(axis=(1, 2, 3, 4, 5))) == 2
    b = ti.gauss_spinor(dims, 4)
    full = oracle.loop(eta, b)
    for t0 in (0, 3, 7):
        assert rel(oracle.loop_slice(eta, b, t0), full[:, t0]) < 1e-13
        assert rel(oracle.loop(parts[t0], b)[:, t0], full[:, t0]) < 1e-13


# ---- P23 hopping-parameter expansion ------------------------------------------------------------------------------
@pytest.fixture(scope="module")
def dense_hpe():
    U = ti.gauge(D4)
    Mat = dense.dense_M(U, KAPPA, MU, ap=True)
    Binv = np.kron(np.eye(256), np.kron(np.eye(4) + 1j * A * dense.GAMMA5, np.eye(3)))
    B = np.linalg.inv(Binv)
    H = Mat - Binv
    BH = B @ H
    BH2 = BH @ BH
    series = B - BH @ B + BH2 @ B - BH2 @ BH @ B
    return U, Mat, np.linalg.inv(Mat), series, BH2 @ BH2


def test_P23_hpe_identity_dense_and_vectors(dense_hpe):
    """Eq. (16) as a matrix identity on 4^4, and the oracle's vector routines against those matrices."""
    U, Mat, Minv, series, BH4 = dense_hpe
    assert rel(series + BH4 @ Minv, Minv) < 1e-12
    eta = ti.z4(D4, seed=8)
    v = eta.reshape(-1)
    assert rel(oracle.hpe_series(U, eta, KAPPA, MU).reshape(-1), series @ v) < 1e-13
    s = (Minv @ v).reshape(eta.shape)
    assert rel(oracle.hpe_remainder(U, s, KAPPA, MU).reshape(-1), BH4 @ (Minv @ v)) < 1e-13
    # with the CG solution instead of the dense one (Eq. 17: the stochastic term uses s_r)
    s_cg, _ = oracle.cg_solve(U, eta, KAPPA, MU, 1e-12, 2000)
    assert rel(oracle.hpe_series(U, eta, KAPPA, MU) + oracle.hpe_remainder(U, s_cg, KAPPA, MU), s_cg) < 1e-10


def test_P23_hpe_local_traces_are_the_dense_ones(dense_hpe):
    """Tr_t[Gamma_n (B - BHB + (BH)^2 B - (BH)^3 B)] from the dense matrices on a RANDOM gauge field equals
    V3 x the gauge-independent per-site closed form; only Gamma = 1, g5 survive."""
    U, Mat, Minv, series, BH4 = dense_hpe
    tr = dense.timeslice_traces(series, D4)
    loc = oracle.hpe_local_traces(KAPPA, MU)
    assert np.allclose(tr, 64 * loc[:, None], atol=1e-10)
    nz = [n for n in range(16) if abs(loc[n]) > 1e-12]
    assert nz == [0, 15]
    # exact split of the loop: Tr_t[Gamma M^-1] = local part + Tr_t[Gamma (BH)^4 M^-1]
    assert np.allclose(dense.timeslice_traces(Minv, D4), 64 * loc[:, None] + dense.timeslice_traces(BH4 @ Minv, D4), atol=1e-10)
    # leading term alone: Tr[Gamma_n B] = 12/(1+a^2) for 1, -12 i a/(1+a^2) for g5 ; the (BH)^2 B term is O(kappa^2 a)
    assert abs(loc[0] - 12 / (1 + A * A)) < 1000 * KAPPA ** 2 * A ** 2
    assert abs(loc[15] + 12j * A / (1 + A * A)) < 200 * KAPPA ** 2 * A


# ---- P24 symmetric preconditioning, PAPER.md:376 Eq. (A3) ----------------------------------------------------------
def test_P24_symmetric_preconditioning_is_a_rescaling_of_the_normal_operator():
    """M_sym = R^-1 M_pc and R^dag R = (1 + a^2) 1 for the degenerate twist R = 1 + i a g5, hence
    M_sym^dag M_sym = M_pc^dag M_pc / (1 + a^2): CG on either normal system produces the same iterates, which is why the
    library implements (A2) only (reading 7).  Checked with a large twist so that the factor is visible."""
    dims = (4, 4, 6, 4)
    U = ti.gauge(dims)
    v = oracle.project(ti.gauss_spinor(dims, 5), 0)
    phi = oracle.project(ti.gauss_spinor(dims, 6), 0)
    for mu in (MU, 0.9):
        a = 2 * KAPPA * mu
        ms = oracle.Mpc_sym(U, v, KAPPA, mu)
        assert rel(ms, oracle.twist(oracle.Mpc(U, v, KAPPA, mu), a, inverse=True)) < 1e-13      # M_sym = R^-1 M_pc
        assert abs(vdot(phi, ms) - vdot(oracle.Mpc_sym(U, phi, KAPPA, mu, dagger=True), v)) < 1e-12 * abs(vdot(phi, phi))
        lhs = oracle.Mpc_sym(U, ms, KAPPA, mu, dagger=True)
        assert rel(lhs, oracle.MdagM(U, v, KAPPA, mu) / (1 + a * a)) < 1e-13


def test_P25_temporal_gauge_is_a_gauge_transformation_of_the_oracle_operator():
    """oracle.temporal_gauge (a non-random, time-ordered transformation: g(x,t) = prod_{t'<t} U_t(x,t')) against the oracle:
    U' stays in SU(3), U'_t = 1 on every slice but the last, the last slice carries the Polyakov loop (its trace equals that of the
    ordered product of the original temporal links), M(U') g = g M(U) with the antiperiodic sign left on the fermions, and the
    truncated CG takes the same number of iterations on both fields (the Krylov spaces are unitarily equivalent)."""
    dims = (4, 4, 6, 8)
    U = ti.gauge(dims)
    Up, g = oracle.temporal_gauge(U)
    eye = np.eye(3)
    assert np.abs(Up @ np.conj(np.swapaxes(Up, -1, -2)) - eye).max() < 1e-13
    assert np.abs(np.linalg.det(Up) - 1).max() < 1e-13
    assert not np.abs(Up[:-1, ..., 3, :, :] - eye).any()
    P = np.broadcast_to(eye, U.shape[1:4] + (3, 3)).astype(np.complex128)
    for t in range(dims[3]):
        P = P @ U[t, ..., 3, :, :]
    assert np.abs(np.trace(P, axis1=-2, axis2=-1) - np.trace(Up[-1, ..., 3, :, :], axis1=-2, axis2=-1)).max() < 1e-12
    rot = lambda v: np.einsum("tzyxab,tzyxsb->tzyxsa", g, v)
    psi = ti.gauss_spinor(dims, 41)
    for dagger in (False, True):
        lhs = oracle.M(Up, rot(psi), ti.KAPPA, ti.MU, ap=True, dagger=dagger)
        rhs = rot(oracle.M(U, psi, ti.KAPPA, ti.MU, ap=True, dagger=dagger))
        assert np.linalg.norm(lhs - rhs) / np.linalg.norm(rhs) < 1e-14
    eta = ti.z4(dims, seed=5)
    s0, i0 = oracle.cg_solve(U, eta, ti.KAPPA, ti.MU, 1e-6, 500)
    s1, i1 = oracle.cg_solve(Up, rot(eta), ti.KAPPA, ti.MU, 1e-6, 500)
    assert i0["iters"] == i1["iters"]
    assert np.linalg.norm(s1 - rot(s0)) / np.linalg.norm(s0) < 1e-10
    assert np.linalg.norm(oracle.loop(rot(eta), s1) - oracle.loop(eta, s0)) / np.linalg.norm(oracle.loop(eta, s0)) < 1e-10
