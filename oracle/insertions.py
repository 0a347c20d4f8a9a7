"""fp64 CPU oracle, part 2 -- TEST INFRASTRUCTURE ONLY (same rules as oracle/__init__.py).

Plain numpy definitions of the SURVEY.md 8(f) NEXT-2 / NEXT-3 rows: the colour-traced Dirac-open contraction field,
its momentum projection, the covariant derivative for one-derivative insertions,
time-dilution masks and the hopping-parameter expansion (Eq. 16-17).

Everything here is written from the definitions with np.roll / nested loops over small index sets; nothing is blocked,
fused or reordered.  Fields are complex128 in the canonical layout U[T][Z][Y][X][4][3][3], psi[T][Z][Y][X][4][3].
Readings of the paper (items 27-31) are repeated in the docstrings.
"""
import numpy as np

# numpy axis of direction mu = 0..3 = x,y,z,t in the canonical layout [T][Z][Y][X]
_AXIS = (3, 2, 1, 0)


def _c(a):
    return np.ascontiguousarray(a, dtype=np.complex128)


def _boundary_sign(shape4, mu, ap, forward):
    """s_mu(x) of the hop leaving x forward (or arriving from x - mu backward): -1 only for mu = t across t = T-1 <-> 0."""
    s = np.ones(shape4)
    if ap and mu == 3:
        T = shape4[0]
        if forward:
            s[T - 1] = -1.0  # hop from t = T-1 to t = 0
        else:
            s[0] = -1.0      # hop from t = 0 back to t = T-1
    return s


def covdev(U, psi, mu, ap=True):
    """Symmetric lattice covariant derivative, acting on colour only (spin untouched):

        (D_mu psi)(x) = 1/2 [ s_mu(x) U_mu(x) psi(x + mu) - s_mu(x - mu) U_mu(x - mu)^dag psi(x - mu) ].

    PAPER.md:411 only says "A covariant-derivative kernel was also developed to allow the calculation of one-derivative
    insertions"; this central difference is the reading taken (reading 27).  The antiperiodic sign rides on
    the hop exactly as in the hopping term."""
    U, psi = _c(U), _c(psi)
    ax = _AXIS[mu]
    sh = psi.shape[:4]
    Umu = U[..., mu, :, :]
    fwd = np.einsum("...ab,...sb->...sa", Umu, np.roll(psi, -1, axis=ax))
    fwd = fwd * _boundary_sign(sh, mu, ap, True)[..., None, None]
    Udn = np.roll(Umu, 1, axis=ax)  # U_mu(x - mu)
    bwd = np.einsum("...ba,...sb->...sa", Udn.conj(), np.roll(psi, 1, axis=ax))
    bwd = bwd * _boundary_sign(sh, mu, ap, False)[..., None, None]
    return 0.5 * (fwd - bwd)


def contract_field(a, b):
    """C[t][z][y][x][al][be] = sum_c conj(a_{al c}(x)) b_{be c}(x): colour traced, Dirac and volume indices open
    ("Traces were taken in color space, leaving the Dirac and volume indices open")."""
    return np.einsum("...ac,...bc->...ab", _c(a).conj(), _c(b))


def loop_momentum(a, b, momenta, Gammas):
    """L[n][t][k] = sum_{xvec} exp(-i p_k . xvec) a(x)^dag Gamma_n b(x), p_k = 2 pi (n_x/X, n_y/Y, n_z/Z), n integer.

    The paper Fourier-transforms the contraction field with cuFFT and keeps p^2 <= 9 without stating the
    sign of the exponent; exp(-i p x) (the forward DFT, what an un-normalised FFT computes) is the reading taken (reading 28).
    momenta: integer array [K][3] = (n_x, n_y, n_z); Gammas: [16][4][4].  Plain nested sums."""
    a, b = _c(a), _c(b)
    T, Z, Y, X = a.shape[:4]
    C = contract_field(a, b)
    out = np.zeros((16, T, len(momenta)), dtype=np.complex128)
    x = np.arange(X)[None, None, :]
    y = np.arange(Y)[None, :, None]
    z = np.arange(Z)[:, None, None]
    for k, (nx, ny, nz) in enumerate(momenta):
        ph = np.exp(-2j * np.pi * (nx * x / X + ny * y / Y + nz * z / Z))
        Ct = np.einsum("tzyxab,zyx->tab", C, ph)
        for n in range(16):
            out[n, :, k] = np.einsum("ab,tab->t", Gammas[n], Ct)
    return out


def momenta_p2_max(p2max):
    """All integer 3-vectors with n.n <= p2max, ordered by (n.n, n_x, n_y, n_z) ("p^2 <= 9")."""
    r = int(np.floor(np.sqrt(p2max)))
    lst = [(nx, ny, nz) for nx in range(-r, r + 1) for ny in range(-r, r + 1) for nz in range(-r, r + 1)
           if nx * nx + ny * ny + nz * nz <= p2max]
    lst.sort(key=lambda p: (p[0] ** 2 + p[1] ** 2 + p[2] ** 2, p[0], p[1], p[2]))
    return np.array(lst, dtype=np.int32)


# ---- NEXT-3: time dilution ---------------------------------------------------------------------------------------

def time_dilute(eta, slices):
    """Noise source restricted to the listed time slices (PAPER.md:150 dilution; :154 coherent sources = several
    well-separated slices in one vector): entries on every other slice are set to zero."""
    eta = _c(eta)
    out = np.zeros_like(eta)
    for t in slices:
        out[t] = eta[t]
    return out


def loop_slice(a, b, t0, Gammas):
    """Single-time-slice contraction: L[n] = sum_{x: x4 = t0} a(x)^dag Gamma_n b(x)."""
    C = contract_field(a[t0], b[t0]).sum(axis=(0, 1, 2))
    return np.array([np.einsum("ab,ab->", Gammas[n], C) for n in range(16)])


# ---- NEXT-3: hopping-parameter expansion, Eq. (16)-(17) ---------------------------------------------
# B = (1 + i 2 kappa mu g5)^-1, H = 2 kappa D with D = -1/2 Dslash (reading 2), i.e. H = -kappa Dslash,
# M_u = B^-1 + H.

def hpe_BH(hop_fn, twist_inv_fn, psi, kappa):
    """(B H) psi = B (-kappa Dslash psi).  hop_fn(psi) = Dslash psi, twist_inv_fn(psi) = B psi are passed in so that this
    module holds only the expansion's bookkeeping."""
    return twist_inv_fn(-kappa * hop_fn(psi))


def hpe_remainder(hop_fn, twist_inv_fn, s, kappa):
    """(B H)^4 s: the factor in front of M_u^-1 in the fifth term of Eq. (16); with s = M_u^-1 eta this is the vector whose
    contraction with eta estimates Tr[X (BH)^4 M_u^-1] (Eq. 17)."""
    v = s
    for _ in range(4):
        v = hpe_BH(hop_fn, twist_inv_fn, v, kappa)
    return v


def hpe_series(hop_fn, twist_inv_fn, eta, kappa):
    """The four exact terms of Eq. (16) applied to eta: B eta - B H B eta + (BH)^2 B eta - (BH)^3 B eta."""
    term = twist_inv_fn(eta)
    total = term.copy()
    for k in range(1, 4):
        term = hpe_BH(hop_fn, twist_inv_fn, term, kappa)
        total = total + ((-1) ** k) * term
    return total


def hpe_local_traces(kappa, mu, gammas, Gammas):
    """Per-site value of Tr_{spin,colour}[Gamma_n (B - B H B + (BH)^2 B - (BH)^3 B)]_{xx} for an ultra-local insertion.

    Odd powers of the hopping matrix have no site-diagonal part ("the hopping matrix ... is traceless, so only the
    even powers (third term) will survive").  The second-order return paths x -> x +- mu -> x multiply U U^dag = 1 and a squared
    boundary sign, so the term is gauge independent ("do not depend on the gauge configuration for local operators"):
        [(BH)^2 B]_{xx} = kappa^2 sum_mu [ B (1 - g_mu) B (1 + g_mu) B + B (1 + g_mu) B (1 - g_mu) B ]  (x) 1_colour.
    Returns complex [16]: 3 * tr_spin[Gamma_n (B + that)].  gammas: [4][4][4] g_mu and g5 as gammas[4]."""
    a = 2 * kappa * mu
    one = np.eye(4, dtype=np.complex128)
    B = np.linalg.inv(one + 1j * a * gammas[4])
    second = np.zeros((4, 4), dtype=np.complex128)
    for m in range(4):
        second += B @ (one - gammas[m]) @ B @ (one + gammas[m]) @ B
        second += B @ (one + gammas[m]) @ B @ (one - gammas[m]) @ B
    S = B + kappa * kappa * second
    return np.array([3.0 * np.trace(Gammas[n] @ S) for n in range(16)])
