"""Dense matrix-element construction of the twisted-mass operator on tiny lattices (numpy).

TEST INFRASTRUCTURE ONLY.  A second, independent statement of the operator (a loop nest over matrix
elements rather than a stencil applied to a vector, with its own gamma table typed entry by entry), used to
pin oracle/tm_oracle.cpp by brute force on 4^4 (north_star "a dense-matrix brute force on a 4^4 lattice";
SURVEY.md P5, P14).  Row/column index = ((site*4 + spin)*3 + colour), site = x + X*(y + Y*(z + Z*t)).

  M[(x,al,c),(y,be,d)] = delta_xy [delta + i 2 kappa mu (g5)_{al be}] delta_cd
        - kappa sum_mu [ (1-g_mu)_{al be} s_mu(x) U_mu(x)_{cd} delta_{y,x+mu}
                       + (1+g_mu)_{al be} s_mu(y) conj(U_mu(y)_{dc}) delta_{y,x-mu} ]
"""
import numpy as np

_i = 1j
# explicit entries, chiral basis (reading 3)
GAMMA = np.array([
    [[0, 0, 0, -_i], [0, 0, -_i, 0], [0, _i, 0, 0], [_i, 0, 0, 0]],
    [[0, 0, 0, -1], [0, 0, 1, 0], [0, 1, 0, 0], [-1, 0, 0, 0]],
    [[0, 0, -_i, 0], [0, 0, 0, _i], [_i, 0, 0, 0], [0, -_i, 0, 0]],
    [[0, 0, 1, 0], [0, 0, 0, 1], [1, 0, 0, 0], [0, 1, 0, 0]],
], dtype=np.complex128)
GAMMA5 = np.diag([1.0, 1.0, -1.0, -1.0]).astype(np.complex128)


def Gamma_n(n):
    g = np.eye(4, dtype=np.complex128)
    for k in range(4):
        if (n >> k) & 1:
            g = g @ GAMMA[k]
    return g


def dense_M(U, kappa, mu, ap=True):
    """U[T][Z][Y][X][4][3][3] -> dense (12V x 12V) complex matrix of M(kappa, mu)."""
    T, Z, Y, X = U.shape[:4]
    dims = (X, Y, Z, T)
    V = X * Y * Z * T
    Uf = U.reshape(V, 4, 3, 3)
    Mat = np.zeros((V, 12, V, 12), dtype=np.complex128)
    one = np.eye(4)
    diag = np.kron(one + 1j * 2 * kappa * mu * GAMMA5, np.eye(3))
    for t in range(T):
        for z in range(Z):
            for y in range(Y):
                for x in range(X):
                    c = [x, y, z, t]
                    i = x + X * (y + Y * (z + Z * t))
                    Mat[i, :, i, :] += diag
                    for m in range(4):
                        cf = list(c)
                        cf[m] = (c[m] + 1) % dims[m]
                        j = cf[0] + X * (cf[1] + Y * (cf[2] + Z * cf[3]))
                        s = -1.0 if (ap and m == 3 and c[3] == T - 1) else 1.0
                        # forward element (row i, column j) and its backward partner (row j, column i)
                        Mat[i, :, j, :] += -kappa * s * np.kron(one - GAMMA[m], Uf[i, m])
                        Mat[j, :, i, :] += -kappa * s * np.kron(one + GAMMA[m], Uf[i, m].conj().T)
    return Mat.reshape(12 * V, 12 * V)


def timeslice_traces(Minv, dims):
    """Tr_t[Gamma_n M^-1] = sum_{x: x4=t} sum_{al be c} (Gamma_n)_{al be} Minv[(x,be,c),(x,al,c)] -> [16][T]."""
    X, Y, Z, T = dims
    V = X * Y * Z * T
    V3 = X * Y * Z
    blocks = Minv.reshape(V, 4, 3, V, 4, 3)
    out = np.zeros((16, T), dtype=np.complex128)
    for i in range(V):
        t = i // V3
        B = np.einsum("bcac->ba", blocks[i, :, :, i, :, :])  # B[be][al] = sum_c Minv[(x,be,c),(x,al,c)]
        for n in range(16):
            out[n, t] += np.sum(Gamma_n(n) * B.T)
    return out
