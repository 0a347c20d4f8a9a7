"""fp64 CPU oracle -- TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It shares no code with paper_1309_2256_b200 (the CUDA path) and neither imports the other.

`tm_oracle.cpp` holds the plain stencil definitions (ctypes-loaded below); `dense.py` holds an independent
numpy matrix-element construction of the same operator used to pin the stencil on 4^4.

Fields are numpy complex128 arrays in the canonical layout of tm_inputs:
    U[T][Z][Y][X][4][3][3], psi[T][Z][Y][X][4][3].
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tm_oracle.cpp")
_LIB = os.path.join(_HERE, "libtm_oracle.so")
_lib = None


def build(force=False):
    """g++ -O2 (no intrinsics, no fast-math beyond limited-range complex multiply) -> libtm_oracle.so."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["g++", "-O2", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC", "-o", tmp, _SRC])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        vp, i, d = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        lib.orc_gamma.argtypes = [i, vp]
        lib.orc_Gamma.argtypes = [i, vp]
        lib.orc_hop.argtypes = [vp, i, vp, vp, vp, i]
        lib.orc_hop_gathered.argtypes = [vp, vp, vp, vp, vp, vp, i, vp]
        lib.orc_twist.argtypes = [vp, d, i, vp, vp]
        lib.orc_M.argtypes = [vp, i, vp, d, d, i, vp, vp]
        lib.orc_Mpc.argtypes = [vp, i, vp, d, d, i, i, vp, vp]
        lib.orc_MdagM.argtypes = [vp, i, vp, d, d, i, vp, vp]
        lib.orc_cg_solve.argtypes = [vp, i, vp, d, d, vp, d, i, vp, vp, vp]
        lib.orc_loop.argtypes = [vp, vp, vp, vp]
        for f in ("orc_gamma", "orc_Gamma", "orc_hop", "orc_hop_gathered", "orc_twist", "orc_M", "orc_Mpc",
                  "orc_MdagM", "orc_cg_solve", "orc_loop"):
            getattr(lib, f).restype = None
        _lib = lib
    return _lib


def _dims(psi):
    T, Z, Y, X = psi.shape[:4]
    return (ctypes.c_int * 4)(X, Y, Z, T)


def _c(a):
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a


def gamma(mu):
    """gamma_mu, mu = 0..3 (x,y,z,t); mu = 4 -> gamma5 = g1 g2 g3 g4."""
    out = np.empty((4, 4), dtype=np.complex128)
    _load().orc_gamma(mu, out.ctypes.data)
    return out


def Gamma(n):
    """Gamma_n = g1^b0 g2^b1 g3^b2 g4^b3, n = b0 + 2 b1 + 4 b2 + 8 b3."""
    out = np.empty((4, 4), dtype=np.complex128)
    _load().orc_Gamma(n, out.ctypes.data)
    return out


def hop(U, psi, ap=True, dagger=False):
    """Full-lattice positive hopping sum Dslash psi (or Dslash^dag psi)."""
    U, psi = _c(U), _c(psi)
    out = np.empty_like(psi)
    _load().orc_hop(_dims(psi), int(ap), U.ctypes.data, psi.ctypes.data, out.ctypes.data, int(dagger))
    return out


def hop_gathered(Ufwd, Ubwd, nf, nb, sf, sb, dagger=False):
    """Single-site Dslash from gathered links/neighbours: Ufwd[4][3][3], Ubwd[4][3][3], nf[4][4][3], nb[4][4][3]."""
    Ufwd, Ubwd, nf, nb = _c(Ufwd), _c(Ubwd), _c(nf), _c(nb)
    sf = np.ascontiguousarray(sf, dtype=np.float64)
    sb = np.ascontiguousarray(sb, dtype=np.float64)
    out = np.empty((4, 3), dtype=np.complex128)
    _load().orc_hop_gathered(Ufwd.ctypes.data, Ubwd.ctypes.data, nf.ctypes.data, nb.ctypes.data, sf.ctypes.data,
                             sb.ctypes.data, int(dagger), out.ctypes.data)
    return out


def twist(psi, a, inverse=False):
    """R(a) psi = (1 + i a g5) psi, or R(a)^-1 psi."""
    psi = _c(psi)
    out = np.empty_like(psi)
    _load().orc_twist(_dims(psi), float(a), int(inverse), psi.ctypes.data, out.ctypes.data)
    return out


def project(psi, parity):
    """Keep sites of the given parity ((x+y+z+t)&1), zero the rest."""
    T, Z, Y, X = psi.shape[:4]
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    m = ((x + y + z + t) & 1) == parity
    return psi * m[..., None, None]


def M(U, psi, kappa, mu, ap=True, dagger=False):
    """Full twisted-mass operator M(kappa, mu) psi = psi + i 2 kappa mu g5 psi - kappa Dslash psi."""
    U, psi = _c(U), _c(psi)
    out = np.empty_like(psi)
    _load().orc_M(_dims(psi), int(ap), U.ctypes.data, kappa, mu, int(dagger), psi.ctypes.data, out.ctypes.data)
    return out


def Mpc(U, psi, kappa, mu, parity=0, ap=True, dagger=False):
    """Asymmetric even-odd preconditioned operator on `parity` (Eq. A2 lhs); full-lattice arrays in and out."""
    U, psi = _c(U), _c(psi)
    out = np.empty_like(psi)
    _load().orc_Mpc(_dims(psi), int(ap), U.ctypes.data, kappa, mu, int(parity), int(dagger), psi.ctypes.data,
                    out.ctypes.data)
    return out


def MdagM(U, psi, kappa, mu, parity=0, ap=True):
    U, psi = _c(U), _c(psi)
    out = np.empty_like(psi)
    _load().orc_MdagM(_dims(psi), int(ap), U.ctypes.data, kappa, mu, int(parity), psi.ctypes.data, out.ctypes.data)
    return out


def cg_solve(U, eta, kappa, mu, tol, max_iter, ap=True, history=False):
    """Solve M s = eta through the even-even Schur system with textbook CG on M_pc^dag M_pc, x0 = 0.

    Returns (s, info) with info = dict(iters, iterated_resid, true_resid_normal, true_resid_full[, history])."""
    U, eta = _c(U), _c(eta)
    s = np.empty_like(eta)
    info = np.zeros(4)
    hist = np.zeros(max_iter + 1) if history else None
    _load().orc_cg_solve(_dims(eta), int(ap), U.ctypes.data, kappa, mu, eta.ctypes.data, tol, int(max_iter),
                         s.ctypes.data, info.ctypes.data, hist.ctypes.data if history else None)
    d = dict(iters=int(info[0]), iterated_resid=info[1], true_resid_normal=info[2], true_resid_full=info[3])
    if history:
        d["history"] = hist[: d["iters"] + 1]
    return s, d


def loop(a, b):
    """L[n][t] = sum_{x: x4=t} a(x)^dag (Gamma_n (x) 1) b(x); returns complex128 [16][T]."""
    a, b = _c(a), _c(b)
    T = a.shape[0]
    out = np.empty((16, T), dtype=np.complex128)
    _load().orc_loop(_dims(a), a.ctypes.data, b.ctypes.data, out.ctypes.data)
    return out


# ---- NEXT-1: estimators, written out in the paper's order -------------------------------------

def gamma5(psi):
    """g5 psi with g5 = gamma(4) = g1 g2 g3 g4 as a full 4x4 matrix acting on the spin index."""
    return np.einsum("ab,...bc->...ac", gamma(4), _c(psi))


def loop_oneend_tau3(s, kappa, mu):
    """PAPER.md:127 Eq. (13), kappa-normalised (2 mu a -> 2 (2 kappa mu)): 2 i (2 kappa mu) sum_x s^dag g5 Gamma_n s, [16][T]."""
    return 2j * (2 * kappa * mu) * loop(gamma5(s), s)


def loop_oneend_general(U, s, kappa, ap=True):
    """PAPER.md:141 Eq. (15): 2 sum_x s^dag g5 Gamma_n g5 D_W s with D_W = (M_u + M_d)/2 = M(kappa, 0) (Eq. 14)."""
    DWs = M(U, s, kappa, 0.0, ap=ap)
    return 2.0 * loop(gamma5(s), gamma5(DWs))


def tsm_combine(L_hp, L_lp_same, L_lp):
    """PAPER.md:75-77 Eq. (8) applied to loops: 1/N_HP sum_r [L_HP(r) - L_LP(r)] + 1/N_LP sum_j L_LP(j).
    L_hp, L_lp_same: [N_HP][16][T] of the same sources; L_lp: [N_LP][16][T]."""
    out = 0
    if len(L_hp):
        c = 0
        for r in range(len(L_hp)):
            c = c + (L_hp[r] - L_lp_same[r])
        out = out + c / len(L_hp)
    if len(L_lp):
        l = 0
        for j in range(len(L_lp)):
            l = l + L_lp[j]
        out = out + l / len(L_lp)
    return out


# ---- NEXT-2 / NEXT-3: plain numpy definitions in oracle/insertions.py ---------------------------
from . import insertions as _ins  # noqa: E402
from .gaugefix import temporal_gauge  # noqa: E402,F401

covdev = _ins.covdev
contract_field = _ins.contract_field
momenta_p2_max = _ins.momenta_p2_max
time_dilute = _ins.time_dilute


def _Gammas():
    return np.array([Gamma(n) for n in range(16)])


def loop_momentum(a, b, momenta):
    """L[n][t][k] = sum_xvec exp(-i p_k xvec) a^dag Gamma_n b; momenta int [K][3]."""
    return _ins.loop_momentum(a, b, momenta, _Gammas())


def loop_derivative(U, a, b, mu, ap=True):
    """One-derivative insertion: L[n][t] = sum_x a(x)^dag Gamma_n (D_mu b)(x)."""
    return loop(a, covdev(U, b, mu, ap=ap))


def loop_slice(a, b, t0):
    """Single-time-slice contraction, complex [16]."""
    return _ins.loop_slice(_c(a), _c(b), t0, _Gammas())


def hpe_remainder(U, s, kappa, mu, ap=True):
    """(B H)^4 s of PAPER.md:160 Eq. (16)/(17): B = R(2 kappa mu)^-1, H = -kappa Dslash."""
    a = 2 * kappa * mu
    return _ins.hpe_remainder(lambda v: hop(U, v, ap=ap), lambda v: twist(v, a, inverse=True), _c(s), kappa)


def hpe_series(U, eta, kappa, mu, ap=True):
    """B eta - B H B eta + (BH)^2 B eta - (BH)^3 B eta (first four terms of Eq. 16)."""
    a = 2 * kappa * mu
    return _ins.hpe_series(lambda v: hop(U, v, ap=ap), lambda v: twist(v, a, inverse=True), _c(eta), kappa)


def hpe_local_traces(kappa, mu):
    """Per-site Tr[Gamma_n (B - BHB + (BH)^2 B - (BH)^3 B)]_xx, complex [16] (gauge independent)."""
    return _ins.hpe_local_traces(kappa, mu, np.array([gamma(m) for m in range(5)]), _Gammas())


def Mpc_sym(U, psi, kappa, mu, parity=0, ap=True, dagger=False):
    """Symmetric even-odd preconditioned operator, PAPER.md:376 Eq. (A3) lhs: M_sym = 1 - kappa^2 R^-1 Dslash R^-1 Dslash on
    `parity` (full-lattice arrays, zero elsewhere); dagger: 1 - kappa^2 Dslash^dag R^-dag Dslash^dag R^-dag."""
    a = 2 * kappa * mu
    v = project(_c(psi), parity)
    if not dagger:
        w = twist(project(hop(U, v, ap=ap), 1 - parity), a, inverse=True)
        w = twist(project(hop(U, w, ap=ap), parity), a, inverse=True)
    else:
        w = project(hop(U, twist(v, -a, inverse=True), ap=ap, dagger=True), 1 - parity)
        w = project(hop(U, twist(w, -a, inverse=True), ap=ap, dagger=True), parity)
    return v - kappa ** 2 * w
