"""Seeded synthetic input generators (DATA ONLY -- none of the method's arithmetic lives here).

Serves both the oracle-side tests and the CUDA-side tests / bench.  Imports neither.
Recipe: BASELINE.json configs[0]; stated in DESIGN.md.

Canonical host layout (fp64, C order):
    gauge   U[T][Z][Y][X][mu][row][col] complex128   (site = x + X*(y + Y*(z + Z*t)), mu = 0..3 = x,y,z,t)
    spinor  psi[T][Z][Y][X][spin][colour] complex128
"""
import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gen.c")
_LIB = os.path.join(_HERE, "libtm_inputs.so")
_lib = None

GAUGE_SEED = 1309
NOISE_SEED = 2256
EPS = 0.5
KAPPA = 0.161236
MU = 0.0055


def build(force=False):
    """Compile gen.c with gcc (OpenMP) into libtm_inputs.so next to this file."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        u64, i64, dbl, vp = ctypes.c_uint64, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        lib.tmi_gauge_range.argtypes = [u64, dbl, dbl, i64, i64, vp]
        lib.tmi_gauge_sites.argtypes = [u64, dbl, dbl, i64, vp, vp]
        lib.tmi_su3_range.argtypes = [u64, dbl, dbl, i64, i64, vp]
        lib.tmi_z4_codes_range.argtypes = [u64, i64, i64, vp]
        lib.tmi_z4_range.argtypes = [u64, i64, i64, vp]
        lib.tmi_z4_sites.argtypes = [u64, i64, vp, vp]
        lib.tmi_gauss_range.argtypes = [u64, i64, i64, vp]
        for f in ("tmi_gauge_range", "tmi_gauge_sites", "tmi_su3_range", "tmi_z4_codes_range", "tmi_z4_range",
                  "tmi_z4_sites", "tmi_gauss_range"):
            getattr(lib, f).restype = None
        _lib = lib
    return _lib


def volume(dims):
    X, Y, Z, T = dims
    return X * Y * Z * T


def _slab(dims, t0, t1):
    X, Y, Z, T = dims
    t0 = 0 if t0 is None else t0
    t1 = T if t1 is None else t1
    v3 = X * Y * Z
    return t0, t1, t0 * v3, t1 * v3


def gauge(dims, seed=GAUGE_SEED, eps=EPS, w=1.0, t0=None, t1=None):
    """SU(3) links = Gram-Schmidt projection of (w*1 + eps*complex Gaussian); time slab [t0, t1)."""
    X, Y, Z, T = dims
    t0, t1, s0, s1 = _slab(dims, t0, t1)
    out = np.empty((t1 - t0, Z, Y, X, 4, 3, 3), dtype=np.complex128)
    _load().tmi_gauge_range(seed, w, eps, s0, s1, out.ctypes.data)
    return out


def unit_gauge(dims):
    X, Y, Z, T = dims
    out = np.zeros((T, Z, Y, X, 4, 3, 3), dtype=np.complex128)
    out[..., 0, 0] = out[..., 1, 1] = out[..., 2, 2] = 1.0
    return out


def gauge_sites(sites, seed=GAUGE_SEED, eps=EPS, w=1.0):
    """Links U[k][mu][3][3] of the listed global site indices (same values as gauge())."""
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((sites.size, 4, 3, 3), dtype=np.complex128)
    _load().tmi_gauge_sites(seed, w, eps, sites.size, sites.ctypes.data, out.ctypes.data)
    return out


def su3_field(dims, seed):
    """One random SU(3) matrix per site (a gauge transformation g(x)): Gram-Schmidt of a pure Gaussian matrix."""
    X, Y, Z, T = dims
    out = np.empty((T, Z, Y, X, 3, 3), dtype=np.complex128)
    _load().tmi_su3_range(seed, 0.0, 1.0, 0, volume(dims), out.ctypes.data)
    return out


def z4(dims, seed=NOISE_SEED, t0=None, t1=None):
    """Z2 (x) iZ2 noise spinor, (+-1 +- i)/sqrt(2) per (site, spin, colour)."""
    X, Y, Z, T = dims
    t0, t1, s0, s1 = _slab(dims, t0, t1)
    out = np.empty((t1 - t0, Z, Y, X, 4, 3), dtype=np.complex128)
    _load().tmi_z4_range(seed, s0, s1, out.ctypes.data)
    return out


def z4_codes(dims, seed=NOISE_SEED, t0=None, t1=None):
    """The same noise as z4() as 2-bit codes in bytes: bit0 = re negative, bit1 = im negative."""
    X, Y, Z, T = dims
    t0, t1, s0, s1 = _slab(dims, t0, t1)
    out = np.empty((t1 - t0, Z, Y, X, 4, 3), dtype=np.uint8)
    _load().tmi_z4_codes_range(seed, s0, s1, out.ctypes.data)
    return out


def z4_bits(dims, seed=NOISE_SEED, t0=None, t1=None):
    """z4_codes() bit-packed: 3 bytes per site, component k = spin*3 + colour in bits 2k (re < 0), 2k+1 (im < 0), little endian.
    Packaging only (the 4x smaller host->device format of tm_spinor_pack_z4_bits)."""
    c = z4_codes(dims, seed=seed, t0=t0, t1=t1).astype(np.uint32)
    flat = c.reshape(-1, 12)
    w = np.zeros(flat.shape[0], dtype=np.uint32)
    for k in range(12):
        w |= (flat[:, k] & 3) << (2 * k)
    out = np.empty((flat.shape[0], 3), dtype=np.uint8)
    out[:, 0] = w & 0xFF
    out[:, 1] = (w >> 8) & 0xFF
    out[:, 2] = (w >> 16) & 0xFF
    return out.reshape(c.shape[:-2] + (3,))


def z4_sites(sites, seed=NOISE_SEED):
    sites = np.ascontiguousarray(sites, dtype=np.int64)
    out = np.empty((sites.size, 4, 3), dtype=np.complex128)
    _load().tmi_z4_sites(seed, sites.size, sites.ctypes.data, out.ctypes.data)
    return out


def gauss_spinor(dims, seed):
    """Complex Gaussian spinor (unit variance per real component)."""
    X, Y, Z, T = dims
    out = np.empty((T, Z, Y, X, 4, 3), dtype=np.complex128)
    _load().tmi_gauss_range(seed, 0, volume(dims), out.ctypes.data)
    return out


def site_index(dims, x, y, z, t):
    X, Y, Z, T = dims
    return x + X * (y + Y * (z + Z * t))


def parity_mask(dims):
    """mask[T][Z][Y][X] = (x+y+z+t) & 1."""
    X, Y, Z, T = dims
    t, z, y, x = np.meshgrid(np.arange(T), np.arange(Z), np.arange(Y), np.arange(X), indexing="ij")
    return ((x + y + z + t) & 1).astype(np.int8)
