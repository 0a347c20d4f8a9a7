"""Temporal gauge -- fp64 numpy checker of the product call tm_gauge_fix_temporal.  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Not in the paper (reading 33): the loops eta^dag Gamma s of PAPER.md:116 Eq. (10) are gauge invariant and Z2 x iZ2 noise
 is noise in any gauge, so a configuration may be gauge-fixed before its solves.  The definition is written out
as it stands: g(x, t) = prod_{t' < t} U_t(x, t') (time-ordered product from slice 0), U'_mu(x) = g(x) U_mu(x) g(x + mu)^dagger
with periodic wrap (the antiperiodic sign belongs to the fermions, not to the links).

Pinned by P25 (tests/test_oracle_pins2.py): M(U') g = g M(U) with the pinned oracle operator, the Polyakov-loop trace is
preserved, CG iteration counts and loops are equal -- a wrong order of the product, a transposed g or a wrong shift fails it.
"""
import numpy as np


def temporal_gauge(U):
    """U[T][Z][Y][X][4][3][3] complex128 -> (U', g): unit temporal links on every slice but the last (set to exactly 1; they
    are 1 up to rounding), slice T - 1 carries the Polyakov loop; g[T][Z][Y][X][3][3] is the transformation."""
    T = U.shape[0]
    eye = np.eye(3, dtype=np.complex128)
    g = np.empty(U.shape[:4] + (3, 3), dtype=np.complex128)
    g[0] = eye
    for t in range(T - 1):
        g[t + 1] = g[t] @ U[t, ..., 3, :, :]
    Up = np.empty_like(U)
    for mu in range(4):
        gs = np.roll(g, -1, axis=3 - mu)  # g(x + mu); array axes are (t, z, y, x)
        Up[..., mu, :, :] = g @ U[..., mu, :, :] @ np.conj(np.swapaxes(gs, -1, -2))
    Up[:T - 1, ..., 3, :, :] = eye
    return Up, g
