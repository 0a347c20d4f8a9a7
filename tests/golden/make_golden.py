"""Writes tests/golden/config0_4x4.json from the fp64 CPU oracle ONLY (never from the CUDA path).

BASELINE.json configs[0]: 4^4 lattice, antiperiodic in time, links = Gram-Schmidt SU(3) projection of (1 + 0.5 x complex
Gaussian) from gauge seed 1309, one Z2xiZ2 noise spinor from noise seed 2256, kappa = 0.161236, a mu = 0.0055: one dslash, CG to
1e-12, loops for the 16 Gamma_n per time slice.  The paper prints no worked numerical example, so nothing
here is "the paper's value": the file freezes the pinned oracle's output for this configuration, (a) as a regression guard on the
oracle itself (tests/test_golden.py, CPU) and (b) as an oracle-free expected value for the GPU run of configs[0].

    python tests/golden/make_golden.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle  # noqa: E402
import tm_inputs as ti  # noqa: E402


def cplx(a):
    a = np.asarray(a, dtype=np.complex128)
    return [[float(z.real), float(z.imag)] for z in a.ravel()]


def main():
    dims = (4, 4, 4, 4)
    U = ti.gauge(dims, seed=1309)
    eta = ti.z4(dims, seed=2256)
    kappa, mu = ti.KAPPA, ti.MU
    hop_e = oracle.project(oracle.hop(U, oracle.project(eta, 1)), 0)
    mdagm = oracle.MdagM(U, oracle.project(eta, 0), kappa, mu, parity=0)
    s, info = oracle.cg_solve(U, eta, kappa, mu, 1e-12, 5000)
    loops = oracle.loop(eta, s)
    sample = [(0, 0, 0, 0), (1, 2, 3, 0), (3, 3, 3, 3), (2, 0, 1, 3)]  # (x, y, z, t)
    out = {
        "citation": "BASELINE.json configs[0]; operator PAPER.md:162 Eq. (16) / :367 Eq. (A1), loop PAPER.md:116 Eq. (10); "
                    "written by tests/golden/make_golden.py from oracle/ only",
        "dims": dims, "gauge_seed": 1309, "noise_seed": 2256, "kappa": kappa, "mu": mu,
        "plaquette_like_stat_mean_re_tr_U_over_3": float(np.mean(np.einsum("...ii->...", U).real) / 3),
        "norm2_dslash_even": float(np.vdot(hop_e, hop_e).real),
        "norm2_MdagM_even": float(np.vdot(mdagm, mdagm).real),
        "cg_iters": int(info["iters"]),
        "norm2_solution": float(np.vdot(s, s).real),
        "sample_sites_xyzt": sample,
        "dslash_even_at_samples": [cplx(hop_e[t, z, y, x]) for (x, y, z, t) in sample],
        "solution_at_samples": [cplx(s[t, z, y, x]) for (x, y, z, t) in sample],
        "loops_16x4": cplx(loops),
    }
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_4x4.json")
    with open(path, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", path)


if __name__ == "__main__":
    main()
