"""-m gpu: tm_gauge_synthetic (on-device gauge generator) against the host generator of tm_inputs.

The two share the counter-based hashes bit for bit and differ in the last bits of log / cos / sin and in FMA contraction, so
the comparison is to rounding: every real within 1e-13, unitarity and det = 1 within 5e-14 (the tolerances tm.h states)."""
import numpy as np
import pytest
import torch

import tm_inputs as ti
import paper_1309_2256_b200 as tm
from tm_harness import to_dev

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("dims,seed,eps,w", [((4, 4, 4, 8), ti.GAUGE_SEED, ti.EPS, 1.0), ((6, 4, 8, 10), 77, 0.9, 0.3), ((16, 16, 16, 32), ti.GAUGE_SEED, ti.EPS, 1.0)])
def test_device_links_equal_host_links_to_rounding(dims, seed, eps, w):
    L = tm.tm_lattice_create(dims, True)
    U = torch.empty(L.V * 4 * 18, dtype=torch.float64, device="cuda")
    tm.tm_gauge_synthetic(L, seed, w, eps, U)
    got = U.cpu().numpy().view(np.complex128).reshape(-1, 3, 3)
    ref = ti.gauge(dims, seed=seed, eps=eps, w=w).reshape(-1, 3, 3)
    assert np.abs(got - ref).max() < 1e-13
    eye = np.eye(3)
    assert np.abs(got @ np.conj(np.swapaxes(got, -1, -2)) - eye).max() < 5e-14
    assert np.abs(np.linalg.det(got) - 1.0).max() < 5e-14
    # the generator's sanity statistic: <Re tr U>/3 = 0.563 at eps = 0.5, w = 1
    if eps == 0.5 and w == 1.0:
        assert abs(np.real(np.trace(got, axis1=1, axis2=2)).mean() / 3 - 0.563) < 0.01


def test_device_field_packs_and_drives_the_operator():
    """The generated field goes through tm_gauge_pack (SU(3) check at 1e-10, 12-real storage) and gives the hopping term of the host field."""
    import oracle
    from tm_harness import Fields, TOL, rel
    dims = (8, 8, 8, 16)
    Uh = ti.gauge(dims)
    F = Fields(dims, Uh, True)
    tm.tm_gauge_synthetic(F.L, ti.GAUGE_SEED, 1.0, ti.EPS, F.U_dev)  # replaces the uploaded host field
    psi = ti.gauss_spinor(dims, 5)
    pin = F.pack(psi, 8)
    out = F.zeros_full(8)
    tm.tm_dslash(F.L, F.gauge(8, 12), 8, 12, F.half(out, 8, 0), F.half(pin, 8, 1), None, 0, 0, tm.TM_KIND_PLAIN, ti.KAPPA, ti.MU)
    ref = oracle.project(oracle.hop(Uh, oracle.project(psi, 1), ap=True), 0)
    assert rel(F.unpack(out, 8), ref) < TOL[8]
