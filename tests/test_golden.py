"""tests/golden/config0_4x4.json (BASELINE.json configs[0]): the oracle reproduces it (CPU regression guard); the CUDA path
reproduces it at fp64 without the oracle in the loop (-m gpu)."""
import json
import os

import numpy as np
import pytest

import tm_inputs as ti

HERE = os.path.dirname(os.path.abspath(__file__))
G = json.load(open(os.path.join(HERE, "golden", "config0_4x4.json")))
DIMS = tuple(G["dims"])


def c(lst):
    a = np.array(lst, dtype=np.float64)
    return a[..., 0] + 1j * a[..., 1]


def test_golden_is_what_the_oracle_computes():
    import oracle
    U = ti.gauge(DIMS, seed=G["gauge_seed"])
    eta = ti.z4(DIMS, seed=G["noise_seed"])
    hop_e = oracle.project(oracle.hop(U, oracle.project(eta, 1)), 0)
    assert abs(np.vdot(hop_e, hop_e).real / G["norm2_dslash_even"] - 1) < 1e-13
    s, info = oracle.cg_solve(U, eta, G["kappa"], G["mu"], 1e-12, 5000)
    assert info["iters"] == G["cg_iters"]
    loops = oracle.loop(eta, s)
    assert np.allclose(loops.ravel(), c(G["loops_16x4"]), rtol=0, atol=1e-9 * np.abs(loops).max())
    for k, (x, y, z, t) in enumerate(G["sample_sites_xyzt"]):
        assert np.allclose(hop_e[t, z, y, x].ravel(), c(G["dslash_even_at_samples"][k]), atol=1e-12)
        assert np.allclose(s[t, z, y, x].ravel(), c(G["solution_at_samples"][k]), atol=1e-9)
    # the gauge generator's sanity statistic at eps = 0.5 (about 0.563 in the infinite-volume mean)
    assert abs(G["plaquette_like_stat_mean_re_tr_U_over_3"] - 0.563) < 0.02


@pytest.mark.gpu
def test_config0_on_the_gpu_against_the_golden_file():
    import torch
    import paper_1309_2256_b200 as tm
    from tm_harness import Fields
    U = ti.gauge(DIMS, seed=G["gauge_seed"])
    eta = ti.z4(DIMS, seed=G["noise_seed"])
    F = Fields(DIMS, U, True)
    kappa, mu = G["kappa"], G["mu"]
    for recon in (18, 12, 8):
        g = F.gauge(8, recon)
        pe = F.pack(eta, 8)
        out = F.zeros_full(8)
        tm.tm_dslash(F.L, g, 8, recon, F.half(out, 8, 0), F.half(pe, 8, 1), None, 0, 0, tm.TM_KIND_PLAIN, kappa, mu)
        d = F.unpack(out, 8)
        assert abs(np.vdot(d, d).real / G["norm2_dslash_even"] - 1) < 1e-12
        for k, (x, y, z, t) in enumerate(G["sample_sites_xyzt"]):
            assert np.allclose(d[t, z, y, x].ravel(), c(G["dslash_even_at_samples"][k]), atol=1e-11)
        tmp = tm.device_buffer(2 * F.pb(8))
        tm.tm_MdagM(F.L, g, 8, recon, F.half(out, 8, 0), F.half(pe, 8, 0), tmp, 0, kappa, mu)
        m = F.unpack(out, 8)
        m[(np.indices(m.shape[:4]).sum(axis=0) & 1) == 1] = 0  # odd block of `out` still holds nothing meaningful
        assert abs(np.vdot(m, m).real / G["norm2_MdagM_even"] - 1) < 1e-12
        s = F.zeros_full(8)
        ws = tm.device_buffer(tm.tm_cg_workspace_bytes(F.L, 8, 8, tm.TM_CG_LP_TRUNCATED, 1))
        prm = tm.make_cg_params(kappa, mu, 1e-12, 5000, tm.TM_CG_LP_TRUNCATED)
        rc, info = tm.tm_cg(F.L, g, 8, g, 8, recon, s, pe, prm, ws)
        assert rc == tm.TM_OK and abs(info.iters - G["cg_iters"]) <= 1
        sol = F.unpack(s, 8)
        assert abs(np.vdot(sol, sol).real / G["norm2_solution"] - 1) < 1e-9
        loops = torch.zeros((1, 16, DIMS[3], 2), dtype=torch.float64, device="cuda")
        lws = tm.device_buffer(tm.tm_loop_workspace_bytes(F.L, 1))
        tm.tm_loop_contract(F.L, pe, s, 8, 1, loops, lws)
        got = loops.cpu().numpy().view(np.complex128)[0, ..., 0]
        ref = c(G["loops_16x4"]).reshape(16, DIMS[3])
        assert np.abs(got - ref).max() < 1e-8 * np.abs(ref).max()
