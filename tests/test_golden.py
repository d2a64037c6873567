"""tests/golden/cfg0_oracle.txt: the oracle reproduces its stored configs[0] outputs (CPU), and the CUDA path matches the
stored values (GPU).  The file is written by tests/golden/make_golden.py, which calls only oracle/."""
import os

import numpy as np
import pytest

GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg0_oracle.txt")


def load_golden():
    out = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, v = line.split()
        out[k] = float.fromhex(v)
    return out


def test_oracle_reproduces_golden_cfg0():
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(os.path.dirname(GOLD), "make_golden.py"))
    mg = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mg)
    got, want = mg.compute(), load_golden()
    assert set(got) == set(want)
    for k in want:
        # libm / compiler differences between boxes stay at rounding level; anything larger is a changed oracle
        assert abs(got[k] - want[k]) <= 1e-12 * max(1.0, abs(want[k])), k


@pytest.mark.gpu
def test_cuda_path_matches_golden_cfg0(cuda_device):
    import torch
    import paper_1910_13908_b200 as sg
    from sagecal_inputs import make_config
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host

    want = load_golden()
    p = make_config(0)
    coh = gpu_predict(p)
    vis = gpu_simulate(p, coh)
    c = host(coh)
    assert abs(np.vdot(c, c).real - want["coh_norm2"]) <= 1e-10 * want["coh_norm2"]
    v = host(vis)
    assert abs(np.vdot(v, v).real - want["vis_norm2"]) <= 1e-10 * want["vis_norm2"]
    cost, G, M = sg.lm_cost_grad_jtj(p.N, p.T, p.F, vis, coh[0], dev(p.jones_init()[0]))
    assert abs(float(cost) - want["phi_identity"]) <= 1e-10 * want["phi_identity"]
    g = host(G)
    assert abs(np.vdot(g, g).real - want["G_norm2_identity"]) <= 1e-10 * want["G_norm2_identity"]
    out = sg.sage_calibrate(p.N, p.T, p.F, vis, coh, dev(p.jones_init()), p.n_em, p.n_lm, p.tau, trace=True)
    torch.cuda.synchronize()
    assert abs(float(out["cost_per_cluster"][0]) - want["cost_cluster0"]) <= 1e-8 * want["cost_cluster0"]
    tr = host(out["cost_trace"])
    for i in range(tr.size):
        assert abs(tr[i] - want[f"cost_trace_{i}"]) <= 1e-8 * want[f"cost_trace_{i}"], i


GOLD4 = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg4_oracle.txt")


def _load(path):
    out = {}
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            out[k] = float.fromhex(v)
    return out


def test_cfg4_fixture_is_a_parity_seed():
    """The stored full-size oracle run (tests/golden/make_golden_full.py cfg4, oracle only) took no accept/reject decision
    within rounding of zero, and its cost trace falls monotonically (P11)."""
    g = _load(GOLD4)
    assert g["min_abs_rho"] > 1e-6
    tr = np.array([g[f"cost_trace_{i}"] for i in range(151)])
    assert np.all(np.diff(tr) <= 1e-12 * tr[:-1])
    assert abs(tr[-1] - g["residual_norm2"]) <= 1e-12 * tr[-1]


@pytest.mark.gpu
@pytest.mark.parametrize("coh", ["full", "scalar"])
def test_cuda_path_matches_oracle_at_full_cfg4(cuda_device, coh):
    """The whole bench workload (configs[4]: N=512, T=20, F=8, K=50 x 40 sources, 3 EM x 10 LM), default lm_mode, in the
    launch configuration bench.py times (and, second, with the prediction fused with the initial residual:
    sagecal_predict_residual, then sagecal_sage_calibrate on that residual) against the stored oracle run: all 50 per-cluster costs and the 151-entry cost trace, ALL 25 600
    Jones matrices and sampled residual entries to 1e-8."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate
    g, J_want, p, rows = _fixture("cfg4")
    fmt = sg.COH_FULL if coh == "full" else sg.COH_SCALAR
    coh_d = gpu_predict(p, fmt)
    vis = gpu_simulate(p, coh_d, fmt)
    v2 = float((vis.abs() ** 2).sum())
    assert abs(v2 - g["vis_norm2"]) <= 1e-10 * g["vis_norm2"]
    out = sg.sage_calibrate(p.N, p.T, p.F, vis, coh_d, dev(p.jones_init()), p.n_em, p.n_lm, p.tau, coh_format=fmt)
    torch.cuda.synchronize()
    _compare_with_fixture(sg, p, g, J_want, rows, out, coh)
    del out
    jones = dev(p.jones_init())
    coh_d.zero_()
    _, res = sg.predict_residual(p.N, p.T, p.freqs, p.f0, dev(p.uvw), p.cluster_offset, dev(p.src_l), dev(p.src_m),
                                 dev(p.src_I), dev(p.src_alpha), jones, vis, coh_format=fmt, out=coh_d)
    out = sg.sage_calibrate(p.N, p.T, p.F, None, coh_d, jones, p.n_em, p.n_lm, p.tau, coh_format=fmt, residual=res)
    torch.cuda.synchronize()
    _compare_with_fixture(sg, p, g, J_want, rows, out, coh + " fused")
    del coh_d, vis, out, res
    torch.cuda.empty_cache()


# ---- full-budget fixtures of tests/golden/make_golden_full.py (oracle only): configs[3], polarised configs[4] shape ----
GOLD_DIR = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def _fixture(name):
    import importlib.util
    spec = importlib.util.spec_from_file_location("make_golden_full", os.path.join(GOLD_DIR, "make_golden_full.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    g = _load(os.path.join(GOLD_DIR, f"{name}_oracle.txt"))
    J = np.load(os.path.join(GOLD_DIR, f"{name}_oracle_jones.npy"))
    p = mod.problem(name)
    return g, J, p, mod.sample_rows(name, p)


@pytest.mark.parametrize("name", ["cfg3", "cfg4pol", "cfg4"])
def test_full_budget_fixtures_are_parity_seeds(name):
    """No accept/reject decision of the stored oracle runs was within rounding of zero (Q18), the traces fall
    monotonically (P11) and end at ||R||^2 (P13); the polarised fixture does carry off-diagonal coherencies."""
    g, J, p, rows = _fixture(name)
    n = p.n_em * p.K + 1
    assert g["min_abs_rho"] > 1e-6
    tr = np.array([g[f"cost_trace_{i}"] for i in range(n)])
    assert np.all(np.diff(tr) <= 1e-12 * tr[:-1])
    assert abs(tr[-1] - g["residual_norm2"]) <= 1e-12 * tr[-1]
    assert J.shape == (p.K, p.N, 2, 2)
    for k in range(p.K):
        assert abs(float(np.vdot(J[k], J[k]).real) - g[f"jones_norm2_{k}"]) <= 1e-13 * g[f"jones_norm2_{k}"]
    assert (g["offdiag_coh_norm2"] > 0) == (name == "cfg4pol")


def _compare_with_fixture(sg, p, g, J_want, rows, out, fmt_name):
    import torch
    from tests.gpu_util import host
    cpc = host(out["cost_per_cluster"])
    want = np.array([g[f"cost_cluster_{k}"] for k in range(p.K)])
    assert np.max(np.abs(cpc - want) / want) < 1e-8, fmt_name
    tr = host(out["cost_trace"])
    want_tr = np.array([g[f"cost_trace_{i}"] for i in range(tr.size)])
    assert np.max(np.abs(tr - want_tr) / want_tr) < 1e-8, fmt_name
    J = host(out["jones"])                                         # EVERY Jones matrix, same fixed trajectory (Q17)
    assert np.linalg.norm(J - J_want) <= 1e-8 * np.linalg.norm(J_want)
    assert np.abs(J - J_want).max() <= 1e-8 * np.abs(J_want).max()
    res = host(out["residual"][torch.from_numpy(rows).to(out["residual"].device)])
    assert abs(float(np.vdot(res, res).real) - g["residual_sample_norm2"]) <= 1e-8 * g["residual_sample_norm2"]
    scale = np.sqrt(g["residual_sample_norm2"] / res.size)
    for i, r in enumerate(rows):
        for c in (0, p.F - 1):
            for e in range(4):
                z = g[f"residual_{r}_{c}_{e}_re"] + 1j * g[f"residual_{r}_{c}_{e}_im"]
                assert abs(res[i, c, e] - z) <= 1e-8 * max(abs(z), scale)


@pytest.mark.gpu
@pytest.mark.parametrize("lm", ["compressed", "percluster", "direct"])
@pytest.mark.parametrize("coh", ["full", "scalar"])
def test_cuda_path_matches_oracle_at_full_cfg3(cuda_device, coh, lm):
    """configs[3] with its full budget (N=256, T=20, F=4, K=50 x 20 sources, 3 EM x 10 LM) against the stored oracle
    run, in every lm_mode that follows the oracle's trajectory and both coherency formats: all 50 costs, the 151-entry
    trace, the WHOLE Jones array and sampled residual entries to 1e-8."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate
    g, J_want, p, rows = _fixture("cfg3")
    fmt = sg.COH_FULL if coh == "full" else sg.COH_SCALAR
    mode = {"compressed": sg.LM_COMPRESSED, "percluster": sg.LM_PERCLUSTER, "direct": sg.LM_DIRECT}[lm]
    coh_d = gpu_predict(p, fmt)
    vis = gpu_simulate(p, coh_d, fmt)
    v2 = float((vis.abs() ** 2).sum())
    assert abs(v2 - g["vis_norm2"]) <= 1e-10 * g["vis_norm2"]
    out = sg.sage_calibrate(p.N, p.T, p.F, vis, coh_d, dev(p.jones_init()), p.n_em, p.n_lm, p.tau, coh_format=fmt, lm_mode=mode)
    torch.cuda.synchronize()
    _compare_with_fixture(sg, p, g, J_want, rows, out, f"{coh}/{lm}")
    del coh_d, vis, out
    torch.cuda.empty_cache()


@pytest.mark.gpu
@pytest.mark.parametrize("lm", ["compressed", "percluster"])
def test_cuda_path_matches_oracle_at_polarised_cfg4_shape(cuda_device, lm):
    """configs[4]'s N, T, F and sources per cluster with POLARISED sources (K cut to 4 so that the oracle run fits a
    test fixture): the tensor-core statistics kernel (wbgroup_mma, the default route) and the cluster-by-cluster kernel
    see non-zero XY / YX coherencies at the bench's launch configuration.  Costs, trace, the whole Jones array and
    sampled residual entries against the stored oracle run to 1e-8."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate
    g, J_want, p, rows = _fixture("cfg4pol")
    assert p.polarised and p.N == 512 and p.T == 20 and p.F == 8
    mode = {"compressed": sg.LM_COMPRESSED, "percluster": sg.LM_PERCLUSTER}[lm]
    coh_d = gpu_predict(p)
    off = float((coh_d[..., 1:3].abs() ** 2).sum())
    assert abs(off - g["offdiag_coh_norm2"]) <= 1e-10 * g["offdiag_coh_norm2"] and off > 0
    vis = gpu_simulate(p, coh_d)
    v2 = float((vis.abs() ** 2).sum())
    assert abs(v2 - g["vis_norm2"]) <= 1e-10 * g["vis_norm2"]
    out = sg.sage_calibrate(p.N, p.T, p.F, vis, coh_d, dev(p.jones_init()), p.n_em, p.n_lm, p.tau, lm_mode=mode)
    torch.cuda.synchronize()
    _compare_with_fixture(sg, p, g, J_want, rows, out, lm)
    del coh_d, vis, out
    torch.cuda.empty_cache()
