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
