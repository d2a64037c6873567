"""-m gpu parity of lm_mode = SAGECAL_LM_FULLGN (full 8N x 8N Gauss-Newton M-step, cuSOLVER Cholesky; SURVEY.md §8(f)
NEXT-2) against oracle/fullgn.py on the same seeded inputs and iteration counts.  Tolerance 1e-8 relative on the final
per-cluster cost, the Jones, the residual and the cost trace, as for the block-diagonal modes."""
import numpy as np
import pytest

from oracle import fullgn, oracle
from sagecal_inputs import make_config, make_problem
from tests.helpers import procrustes_err, rel_l2, rel_max

pytestmark = pytest.mark.gpu
TOL = 1e-8


def _run_both(p, n_em, n_lm, scalar=False):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, host
    fmt = sg.COH_SCALAR if scalar else sg.COH_FULL
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    want = fullgn.sage(p.N, p.T, p.F, V, coh, p.jones_init(), n_em, n_lm, p.tau)
    assert want["min_abs_rho"] > 1e-6, "seed has an accept/reject decision within rounding of 0: not a parity seed"
    got = sg.sage_calibrate(p.N, p.T, p.F, dev(V), gpu_predict(p, fmt), dev(p.jones_init()), n_em, n_lm, p.tau,
                            coh_format=fmt, lm_mode=sg.LM_FULLGN)
    return want, {k: (None if v is None else host(v)) for k, v in got.items()}


def _compare(want, got):
    assert np.max(np.abs(got["cost_per_cluster"] - want["cost_per_cluster"]) / want["cost_per_cluster"]) < TOL
    assert rel_max(got["cost_trace"], want["cost_trace"]) < TOL
    assert rel_l2(got["jones"], want["jones"]) < TOL
    assert rel_l2(got["residual"], want["residual"]) < TOL


def test_fullgn_cfg0(cuda_device):
    p = make_config(0)
    _compare(*_run_both(p, 2, 4))


def test_fullgn_multi_cluster_polarised(cuda_device):
    p = make_problem(14, 4, 3, 3, 4, seed=41, sigma=0.05, layout="disc:4000", field_deg=4.0, patch_deg=0.5, polarised=True)
    _compare(*_run_both(p, 2, 3))


def test_fullgn_scalar_format_ragged_tiles(cuda_device):
    p = make_problem(37, 2, 5, 2, 4, seed=43, sigma=0.05, layout="disc:6000", field_deg=4.0, patch_deg=0.5)
    _compare(*_run_both(p, 1, 3, scalar=True))


def test_fullgn_recentres_long_msteps(cuda_device):
    """n_lm = 12 > SAGECAL_LM_RECENTRE: the statistics are re-taken once inside the M-step."""
    p = make_problem(10, 3, 2, 2, 4, seed=47, sigma=0.05, layout="disc:3000", field_deg=4.0, patch_deg=0.5,
                     jones_std=0.3)
    want, got = _run_both(p, 1, 12)
    _compare(want, got)


def test_fullgn_noiseless_recovery_on_gpu(cuda_device):
    """Noiseless single-cluster data: the full solve reaches < 1e-20 relative cost within 12 trial steps and recovers
    the true Jones up to a unitary (the block-diagonal modes need about 45 steps)."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host
    p = make_config(0, sigma=0.0)
    coh_d = gpu_predict(p)
    V = gpu_simulate(p, coh_d, noise=False)
    phi0 = float((V.abs() ** 2).sum())
    got = sg.sage_calibrate(p.N, p.T, p.F, V, coh_d, dev(p.jones_init()), 1, 12, p.tau, lm_mode=sg.LM_FULLGN)
    assert float(got["cost_per_cluster"][0]) / phi0 < 1e-20
    assert procrustes_err(host(got["jones"])[0], p.jones_true[0]) < 1e-12


def test_fullgn_cfg1_512x512_system(cuda_device):
    """configs[1] (N=64: a 512 x 512 normal matrix), 1 EM x 3 LM."""
    p = make_config(1)
    _compare(*_run_both(p, 1, 3))
