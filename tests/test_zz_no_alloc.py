"""-m gpu: sagecal_predict_coherencies_static, the entry point for callers that cannot allocate device memory (its
scratch -- the prepared source table -- is a fixed device array of the library), against the existing path
sagecal_predict_coherencies on the same seeded inputs, on calls in a row that share the array, and against the oracle.
Tolerance as in tests/test_gpu_predict.py: 1e-10 relative (BASELINE.json:5).  Collected last on purpose (the file name):
the suite runs with pytest -x."""
import numpy as np
import pytest

from oracle import oracle
from sagecal_inputs import make_config, make_problem
from tests.helpers import rel_l2, rel_max

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _check(got, want, tol=TOL):
    assert got.shape == want.shape
    assert rel_l2(got, want) < tol, rel_l2(got, want)
    assert rel_max(got, want) < tol, rel_max(got, want)


def _inputs(p):
    """The problem's device arrays, made BEFORE the calls that are checked for allocating nothing."""
    from tests.gpu_util import dev
    d = {k: dev(getattr(p, k)) for k in ("src_l", "src_m", "src_I", "src_alpha", "src_Q", "src_U", "src_V")}
    d["uvw"] = dev(p.uvw)
    return d


def _static(sg, p, d, fmt, out):
    return sg.predict_coherencies_static(p.N, p.T, p.freqs, p.f0, d["uvw"], p.cluster_offset, d["src_l"], d["src_m"],
                                         d["src_I"], d["src_alpha"], out, d["src_Q"], d["src_U"], d["src_V"],
                                         coh_format=fmt)


def test_static_scratch_predict_matches_the_workspace_path_on_calls_in_a_row(cuda_device):
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import gpu_predict, host, per_baseline_form

    # three different sky models one after the other through the ONE shared array: a large unpolarised table, then a
    # smaller polarised one with non-uniform channels (the first call's entries are still behind it), then scalar output
    a = make_config(1)
    b = make_problem(12, 3, 5, 2, 9, seed=10, layout="disc:30000", field_deg=5.0, patch_deg=0.5, polarised=True,
                     freqs=np.array([120e6, 131e6, 150e6, 151e6, 178e6]))
    c = make_config(2, K=5)
    cases = [(a, sg.COH_FULL), (b, sg.COH_FULL), (c, sg.COH_SCALAR), (a, sg.COH_FULL)]
    with per_baseline_form():                                               # the static entry predicts per baseline
        want = [host(gpu_predict(p, fmt)) for p, fmt in cases]              # the existing path, its own workspace
    outs = [torch.full(w.shape, float("nan"), dtype=torch.complex128, device=cuda_device) for w in want]
    ins = [_inputs(p) for p, _ in cases]
    torch.cuda.synchronize()
    free = []
    for (p, fmt), d, out in zip(cases, ins, outs):                          # calls in a row, nothing in between
        _static(sg, p, d, fmt, out)
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    for out, w in zip(outs, want):
        _check(host(out), w)
        assert np.array_equal(host(out), w)                                 # same kernels, same inputs: same bits
    _check(host(outs[0]), oracle.predict(a))
    _check(host(outs[1]), oracle.predict(b))
    # the repeated call of the first sky model gives the first call's answer again
    assert np.array_equal(host(outs[0]), host(outs[3]))
    # nothing was allocated on the device by the calls after the first (which may still load the module lazily)
    assert free[1] == free[2] == free[3], free


def test_static_scratch_predict_refuses_what_does_not_fit(cuda_device):
    import torch
    import paper_1910_13908_b200 as sg

    limit = sg.predict_static_bytes()
    assert limit == 2 * 1024 * 1024
    F, S = 8, 8000                                                          # 8000 x 8 x 4 x 8 B of fluxes alone > 2 MiB
    L = sg.load_library()
    assert L.sagecal_predict_workspace_bytes(F, S) > limit
    N, T = 3, 1
    rows = T * N * (N - 1) // 2
    z = torch.zeros(S, dtype=torch.float64, device=cuda_device)
    out = torch.full((1, rows, F, 4), 7.0, dtype=torch.complex128, device=cuda_device)
    uvw = torch.zeros((rows, 3), dtype=torch.float64, device=cuda_device)
    freqs = np.linspace(120e6, 160e6, F)
    with pytest.raises(sg.SagecalError) as e:
        sg.predict_coherencies_static(N, T, freqs, 140e6, uvw, [0, S], z, z, z, z, out)
    assert e.value.code == -5 and "scratch" in str(e.value)          # SAGECAL_ESTATICLIMIT
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                                         # nothing was launched
    # the largest table that fits is accepted
    S_ok = 7900
    assert L.sagecal_predict_workspace_bytes(F, S_ok) <= limit
    z = torch.zeros(S_ok, dtype=torch.float64, device=cuda_device)
    sg.predict_coherencies_static(N, T, freqs, 140e6, uvw, [0, S_ok], z, z, z, z, out)
    torch.cuda.synchronize()
    assert bool((out == 0.0).all())                                         # zero fluxes: zero coherencies
