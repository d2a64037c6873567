"""-m gpu parity: sagecal_predict_coherencies (CUDA, through the C ABI) against oracle.predict on the same seeded
inputs.  Tolerance: 1e-10 relative (BASELINE.json:5 'to within 1e-10 relative for float64'), measured as in
DESIGN.md §3 Q16: ||gpu-oracle||_2/||oracle||_2 and max|gpu-oracle|/max|oracle| over the whole array."""
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


@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_predict_configs_full_and_scalar(cuda_device, cfg):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import gpu_predict, host

    p = make_config(cfg)
    want = oracle.predict(p)                                  # [K, rows, F, 4]
    got = host(gpu_predict(p, sg.COH_FULL))
    _check(got, want)
    # unpolarised: XY = YX = 0 exactly, XX = YY
    assert np.all(got[..., 1] == 0) and np.all(got[..., 2] == 0) and np.array_equal(got[..., 0], got[..., 3])
    got_s = host(gpu_predict(p, sg.COH_SCALAR))
    assert np.array_equal(got_s, got[..., 0])                 # the scalar format is the same numbers


@pytest.mark.parametrize("F,uniform", [(1, True), (3, True), (5, False), (9, True), (13, False)])
def test_predict_polarised_ragged(cuda_device, F, uniform):
    """Polarised sources (general 2x2 brightness), rows not a multiple of the CTA size, channel counts that are not
    a multiple of the register tile, non-uniform channel spacing (no recurrence), clusters of unequal size
    including an empty one."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host

    rng = np.random.default_rng(100 + F)
    freqs = np.linspace(120e6, 170e6, F) if uniform else np.sort(rng.uniform(120e6, 170e6, F))
    if F == 1:
        freqs = np.array([143.7e6])
    p = make_problem(11, 3, F, 4, 7, seed=55 + F, polarised=True, layout="disc:20000", field_deg=5.0,
                     patch_deg=0.7, freqs=freqs)
    # ragged clusters: sizes 7, 0, 12, 9
    off = np.array([0, 7, 7, 19, 28], dtype=np.int32)
    p.cluster_offset = off
    p.K = 4
    want = oracle.predict(p)
    d = {k: dev(getattr(p, k)) for k in ("src_l", "src_m", "src_I", "src_alpha", "src_Q", "src_U", "src_V")}
    got = host(sg.predict_coherencies(p.N, p.T, p.freqs, p.f0, dev(p.uvw), off, d["src_l"], d["src_m"], d["src_I"],
                                      d["src_alpha"], d["src_Q"], d["src_U"], d["src_V"]))
    _check(got, want)
    assert np.all(got[1] == 0)                                # empty cluster


def test_predict_closed_forms_on_gpu(cuda_device):
    """P1/P2 on the CUDA path itself: a source at the phase centre gives C = B_s (f/f0)^alpha on every row;
    negating uvw gives the Hermitian transpose."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host

    p = make_problem(9, 2, 4, 1, 1, seed=9, polarised=True, layout="disc:30000")
    p.src_l[:] = 0.0
    p.src_m[:] = 0.0
    d = {k: dev(getattr(p, k)) for k in ("src_l", "src_m", "src_I", "src_alpha", "src_Q", "src_U", "src_V")}
    args = (p.N, p.T, p.freqs, p.f0)
    got = host(sg.predict_coherencies(*args, dev(p.uvw), p.cluster_offset, d["src_l"], d["src_m"], d["src_I"],
                                      d["src_alpha"], d["src_Q"], d["src_U"], d["src_V"]))[0]
    sc = (p.freqs / p.f0) ** p.src_alpha[0]
    I, Q, U, V = p.src_I[0], p.src_Q[0], p.src_U[0], p.src_V[0]
    Bm = np.array([I + Q, U + 1j * V, U - 1j * V, I - Q])
    want = np.broadcast_to(sc[None, :, None] * Bm[None, None, :], got.shape)
    assert rel_max(got, want) < 1e-14
    # Hermitian symmetry under uvw -> -uvw with sources off centre
    p2 = make_problem(9, 2, 4, 1, 6, seed=10, polarised=True, layout="disc:30000", field_deg=4.0)
    d = {k: dev(getattr(p2, k)) for k in ("src_l", "src_m", "src_I", "src_alpha", "src_Q", "src_U", "src_V")}
    a = host(sg.predict_coherencies(*args, dev(p2.uvw), p2.cluster_offset, d["src_l"], d["src_m"], d["src_I"],
                                    d["src_alpha"], d["src_Q"], d["src_U"], d["src_V"]))[0]
    b = host(sg.predict_coherencies(*args, dev(-p2.uvw), p2.cluster_offset, d["src_l"], d["src_m"], d["src_I"],
                                    d["src_alpha"], d["src_Q"], d["src_U"], d["src_V"]))[0]
    bh = b.reshape(-1, 4, 2, 2).conj().transpose(0, 1, 3, 2).reshape(b.shape)
    assert rel_max(a, bh) < 1e-14


def test_predict_full_size_sampled(cuda_device):
    """configs[4] (N=512, T=20, F=8, K=50, S=40) in the launch configuration bench.py times: all 4.19e10 vis*src
    predicted on the device (scalar format, 16.7 GB), a random sample of rows checked against the oracle."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import gpu_predict, host

    p = make_config(4)
    coh = gpu_predict(p, sg.COH_SCALAR)                       # [K, rows, F]
    rng = np.random.default_rng(4)
    rows = np.sort(rng.choice(p.rows, 192, replace=False))
    rows[0], rows[-1] = 0, p.rows - 1
    want = oracle.predict(p, rows=rows)[..., 0]               # [K, 192, F]
    import torch
    got = host(coh[:, torch.from_numpy(rows).to(coh.device), :])
    _check(got, want)
    del coh
    torch.cuda.empty_cache()


def test_predict_errors(cuda_device):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev

    p = make_config(0)
    d = {k: dev(getattr(p, k)) for k in ("src_l", "src_m", "src_I", "src_alpha")}
    with pytest.raises(sg.SagecalError) as e:   # bad reference frequency
        sg.predict_coherencies(p.N, p.T, p.freqs, -1.0, dev(p.uvw), p.cluster_offset, d["src_l"], d["src_m"],
                               d["src_I"], d["src_alpha"])
    assert e.value.code == -1
    with pytest.raises(sg.SagecalError):        # offsets must start at 0 and not decrease
        sg.predict_coherencies(p.N, p.T, p.freqs, p.f0, dev(p.uvw), [3, 0, 3], d["src_l"], d["src_m"],
                               d["src_I"], d["src_alpha"])


@pytest.mark.parametrize("case", ["cfg1", "cfg2-scalar", "polarised", "nonuniform"])
def test_predict_mixed_precision_variant(cuda_device, case):
    """precision=1 (float64 phase and range reduction, float32 phasor (sin.approx / cos.approx) / recurrence / flux products, float64
    accumulation of 32-source partial sums): 1e-5 relative against the float64 oracle (BASELINE.json:5), and
    clearly not the float64 path (error above 1e-10)."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import gpu_predict, host
    freqs = None
    fmt = sg.COH_FULL
    if case == "cfg1":
        p = make_config(1)
    elif case == "cfg2-scalar":
        p = make_config(2, K=5)
        fmt = sg.COH_SCALAR
    elif case == "polarised":
        p = make_problem(12, 3, 6, 3, 37, seed=9, layout="disc:20000", field_deg=5.0, patch_deg=0.5, polarised=True)
    else:
        p = make_problem(12, 3, 5, 2, 9, seed=10, layout="disc:30000", field_deg=5.0, patch_deg=0.5,
                         freqs=np.array([120e6, 131e6, 150e6, 151e6, 178e6]))
    want = oracle.predict(p)
    got = host(gpu_predict(p, fmt, precision=1))
    if fmt == sg.COH_SCALAR:
        want = want[..., 0]
    got = got.reshape(want.shape)
    assert rel_l2(got, want) < 1e-5 and rel_max(got, want) < 1e-5
    assert rel_l2(got, want) > 1e-10


# ---- sagecal_predict_residual: prediction fused with the initial residual (rows 8a-0 .. 8a-2 in one pass) ----------
def _fused(sg, p, fmt, jones, vis):
    from tests.gpu_util import dev
    d = {k: dev(getattr(p, k)) for k in ("src_l", "src_m", "src_I", "src_alpha", "src_Q", "src_U", "src_V")}
    return sg.predict_residual(p.N, p.T, p.freqs, p.f0, dev(p.uvw), p.cluster_offset, d["src_l"], d["src_m"], d["src_I"],
                               d["src_alpha"], dev(jones), dev(vis), d["src_Q"], d["src_U"], d["src_V"], coh_format=fmt)


@pytest.mark.parametrize("cfg,fmt_name", [(0, "full"), (1, "full"), (2, "full"), (2, "scalar")])
def test_predict_residual_matches_oracle(cuda_device, cfg, fmt_name):
    """coh = the oracle's prediction and residual = V - sum_k J_k C_k J_k^H by the oracle's corrupt/subtract (1e-10), with
    Jones that are not the identity; the coherencies are bit-identical to sagecal_predict_coherencies'."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import gpu_predict, host, per_baseline_form
    p = make_config(cfg)
    fmt = sg.COH_FULL if fmt_name == "full" else sg.COH_SCALAR
    coh_ref = oracle.predict(p)
    V = oracle.simulate(p, coh_ref)
    J = p.jones_true * (1.0 + 0.05j) + 0.02
    want = oracle.corrupt_subtract(p.N, p.T, p.F, coh_ref, J, V, sign=-1.0)
    coh, res = _fused(sg, p, fmt, J, V)
    with per_baseline_form():                                 # the fused arm predicts per baseline
        assert np.array_equal(host(coh), host(gpu_predict(p, fmt)))
    _check(host(coh).reshape(coh_ref[..., 0].shape if fmt == sg.COH_SCALAR else coh_ref.shape),
           coh_ref[..., 0] if fmt == sg.COH_SCALAR else coh_ref)
    _check(host(res), want)


@pytest.mark.parametrize("F,uniform", [(3, True), (5, False), (9, True)])
def test_predict_residual_polarised_ragged(cuda_device, F, uniform):
    """General 2x2 coherencies (model = J_p C J_q^H by two products), channel counts off the register tile, rows off the
    CTA size, an empty cluster."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import host
    rng = np.random.default_rng(300 + F)
    freqs = np.linspace(120e6, 170e6, F) if uniform else np.sort(rng.uniform(120e6, 170e6, F))
    p = make_problem(11, 3, F, 4, 7, seed=77 + F, polarised=True, layout="disc:20000", field_deg=5.0,
                     patch_deg=0.7, freqs=freqs)
    p.cluster_offset = np.array([0, 7, 7, 19, 28], dtype=np.int32)
    coh_ref = oracle.predict(p)
    V = oracle.simulate(p, coh_ref)
    J = p.jones_true * (0.9 - 0.1j)
    want = oracle.corrupt_subtract(p.N, p.T, p.F, coh_ref, J, V, sign=-1.0)
    coh, res = _fused(sg, p, sg.COH_FULL, J, V)
    _check(host(coh), coh_ref)
    _check(host(res), want)


@pytest.mark.parametrize("fmt_name", ["full", "scalar"])
def test_calibrate_from_fused_residual_is_the_same_run(cuda_device, fmt_name):
    """sagecal_sage_calibrate(vis = NULL) on the residual sagecal_predict_residual wrote follows the very trajectory of
    the unfused route: costs, trace, Jones and residual agree to rounding of the initial residual (1e-11)."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host, per_baseline_form
    p = make_config(2)
    fmt = sg.COH_FULL if fmt_name == "full" else sg.COH_SCALAR
    with per_baseline_form():                                 # the same coherencies, bit for bit, on both routes
        coh_d = gpu_predict(p, fmt)
    vis = gpu_simulate(p, coh_d, fmt)
    a = sg.sage_calibrate(p.N, p.T, p.F, vis, coh_d, dev(p.jones_init()), p.n_em, p.n_lm, p.tau, coh_format=fmt)
    coh2, res = _fused(sg, p, fmt, p.jones_init(), host(vis))
    b = sg.sage_calibrate(p.N, p.T, p.F, None, coh2, dev(p.jones_init()), p.n_em, p.n_lm, p.tau, coh_format=fmt, residual=res)
    torch.cuda.synchronize()
    for key in ("cost_per_cluster", "cost_trace", "jones", "residual"):
        assert rel_l2(host(b[key]), host(a[key])) < 1e-11, key


# ---- station form (DMMA contraction of station phasors) and its fall-backs ------------------------------------------
@pytest.mark.parametrize("shape", [(2, 1, 1, 1, 1), (3, 2, 3, 2, 5), (17, 2, 8, 3, 7), (33, 3, 5, 2, 9), (50, 2, 9, 4, 6),
                                   (70, 1, 13, 2, 11)])
@pytest.mark.parametrize("fmt_name", ["full", "scalar"])
def test_predict_station_form_ragged_shapes(cuda_device, shape, fmt_name):
    """Station counts off the 16 x 32 tile, channel counts off the register tile (and several channel tiles), odd source
    counts (a padding source per cluster), an empty cluster: both forms against the oracle, and against each other."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import gpu_predict, host, per_baseline_form
    N, T, F, K, S = shape
    p = make_problem(N, T, F, K, S, seed=500 + N, layout="disc:20000", field_deg=5.0, patch_deg=0.7)
    if K >= 3:
        off = p.cluster_offset.copy()
        off[2] = off[1]                                       # cluster 1 is empty
        p.cluster_offset = off
    fmt = sg.COH_FULL if fmt_name == "full" else sg.COH_SCALAR
    want = oracle.predict(p)
    if fmt == sg.COH_SCALAR:
        want = want[..., 0]
    got = host(gpu_predict(p, fmt)).reshape(want.shape)
    with per_baseline_form():
        got_b = host(gpu_predict(p, fmt)).reshape(want.shape)
    _check(got, want)
    _check(got_b, want)
    assert not np.array_equal(got, got_b) or N <= 2           # two different computations (the station form DID run)
    if K >= 3:
        assert np.all(got[1] == 0)


def test_predict_falls_back_when_uvw_are_not_station_differences(cuda_device):
    """One baseline's uvw moved by a metre: the rows are no longer differences of station coordinates, the device-side
    check sends the call to the per-baseline form, and the answer is the definition's (the station form would be off by
    a whole phase turn on that row)."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import gpu_predict, host, per_baseline_form
    p = make_problem(20, 2, 8, 3, 9, seed=611, layout="disc:20000", field_deg=5.0, patch_deg=0.7)
    uvw = p.uvw.copy()
    uvw[p.B + 57] += np.array([1.0, -2.0, 0.5])               # (t = 1, baseline 57), not a (0, q) row
    p.uvw = uvw
    want = oracle.predict(p)
    got = host(gpu_predict(p, sg.COH_FULL))
    _check(got, want)
    with per_baseline_form():
        assert np.array_equal(got, host(gpu_predict(p, sg.COH_FULL)))      # it WAS the per-baseline form
    # NaN anywhere in the uvw: inconsistent, never the station form
    uvw[3, 1] = np.nan
    p.uvw = uvw
    got = host(gpu_predict(p, sg.COH_FULL))
    with per_baseline_form():
        assert np.array_equal(got, host(gpu_predict(p, sg.COH_FULL)), equal_nan=True)


def test_predict_with_the_small_workspace_predicts_per_baseline(cuda_device):
    """sagecal_predict_workspace_bytes() (no room for station phasors) still works: per-baseline form, same bits."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, host, per_baseline_form
    p = make_config(1)
    L = sg.load_library()
    S = int(p.cluster_offset[-1])
    wsb = int(L.sagecal_predict_workspace_bytes(p.F, S))
    assert int(L.sagecal_predict_workspace_bytes_station(p.N, p.T, p.F, p.K, S)) > wsb
    ws = torch.empty(wsb, dtype=torch.uint8, device=cuda_device)
    out = torch.empty((p.K, p.rows, p.F, 4), dtype=torch.complex128, device=cuda_device)
    fr = np.ascontiguousarray(p.freqs, dtype=np.float64)
    co = np.ascontiguousarray(p.cluster_offset, dtype=np.int32)
    d = {k: dev(getattr(p, k)) for k in ("uvw", "src_l", "src_m", "src_I", "src_alpha")}
    rc = L.sagecal_predict_coherencies(p.N, p.T, p.F, fr.ctypes.data, float(p.f0), d["uvw"].data_ptr(), p.K, co.ctypes.data,
                                       d["src_l"].data_ptr(), d["src_m"].data_ptr(), d["src_I"].data_ptr(), None, None,
                                       None, d["src_alpha"].data_ptr(), sg.COH_FULL, out.data_ptr(), 0, ws.data_ptr(), wsb,
                                       torch.cuda.current_stream().cuda_stream)
    assert rc == 0
    with per_baseline_form():
        assert np.array_equal(host(out), host(gpu_predict(p, sg.COH_FULL)))
    _check(host(gpu_predict(p, sg.COH_FULL)), oracle.predict(p))
