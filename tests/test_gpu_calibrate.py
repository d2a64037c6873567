"""-m gpu parity: sagecal_sage_calibrate (CUDA, device-resident EM/LM loop) against oracle.sage on the same seeded
inputs and the same fixed iteration counts.  Tolerance: 1e-8 relative on the final per-cluster cost
(BASELINE.json:5); the same bound is applied to the Jones, the residual and the cost trace.  A parity seed is only
valid if no accept/reject decision sat within rounding of zero (DESIGN.md §3 Q18): min |rho| > 1e-6."""
import numpy as np
import pytest

from oracle import oracle
from sagecal_inputs import make_config, make_problem
from tests.helpers import rel_l2, rel_max

pytestmark = pytest.mark.gpu
TOL = 1e-8
MODES = ["compressed", "direct", "percluster"]      # lm_mode of sagecal_sage_calibrate: all follow the oracle's trajectory


def _mode(name):
    import paper_1910_13908_b200 as sg
    return {"compressed": sg.LM_COMPRESSED, "direct": sg.LM_DIRECT, "percluster": sg.LM_PERCLUSTER}[name]


def _run_both(p, n_em, n_lm, coh_format=None, polarised=False, mode="compressed"):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, host

    fmt = sg.COH_FULL if coh_format is None else coh_format
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)                       # the oracle's V feeds both sides (never the other way round)
    want = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), n_em, n_lm, p.tau)
    assert want["min_abs_rho"] > 1e-6, "seed has an accept/reject decision within rounding of 0: not a parity seed"
    coh_d = gpu_predict(p, fmt)                        # the CUDA path predicts its own coherencies
    got = sg.sage_calibrate(p.N, p.T, p.F, dev(V), coh_d, dev(p.jones_init()), n_em, n_lm, p.tau, coh_format=fmt,
                            lm_mode=_mode(mode))
    return want, {k: (None if v is None else host(v)) for k, v in got.items()}, V, coh


def _compare(want, got):
    cpc_err = np.max(np.abs(got["cost_per_cluster"] - want["cost_per_cluster"]) / want["cost_per_cluster"])
    assert cpc_err < TOL, cpc_err
    assert rel_max(got["cost_trace"], want["cost_trace"]) < TOL
    assert rel_l2(got["jones"], want["jones"]) < TOL
    assert rel_l2(got["residual"], want["residual"]) < TOL


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("cfg", [0, 1, 2])
def test_calibrate_configs(cuda_device, cfg, mode):
    """configs[0..2] with their own iteration budget (3 EM x 10 LM)."""
    p = make_config(cfg)
    want, got, V, coh = _run_both(p, p.n_em, p.n_lm, mode=mode)
    _compare(want, got)
    tr = got["cost_trace"]
    assert np.all(np.diff(tr) <= 1e-12 * tr[:-1])            # P11 on the CUDA path


@pytest.mark.parametrize("mode", MODES)
def test_calibrate_scalar_format(cuda_device, mode):
    import paper_1910_13908_b200 as sg
    p = make_config(2, K=6)
    want, got, _, _ = _run_both(p, 2, 6, coh_format=sg.COH_SCALAR, mode=mode)
    _compare(want, got)


@pytest.mark.parametrize("mode", MODES)
def test_calibrate_polarised_small(cuda_device, mode):
    p = make_problem(10, 4, 3, 3, 4, seed=31, sigma=0.05, layout="disc:3000", field_deg=4.0, patch_deg=0.5,
                     polarised=True)
    want, got, _, _ = _run_both(p, 3, 5, mode=mode)
    _compare(want, got)


@pytest.mark.parametrize("mode", ["compressed", "percluster"])
@pytest.mark.parametrize("shape", [(37, 3, 3), (33, 2, 5), (70, 2, 8), (6, 2, 40)])
def test_calibrate_compressed_ragged_shapes(cuda_device, shape, mode):
    """Compressed mode on shapes that leave ragged pieces everywhere: N not a multiple of the 32-station column segment,
    F not a power of two (idle lanes in a baseline's lane group) and F > 32 (a lane walks several channels);
    polarised sources so all 16 + 16 statistics of a baseline matter."""
    N, T, F = shape
    p = make_problem(N, T, F, 3, 4, seed=77 + N, sigma=0.05, layout="disc:5000", field_deg=4.0, patch_deg=0.5,
                     polarised=True)
    want, got, _, _ = _run_both(p, 2, 4, mode=mode)
    _compare(want, got)


@pytest.mark.parametrize("K", [1, 2, 5, 7, 9])
@pytest.mark.parametrize("scalar", [False, True])
def test_calibrate_grouped_ragged_groups(cuda_device, K, scalar):
    """Cluster groups of 4: K = 1, 2 (one short group), 5 (4 + 1), 7 (4 + 3), 9 (4 + 4 + 1) exercise every
    (previous group, next group) size pair of the streaming kernel and the cross-gram slots of short groups."""
    import paper_1910_13908_b200 as sg
    p = make_problem(12, 3, 3, K, 3, seed=500 + K, sigma=0.05, layout="disc:5000", field_deg=4.0, patch_deg=0.5,
                     polarised=not scalar)
    want, got, _, _ = _run_both(p, 2, 4, coh_format=sg.COH_SCALAR if scalar else sg.COH_FULL, mode="compressed")
    _compare(want, got)


def test_calibrate_compressed_more_tiles_than_ctas(cuda_device):
    """N = 700: 8070 units for at most 1184 co-resident warps, so every warp of the M-step kernel owns a chunk of 7 rows
    whose statistics are streamed through its two shared-memory slots; the last column segment is ragged
    (700 = 21*32 + 28)."""
    p = make_problem(700, 1, 2, 2, 3, seed=123, sigma=0.05, layout="disc:20000", field_deg=4.0, patch_deg=0.5)
    want, got, _, _ = _run_both(p, 1, 4, mode="compressed")
    _compare(want, got)


@pytest.mark.parametrize("N,what", [(64, "one thread-block cluster of 16 CTAs, every warp a row (94 chunks)"),
                                    (65, "first shape past the cluster (158 chunks): cooperative launch, 40 CTAs of 4 warps"),
                                    (130, "cooperative, 1 row per warp, 5 column segments, ragged last one"),
                                    (345, "2 rows per warp, statistics resident in two slots"),
                                    (400, "3 rows per warp: more rows than slots, statistics streamed")])
@pytest.mark.parametrize("scalar", [False, True])
def test_calibrate_mstep_launch_regimes(cuda_device, N, what, scalar):
    """The M-step kernel's launch plans (mstep.cu make_plan: cluster / cooperative launch, resident / streamed
    statistics, chunk lengths 1, 2, 3) each against the oracle: one time slot, one channel, two clusters, so that the
    oracle's pass over N(N-1)/2 baselines stays a matter of seconds."""
    import paper_1910_13908_b200 as sg
    p = make_problem(N, 1, 1, 2, 3, seed=900 + N, sigma=0.05, layout="disc:20000", field_deg=4.0, patch_deg=0.5,
                     polarised=not scalar)
    want, got, _, _ = _run_both(p, 2, 5, coh_format=sg.COH_SCALAR if scalar else sg.COH_FULL, mode="compressed")
    _compare(want, got)


def test_calibrate_compressed_recentres_long_msteps(cuda_device):
    """n_lm = 25 > SAGECAL_LM_RECENTRE: the statistics are re-taken at the accepted Jones twice inside every M-step;
    the trajectory must still be the oracle's."""
    p = make_config(1)
    want, got, _, _ = _run_both(p, 2, 25, mode="compressed")
    _compare(want, got)


@pytest.mark.parametrize("mode", MODES)
def test_calibrate_cfg3_multi_tile(cuda_device, mode):
    """configs[3] shape (N=256, F=4: 8 column tiles, time-chunked units), K cut to 4 and 1 EM x 5 LM so the oracle
    finishes in seconds."""
    p = make_config(3, K=4)
    want, got, _, _ = _run_both(p, 1, 5, mode=mode)
    _compare(want, got)


def test_calibrate_modes_agree_to_rounding(cuda_device):
    """The two lm_modes are the same sums re-associated: on the same inputs they agree far inside the parity bound."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host
    p = make_config(2, K=8)
    coh_d = gpu_predict(p)
    V = gpu_simulate(p, coh_d)
    out = [sg.sage_calibrate(p.N, p.T, p.F, V, coh_d, dev(p.jones_init()), 2, 6, p.tau, lm_mode=m)
           for m in (sg.LM_COMPRESSED, sg.LM_PERCLUSTER, sg.LM_DIRECT)]
    a, c, b = [{k: host(v) for k, v in o.items()} for o in out]
    for x in (a, c):
        assert np.max(np.abs(x["cost_per_cluster"] - b["cost_per_cluster"]) / b["cost_per_cluster"]) < 1e-11
        assert rel_l2(x["jones"], b["jones"]) < 1e-11
        assert rel_l2(x["residual"], b["residual"]) < 1e-11


@pytest.mark.parametrize("mode", MODES)
def test_calibrate_noiseless_recovery_on_gpu(cuda_device, mode):
    """P10 on the CUDA path: noiseless single-cluster data, the cost falls below 1e-20 relative and the true Jones
    are recovered up to a unitary matrix.  60 trial steps of one M-step; compressed mode re-centres its statistics
    every 10 of them, which is what lets the cost fall 20 decades below the starting residual."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host
    from tests.helpers import procrustes_err

    p = make_config(0, sigma=0.0)
    coh_d = gpu_predict(p)
    V = gpu_simulate(p, coh_d, noise=False)
    phi0 = float((V.abs() ** 2).sum())
    got = sg.sage_calibrate(p.N, p.T, p.F, V, coh_d, dev(p.jones_init()), 1, 60, p.tau, lm_mode=_mode(mode))
    assert float(got["cost_per_cluster"][0]) / phi0 < 1e-20
    assert procrustes_err(host(got["jones"])[0], p.jones_true[0]) < 1e-12


@pytest.mark.parametrize("mode", MODES)
def test_calibrate_full_size_properties(cuda_device, mode):
    """configs[4] (N=512, T=20, F=8, K=50 x 40 sources) in the launch configuration bench.py times, scalar
    coherencies, 1 EM x 2 LM to bound the time.  The oracle cannot run this size inside a test, so: sampled outputs
    (the residual on random rows, recomputed by the oracle from the returned Jones; the gradient of one LM pass for
    sampled stations, by the oracle on those stations' baselines) and properties that hold at any size
    (P11 monotone trace, P13 residual bookkeeping, cost == ||residual||^2)."""
    import torch
    import paper_1910_13908_b200 as sg
    from sagecal_inputs import baseline_index, noise_rows
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host

    p = make_config(4)
    N, T, F, K = p.N, p.T, p.F, p.K
    coh_d = gpu_predict(p, sg.COH_SCALAR)
    V = gpu_simulate(p, coh_d, sg.COH_SCALAR)
    J0 = dev(p.jones_init())
    got = sg.sage_calibrate(N, T, F, V, coh_d, J0, 1, 2, p.tau, coh_format=sg.COH_SCALAR, lm_mode=_mode(mode))
    tr = host(got["cost_trace"])
    assert np.all(np.isfinite(tr)) and np.all(np.diff(tr) <= 1e-12 * tr[:-1])
    # cost_per_cluster[K-1] is ||R||^2 after the last M-step
    r2 = float((got["residual"].abs() ** 2).sum())
    assert abs(r2 - tr[-1]) < 1e-9 * r2
    assert abs(float(got["cost_per_cluster"][-1]) - tr[-1]) <= 1e-15 * tr[-1]
    # P13 / sampled parity: residual rows recomputed from scratch by the oracle from the returned Jones
    rng = np.random.default_rng(44)
    rows = np.sort(rng.choice(p.rows, 64, replace=False))
    rows_d = torch.from_numpy(rows).to(V.device)
    coh_rows = oracle.predict(p, rows=rows)                       # [K, 64, F, 4]
    Jt, Jn = p.jones_true, host(got["jones"])
    P_, Q_ = np.triu_indices(N, 1)
    bidx = rows % p.B
    def model(J):
        C = coh_rows.reshape(K, rows.size, F, 2, 2)
        return np.einsum("krij,krfjl,krml->rfim", J[:, P_[bidx]], C, J[:, Q_[bidx]].conj()).reshape(rows.size, F, 4)
    v_rows = model(Jt) + noise_rows(p, rows)
    assert rel_l2(host(V[rows_d]), v_rows) < 1e-10
    assert rel_l2(host(got["residual"][rows_d]), v_rows - model(Jn)) < 1e-9
    # one LM pass at full size: gradient / J^H J of sampled stations against the oracle on their baselines
    x = V  # any data serves
    cost, grad, jtj = sg.lm_cost_grad_jtj(N, T, F, x, coh_d[7], got["jones"][7], coh_format=sg.COH_SCALAR)
    for s in (0, 255, 511):
        others = [o for o in range(N) if o != s]
        bl = np.array([baseline_index(N, min(s, o), max(s, o)) for o in others])
        rr = (np.arange(T)[:, None] * p.B + bl[None, :]).reshape(-1)
        rr_d = torch.from_numpy(rr).to(V.device)
        xs = host(x[rr_d]).reshape(T, N - 1, F, 4)
        cs = host(coh_d[7][rr_d]).reshape(T, N - 1, F)
        Js = Jn[7]
        G = np.zeros((2, 2), complex)
        M = np.zeros((2, 2), complex)
        for j, o in enumerate(others):
            Xm = xs[:, j].reshape(-1, 2, 2)
            c = cs[:, j].reshape(-1)
            if s < o:   # s is the row station p
                A = c[:, None, None] * Js[o].conj().T[None]
                E = Xm - Js[s][None] @ A
                G += np.einsum("nij,nkj->ik", E, A.conj())
                M += np.einsum("nij,nkj->ik", A, A.conj())
            else:       # s is the column station q
                T1 = c[:, None, None] * Js[o][None]
                E = Xm - T1 @ Js[s].conj().T[None]
                G += np.einsum("nji,njk->ik", E.conj(), T1)
                M += np.einsum("nji,njk->ik", T1.conj(), T1)
        assert rel_l2(host(grad[s]), G) < 1e-10
        assert rel_l2(host(jtj[s]), M) < 1e-10
    del coh_d, V
    torch.cuda.empty_cache()


def test_calibrate_host_entry(cuda_device):
    """sagecal_calibrate_interval_host (host buffers, copies inside) gives the same answer as the device API."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, host

    p = make_config(1)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    ref = sg.sage_calibrate(p.N, p.T, p.F, dev(V), gpu_predict(p), dev(p.jones_init()), 2, 4, p.tau)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    J = t(p.jones_init())
    R = torch.empty((p.rows, p.F, 4), dtype=torch.complex128).pin_memory()
    out = sg.calibrate_interval_host(p.N, p.T, p.freqs, p.f0, t(p.uvw), p.cluster_offset, t(p.src_l), t(p.src_m),
                                     t(p.src_I), t(p.src_alpha), t(V), J, 2, 4, p.tau, residual=R)
    assert np.array_equal(J.numpy(), host(ref["jones"]))
    assert np.array_equal(R.numpy(), host(ref["residual"]))
    assert np.array_equal(out["cost_per_cluster"].numpy(), host(ref["cost_per_cluster"]))


def test_calibrate_host_entry_async_stream_of_intervals(cuda_device):
    """sagecal_calibrate_interval_host_async: five different intervals enqueued back to back (two sets of host buffers,
    alternating; never more than two in flight), one sagecal_host_sync between reuse: each comes back bit-identical to
    the synchronous entry on the same inputs."""
    import torch
    import paper_1910_13908_b200 as sg
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    probs, want = [], []
    for i in range(5):
        p = make_config(1, seed=4000 + i)
        V = oracle.simulate(p, oracle.predict(p))
        args = (p.N, p.T, p.freqs, p.f0, t(p.uvw), p.cluster_offset, t(p.src_l), t(p.src_m), t(p.src_I), t(p.src_alpha), t(V))
        J = t(p.jones_init())
        R = torch.empty((p.rows, p.F, 4), dtype=torch.complex128).pin_memory()
        out = sg.calibrate_interval_host(*args, J, 2, 4, p.tau, residual=R)
        want.append((J.numpy().copy(), R.numpy().copy(), out["cost_per_cluster"].numpy().copy()))
        probs.append((p, args))
    sets = [dict(J=t(probs[0][0].jones_init()), R=torch.empty_like(R).pin_memory(),
                 C=torch.zeros(1, dtype=torch.float64).pin_memory()) for _ in range(2)]
    snap = lambda b: (b["J"].numpy().copy(), b["R"].numpy().copy(), b["C"].numpy().copy())
    got, pending = {}, {}                                # pending: buffer set -> the interval it carries
    for i, (p, args) in enumerate(probs):
        k = i & 1
        if k in pending:                                 # the set is reused: everything in flight must be home first
            sg.host_sync()
            for kk, ii in pending.items():
                got[ii] = snap(sets[kk])
            pending.clear()
        b = sets[k]
        b["J"].copy_(torch.from_numpy(p.jones_init()))
        sg.calibrate_interval_host(*args, b["J"], 2, 4, p.tau, residual=b["R"], cost_per_cluster=b["C"], asynchronous=True)
        pending[k] = i
    sg.host_sync()
    for kk, ii in pending.items():
        got[ii] = snap(sets[kk])
    assert sorted(got) == [0, 1, 2, 3, 4]
    for i in range(5):
        for a, w in zip(got[i], want[i]):
            assert np.array_equal(a, w), i


@pytest.mark.parametrize("fmt", ["full", "scalar"])
def test_calibrate_compressed_is_bit_reproducible(cuda_device, fmt):
    """No atomics in any sum and a fixed summation order: repeated runs on the same inputs give bit-identical Jones,
    residual and costs (a cross-CTA race in the M-step kernel would show up here)."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host
    f = sg.COH_FULL if fmt == "full" else sg.COH_SCALAR
    p = make_config(3, K=3)
    coh_d = gpu_predict(p, f)
    V = gpu_simulate(p, coh_d, f)
    runs = []
    for _ in range(3):
        o = sg.sage_calibrate(p.N, p.T, p.F, V, coh_d, dev(p.jones_init()), 2, 10, p.tau, coh_format=f)
        runs.append({k: host(v) for k, v in o.items()})
    for r in runs[1:]:
        for k in ("jones", "residual", "cost_per_cluster", "cost_trace"):
            assert np.array_equal(r[k], runs[0][k]), k


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("scalar", [False, True])
def test_calibrate_degenerate_iteration_counts(cuda_device, mode, scalar):
    """n_lm = 0 (every M-step is one evaluation, no trial step: Jones stay at the start values, the per-cluster
    cost is ||R||^2 of the initial residual) and n_em = 0 (initial residual only) in every mode and format; K = 0
    returns the visibilities as residual."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host
    p = make_problem(9, 3, 2, 5, 3, seed=61, sigma=0.05, layout="disc:5000", field_deg=4.0, patch_deg=0.5)
    fmt = sg.COH_SCALAR if scalar else sg.COH_FULL
    want, got, V, coh = _run_both_nocheck(p, 2, 0, fmt, mode)
    assert np.array_equal(got["jones"], p.jones_init())
    assert rel_l2(got["residual"], want["residual"]) < 1e-12
    assert np.allclose(got["cost_per_cluster"], want["cost_per_cluster"], rtol=1e-12)
    assert np.allclose(got["cost_trace"], want["cost_trace"], rtol=1e-12)
    want0, got0, _, _ = _run_both_nocheck(p, 0, 3, fmt, mode)
    assert rel_l2(got0["residual"], want0["residual"]) < 1e-12 and np.array_equal(got0["jones"], p.jones_init())
    # K = 0: nothing to subtract
    Vd = dev(V)
    out = sg.sage_calibrate(p.N, p.T, p.F, Vd, torch.empty((0, p.rows, p.F, 4), dtype=torch.complex128, device="cuda:0"),
                            torch.empty((0, p.N, 2, 2), dtype=torch.complex128, device="cuda:0"), 2, 3, p.tau,
                            lm_mode=_mode(mode))
    assert np.array_equal(host(out["residual"]), V)


def _run_both_nocheck(p, n_em, n_lm, fmt, mode):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, host
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    want = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), n_em, n_lm, p.tau)
    got = sg.sage_calibrate(p.N, p.T, p.F, dev(V), gpu_predict(p, fmt), dev(p.jones_init()), n_em, n_lm, p.tau,
                            coh_format=fmt, lm_mode=_mode(mode))
    return want, {k: (None if v is None else host(v)) for k, v in got.items()}, V, coh


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("scalar", [False, True])
def test_calibrate_writes_nothing_outside_its_buffers(cuda_device, mode, scalar):
    """Every buffer the call may write (residual, Jones, costs, trace, workspace of exactly sagecal_workspace_bytes)
    sits between guard bands of a known byte pattern; ragged shape (N, T*F and K not multiples of any tile, warp or
    group size).  The guards must come back untouched, the read-only inputs unchanged, and the result must still be
    the oracle's."""
    import torch
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, gpu_predict, host
    p = make_problem(13, 3, 3, 5, 3, seed=71, sigma=0.05, layout="disc:5000", field_deg=4.0, patch_deg=0.5,
                     polarised=not scalar)
    fmt = sg.COH_SCALAR if scalar else sg.COH_FULL
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    want = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), 2, 4, p.tau)
    G = 4096

    def guarded(nbytes):
        buf = torch.full((G + ((nbytes + 255) // 256) * 256 + G,), 0xA5, dtype=torch.uint8, device="cuda:0")
        return buf, buf[G:G + nbytes]

    def carve(arr_shape, dtype):
        n = int(np.prod(arr_shape)) * torch.empty((), dtype=dtype).element_size()
        buf, body = guarded(n)
        return buf, body.view(dtype).view(*arr_shape)

    wsb = sg.workspace_bytes(2, p.N, p.T, p.F, p.K)
    ws_buf, ws = guarded(wsb)
    res_buf, res = carve((p.rows, p.F, 4), torch.complex128)
    j_buf, J = carve((p.K, p.N, 2, 2), torch.complex128)
    J.copy_(dev(p.jones_init()))
    coh_d, V_d = gpu_predict(p, fmt), dev(V)
    coh0, V0 = coh_d.clone(), V_d.clone()
    got = sg.sage_calibrate(p.N, p.T, p.F, V_d, coh_d, J, 2, 4, p.tau, coh_format=fmt, residual=res, workspace=ws,
                            lm_mode=_mode(mode))
    torch.cuda.synchronize()
    for name, buf, n in (("workspace", ws_buf, wsb), ("residual", res_buf, res.numel() * 16), ("jones", j_buf, J.numel() * 16)):
        body_end = G + n
        assert bool((buf[:G] == 0xA5).all()), f"{name}: bytes before the buffer were written"
        assert bool((buf[G + ((n + 255) // 256) * 256:] == 0xA5).all()), f"{name}: bytes after the buffer were written"
        assert bool((buf[body_end:G + ((n + 255) // 256) * 256] == 0xA5).all()), f"{name}: padding after the buffer was written"
    assert torch.equal(coh_d, coh0) and torch.equal(V_d, V0)
    _compare(want, {k: (None if v is None else host(v)) for k, v in got.items()})


@pytest.mark.parametrize("mode", MODES)
@pytest.mark.parametrize("scalar", [False, True])
@pytest.mark.parametrize("shape", [(2, 1, 1, 1), (3, 1, 2, 2), (4, 2, 1, 5), (2, 3, 3, 2)])
def test_calibrate_smallest_shapes(cuda_device, shape, scalar, mode):
    """The smallest problems there are: one baseline, one sample (a tensor-core chunk with 7 of 8 sample slots empty,
    three of a CTA's four warps without a baseline), more clusters than stations."""
    import paper_1910_13908_b200 as sg
    N, T, F, K = shape
    p = make_problem(N, T, F, K, 2, seed=900 + N + T, sigma=0.05, layout="disc:5000", field_deg=4.0,
                     patch_deg=0.5 if K > 1 else None, polarised=not scalar)
    want, got, _, _ = _run_both(p, 1, 3, coh_format=sg.COH_SCALAR if scalar else sg.COH_FULL, mode=mode)
    _compare(want, got)
