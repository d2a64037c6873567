"""-m gpu parity: measurement-set row lists (second part).

The CUDA path brings the rows into canonical order (sagecal_rows_to_canonical), predicts on the canonical uvw, zeroes
what is flagged (sagecal_apply_flags), calibrates with the unchanged hot kernels and hands the residual back in the
caller's row order (sagecal_canonical_to_rows).  The oracle (oracle/rows.py) does none of that: it applies the
definitions to the row list directly.  Index and byte work is compared bit for bit, the calibration to 1e-8."""
import numpy as np
import pytest

import sagecal_inputs as si
from oracle import rows as orw
from tests.helpers import crandn, rel_l2, rel_max

pytestmark = pytest.mark.gpu
TOL = 1e-8


def _rowlist(N, T, F, K, S, seed, polarised=False, **kw):
    prob = si.make_problem(N, T, F, K, S, seed=seed, sigma=0.05, layout="disc:3000", field_deg=4.0,
                           patch_deg=0.5 if K > 1 else None, polarised=polarised)
    rl = si.make_rowlist(prob, seed=seed + 1, **kw)
    return prob, rl


def _to_canonical(prob, rl, vis, flags=True):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev
    return sg.rows_to_canonical(prob.N, prob.T, prob.F, dev(rl.ant1), dev(rl.ant2), dev(rl.tslot), dev(rl.uvw),
                                dev(vis), dev(rl.flags) if flags else None)


@pytest.mark.parametrize("shape", [(5, 3, 2), (12, 4, 8), (33, 2, 5), (64, 3, 1)])
def test_rows_to_canonical_is_bit_exact(cuda_device, shape):
    from tests.gpu_util import host
    N, T, F = shape
    prob, rl = _rowlist(N, T, F, 1, 2, seed=100 + N, drop_frac=0.2, swap_frac=0.5, flag_frac=0.2)
    rng = np.random.default_rng(N)
    n = len(rl.ant1)
    vis = crandn(rng, n, F, 4)
    # an auto-correlation, an out-of-range row and a duplicate of row 0 at the end of the list
    import dataclasses
    rl = dataclasses.replace(
        rl, ant1=np.concatenate([rl.ant1, [2, N + 4, rl.ant1[0]]]).astype(np.int32),
        ant2=np.concatenate([rl.ant2, [2, 1, rl.ant2[0]]]).astype(np.int32),
        tslot=np.concatenate([rl.tslot, [0, 0, rl.tslot[0]]]).astype(np.int32),
        uvw=np.concatenate([rl.uvw, np.ones((3, 3))]),
        flags=np.concatenate([rl.flags, np.zeros((3, F), np.uint8)]))
    vis = np.concatenate([vis, crandn(rng, 3, F, 4)])
    want = orw.canonical_from_rows(N, T, F, rl.ant1, rl.ant2, rl.tslot, rl.uvw, vis, rl.flags)
    got = _to_canonical(prob, rl, vis)
    assert np.array_equal(host(got["status"]), want[4])
    assert np.array_equal(host(got["row_map"]), want[3])
    assert np.array_equal(host(got["flags"]), want[2])
    assert np.array_equal(host(got["uvw"]), want[0])            # -0.0 == 0.0
    assert np.array_equal(host(got["vis"]), want[1])


def test_canonical_to_rows_round_trip_and_untouched_dropped_rows(cuda_device):
    import paper_1910_13908_b200 as sg
    import torch
    from tests.gpu_util import dev, host
    prob, rl = _rowlist(9, 3, 4, 1, 2, seed=7, drop_frac=0.1, swap_frac=0.5, flag_frac=0.0)
    rng = np.random.default_rng(3)
    n = len(rl.ant1)
    vis = crandn(rng, n, prob.F, 4)
    can = _to_canonical(prob, rl, vis, flags=False)
    out = torch.full((n, prob.F, 4), 7.0 + 0j, dtype=torch.complex128, device="cuda:0")
    sg.canonical_to_rows(prob.N, prob.T, prob.F, can["row_map"], can["vis"], out)
    assert np.array_equal(host(out), vis)                       # conj-transpose twice is the identity, bit for bit
    rm = host(can["row_map"]).copy()
    rm[::3] = -1
    out2 = torch.full((n, prob.F, 4), 7.0 + 0j, dtype=torch.complex128, device="cuda:0")
    sg.canonical_to_rows(prob.N, prob.T, prob.F, dev(rm), can["vis"], out2)
    o2 = host(out2)
    assert np.all(o2[::3] == 7.0) and np.array_equal(o2[rm >= 0], vis[rm >= 0])


@pytest.mark.parametrize("scalar", [False, True])
def test_apply_flags_zeroes_exactly_the_flagged_samples(cuda_device, scalar):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host
    N, T, F, K = 11, 3, 5, 3
    rows = T * N * (N - 1) // 2
    rng = np.random.default_rng(9)
    coh = crandn(rng, K, rows, F) if scalar else crandn(rng, K, rows, F, 4)
    vis = crandn(rng, rows, F, 4)
    fl = (rng.random((rows, F)) < 0.3).astype(np.uint8) * 5     # any non-zero byte flags
    cd, vd = dev(coh), dev(vis)
    sg.apply_flags(N, T, F, dev(fl), cd, vd, coh_format=sg.COH_SCALAR if scalar else sg.COH_FULL)
    wc, wv = coh.copy(), vis.copy()
    wc[:, fl != 0] = 0
    wv[fl != 0] = 0
    assert np.array_equal(host(cd), wc) and np.array_equal(host(vd), wv)


def _pipeline(prob, rl, vis, n_em, n_lm, mode, fmt):
    """rows -> canonical -> predict -> flags -> calibrate -> rows, all through the C ABI."""
    import paper_1910_13908_b200 as sg
    import torch
    from tests.gpu_util import dev, host
    can = _to_canonical(prob, rl, vis)
    src = {k: dev(getattr(prob, k)) for k in ("src_l", "src_m", "src_I", "src_alpha", "src_Q", "src_U", "src_V")}
    coh = sg.predict_coherencies(prob.N, prob.T, prob.freqs, prob.f0, can["uvw"], prob.cluster_offset, src["src_l"],
                                 src["src_m"], src["src_I"], src["src_alpha"], src["src_Q"], src["src_U"],
                                 src["src_V"], coh_format=fmt)
    sg.apply_flags(prob.N, prob.T, prob.F, can["flags"], coh, None, coh_format=fmt)   # vis is already zero there
    got = sg.sage_calibrate(prob.N, prob.T, prob.F, can["vis"], coh, dev(prob.jones_init()), n_em, n_lm, prob.tau,
                            coh_format=fmt, lm_mode=mode)
    res = torch.zeros((len(rl.ant1), prob.F, 4), dtype=torch.complex128, device="cuda:0")
    sg.canonical_to_rows(prob.N, prob.T, prob.F, can["row_map"], got["residual"], res)
    return dict(jones=host(got["jones"]), cost_per_cluster=host(got["cost_per_cluster"]),
                cost_trace=host(got["cost_trace"]), residual=host(res), status=host(can["status"]))


def _oracle(prob, rl, n_em, n_lm):
    coh = orw.predict_rows(prob, rl.uvw)
    vis = orw.simulate_rows(coh, prob.jones_true, rl.ant1, rl.ant2, rl.noise)
    want = orw.sage_rows(prob.N, rl.ant1, rl.ant2, rl.flags, vis, coh, prob.jones_init(), n_em, n_lm, prob.tau)
    assert want["min_abs_rho"] > 1e-6, "seed has an accept/reject decision within rounding of 0: not a parity seed"
    return vis, want


def _compare(want, got):
    cpc_err = np.max(np.abs(got["cost_per_cluster"] - want["cost_per_cluster"]) / want["cost_per_cluster"])
    assert cpc_err < TOL, cpc_err
    assert rel_max(got["cost_trace"], want["cost_trace"]) < TOL
    assert rel_l2(got["jones"], want["jones"]) < TOL
    assert rel_l2(got["residual"], want["residual"]) < TOL


@pytest.mark.parametrize("mode", ["compressed", "direct"])
@pytest.mark.parametrize("case", [
    dict(N=8, T=5, F=2, K=1, S=3, pol=False, scalar=False),
    dict(N=14, T=4, F=3, K=3, S=4, pol=True, scalar=False),
    dict(N=37, T=3, F=8, K=2, S=3, pol=False, scalar=True),
    dict(N=40, T=3, F=4, K=2, S=3, pol=True, scalar=False),
])
def test_row_list_calibration_matches_the_row_list_oracle(cuda_device, case, mode):
    import paper_1910_13908_b200 as sg
    prob, rl = _rowlist(case["N"], case["T"], case["F"], case["K"], case["S"], seed=300 + case["N"],
                        polarised=case["pol"], drop_frac=0.15, swap_frac=0.4, flag_frac=0.1)
    vis, want = _oracle(prob, rl, 2, 5)
    got = _pipeline(prob, rl, vis, 2, 5, {"compressed": sg.LM_COMPRESSED, "direct": sg.LM_DIRECT}[mode],
                    sg.COH_SCALAR if case["scalar"] else sg.COH_FULL)
    assert got["status"][3] == prob.rows - len(rl.ant1) and not got["status"][:3].any()
    _compare(want, got)
    assert np.all(got["residual"][rl.flags != 0] == 0)


def test_fully_flagged_station_keeps_its_start_jones(cuda_device):
    """Degenerate case: every row of one station is absent.  Its gradient and J^H J block are exactly zero, the 2x2
    solve is G (0 + mu I)^-1 = 0, so its Jones must come back as the start value, bit for bit, on both sides."""
    import paper_1910_13908_b200 as sg
    prob, rl = _rowlist(10, 4, 2, 1, 3, seed=55, drop_frac=0.0, swap_frac=0.3, flag_frac=0.05)
    dead = 4
    keep = (rl.ant1 != dead) & (rl.ant2 != dead)
    import dataclasses
    rl = dataclasses.replace(rl, **{f.name: getattr(rl, f.name)[keep] for f in dataclasses.fields(rl)})
    vis, want = _oracle(prob, rl, 1, 6)
    got = _pipeline(prob, rl, vis, 1, 6, sg.LM_COMPRESSED, sg.COH_FULL)
    _compare(want, got)
    assert np.array_equal(got["jones"][0, dead], np.eye(2)) and np.array_equal(want["jones"][0, dead], np.eye(2))


def test_rows_front_end_at_the_bench_size(cuda_device):
    """configs[4]'s shape (2.6 M slots x 8 channels), the row list bench.py --rows times.  The loop oracle is too slow
    here, so: everything that is index work is checked in full against the generator's own bookkeeping (which slot a
    row belongs to, whether it was swapped), the sample contents on 4096 sampled rows and on sampled empty slots, and
    the round trip back to row order bit for bit."""
    import paper_1910_13908_b200 as sg
    import torch
    from tests.gpu_util import dev, host
    prob = si.make_config(4)
    rl = si.make_rowlist(prob, seed=prob.seed + 1000, drop_frac=0.05, swap_frac=0.3, flag_frac=0.05)
    n, F = len(rl.ant1), prob.F
    vis = rl.noise                                             # any content will do: this is index work
    can = _to_canonical(prob, rl, vis)
    swapped = rl.ant1 > rl.ant2
    assert np.array_equal(host(can["row_map"]), 2 * rl.canonical_row + swapped)
    st = host(can["status"])
    assert list(st[:3]) == [0, 0, 0] and st[3] == prob.rows - n
    fl_c = host(can["flags"])
    want_fl = np.ones((prob.rows, F), np.uint8)
    want_fl[rl.canonical_row] = rl.flags
    assert np.array_equal(fl_c, want_fl)
    rng = np.random.default_rng(8)
    pick = np.sort(rng.choice(n, 4096, replace=False))
    slots = torch.from_numpy(rl.canonical_row[pick]).to("cuda:0")
    got_v, got_u = host(can["vis"][slots]), host(can["uvw"][slots])
    want_v = np.where(swapped[pick, None, None], vis[pick][:, :, [0, 2, 1, 3]].conj(), vis[pick])
    want_v = np.where(rl.flags[pick][:, :, None] != 0, 0.0, want_v)
    assert np.array_equal(got_v, want_v)
    assert np.array_equal(got_u, prob.uvw[rl.canonical_row[pick]])        # the swap negated uvw back
    empty = np.setdiff1d(np.arange(prob.rows), rl.canonical_row)[:2048]
    e_d = torch.from_numpy(empty).to("cuda:0")
    assert not host(can["vis"][e_d]).any() and not host(can["uvw"][e_d]).any()
    back = torch.zeros((n, F, 4), dtype=torch.complex128, device="cuda:0")
    sg.canonical_to_rows(prob.N, prob.T, F, can["row_map"], can["vis"], back)
    got_b = host(back[torch.from_numpy(pick).to("cuda:0")])
    assert np.array_equal(got_b, np.where(rl.flags[pick][:, :, None] != 0, 0.0, vis[pick]))
    del can, back
    torch.cuda.empty_cache()
