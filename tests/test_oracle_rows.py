"""-m "not gpu": pins of the row-list oracle (oracle/rows.py, second part).

Each pin is something other than the function itself: the C oracle (independent implementation) on the special case
it covers, finite differences, mathematical identities (orientation, flag == deletion), a dense-Jacobian norm,
noiseless recovery."""
import numpy as np
import pytest

import sagecal_inputs as si
from oracle import oracle as orc
from oracle import rows as orw
from tests.helpers import crandn, procrustes_err, rel_l2


def _canon_rowlist(prob):
    p, q = si.baseline_pairs(prob.N)
    a1 = np.tile(p, prob.T)
    a2 = np.tile(q, prob.T)
    ts = np.repeat(np.arange(prob.T, dtype=np.int32), prob.B)
    return a1, a2, ts


def _setup(N=6, T=3, F=2, K=1, S=3, seed=5, polarised=True, **kw):
    prob = si.make_problem(N, T, F, K, S, seed=seed, polarised=polarised, sigma=0.05)
    rl = si.make_rowlist(prob, seed=seed + 1, **kw)
    coh = orw.predict_rows(prob, rl.uvw)
    return prob, rl, coh


def test_canonical_unflagged_rows_reproduce_the_c_oracle():
    prob = si.make_problem(7, 4, 3, 1, 4, seed=11, polarised=True)
    a1, a2, _ = _canon_rowlist(prob)
    coh = orc.predict(prob)[0]
    rng = np.random.default_rng(0)
    x = crandn(rng, prob.rows, prob.F, 4)
    J = np.eye(2) + 0.3 * crandn(rng, prob.N, 2, 2)
    phi_c, G_c, M_c = orc.cost_grad_jtj(prob.N, prob.T, prob.F, x, coh, J)
    phi, G, M = orw.cost_grad_jtj_rows(prob.N, a1, a2, None, x, coh, J)
    assert abs(phi - phi_c) <= 1e-13 * phi_c
    assert rel_l2(G, G_c) < 1e-13 and rel_l2(M, M_c) < 1e-13


def test_sage_on_canonical_rows_reproduces_the_c_oracle():
    prob = si.make_problem(6, 4, 2, 2, 3, seed=21, sigma=0.02)
    a1, a2, _ = _canon_rowlist(prob)
    coh = orc.predict(prob)
    vis = orc.simulate(prob, coh)
    ref = orc.sage(prob.N, prob.T, prob.F, vis, coh, prob.jones_init(), 2, 5)
    got = orw.sage_rows(prob.N, a1, a2, None, vis, coh, prob.jones_init(), 2, 5)
    assert ref["min_abs_rho"] > 1e-6
    assert np.allclose(got["cost_per_cluster"], ref["cost_per_cluster"], rtol=1e-10)
    assert np.allclose(got["cost_trace"], ref["cost_trace"], rtol=1e-10)
    assert rel_l2(got["jones"], ref["jones"]) < 1e-10
    assert rel_l2(got["residual"], ref["residual"]) < 1e-9


def test_finite_difference_gradient_with_flags_swaps_and_gaps():
    prob, rl, coh = _setup(drop_frac=0.2, swap_frac=0.5, flag_frac=0.2)
    rng = np.random.default_rng(1)
    x = crandn(rng, len(rl.ant1), prob.F, 4)
    J = np.eye(2) + 0.3 * crandn(rng, prob.N, 2, 2)
    phi, G, _ = orw.cost_grad_jtj_rows(prob.N, rl.ant1, rl.ant2, rl.flags, x, coh[0], J)
    h = 1e-6
    for p in range(prob.N):
        for i in range(2):
            for j in range(2):
                for part in (1.0, 1j):
                    Jp, Jm = J.copy(), J.copy()
                    Jp[p, i, j] += h * part
                    Jm[p, i, j] -= h * part
                    fp = orw.cost_grad_jtj_rows(prob.N, rl.ant1, rl.ant2, rl.flags, x, coh[0], Jp)[0]
                    fm = orw.cost_grad_jtj_rows(prob.N, rl.ant1, rl.ant2, rl.flags, x, coh[0], Jm)[0]
                    fd = (fp - fm) / (2 * h)
                    g = G[p, i, j]
                    want = -2.0 * (g.real if part == 1.0 else g.imag)     # d phi = -2 Re tr(G^H dJ)
                    assert abs(fd - want) <= 1e-6 * max(1.0, abs(want)), (p, i, j, part, fd, want)


def test_row_orientation_identity():
    """Row (q,p) carrying x^H and C^H is the same measurement as row (p,q): cost, G and M must not change."""
    prob, rl, coh = _setup(drop_frac=0.0, swap_frac=0.0, flag_frac=0.1)
    rng = np.random.default_rng(2)
    n = len(rl.ant1)
    x = crandn(rng, n, prob.F, 4)
    J = np.eye(2) + 0.3 * crandn(rng, prob.N, 2, 2)
    ref = orw.cost_grad_jtj_rows(prob.N, rl.ant1, rl.ant2, rl.flags, x, coh[0], J)
    sw = rng.random(n) < 0.5
    herm = lambda a: a.reshape(n, prob.F, 4)[:, :, [0, 2, 1, 3]].conj()
    x2 = np.where(sw[:, None, None], herm(x), x)
    c2 = np.where(sw[:, None, None], herm(coh[0]), coh[0])
    b1 = np.where(sw, rl.ant2, rl.ant1)
    b2 = np.where(sw, rl.ant1, rl.ant2)
    got = orw.cost_grad_jtj_rows(prob.N, b1, b2, rl.flags, x2, c2, J)
    assert abs(got[0] - ref[0]) <= 1e-13 * ref[0]
    assert rel_l2(got[1], ref[1]) < 1e-13 and rel_l2(got[2], ref[2]) < 1e-13
    # and the coherency of the negated uvw IS C^H (pin P2 of the predict oracle), so a swapped row list is consistent
    c_neg = orw.predict_rows(prob, -rl.uvw)[0]
    assert rel_l2(c_neg, herm(coh[0])) < 1e-13


def test_whole_row_flags_equal_deleted_rows():
    prob, rl, coh = _setup(drop_frac=0.1, swap_frac=0.4, flag_frac=0.0)
    rng = np.random.default_rng(3)
    n = len(rl.ant1)
    x = crandn(rng, n, prob.F, 4)
    J = np.eye(2) + 0.3 * crandn(rng, prob.N, 2, 2)
    dead = rng.random(n) < 0.3
    fl = np.repeat(dead[:, None], prob.F, axis=1).astype(np.uint8)
    a = orw.cost_grad_jtj_rows(prob.N, rl.ant1, rl.ant2, fl, x, coh[0], J)
    k = ~dead
    b = orw.cost_grad_jtj_rows(prob.N, rl.ant1[k], rl.ant2[k], None, x[k], coh[0][k], J)
    assert abs(a[0] - b[0]) <= 1e-13 * b[0]
    assert rel_l2(a[1], b[1]) < 1e-13 and rel_l2(a[2], b[2]) < 1e-13


def test_jtj_block_is_the_norm_of_a_one_station_perturbation():
    """||d model||^2 over unflagged samples for a perturbation D of station p alone = Re tr(D M_p D^H)."""
    prob, rl, coh = _setup(drop_frac=0.2, swap_frac=0.5, flag_frac=0.2)
    rng = np.random.default_rng(4)
    J = np.eye(2) + 0.3 * crandn(rng, prob.N, 2, 2)
    n = len(rl.ant1)
    x = np.zeros((n, prob.F, 4), np.complex128)
    _, _, M = orw.cost_grad_jtj_rows(prob.N, rl.ant1, rl.ant2, rl.flags, x, coh[0], J)
    w = (rl.flags == 0)[:, :, None, None]
    for p in range(prob.N):
        D = crandn(rng, 2, 2)
        J2 = J.copy()
        J2[p] += D
        # the model is linear in J_p when only station p moves (p never pairs with itself)
        dmod = (orw.model_rows(coh[0], J2, rl.ant1, rl.ant2) - orw.model_rows(coh[0], J, rl.ant1, rl.ant2)) * w
        lhs = float(np.sum(np.abs(dmod) ** 2))
        rhs = float(np.trace(D @ M[p] @ D.conj().T).real)
        assert abs(lhs - rhs) <= 1e-12 * lhs


def test_noiseless_recovery_on_an_incomplete_flagged_row_list():
    prob = si.make_problem(8, 6, 2, 1, 3, seed=31, polarised=False)
    rl = si.make_rowlist(prob, seed=32, drop_frac=0.15, swap_frac=0.5, flag_frac=0.1)
    coh = orw.predict_rows(prob, rl.uvw)
    vis = orw.simulate_rows(coh, prob.jones_true, rl.ant1, rl.ant2)
    out = orw.sage_rows(prob.N, rl.ant1, rl.ant2, rl.flags, vis, coh, prob.jones_init(), 1, 80)
    v2 = float(np.sum(np.abs(vis * (rl.flags == 0)[:, :, None]) ** 2))
    assert out["cost_per_cluster"][0] < 1e-20 * v2
    assert procrustes_err(out["jones"][0], prob.jones_true[0]) < 1e-10
    assert np.all(out["residual"][rl.flags != 0] == 0)


def test_canonical_from_rows_bookkeeping():
    prob = si.make_problem(5, 3, 2, 1, 2, seed=41)
    rl = si.make_rowlist(prob, seed=42, drop_frac=0.2, swap_frac=0.5, flag_frac=0.2)
    n = len(rl.ant1)
    rng = np.random.default_rng(5)
    vis = crandn(rng, n, prob.F, 4)
    # append an auto-correlation, an out-of-range row and a duplicate of row 0
    a1 = np.concatenate([rl.ant1, [2, 9, rl.ant1[0]]]).astype(np.int32)
    a2 = np.concatenate([rl.ant2, [2, 1, rl.ant2[0]]]).astype(np.int32)
    ts = np.concatenate([rl.tslot, [0, 0, rl.tslot[0]]]).astype(np.int32)
    uvw = np.concatenate([rl.uvw, np.ones((3, 3))])
    v = np.concatenate([vis, crandn(rng, 3, prob.F, 4)])
    fl = np.concatenate([rl.flags, np.zeros((3, prob.F), np.uint8)])
    uvw_c, vis_c, fl_c, rmap, status = orw.canonical_from_rows(prob.N, prob.T, prob.F, a1, a2, ts, uvw, v, fl)
    assert list(status[:3]) == [1, 1, 1] and status[3] == prob.rows - n
    assert rmap[0] == -1 and rmap[n] == -1 and rmap[n + 1] == -1 and rmap[n + 2] >= 0
    ok = rmap >= 0
    # every surviving row sits in its own slot, with the generator's canonical uvw
    slots = rmap[ok] >> 1
    assert len(set(slots.tolist())) == slots.size
    keep = np.nonzero(ok)[0]
    keep = keep[keep < n]
    assert np.array_equal(rmap[keep] >> 1, rl.canonical_row[keep])
    assert np.array_equal(uvw_c[rl.canonical_row[keep]], prob.uvw[rl.canonical_row[keep]])
    empty = np.ones(prob.rows, bool)
    empty[slots] = False
    assert np.all(fl_c[empty] == 1) and np.all(vis_c[empty] == 0) and np.all(vis_c[fl_c != 0] == 0)
