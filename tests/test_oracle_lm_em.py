"""Pins for the oracle's LM (A7) and SAGE-EM (A8): SURVEY.md §8(c) P10-P13.
The LM constants (tau, Nielsen rule) are conventions ('parity unpinned');
what is pinned here is that the iteration solves the problem it claims to solve."""
import numpy as np
import pytest

from oracle import oracle
from sagecal_inputs import make_config, make_problem
from tests.helpers import crandn, np_model, procrustes_err, rel_l2


def test_p10_noiseless_single_cluster_recovers_true_jones():
    """P10 (BASELINE.json:5: 'On noiseless data it must recover the true Jones up to the
    unitary ambiguity, with the cost falling to below 1e-20 relative')."""
    p = make_config(0, sigma=0.0)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh, noise=False)
    phi0 = np.sum(np.abs(V) ** 2)
    J, phi, _, nacc = oracle.lm(p.N, p.T, p.F, V, coh[0], p.jones_init()[0], 60)
    assert phi / phi0 < 1e-20
    assert procrustes_err(J, p.jones_true[0]) < 1e-12
    assert nacc >= 40


def test_p10_noiseless_multi_cluster_em_converges():
    p = make_problem(16, 10, 2, 4, 5, seed=7, sigma=0.0, layout="disc:2500", field_deg=4.0, patch_deg=0.5)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh, noise=False)
    phi0 = np.sum(np.abs(V) ** 2)
    r = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), 100, 10)
    assert r["cost_trace"][-1] / phi0 < 1e-20
    for k in range(p.K):
        assert procrustes_err(r["jones"][k], p.jones_true[k]) < 1e-12


def test_p11_p13_em_monotone_and_residual_bookkeeping():
    """P11: total cost after each M-step is non-increasing.  P13: the residual carried
    through add-back/write-back equals V - sum_k J C J^H recomputed from scratch (numpy).
    Also: cost_per_cluster[k] is ||R||^2 right after cluster k's last M-step (Q15)."""
    p = make_problem(10, 4, 3, 3, 4, seed=31, sigma=0.05, layout="disc:3000", field_deg=4.0,
                     patch_deg=0.5, polarised=True)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    r = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), 3, 5)
    tr = r["cost_trace"]
    assert np.all(np.diff(tr) <= 1e-12 * tr[:-1])
    scratch = V - sum(np_model(p.N, p.T, p.F, coh[k], r["jones"][k]) for k in range(p.K))
    assert rel_l2(r["residual"], scratch) < 1e-12
    assert abs(tr[0] - np.sum(np.abs(V - coh.sum(0)) ** 2)) < 1e-12 * tr[0]  # identity start
    K = p.K
    last = tr[1:].reshape(3, K)[-1]
    assert np.allclose(r["cost_per_cluster"], last, rtol=1e-12)


def test_p12_noise_floor_statistic():
    """P12: converged cost / (sigma^2 dof) = 1 +- few sqrt(2/dof),
    dof = 8 samples - (8N-4) K for unpolarised clusters."""
    sig = 0.01
    p = make_problem(16, 10, 2, 4, 5, seed=7, sigma=sig, layout="disc:2500", field_deg=4.0, patch_deg=0.5)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    dof = 8 * p.samples - (8 * p.N - 4) * p.K
    r = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), 30, 10)
    stat = r["cost_trace"][-1] / (sig ** 2 * dof)
    assert abs(stat - 1.0) < 4 * np.sqrt(2.0 / dof)


def test_lm_zero_iterations_and_first_step():
    """n_lm = 0 returns the start point and its cost.  One LM step from J reproduces
    J + G (M + mu I)^-1 with mu = tau max diag M, with G, M as pinned by P6/P7, and is
    the minimiser of the damped block-diagonal quadratic model: for each station the
    damped normal equations D (M_p + mu I) = G_p hold."""
    rng = np.random.default_rng(41)
    N, T, F = 6, 3, 2
    B = N * (N - 1) // 2
    coh = crandn(rng, T * B, F, 4)
    Jt = np.eye(2) + 0.1 * crandn(rng, N, 2, 2)
    x = np_model(N, T, F, coh, Jt) + 0.01 * crandn(rng, T * B, F, 4)
    J0 = np.tile(np.eye(2, dtype=complex), (N, 1, 1))
    J, phi, _, _ = oracle.lm(N, T, F, x, coh, J0, 0)
    phi0, G, M = oracle.cost_grad_jtj(N, T, F, x, coh, J0)
    assert np.array_equal(J, J0) and phi == phi0
    tau = 1e-3
    J1, phi1, mar, nacc = oracle.lm(N, T, F, x, coh, J0, 1, tau)
    mu = tau * max(M[:, 0, 0].real.max(), M[:, 1, 1].real.max())
    assert nacc == 1 and phi1 < phi0
    D = J1 - J0
    for p in range(N):
        assert rel_l2(D[p] @ (M[p] + mu * np.eye(2)), G[p]) < 1e-13


def test_lm_rejects_uphill_and_keeps_cost_monotone():
    """Accepted cost never increases, whatever tau; a huge tau (tiny steps) still descends."""
    p = make_config(0)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    prev = None
    for n in range(0, 12):
        _, phi, _, _ = oracle.lm(p.N, p.T, p.F, V, coh[0], p.jones_init()[0], n, 1e-3)
        if prev is not None:
            assert phi <= prev * (1 + 1e-14)
        prev = phi
    _, phi_small, _, _ = oracle.lm(p.N, p.T, p.F, V, coh[0], p.jones_init()[0], 3, 1e6)
    phi0, _, _ = oracle.cost_grad_jtj(p.N, p.T, p.F, V, coh[0], p.jones_init()[0])
    assert phi_small < phi0


def test_branch_margin_of_parity_seeds():
    """Q18: a parity seed is valid only if no accept/reject decision is within rounding
    of the threshold: min |rho| over all decisions > 1e-6 for the configs the GPU parity
    tests use."""
    for idx in (0, 1):
        p = make_config(idx)
        coh = oracle.predict(p)
        V = oracle.simulate(p, coh)
        r = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), p.n_em, p.n_lm, p.tau)
        assert r["min_abs_rho"] > 1e-6
