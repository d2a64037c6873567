"""Pins for the oracle's corrupt/residual (A4) and cost, gradient, per-station J^H J
(A5-A6): SURVEY.md §8(c) P3, P6, P7, P8, P9, P14.  Coherencies here are arbitrary
complex 2x2 matrices (not Hermitian, not scalar) unless the pin needs otherwise, so a
transposed or conjugated operand anywhere changes the result."""
import numpy as np
import pytest

from oracle import oracle
from sagecal_inputs import baseline_pairs, make_problem
from tests.helpers import crandn, np_model, rel_l2


def _random_case(seed, N=5, T=3, F=2):
    rng = np.random.default_rng(seed)
    B = N * (N - 1) // 2
    coh = crandn(rng, T * B, F, 4)
    x = crandn(rng, T * B, F, 4)
    J = (np.eye(2) + 0.3 * crandn(rng, N, 2, 2))
    return rng, coh, x, J


def test_p3_identity_jones_model_equals_coherency():
    """P3 (BASELINE.json:5: 'identity Jones give V=C')."""
    prob = make_problem(6, 2, 2, 3, 2, seed=3, polarised=True)
    coh = oracle.predict(prob)
    V = oracle.simulate(prob, coh, jones=prob.jones_init(), noise=False)
    assert np.array_equal(V, coh[0] + coh[1] + coh[2]) or rel_l2(V, coh.sum(0)) < 1e-15
    R = oracle.corrupt_subtract(prob.N, prob.T, prob.F, coh, prob.jones_init(), V)
    assert np.max(np.abs(R)) < 1e-13 * np.max(np.abs(V))


def test_corrupt_matches_einsum_and_index_order():
    """A4 against an independent numpy einsum over baseline_pairs: pins b(p,q) order,
    which side carries the Hermitian transpose, and the sign argument."""
    N, T, F = 5, 3, 2
    rng, coh, x, J = _random_case(21, N, T, F)
    model = np_model(N, T, F, coh, J)
    got = oracle.corrupt_accumulate(N, T, F, coh, J, -1.0, x.copy())
    assert rel_l2(got, x - model) < 1e-15
    got = oracle.corrupt_accumulate(N, T, F, coh, J, +1.0, x.copy())
    assert rel_l2(got, x + model) < 1e-15
    # mask: only the selected clusters are applied
    coh3 = np.stack([coh, 2 * coh, -0.5j * coh])
    J3 = np.stack([J, J, J])
    got = oracle.corrupt_subtract(N, T, F, coh3, J3, x, mask=[1, 0, 1])
    assert rel_l2(got, x - (1 - 0.5j) * model) < 1e-15


def test_hermitian_symmetry_of_model():
    """V_qp = V_pq^H (BASELINE.json:5): with Hermitian-symmetric coherencies C_qp = C_pq^H the
    model of the swapped baseline is the Hermitian transpose."""
    rng = np.random.default_rng(5)
    N, T, F = 2, 1, 1
    C = crandn(rng, 2, 2)
    J = np.eye(2) + 0.3 * crandn(rng, 2, 2, 2)
    v_pq = oracle.corrupt_accumulate(N, T, F, C.reshape(1, 1, 4), J, 1.0, np.zeros((1, 1, 4), complex)).reshape(2, 2)
    v_qp = oracle.corrupt_accumulate(N, T, F, C.conj().T.reshape(1, 1, 4).copy(), J[::-1].copy(), 1.0,
                                     np.zeros((1, 1, 4), complex)).reshape(2, 2)
    assert np.allclose(v_qp, v_pq.conj().T, rtol=1e-15, atol=1e-16)


def test_cost_is_frobenius_norm_of_residual():
    N, T, F = 5, 3, 2
    rng, coh, x, J = _random_case(22, N, T, F)
    phi, G, M = oracle.cost_grad_jtj(N, T, F, x, coh, J)
    E = x - np_model(N, T, F, coh, J)
    assert abs(phi - np.sum(np.abs(E) ** 2)) < 1e-13 * phi


def test_p6_gradient_by_central_finite_differences():
    """P6 (BASELINE.json:5 'finite-difference gradients'): d phi/d Re J = -2 Re G,
    d phi/d Im J = -2 Im G, for each of the 8N real parameters.  phi is evaluated with
    numpy (np_model), not with the oracle."""
    N, T, F = 5, 3, 2
    rng, coh, x, J = _random_case(23, N, T, F)
    _, G, _ = oracle.cost_grad_jtj(N, T, F, x, coh, J)

    def phi_np(Jx):
        return np.sum(np.abs(x - np_model(N, T, F, coh, Jx)) ** 2)

    h = 1e-6
    worst = 0.0
    for p in range(N):
        for i in range(2):
            for j in range(2):
                for d, part in ((1.0, "re"), (1j, "im")):
                    Jp, Jm = J.copy(), J.copy()
                    Jp[p, i, j] += h * d
                    Jm[p, i, j] -= h * d
                    fd = (phi_np(Jp) - phi_np(Jm)) / (2 * h)
                    an = -2 * (G[p, i, j].real if part == "re" else G[p, i, j].imag)
                    worst = max(worst, abs(fd - an) / max(1.0, abs(an)))
    assert worst < 1e-6


def test_p7_brute_force_jacobian_n4():
    """P7 (BASELINE.json:5 'brute force on N=4'): dense real Jacobian of
    r(theta) = [Re vec E; Im vec E] by central differences of the numpy model;
    J^T r = -[Re G; Im G]; every diagonal 8x8 block acts as D -> D M_p (A6)."""
    N, T, F = 4, 2, 2
    rng, coh, x, J = _random_case(24, N, T, F)
    _, G, M = oracle.cost_grad_jtj(N, T, F, x, coh, J)

    def rvec(theta):
        Jt = (theta[: 4 * N] + 1j * theta[4 * N:]).reshape(N, 2, 2)
        E = x - np_model(N, T, F, coh, Jt)
        return np.concatenate([E.real.ravel(), E.imag.ravel()])

    th = np.concatenate([J.real.ravel(), J.imag.ravel()])
    h = 1e-6
    Jac = np.zeros((rvec(th).size, 8 * N))
    for k in range(8 * N):  # the model is bilinear in theta: central differences are exact up to rounding
        tp, tm = th.copy(), th.copy()
        tp[k] += h
        tm[k] -= h
        Jac[:, k] = (rvec(tp) - rvec(tm)) / (2 * h)
    g = Jac.T @ rvec(th)
    want_g = -np.concatenate([G.real.ravel(), G.imag.ravel()])
    assert np.max(np.abs(g - want_g)) < 1e-8 * np.max(np.abs(g))
    H = Jac.T @ Jac
    for p in range(N):
        idx = np.concatenate([np.arange(4 * p, 4 * p + 4), 4 * N + np.arange(4 * p, 4 * p + 4)])
        Hpp = H[np.ix_(idx, idx)]
        # explicit 8x8 layout of A6: K_p = I2 (x) M_p^T, H_pp = [[Re K, -Im K], [Im K, Re K]]
        Kp = np.kron(np.eye(2), M[p].T)
        want = np.block([[Kp.real, -Kp.imag], [Kp.imag, Kp.real]])
        assert np.max(np.abs(Hpp - want)) < 1e-7 * np.max(np.abs(want))
        assert np.allclose(M[p], M[p].conj().T, rtol=1e-14, atol=1e-14)  # Hermitian
        assert np.linalg.eigvalsh(M[p]).min() > 0  # PSD (full rank here)


def test_p8_gauge_equivariance_unpolarised():
    """P8: C = c I_2, J -> J U (U unitary): phi same, G -> G U, M -> U^H M U."""
    prob = make_problem(6, 3, 2, 1, 3, seed=8, sigma=0.05)
    coh = oracle.predict(prob)[0]
    V = oracle.simulate(prob, coh[None])
    rng = np.random.default_rng(9)
    J = np.eye(2) + 0.2 * crandn(rng, prob.N, 2, 2)
    U, _ = np.linalg.qr(crandn(rng, 2, 2))
    phi, G, M = oracle.cost_grad_jtj(prob.N, prob.T, prob.F, V, coh, J)
    phi2, G2, M2 = oracle.cost_grad_jtj(prob.N, prob.T, prob.F, V, coh, J @ U)
    assert abs(phi2 - phi) < 1e-12 * phi
    assert rel_l2(G2, G @ U) < 1e-12
    assert rel_l2(M2, U.conj().T @ M @ U) < 1e-12


def test_p9_one_station_exact_least_squares():
    """P9: with the other stations fixed the problem is linear in J_p; the undamped
    block step J_p += G_p M_p^-1 zeroes G_p and lowers phi by tr(G_p M_p^-1 G_p^H)."""
    N, T, F = 5, 3, 2
    rng, coh, x, J = _random_case(25, N, T, F)
    phi, G, M = oracle.cost_grad_jtj(N, T, F, x, coh, J)
    p = 2
    J2 = J.copy()
    Minv = np.linalg.inv(M[p])
    J2[p] = J[p] + G[p] @ Minv
    phi2, G2, M2 = oracle.cost_grad_jtj(N, T, F, x, coh, J2)
    assert np.linalg.norm(G2[p]) < 1e-12 * np.linalg.norm(G[p])
    drop = np.trace(G[p] @ Minv @ G[p].conj().T).real
    assert abs((phi - phi2) - drop) < 1e-12 * phi
    assert rel_l2(M2[p], M[p]) < 1e-14  # M_p does not depend on J_p


def test_p14_flux_jones_scaling_invariance():
    """P14: fluxes * a and Jones * a^-1/2 leave V unchanged."""
    prob = make_problem(5, 2, 2, 2, 3, seed=14)
    a = 3.7
    coh = oracle.predict(prob)
    V1 = oracle.simulate(prob, coh, noise=False)
    prob.src_I = prob.src_I * a
    coh2 = oracle.predict(prob)
    V2 = oracle.simulate(prob, coh2, jones=prob.jones_true / np.sqrt(a), noise=False)
    assert rel_l2(V2, V1) < 1e-14


def test_baseline_order_helper_matches_oracle_walk():
    """The oracle's inverse b -> (p,q) walk agrees with numpy.triu_indices: one station
    with a unique Jones only touches the baselines that contain it."""
    N, T, F = 7, 1, 1
    B = N * (N - 1) // 2
    P, Q = baseline_pairs(N)
    coh = np.ones((B, 1, 4), complex)
    for s in (0, 3, 6):
        J = np.zeros((N, 2, 2), complex)
        J[s] = np.eye(2)
        Jall = np.tile(np.eye(2, dtype=complex), (N, 1, 1))
        # model with J_s = I for station s and 0 elsewhere is zero everywhere (needs both ends)
        out = oracle.corrupt_accumulate(N, T, F, coh, J, 1.0, np.zeros((B, 1, 4), complex))
        assert np.all(out == 0)
        Jall[s] = 2 * np.eye(2)
        out = oracle.corrupt_accumulate(N, T, F, coh, Jall, 1.0, np.zeros((B, 1, 4), complex))
        touched = np.abs(out[:, 0, 0]) > 1.5
        assert np.array_equal(touched, (P == s) | (Q == s))
