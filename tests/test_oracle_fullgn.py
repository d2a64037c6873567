"""Pins of the full Gauss-Newton oracle (oracle/fullgn.py).  CPU only."""
import numpy as np
import pytest

from oracle import fullgn, oracle
from sagecal_inputs import make_config, make_problem
from tests.helpers import procrustes_err


def _small(polarised, seed=3, N=4, T=2, F=2):
    p = make_problem(N, T, F, 1, 3, seed=seed, sigma=0.05, layout="disc:3000", field_deg=4.0, patch_deg=0.5,
                     polarised=polarised)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    rng = np.random.default_rng(seed)
    J = p.jones_init()[0] + 0.1 * (rng.standard_normal((N, 2, 2)) + 1j * rng.standard_normal((N, 2, 2)))
    return p, coh[0], V, J


@pytest.mark.parametrize("polarised", [False, True])
def test_normal_equations_against_finite_difference_jacobian(polarised):
    """H = Jac^T Jac and g = -Jac^T r with Jac from central differences of the residual vector r(theta) (N=4)."""
    p, C, V, J = _small(polarised)
    N, T, F = p.N, p.T, p.F
    P, Q = np.triu_indices(N, 1)

    def resid(theta):
        Jm = fullgn.unpack(theta)
        E = V.reshape(T, p.B, F, 2, 2) - np.einsum("bij,tbfjk,blk->tbfil", Jm[P], C.reshape(T, p.B, F, 2, 2), Jm[Q].conj())
        v = E.reshape(-1, 4)
        return np.concatenate([v.real, v.imag], axis=1).reshape(-1)

    th = fullgn.pack(J)
    h = 1e-6
    Jac = np.stack([(resid(th + h * e) - resid(th - h * e)) / (2 * h) for e in np.eye(th.size)], axis=1)
    r = resid(th)
    phi, g, H = fullgn.normal_equations(N, T, F, V, C, J)
    assert abs(phi - r @ r) <= 1e-12 * phi
    assert np.linalg.norm(H - Jac.T @ Jac) <= 1e-7 * np.linalg.norm(H)
    assert np.linalg.norm(g + Jac.T @ r) <= 1e-7 * np.linalg.norm(g)
    assert np.allclose(H, H.T, rtol=0, atol=1e-12 * np.abs(H).max())


def test_diagonal_blocks_and_gradient_match_the_closed_forms():
    """The (p,p) 8x8 blocks are the A6 matrix of the C oracle's M_p, g is [Re G; Im G] (two independent routes)."""
    p, C, V, J = _small(True, seed=8, N=6, T=3, F=2)
    N = p.N
    phi, g, H = fullgn.normal_equations(N, p.T, p.F, V, C, J)
    phi_c, G, M = oracle.cost_grad_jtj(N, p.T, p.F, V, C, J)
    assert abs(phi - phi_c) <= 1e-12 * phi_c
    assert np.linalg.norm(g - fullgn.pack(G)) <= 1e-12 * np.linalg.norm(g)
    for s in range(N):
        K = np.kron(np.eye(2), M[s].T)
        blk = np.block([[K.real, -K.imag], [K.imag, K.real]])
        assert np.linalg.norm(H[8 * s:8 * s + 8, 8 * s:8 * s + 8] - blk) <= 1e-12 * np.linalg.norm(blk)


def test_gauge_directions_are_null_vectors_of_H():
    """Unpolarised cluster: J_p -> J_p U leaves every visibility unchanged, so the four directions J_p X (X
    anti-Hermitian) are in the null space of the Gauss-Newton matrix at any J."""
    p, C, V, J = _small(False, seed=5, N=5)
    _, _, H = fullgn.normal_equations(p.N, p.T, p.F, V, C, J)
    for X in (np.array([[1j, 0], [0, 0]]), np.array([[0, 0], [0, 1j]]), np.array([[0, 1], [-1, 0]]),
              np.array([[0, 1j], [1j, 0]])):
        v = fullgn.pack(J @ X)
        assert np.linalg.norm(H @ v) <= 1e-10 * np.linalg.norm(H) * np.linalg.norm(v)
    w = np.linalg.eigvalsh(H)
    assert w[3] <= 1e-10 * w[-1] < w[4]


def test_noiseless_recovery_in_a_handful_of_steps():
    """P10 for the full solve: relative cost < 1e-20 and the true Jones up to a unitary within 12 trial steps
    (the block-diagonal M-step needs about 45)."""
    p = make_config(0, sigma=0.0)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh, noise=False)
    phi0 = float(np.sum(np.abs(V) ** 2))
    J, phi, _, nacc = fullgn.lm(p.N, p.T, p.F, V, coh[0], p.jones_init()[0], 12, p.tau)
    assert phi / phi0 < 1e-20
    assert procrustes_err(J, p.jones_true[0]) < 1e-12
    Jb, phib, _, _ = oracle.lm(p.N, p.T, p.F, V, coh[0], p.jones_init()[0], 12, p.tau)
    assert phib / phi0 > 1e-10                      # the block-diagonal iteration is nowhere near after 12 steps


def test_sage_fullgn_trace_is_monotone_and_beats_block_diagonal():
    p = make_config(2, N=12, K=3, T=4)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    full = fullgn.sage(p.N, p.T, p.F, V, coh, p.jones_init(), 2, 4, p.tau)
    blk = oracle.sage(p.N, p.T, p.F, V, coh, p.jones_init(), 2, 4, p.tau)
    tr = full["cost_trace"]
    assert np.all(np.diff(tr) <= 1e-12 * tr[:-1])
    assert tr[-1] < blk["cost_trace"][-1]
    assert abs(tr[0] - blk["cost_trace"][0]) <= 1e-12 * tr[0]
