"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Full Gauss-Newton Levenberg-Marquardt M-step (the other reading of Q1 in §8(c):
"per-station-block J^H J ... small dense per-cluster solve" taken as the full 8N x 8N normal matrix with one
off-diagonal 8x8 block per baseline).  Plain numpy, float64, the definition written out:

  theta_p = [Re vec(J_p); Im vec(J_p)]  (row-major vec, 8 reals per station)
  r       = [Re vec(E); Im vec(E)] stacked over all samples,  E = x - J_p C J_q^H           (BASELINE.json:5)
  Jac     = d r / d theta, built per sample from the 16 basis perturbations of (J_p, J_q)
  H = Jac^T Jac,   g = -Jac^T r,   phi = r^T r
  LM (A7 with the full solve):  (H + mu I) delta = g;  J' = J + delta;  pred = delta^T (g + mu delta);
      rho = (phi - phi') / pred;  accept iff rho > 0 (all finite): mu *= max(1/3, 1 - (2 rho - 1)^3), nu = 2;
      else mu *= nu, nu *= 2.   mu0 = tau * max diag(H).  Exactly n_lm trial steps, no early exit.

Pins (tests/test_oracle_fullgn.py): H and g against a central-difference Jacobian of r(theta) on N=4; diagonal blocks and
g against the C oracle's closed forms (A5-A6); four gauge null directions of H for an unpolarised cluster; noiseless
recovery to < 1e-20 relative cost in a handful of steps.  Imports nothing from the CUDA package.
"""
from __future__ import annotations

import numpy as np

from . import oracle as _o


def _pairs(N):
    P, Q = np.triu_indices(N, 1)
    return P, Q


def _real8(dE):
    """[..., 2, 2] complex -> [..., 8] real = [Re vec; Im vec]."""
    v = dE.reshape(dE.shape[:-2] + (4,))
    return np.concatenate([v.real, v.imag], axis=-1)


def normal_equations(N, T, F, x, coh_k, J):
    """phi, g [8N], H [8N, 8N] at Jones J [N,2,2] for data x [T*B, F, 4] and coherencies coh_k [T*B, F, 4]."""
    B = N * (N - 1) // 2
    P, Q = _pairs(N)
    X = np.asarray(x, np.complex128).reshape(T, B, F, 2, 2)
    C = np.asarray(coh_k, np.complex128).reshape(T, B, F, 2, 2)
    J = np.asarray(J, np.complex128).reshape(N, 2, 2)
    H = np.zeros((8 * N, 8 * N))
    g = np.zeros(8 * N)
    phi = 0.0
    basis = np.zeros((4, 2, 2))
    for a in range(2):
        for b in range(2):
            basis[2 * a + b, a, b] = 1.0
    for bl in range(B):
        p, q = P[bl], Q[bl]
        Cb = C[:, bl].reshape(-1, 2, 2)                    # [S, 2, 2]
        Xb = X[:, bl].reshape(-1, 2, 2)
        A = Cb @ J[q].conj().T                             # C J_q^H
        T1 = J[p] @ Cb                                     # J_p C
        E = Xb - J[p] @ A
        r = _real8(E)                                      # [S, 8]
        # d E / d (J_p = e_ab) = -e_ab A ;  d E / d (J_p = i e_ab) = -i e_ab A
        dp_re = -np.einsum("kij,sjl->skil", basis, A)      # [S, 4, 2, 2]
        # d E / d (J_q = e_ab) = -T1 e_ab^H = -T1 e_ba ;  d E / d (J_q = i e_ab) = -T1 (i e_ab)^H = +i T1 e_ba
        dq_re = -np.einsum("sij,klj->skil", T1, basis)     # T1 @ basis[k].T
        Jp = np.concatenate([_real8(dp_re), _real8(1j * dp_re)], axis=1)      # [S, 8 params, 8 residuals]
        Jq = np.concatenate([_real8(dq_re), _real8(-1j * dq_re)], axis=1)
        sp, sq = slice(8 * p, 8 * p + 8), slice(8 * q, 8 * q + 8)
        H[sp, sp] += np.einsum("sar,sbr->ab", Jp, Jp)
        H[sq, sq] += np.einsum("sar,sbr->ab", Jq, Jq)
        Hpq = np.einsum("sar,sbr->ab", Jp, Jq)
        H[sp, sq] += Hpq
        H[sq, sp] += Hpq.T
        g[sp] -= np.einsum("sar,sr->a", Jp, r)
        g[sq] -= np.einsum("sar,sr->a", Jq, r)
        phi += float(np.sum(r * r))
    return phi, g, H


def pack(J):
    """[N,2,2] complex -> theta [8N]."""
    v = np.asarray(J, np.complex128).reshape(-1, 4)
    return np.concatenate([v.real, v.imag], axis=1).reshape(-1)


def unpack(theta):
    t = np.asarray(theta).reshape(-1, 8)
    return (t[:, :4] + 1j * t[:, 4:]).reshape(-1, 2, 2)


def cost(N, T, F, x, coh_k, J):
    P, Q = _pairs(N)
    B = P.size
    X = np.asarray(x, np.complex128).reshape(T, B, F, 2, 2)
    C = np.asarray(coh_k, np.complex128).reshape(T, B, F, 2, 2)
    J = np.asarray(J, np.complex128).reshape(N, 2, 2)
    E = X - np.einsum("bij,tbfjk,blk->tbfil", J[P], C, J[Q].conj())
    return float(np.sum(E.real ** 2 + E.imag ** 2))


def lm(N, T, F, x, coh_k, jones_k, n_lm, tau=1e-3):
    """Returns (J [N,2,2], phi, min|rho|, n_accept)."""
    J = np.array(jones_k, np.complex128).reshape(N, 2, 2)
    phi, g, H = normal_equations(N, T, F, x, coh_k, J)
    mu, nu = tau * float(np.max(np.diag(H))), 2.0
    min_abs_rho, n_accept = np.inf, 0
    for _ in range(n_lm):
        delta = np.linalg.solve(H + mu * np.eye(8 * N), g)
        Jn = J + unpack(delta)
        pred = float(delta @ (g + mu * delta))
        phin, gn, Hn = normal_equations(N, T, F, x, coh_k, Jn)
        rho = (phi - phin) / pred if pred != 0 else np.nan
        ok = np.isfinite(phin) and np.isfinite(pred) and np.isfinite(rho) and pred > 0.0 and rho > 0.0
        if np.isfinite(rho):
            min_abs_rho = min(min_abs_rho, abs(rho))
        if ok:
            J, phi, g, H = Jn, phin, gn, Hn
            mu *= max(1.0 / 3.0, 1.0 - (2.0 * rho - 1.0) ** 3)
            nu = 2.0
            n_accept += 1
        else:
            mu *= nu
            nu *= 2.0
        mu = min(max(mu, 1e-300), 1e300)
        nu = min(nu, 2.0 ** 60)
    return J, phi, min_abs_rho, n_accept


def sage(N, T, F, vis, coh, jones, n_em, n_lm, tau=1e-3):
    """A8 with the full Gauss-Newton M-step.  Same outputs as oracle.sage."""
    K = coh.shape[0]
    J = np.array(jones, np.complex128).reshape(K, N, 2, 2)
    R = _o.corrupt_subtract(N, T, F, coh, J, vis)
    cpc = np.zeros(K)
    trace = [float(np.sum(np.abs(R) ** 2))]
    min_abs_rho, n_accept = np.inf, 0
    for _ in range(n_em):
        for k in range(K):
            _o.corrupt_accumulate(N, T, F, coh[k], J[k], +1.0, R)          # x_k
            J[k], cpc[k], m, na = lm(N, T, F, R, coh[k], J[k], n_lm, tau)
            min_abs_rho, n_accept = min(min_abs_rho, m), n_accept + na
            _o.corrupt_accumulate(N, T, F, coh[k], J[k], -1.0, R)          # back to R
            trace.append(float(np.sum(np.abs(R) ** 2)))
    return dict(jones=J, residual=R, cost_per_cluster=cpc, cost_trace=np.array(trace), min_abs_rho=min_abs_rho,
                n_accept=n_accept)
