"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Row-list form of the calibration hot path (second part: "per-row station index arrays
(non-canonical order, flags)"), in plain numpy float64.  The rows of an interval arrive as a measurement set hands
them over: any order, either station orientation (ant1 < ant2 or ant1 > ant2), some (time slot, baseline) pairs
absent, and a per-sample flag that excludes the sample.  Everything here is the DEFINITION applied to that list
directly -- no canonical reordering, no conjugation of swapped rows, no zero filling -- so that the CUDA path's
"bring the rows into canonical order, zero what is flagged" route is tested against something that does none of it:

    model of row r, channel c   = J_{ant1[r]} C_r,c J_{ant2[r]}^H                       (BASELINE.json:5)
    cost                        = sum over UNFLAGGED samples of ||x - model||_F^2        (reading Q9 + flags)
    G_{ant1} += E A^H,  G_{ant2} += E^H T1,   M_{ant1} += A A^H,  M_{ant2} += T1^H T1    (A5-A6, unflagged samples)
    LM (A7) and SAGE-EM (A8) exactly as oracle/sagecal_oracle.c states them, on these sums.
    Output convention: the residual of a flagged sample is 0.

Pins (tests/test_oracle_rows.py, -m "not gpu"): canonical order without flags reproduces the C oracle (an independent
implementation: C loops with long-double sums) for cost, gradient, J^H J and a whole SAGE run; central finite
differences of the cost in all 8N real parameters with flags, shuffled and swapped rows; the orientation identity
(row (q,p) with x^H, C^H gives the same sums as row (p,q)); whole-row flags == deleted rows; ||dE||^2 of a
one-station perturbation D equals Re tr(D M_p D^H); noiseless recovery on an incomplete, flagged row list.
Parity unpinned: the output convention "residual of a flagged sample is 0" (a convention).

Imports nothing from paper_1910_13908_b200; coherencies of the rows come from oracle.oracle.predict_cluster.
"""
from __future__ import annotations

import numpy as np

from . import oracle as _o


def predict_rows(prob, uvw_rows):
    """Coherencies [K, n, F, 4] of the sky model of `prob` on the given uvw rows (A1-A3, any row subset/order)."""
    return _o.predict(_RowsView(prob, uvw_rows))


class _RowsView:
    """`prob` with its uvw replaced -- attribute forwarding only."""

    def __init__(self, prob, uvw):
        self._p = prob
        self.uvw = np.ascontiguousarray(uvw, dtype=np.float64)

    def __getattr__(self, name):
        return getattr(self._p, name)


def _m(a, n, F):
    return np.asarray(a, dtype=np.complex128).reshape(n, F, 2, 2)


def model_rows(coh_k, jones_k, ant1, ant2):
    """J_{ant1} C J_{ant2}^H for every row and channel: [n, F, 2, 2]."""
    n = len(ant1)
    C = _m(coh_k, n, -1)
    J = np.asarray(jones_k, dtype=np.complex128).reshape(-1, 2, 2)
    return np.einsum("rij,rfjk,rlk->rfil", J[ant1], C, J[ant2].conj())


def simulate_rows(coh, jones, ant1, ant2, noise=None):
    """V = sum_k J C_k J^H (+ noise) on the row list: [n, F, 4]."""
    n = len(ant1)
    F = np.asarray(coh[0]).size // (4 * n)
    v = np.zeros((n, F, 2, 2), np.complex128)
    for k in range(len(coh)):
        v += model_rows(coh[k], jones[k], ant1, ant2)
    v = v.reshape(n, F, 4)
    return v if noise is None else v + noise


def cost_grad_jtj_rows(N, ant1, ant2, flags, x, coh_k, jones_k):
    """A5-A6 on a row list.  flags [n, F] (non-zero = excluded) or None.  Returns (phi, G[N,2,2], M[N,2,2])."""
    n = len(ant1)
    C = _m(coh_k, n, -1)
    F = C.shape[1]
    X = _m(x, n, F)
    J = np.asarray(jones_k, dtype=np.complex128).reshape(N, 2, 2)
    w = np.ones((n, F)) if flags is None else (np.asarray(flags).reshape(n, F) == 0).astype(np.float64)
    Jp, Jq = J[ant1], J[ant2]
    T1 = np.einsum("rij,rfjk->rfik", Jp, C)                  # J_p C
    A = np.einsum("rfij,rkj->rfik", C, Jq.conj())            # C J_q^H
    E = (X - np.einsum("rij,rfjk->rfik", Jp, A)) * w[:, :, None, None]
    phi = float(np.sum(E.real ** 2 + E.imag ** 2))
    Gp = np.einsum("rfij,rfkj->rik", E, A.conj())            # E A^H       (E already carries w)
    Gq = np.einsum("rfji,rfjk->rik", E.conj(), T1)           # E^H T1
    Mp = np.einsum("rf,rfij,rfkj->rik", w, A, A.conj())      # A A^H
    Mq = np.einsum("rf,rfji,rfjk->rik", w, T1.conj(), T1)    # T1^H T1
    G = np.zeros((N, 2, 2), np.complex128)
    M = np.zeros((N, 2, 2), np.complex128)
    np.add.at(G, ant1, Gp)
    np.add.at(G, ant2, Gq)
    np.add.at(M, ant1, Mp)
    np.add.at(M, ant2, Mq)
    return phi, G, M


def lm_rows(N, ant1, ant2, flags, x, coh_k, jones_k, n_lm, tau=1e-3):
    """A7 (block-diagonal Gauss-Newton LM, Nielsen damping, readings Q1, Q12-Q14) on a row list.
    Returns (J[N,2,2], phi, min|rho|, n_accept)."""
    J = np.array(jones_k, dtype=np.complex128).reshape(N, 2, 2)
    phi, G, M = cost_grad_jtj_rows(N, ant1, ant2, flags, x, coh_k, J)
    mu = tau * max(float(np.max(M[:, 0, 0].real)), float(np.max(M[:, 1, 1].real)), 0.0)
    nu = 2.0
    min_rho, n_acc = np.inf, 0
    eye = np.eye(2)
    for _ in range(n_lm):
        D = np.empty_like(J)
        for p in range(N):
            D[p] = G[p] @ np.linalg.inv(M[p] + mu * eye)     # dJ_p = G_p (M_p + mu I)^-1
        pred = float(np.sum(G.real * D.real + G.imag * D.imag) + mu * np.sum(D.real ** 2 + D.imag ** 2))
        Jn = J + D
        phin, Gn, Mn = cost_grad_jtj_rows(N, ant1, ant2, flags, x, coh_k, Jn)
        with np.errstate(all="ignore"):
            rho = (phi - phin) / pred
        ok = np.isfinite(phin) and np.isfinite(pred) and np.isfinite(rho) and pred > 0.0 and rho > 0.0
        if np.isfinite(rho):
            min_rho = min(min_rho, abs(rho))
        if ok:
            J, G, M, phi = Jn, Gn, Mn, phin
            mu *= max(1.0 / 3.0, 1.0 - (2.0 * rho - 1.0) ** 3)
            nu = 2.0
            n_acc += 1
        else:
            mu *= nu
            nu *= 2.0
        if not mu >= 1e-300:
            mu = 1e-300
        mu = min(mu, 1e300)
        nu = min(nu, 2.0 ** 60)
    return J, phi, min_rho, n_acc


def sage_rows(N, ant1, ant2, flags, vis, coh, jones, n_em, n_lm, tau=1e-3):
    """A8 on a row list.  vis [n, F, 4]; coh [K, n, F, 4]; jones [K, N, 2, 2].
    Returns dict(jones, residual [n, F, 4] with flagged samples 0, cost_per_cluster, cost_trace, min_abs_rho)."""
    n = len(ant1)
    K = len(coh)
    F = np.asarray(vis).size // (4 * n)
    J = np.array(jones, dtype=np.complex128).reshape(K, N, 2, 2)
    w = np.ones((n, F)) if flags is None else (np.asarray(flags).reshape(n, F) == 0).astype(np.float64)
    R = np.array(vis, dtype=np.complex128).reshape(n, F, 2, 2)
    for k in range(K):
        R = R - model_rows(coh[k], J[k], ant1, ant2)

    def wnorm2(a):
        a = a * w[:, :, None, None]
        return float(np.sum(a.real ** 2 + a.imag ** 2))

    trace = [wnorm2(R)]
    cpc = np.zeros(K)
    min_rho = np.inf
    for _ in range(n_em):
        for k in range(K):
            x = R + model_rows(coh[k], J[k], ant1, ant2)                       # E-step
            J[k], cpc[k], mr, _ = lm_rows(N, ant1, ant2, flags, x, coh[k], J[k], n_lm, tau)   # M-step
            min_rho = min(min_rho, mr)
            R = x - model_rows(coh[k], J[k], ant1, ant2)
            trace.append(wnorm2(R))
    R = R * w[:, :, None, None]                                               # output convention
    return dict(jones=J, residual=R.reshape(n, F, 4), cost_per_cluster=cpc, cost_trace=np.array(trace),
                min_abs_rho=min_rho)


def canonical_from_rows(N, T, F, ant1, ant2, tslot, uvw, vis, flags):
    """What "bringing a row list into canonical order" means, row by row (index work, written as a loop):
    slot (t, min, max) receives the row (conjugate-transposed and with uvw negated if ant1 > ant2); a slot no row
    maps to is flagged and zero; flagged samples are zero; auto-correlations and out-of-range rows are dropped; of
    several rows on one slot the highest row index wins.
    Returns (uvw_c [T*B,3], vis_c [T*B,F,4], flags_c [T*B,F] uint8, row_map [n] int64 = 2*row + swapped or -1,
    status [4] = {auto-correlations, out of range, duplicates, empty slots})."""
    B = N * (N - 1) // 2
    n = len(ant1)
    uvw_c = np.zeros((T * B, 3))
    vis_c = np.zeros((T * B, F, 4), np.complex128)
    flags_c = np.ones((T * B, F), np.uint8)
    owner = np.full(T * B, -1, np.int64)
    row_map = np.full(n, -1, np.int64)
    status = np.zeros(4, np.int32)
    vis = np.asarray(vis).reshape(n, F, 4)
    for r in range(n):
        a, b, t = int(ant1[r]), int(ant2[r]), int(tslot[r])
        if not (0 <= a < N and 0 <= b < N and 0 <= t < T):
            status[1] += 1
            continue
        if a == b:
            status[0] += 1
            continue
        p, q = min(a, b), max(a, b)
        slot = t * B + p * N - p * (p + 1) // 2 + (q - p - 1)
        if owner[slot] >= 0:
            status[2] += 1
            row_map[owner[slot]] = -1
        owner[slot] = r
        row_map[r] = 2 * slot + (1 if a > b else 0)
    for slot in range(T * B):
        r = owner[slot]
        if r < 0:
            status[3] += 1
            continue
        sw = ant1[r] > ant2[r]
        uvw_c[slot] = -uvw[r] if sw else uvw[r]
        v = vis[r]
        if sw:
            v = v[:, [0, 2, 1, 3]].conj()
        fl = np.zeros(F, np.uint8) if flags is None else (np.asarray(flags)[r] != 0).astype(np.uint8)
        flags_c[slot] = fl
        vis_c[slot] = np.where(fl[:, None] != 0, 0.0, v)
    return uvw_c, vis_c, flags_c, row_map, status
