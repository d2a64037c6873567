"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

numpy/ctypes front end of oracle/sagecal_oracle.c (the plain float64 CPU
statement of the hot path, see that file's header for citations and pins).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the
CUDA package paper_1910_13908_b200.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sagecal_oracle.c")
_SO = os.path.join(_HERE, "liboracle.so")
_lock = threading.Lock()
_lib = None

_c128p = np.ctypeslib.ndpointer(dtype=np.complex128, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp the C oracle into oracle/liboracle.so (idempotent)."""
    with _lock:
        stale = force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC)
        if stale:
            tmp = _SO + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-fcx-limited-range",
                   "-ffp-contract=off", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True)
            os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        i32, i64, dbl, vp = ctypes.c_int, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p
        L.oracle_num_threads.restype = i32
        L.oracle_predict_cluster.argtypes = [i64, i32, _f64p, dbl, _f64p, i32, _f64p, _f64p, _f64p,
                                             vp, vp, vp, _f64p, _c128p]
        L.oracle_predict_cluster.restype = None
        L.oracle_corrupt_accumulate.argtypes = [i32, i32, i32, _c128p, _c128p, dbl, _c128p]
        L.oracle_corrupt_accumulate.restype = None
        L.oracle_cost_grad_jtj.argtypes = [i32, i32, i32, _c128p, _c128p, _c128p,
                                           ctypes.POINTER(dbl), _c128p, _c128p]
        L.oracle_cost_grad_jtj.restype = None
        L.oracle_lm.argtypes = [i32, i32, i32, _c128p, _c128p, _c128p, i32, dbl,
                                ctypes.POINTER(dbl), ctypes.POINTER(dbl), ctypes.POINTER(i32)]
        L.oracle_lm.restype = None
        L.oracle_sage.argtypes = [i32, i32, i32, i32, _c128p, _c128p, _c128p, _c128p, i32, i32, dbl,
                                  _f64p, vp, ctypes.POINTER(dbl), ctypes.POINTER(i32)]
        L.oracle_sage.restype = None
        _lib = L
    return _lib


def num_threads() -> int:
    return int(lib().oracle_num_threads())


def _opt(a):
    if a is None:
        return None
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a.ctypes.data_as(ctypes.c_void_p), a


def predict_cluster(freqs, f0, uvw, l, m, I, Q=None, U=None, V=None, alpha=None):
    """A1-A3 for one cluster.  uvw [nrows,3] m -> coh [nrows, F, 4] complex128."""
    uvw = np.ascontiguousarray(uvw, dtype=np.float64)
    freqs = np.ascontiguousarray(freqs, dtype=np.float64)
    l, m, I = (np.ascontiguousarray(a, dtype=np.float64) for a in (l, m, I))
    alpha = np.ascontiguousarray(alpha, dtype=np.float64)
    nrows, F, S = uvw.shape[0], freqs.size, l.size
    coh = np.zeros((nrows, F, 4), dtype=np.complex128)
    keep = [_opt(Q), _opt(U), _opt(V)]
    ptr = [k[0] if k else None for k in keep]
    if nrows and S >= 0:
        lib().oracle_predict_cluster(nrows, F, freqs, float(f0), uvw.reshape(-1), S, l, m, I,
                                     ptr[0], ptr[1], ptr[2], alpha, coh.reshape(-1))
    return coh


def predict(prob, rows=None, clusters=None):
    """Coherencies of a sagecal_inputs.Problem: [K', nrows, F, 4]."""
    uvw = prob.uvw if rows is None else prob.uvw[np.asarray(rows)]
    ks = range(prob.K) if clusters is None else clusters
    out = []
    for k in ks:
        a, b = int(prob.cluster_offset[k]), int(prob.cluster_offset[k + 1])
        sl = slice(a, b)
        out.append(predict_cluster(
            prob.freqs, prob.f0, uvw, prob.src_l[sl], prob.src_m[sl], prob.src_I[sl],
            None if prob.src_Q is None else prob.src_Q[sl],
            None if prob.src_U is None else prob.src_U[sl],
            None if prob.src_V is None else prob.src_V[sl],
            prob.src_alpha[sl]))
    return np.stack(out) if out else np.zeros((0, uvw.shape[0], prob.F, 4), np.complex128)


def _j(jones):
    return np.ascontiguousarray(jones, dtype=np.complex128).reshape(-1)


def corrupt_accumulate(N, T, F, coh_k, jones_k, sign, vis):
    """A4, in place: vis += sign * J_p C J_q^H (one cluster)."""
    assert vis.dtype == np.complex128 and vis.flags.c_contiguous
    coh_k = np.ascontiguousarray(coh_k, dtype=np.complex128)
    assert coh_k.size == vis.size == T * (N * (N - 1) // 2) * F * 4
    lib().oracle_corrupt_accumulate(N, T, F, coh_k.reshape(-1), _j(jones_k), float(sign), vis.reshape(-1))
    return vis


def corrupt_subtract(N, T, F, coh, jones, vis, sign=-1.0, mask=None):
    """R = V + sign * sum_k J C J^H, clusters in index order (A4)."""
    out = np.array(vis, dtype=np.complex128, order="C", copy=True)
    for k in range(coh.shape[0]):
        if mask is None or mask[k]:
            corrupt_accumulate(N, T, F, coh[k], jones[k], sign, out)
    return out


def simulate(prob, coh=None, jones=None, noise=True):
    """V = sum_k J_true C_k J_true^H (+ noise): the generator's visibilities,
    built with the oracle's own arithmetic."""
    if coh is None:
        coh = predict(prob)
    jones = prob.jones_true if jones is None else jones
    vis = prob.noise() if noise else np.zeros((prob.rows, prob.F, 4), np.complex128)
    for k in range(prob.K):
        corrupt_accumulate(prob.N, prob.T, prob.F, coh[k], jones[k], +1.0, vis)
    return vis


def cost_grad_jtj(N, T, F, x, coh_k, jones_k):
    """A5-A6.  Returns (phi, G[N,2,2], M[N,2,2])."""
    x = np.ascontiguousarray(x, dtype=np.complex128)
    coh_k = np.ascontiguousarray(coh_k, dtype=np.complex128)
    assert coh_k.size == x.size == T * (N * (N - 1) // 2) * F * 4
    cost = ctypes.c_double(0)
    G = np.zeros(4 * N, np.complex128)
    M = np.zeros(4 * N, np.complex128)
    lib().oracle_cost_grad_jtj(N, T, F, x.reshape(-1), coh_k.reshape(-1), _j(jones_k),
                               ctypes.byref(cost), G, M)
    return cost.value, G.reshape(N, 2, 2), M.reshape(N, 2, 2)


def lm(N, T, F, x, coh_k, jones_k, n_lm, tau=1e-3):
    """A7.  Returns (J[N,2,2], phi, min|rho|, n_accept)."""
    x = np.ascontiguousarray(x, dtype=np.complex128)
    coh_k = np.ascontiguousarray(coh_k, dtype=np.complex128)
    J = np.array(jones_k, dtype=np.complex128, order="C", copy=True).reshape(-1)
    cost = ctypes.c_double(0)
    mar = ctypes.c_double(np.inf)
    nacc = ctypes.c_int(0)
    lib().oracle_lm(N, T, F, x.reshape(-1), coh_k.reshape(-1), J, int(n_lm), float(tau),
                    ctypes.byref(cost), ctypes.byref(mar), ctypes.byref(nacc))
    return J.reshape(N, 2, 2), cost.value, mar.value, nacc.value


def sage(N, T, F, vis, coh, jones, n_em, n_lm, tau=1e-3):
    """A8.  Returns dict(jones[K,N,2,2], residual, cost_per_cluster[K],
    cost_trace[n_em*K+1], min_abs_rho, n_accept)."""
    K = coh.shape[0]
    vis = np.ascontiguousarray(vis, dtype=np.complex128)
    coh = np.ascontiguousarray(coh, dtype=np.complex128)
    assert coh.size == K * vis.size
    J = np.array(jones, dtype=np.complex128, order="C", copy=True).reshape(-1)
    res = np.zeros(vis.size, np.complex128)
    cpc = np.zeros(K, np.float64)
    trace = np.zeros(n_em * K + 1, np.float64)
    mar = ctypes.c_double(np.inf)
    nacc = ctypes.c_int(0)
    lib().oracle_sage(N, T, F, K, vis.reshape(-1), coh.reshape(-1), J, res, int(n_em), int(n_lm),
                      float(tau), cpc, trace.ctypes.data_as(ctypes.c_void_p),
                      ctypes.byref(mar), ctypes.byref(nacc))
    return dict(jones=J.reshape(K, N, 2, 2), residual=res.reshape(vis.shape), cost_per_cluster=cpc,
                cost_trace=trace, min_abs_rho=mar.value, n_accept=nacc.value)
