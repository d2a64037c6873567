"""Independent numpy helpers for the pins (no oracle code, no CUDA code)."""
import numpy as np

from sagecal_inputs import baseline_pairs


def crandn(rng, *shape):
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / np.sqrt(2.0)


def np_model(N, T, F, coh, jones):
    """J_p C J_q^H by einsum.  coh [T*B,F,4] -> [T*B,F,4]."""
    P, Q = baseline_pairs(N)
    B = P.size
    C = coh.reshape(T, B, F, 2, 2)
    J = jones.reshape(N, 2, 2)
    out = np.einsum("bij,tbfjk,blk->tbfil", J[P], C, J[Q].conj())
    return out.reshape(T * B, F, 4)


def rel_l2(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


def rel_max(a, b):
    a = np.asarray(a).ravel()
    b = np.asarray(b).ravel()
    mb = np.max(np.abs(b)) if b.size else 0.0
    return (np.max(np.abs(a - b)) if a.size else 0.0) / (mb if mb > 0 else 1.0)


def procrustes_err(Je, Jt):
    """Relative Jones error after removing the unitary ambiguity (Q17):
    U = W Z^H from the SVD of sum_p Je_p^H Jt_p."""
    W, _, Zh = np.linalg.svd(np.einsum("pji,pjk->ik", Je.conj(), Jt))
    U = W @ Zh
    return np.linalg.norm(Je @ U - Jt) / np.linalg.norm(Jt)
