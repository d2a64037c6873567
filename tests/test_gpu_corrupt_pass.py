"""-m gpu parity: sagecal_corrupt_subtract and sagecal_lm_cost_grad_jtj (CUDA, through the C ABI) against the
oracle on the same seeded inputs.  Tolerance 1e-10 relative for residual, cost and gradient (BASELINE.json:5),
norms as in DESIGN.md §3 Q16.  Coherencies are arbitrary complex 2x2 matrices so that a transposed or
conjugated operand fails."""
import numpy as np
import pytest

from oracle import oracle
from sagecal_inputs import make_config
from tests.helpers import crandn, np_model, rel_l2, rel_max

pytestmark = pytest.mark.gpu
TOL = 1e-10


def _case(seed, N, T, F, K=1, scalar=False):
    rng = np.random.default_rng(seed)
    B = N * (N - 1) // 2
    if scalar:
        c = crandn(rng, K, T * B, F)
        coh = np.zeros((K, T * B, F, 4), complex)
        coh[..., 0] = c
        coh[..., 3] = c
    else:
        coh = crandn(rng, K, T * B, F, 4)
    x = crandn(rng, T * B, F, 4)
    J = np.eye(2) + 0.3 * crandn(rng, K, N, 2, 2)
    return coh, x, J


# shapes: tiny; one partial warp; several column tiles with ragged last tile; F not a power of two;
# F > 128 (one station per tile, several sample chunks); N = 2
SHAPES = [(4, 2, 1), (8, 10, 1), (37, 3, 4), (70, 2, 8), (150, 2, 1), (19, 5, 3), (6, 2, 130), (2, 3, 2), (33, 7, 16)]


@pytest.mark.parametrize("N,T,F", SHAPES)
@pytest.mark.parametrize("scalar", [False, True])
def test_lm_pass_matches_oracle(cuda_device, N, T, F, scalar):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host

    coh, x, J = _case(1000 + N + F, N, T, F, 1, scalar)
    phi, G, M = oracle.cost_grad_jtj(N, T, F, x, coh[0], J[0])
    coh_d = dev(coh[0, ..., 0].copy()) if scalar else dev(coh[0])
    cost, grad, jtj = sg.lm_cost_grad_jtj(N, T, F, dev(x), coh_d, dev(J[0]),
                                          coh_format=sg.COH_SCALAR if scalar else sg.COH_FULL)
    assert abs(host(cost)[0] - phi) < TOL * phi
    assert rel_l2(host(grad), G) < TOL and rel_max(host(grad), G) < TOL
    assert rel_l2(host(jtj), M) < TOL and rel_max(host(jtj), M) < TOL
    # bit-reproducible: fixed-order reduction, no atomics
    cost2, grad2, jtj2 = sg.lm_cost_grad_jtj(N, T, F, dev(x), coh_d, dev(J[0]),
                                             coh_format=sg.COH_SCALAR if scalar else sg.COH_FULL)
    assert np.array_equal(host(grad), host(grad2)) and np.array_equal(host(jtj), host(jtj2))
    assert host(cost)[0] == host(cost2)[0]


@pytest.mark.parametrize("N,T,F,K", [(4, 2, 1, 1), (9, 3, 2, 3), (37, 3, 4, 5), (70, 2, 8, 2), (150, 1, 1, 2)])
@pytest.mark.parametrize("scalar", [False, True])
def test_corrupt_subtract_matches_oracle(cuda_device, N, T, F, K, scalar):
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host

    coh, x, J = _case(2000 + N + K, N, T, F, K, scalar)
    fmt = sg.COH_SCALAR if scalar else sg.COH_FULL
    coh_d = dev(coh[..., 0].copy()) if scalar else dev(coh)
    want = oracle.corrupt_subtract(N, T, F, coh, J, x)
    got = host(sg.corrupt_subtract(N, T, F, coh_d, dev(J), dev(x), coh_format=fmt))
    assert rel_l2(got, want) < TOL and rel_max(got, want) < TOL
    # add-back with a mask, in place
    mask = [(k % 2) == 0 for k in range(K)]
    want = oracle.corrupt_subtract(N, T, F, coh, J, x, sign=+1.0, mask=mask)
    xd = dev(x)
    out = sg.corrupt_subtract(N, T, F, coh_d, dev(J), xd, sign=+1.0, cluster_mask=mask, coh_format=fmt, out=xd)
    assert out.data_ptr() == xd.data_ptr()
    assert rel_l2(host(xd), want) < TOL
    # pure model (vis_in = NULL) against an independent einsum
    got = host(sg.corrupt_subtract(N, T, F, coh_d, dev(J), None, sign=+1.0, coh_format=fmt))
    want = sum(np_model(N, T, F, coh[k], J[k]) for k in range(K))
    assert rel_l2(got, want) < TOL


def test_corrupt_identity_jones_and_empty_mask(cuda_device):
    """P3 on the CUDA path: identity Jones give V = sum_k C_k; an all-zero mask copies the input."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host

    N, T, F, K = 7, 2, 3, 3
    coh, x, _ = _case(7, N, T, F, K)
    Jid = np.zeros((K, N, 2, 2), complex)
    Jid[..., 0, 0] = Jid[..., 1, 1] = 1
    got = host(sg.corrupt_subtract(N, T, F, dev(coh), dev(Jid), None, sign=+1.0))
    assert rel_max(got, coh.sum(0)) < 1e-15
    got = host(sg.corrupt_subtract(N, T, F, dev(coh), dev(Jid), dev(x), cluster_mask=[0, 0, 0]))
    assert np.array_equal(got, x)


def test_pass_and_corrupt_cfg2_cluster(cuda_device):
    """configs[2]-shaped data (N=64, T=20, F=4): one cluster's pass on predicted coherencies and noisy data."""
    import paper_1910_13908_b200 as sg
    from tests.gpu_util import dev, host

    p = make_config(2, K=3)
    coh = oracle.predict(p)
    V = oracle.simulate(p, coh)
    x = oracle.corrupt_subtract(p.N, p.T, p.F, coh, p.jones_true, V, mask=[0, 1, 1])
    phi, G, M = oracle.cost_grad_jtj(p.N, p.T, p.F, x, coh[0], p.jones_init()[0])
    cost, grad, jtj = sg.lm_cost_grad_jtj(p.N, p.T, p.F, dev(x), dev(coh[0]), dev(p.jones_init()[0]))
    assert abs(host(cost)[0] - phi) < TOL * phi
    assert rel_l2(host(grad), G) < TOL and rel_l2(host(jtj), M) < TOL
    cost, grad, jtj = sg.lm_cost_grad_jtj(p.N, p.T, p.F, dev(x), dev(coh[0, ..., 0].copy()), dev(p.jones_init()[0]),
                                          coh_format=sg.COH_SCALAR)
    assert abs(host(cost)[0] - phi) < TOL * phi
    assert rel_l2(host(grad), G) < TOL and rel_l2(host(jtj), M) < TOL


def test_pass_errors(cuda_device):
    import torch
    import paper_1910_13908_b200 as sg
    from paper_1910_13908_b200 import _binding as b

    L = sg.load_library()
    z = torch.zeros(64, dtype=torch.complex128, device="cuda:0")
    # workspace too small
    rc = L.sagecal_lm_cost_grad_jtj(4, 1, 1, z.data_ptr(), 0, z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(),
                                    z.data_ptr(), z.data_ptr(), 8, None)
    assert rc == -2
    # N < 2
    rc = L.sagecal_lm_cost_grad_jtj(1, 1, 1, z.data_ptr(), 0, z.data_ptr(), z.data_ptr(), z.data_ptr(), z.data_ptr(),
                                    z.data_ptr(), z.data_ptr(), 1 << 20, None)
    assert rc == -1
    assert b.workspace_bytes(b.WS_LM_PASS, 512, 20, 8) > 0


def test_lm_pass_full_size_tensor_core_form(cuda_device):
    """sagecal_lm_cost_grad_jtj at configs[4]'s shape (N=512, T=20, F=8) with general 2x2 (polarised) coherencies: the
    launch configuration of bench.py --lm direct, tensor-core form with the F = 8 fast path.  Against the oracle on
    the whole array (one cluster: its own prediction of all 20.9 M samples, then one oracle_cost_grad_jtj pass): the
    cost and the gradient and J^H J of ALL 512 stations to 1e-10; and, independently of the oracle's pass routine,
    gradient and J^H J of sampled stations against the definition written out in numpy on those stations' 511
    baselines."""
    import torch
    import paper_1910_13908_b200 as sg
    from sagecal_inputs import baseline_index, make_config
    from tests.gpu_util import dev, gpu_predict, gpu_simulate, host

    p = make_config(4, K=1, polarised=True)
    N, T, F, B = p.N, p.T, p.F, p.B
    coh_d = gpu_predict(p)
    V = gpu_simulate(p, coh_d)
    rng = np.random.default_rng(5)
    J = (np.eye(2) + 0.2 * (rng.standard_normal((N, 2, 2)) + 1j * rng.standard_normal((N, 2, 2)))).astype(np.complex128)
    Jd = dev(J)
    cost, grad, jtj = sg.lm_cost_grad_jtj(N, T, F, V, coh_d[0], Jd)
    C_or = oracle.predict(p)[0]                                               # the oracle's coherencies, all rows
    assert rel_l2(host(coh_d[0]), C_or) < 1e-10
    cost_o, G_o, M_o = oracle.cost_grad_jtj(N, T, F, host(V), C_or, J)
    assert abs(float(cost[0]) - cost_o) <= 1e-10 * cost_o
    assert rel_l2(host(grad), G_o) < 1e-10 and rel_l2(host(jtj), M_o) < 1e-10
    gs, ms = np.abs(G_o).max(), np.abs(M_o).max()
    assert np.abs(host(grad) - G_o).max() <= 1e-10 * gs and np.abs(host(jtj) - M_o).max() <= 1e-10 * ms
    del C_or
    for s in (0, 255, 511):
        others = [o for o in range(N) if o != s]
        bl = np.array([baseline_index(N, min(s, o), max(s, o)) for o in others])
        rows = (np.arange(T)[:, None] * B + bl[None, :]).reshape(-1)
        C = oracle.predict(p, rows=rows)[0].reshape(T, N - 1, F, 2, 2)            # the oracle's coherencies
        X = host(V[torch.from_numpy(rows).to(V.device)]).reshape(T, N - 1, F, 2, 2)
        G = np.zeros((2, 2), complex)
        M = np.zeros((2, 2), complex)
        for j, o in enumerate(others):
            Cm, Xm = C[:, j].reshape(-1, 2, 2), X[:, j].reshape(-1, 2, 2)
            if s < o:   # s is the row station p: E = x - J_s C J_o^H, G += E A^H, M += A A^H, A = C J_o^H
                A = Cm @ J[o].conj().T[None]
                E = Xm - J[s][None] @ A
                G += np.einsum("nij,nkj->ik", E, A.conj())
                M += np.einsum("nij,nkj->ik", A, A.conj())
            else:       # s is the column station q: E = x - J_o C J_s^H, G += E^H T1, M += T1^H T1, T1 = J_o C
                T1 = J[o][None] @ Cm
                E = Xm - T1 @ J[s].conj().T[None]
                G += np.einsum("nji,njk->ik", E.conj(), T1)
                M += np.einsum("nji,njk->ik", T1.conj(), T1)
        assert rel_l2(host(grad[s]), G) < 1e-10, s
        assert rel_l2(host(jtj[s]), M) < 1e-10, s
    del coh_d, V
    torch.cuda.empty_cache()
