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
