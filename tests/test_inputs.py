"""The seeded generator: shapes of BASELINE.json:7-11, determinism, conventions."""
import numpy as np

from sagecal_inputs import C0, CONFIGS, SEED_BASE, baseline_index, baseline_pairs, make_config, make_problem, noise_rows


def test_config_shapes_match_survey_table():
    want = {0: (8, 28, 280, 280, 840), 1: (64, 2016, 40320, 40320, 806400),
            2: (64, 2016, 40320, 161280, 161280000)}
    for idx, (N, B, rows, samples, vs) in want.items():
        p = make_config(idx)
        assert (p.N, p.B, p.rows, p.samples, p.vis_src) == (N, B, rows, samples, vs)
        assert p.uvw.shape == (rows, 3) and p.jones_true.shape == (p.K, N, 2, 2)
        assert p.seed == SEED_BASE + idx
    # sizes of the large configs without generating them
    for idx, vs in ((3, 2.6112e9), (4, 4.1861e10)):
        c = CONFIGS[idx]
        samples = c["T"] * c["N"] * (c["N"] - 1) // 2 * c["F"]
        assert abs(samples * c["K"] * c["S"] / vs - 1) < 1e-4


def test_determinism_and_stream_independence():
    a, b = make_config(1), make_config(1)
    assert a.sha256() == b.sha256()
    c = make_config(1, sigma=0.5)  # sigma does not disturb the other draws
    assert np.array_equal(a.uvw, c.uvw) and np.array_equal(a.jones_true, c.jones_true)
    n1 = a.noise()
    assert n1.shape == (a.rows, a.F, 4) and n1.dtype == np.complex128
    assert abs(n1.real.std() / a.sigma - 1) < 0.02 and abs(n1.imag.std() / a.sigma - 1) < 0.02
    rows = np.array([0, 5, a.B, a.rows - 1, 2 * a.B + 17])
    assert np.array_equal(noise_rows(a, rows), n1[rows])


def test_baseline_order_and_uvw_antisymmetry():
    N = 9
    P, Q = baseline_pairs(N)
    for b, (p, q) in enumerate(zip(P, Q)):
        assert p < q and baseline_index(N, int(p), int(q)) == b
    p = make_problem(N, 3, 1, 1, 2, seed=3)
    uvw = p.uvw.reshape(3, -1, 3)
    # closure: uvw(0,2) = uvw(0,1) + uvw(1,2) for the position(p) - position(q) convention (Q3)
    i01, i12, i02 = baseline_index(N, 0, 1), baseline_index(N, 1, 2), baseline_index(N, 0, 2)
    assert np.allclose(uvw[:, i02], uvw[:, i01] + uvw[:, i12], atol=1e-9)
    # baseline length is preserved by the rotation
    st = p.stations_en
    L = np.linalg.norm(st[P] - st[Q], axis=1)
    assert np.allclose(np.linalg.norm(uvw, axis=2), L[None, :], rtol=1e-12)


def test_channel_centres_and_value_ranges():
    assert np.allclose(make_config(2).freqs, [142.5e6, 147.5e6, 152.5e6, 157.5e6])  # Q6
    assert make_config(0).freqs.tolist() == [150e6]
    p = make_config(2)
    r = np.hypot(p.src_l, p.src_m)
    assert r.max() < np.sin(np.deg2rad(5.6)) and p.src_I.min() >= 0.1 and p.src_I.max() <= 50.0
    assert np.abs(p.uvw).max() <= 30000.0 * 1.0001
    assert np.all(p.src_alpha == -0.7) and p.f0 == 150e6
    assert np.array_equal(p.cluster_offset, np.arange(51) * 20)
