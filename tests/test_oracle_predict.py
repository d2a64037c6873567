"""Pins for the oracle's coherency prediction (A1-A3): SURVEY.md §8(c) P1, P2, P4, P5
plus a DFT special case.  None of these re-types the oracle's loop: each fixes the
result through a closed form, an invariant or a library routine (numpy.fft)."""
import numpy as np
import pytest

from oracle import oracle
from sagecal_inputs import C0, make_problem

F0 = 150e6


def _uvw(rng, n, scale=3000.0):
    return rng.uniform(-scale, scale, (n, 3))


def test_p1_single_source_at_phase_centre_gives_brightness():
    """P1 (BASELINE.json:5: 'a single source at l=m=0 gives C equal to its brightness
    matrix on every baseline').  Polarised source pins the matrix layout of Q4:
    XX=I+Q, XY=U+iV, YX=U-iV, YY=I-Q, and the (f/f0)^alpha law of Q5."""
    rng = np.random.default_rng(1)
    freqs = np.array([120e6, 150e6, 187.5e6])
    I, Q, U, V, alpha = 3.0, 0.4, -0.25, 0.125, -0.7
    coh = oracle.predict_cluster(freqs, F0, _uvw(rng, 37), [0.0], [0.0], [I], [Q], [U], [V], [alpha])
    B = np.array([I + Q, U + 1j * V, U - 1j * V, I - Q])
    for c, f in enumerate(freqs):
        want = B * (f / F0) ** alpha
        assert np.allclose(coh[:, c, :], want[None, :], rtol=4e-16, atol=0)
    # at f = f0 the scale is exactly 1: bit-exact brightness
    assert np.array_equal(coh[:, 1, :], np.broadcast_to(B, (37, 4)))


def test_p2_swapping_p_and_q_gives_hermitian_conjugate():
    """P2: negating uvw (baseline q-p instead of p-q) gives C^H (V_qp = V_pq^H)."""
    rng = np.random.default_rng(2)
    S = 5
    l, m = rng.uniform(-0.05, 0.05, (2, S))
    I = rng.uniform(1, 10, S)
    Q, U, V = (I * rng.uniform(-0.3, 0.3, S) for _ in range(3))
    al = rng.uniform(-1, 0, S)
    freqs = np.array([140e6, 160e6])
    uvw = _uvw(rng, 50)
    a = oracle.predict_cluster(freqs, F0, uvw, l, m, I, Q, U, V, al).reshape(50, 2, 2, 2)
    b = oracle.predict_cluster(freqs, F0, -uvw, l, m, I, Q, U, V, al).reshape(50, 2, 2, 2)
    assert np.array_equal(b, np.conj(np.swapaxes(a, -1, -2)))


def test_p4_integer_phase_and_cosine_pair():
    """P4: (a) uvw chosen so that the phase is an integer number of cycles -> C = B_s;
    (b) two equal sources at +-(l,m) on w=0 baselines -> C = 2 I cos(2 pi (ul+vm) f/c0) I_2."""
    f = 150e6
    lam = C0 / f
    l0 = 0.03125  # exactly representable
    k = np.arange(-8, 9, dtype=np.float64)
    uvw = np.zeros((k.size, 3))
    uvw[:, 0] = k * lam / l0  # u*l*f/c0 = k up to rounding of lam
    coh = oracle.predict_cluster([f], f, uvw, [l0], [0.0], [2.5], None, None, None, [0.0])
    assert np.allclose(coh[:, 0, 0], 2.5, rtol=0, atol=1e-12)
    assert np.allclose(coh[:, 0, 3], 2.5, rtol=0, atol=1e-12)
    assert np.all(coh[:, 0, 1] == 0) and np.all(coh[:, 0, 2] == 0)

    rng = np.random.default_rng(4)
    uvw = _uvw(rng, 64)
    uvw[:, 2] = 0.0
    l, m = 0.0123, -0.0345
    coh = oracle.predict_cluster([f], f, uvw, [l, -l], [m, -m], [1.75, 1.75], None, None, None, [0.0, 0.0])
    want = 2 * 1.75 * np.cos(2 * np.pi * (uvw[:, 0] * l + uvw[:, 1] * m) * f / C0)
    assert np.allclose(coh[:, 0, 0].real, want, rtol=0, atol=2e-12)
    assert np.max(np.abs(coh[:, 0, 0].imag)) < 1e-15
    assert np.array_equal(coh[:, 0, 0], coh[:, 0, 3])


def test_w_term_sign_and_n_minus_1():
    """u=v=0: C = I exp(-2 pi i (f/c0) w (n-1)), n = sqrt(1-l^2-m^2) (Q2: minus sign, w(n-1),
    no 1/n factor).  Pins the w term that the other closed forms do not see."""
    f = 150e6
    l, m = 0.09, -0.04
    n = np.sqrt(np.longdouble(1) - np.longdouble(l) ** 2 - np.longdouble(m) ** 2)
    w = np.array([0.0, 10.0, -250.0, 4321.0])
    uvw = np.zeros((4, 3))
    uvw[:, 2] = w
    coh = oracle.predict_cluster([f], f, uvw, [l], [m], [1.0], None, None, None, [0.0])
    ph = -2 * np.pi * np.longdouble(f) / np.longdouble(C0) * w.astype(np.longdouble) * (n - 1)
    want = (np.cos(ph) + 1j * np.sin(ph)).astype(np.complex128)
    assert np.allclose(coh[:, 0, 0], want, rtol=0, atol=1e-12)
    assert coh[1, 0, 0].imag > 0  # (n-1) < 0, w > 0: phase is positive


def test_dft_special_case_matches_numpy_fft():
    """Sources on a regular l-grid, baselines on the reciprocal u-grid, v=w=0, m=0:
    C(u_k) = sum_j I_j exp(-2 pi i j k / n) = numpy.fft.fft(I)[k]   (library routine)."""
    n = 16
    f = 150e6
    dl = 1.0 / 1024.0
    l = np.arange(n) * dl
    rng = np.random.default_rng(7)
    I = rng.uniform(0.5, 2.0, n)
    k = np.arange(n)
    uvw = np.zeros((n, 3))
    uvw[:, 0] = k / (n * dl) * (C0 / f)
    # w must not contribute: w = 0.  n-1 != 0 for l != 0 but is multiplied by w = 0.
    coh = oracle.predict_cluster([f], f, uvw, l, np.zeros(n), I, None, None, None, np.zeros(n))
    want = np.fft.fft(I)
    assert np.allclose(coh[:, 0, 0], want, rtol=0, atol=1e-11)


def test_p5_brute_force_long_double_direct_sum():
    """P5: N=4, T=2, F=2, S=3.  Direct, un-reduced evaluation of the defining sum in
    numpy long double with n-1 formed as sqrt(1-l^2-m^2)-1 (the textbook form)."""
    prob = make_problem(4, 2, 2, 1, 3, seed=5, polarised=True, field_deg=4.0)
    coh = oracle.predict(prob)[0]
    ld = np.longdouble
    l, m = prob.src_l.astype(ld), prob.src_m.astype(ld)
    n1 = np.sqrt(ld(1) - l * l - m * m) - ld(1)
    u, v, w = (prob.uvw[:, i].astype(ld) for i in range(3))
    two_pi = 2 * np.arctan2(ld(0), ld(-1))
    for c, f in enumerate(prob.freqs):
        acc = np.zeros((prob.rows, 4), dtype=np.clongdouble)
        for s in range(3):
            ph = -two_pi * (ld(f) / ld(C0)) * (u * l[s] + v * m[s] + w * n1[s])
            e = np.cos(ph) + 1j * np.sin(ph)
            sc = (ld(f) / ld(prob.f0)) ** ld(prob.src_alpha[s])
            I, Q, U, V = (ld(a[s]) for a in (prob.src_I, prob.src_Q, prob.src_U, prob.src_V))
            bright = np.array([I + Q, U + 1j * V, U - 1j * V, I - Q], dtype=np.clongdouble)
            acc += sc * e[:, None] * bright[None, :]
        # sqrt(1-r^2)-1 loses ~1e-16/|n-1| relative digits; |w| <= 2 km -> 1e-12 abs is ample
        assert np.allclose(coh[:, c, :], acc.astype(np.complex128), rtol=0, atol=1e-11)


def test_unpolarised_cluster_is_scalar_times_identity():
    """A10: Q=U=V=0 -> C = c I_2 exactly (off-diagonals exactly zero, diagonals equal)."""
    prob = make_problem(6, 3, 2, 2, 4, seed=11)
    coh = oracle.predict(prob)
    assert np.all(coh[..., 1] == 0) and np.all(coh[..., 2] == 0)
    assert np.array_equal(coh[..., 0], coh[..., 3])
    # passing explicit zeros for Q, U, V is the same thing
    z = np.zeros(4)
    c2 = oracle.predict_cluster(prob.freqs, prob.f0, prob.uvw, prob.src_l[:4], prob.src_m[:4],
                                prob.src_I[:4], z, z, z, prob.src_alpha[:4])
    assert np.array_equal(c2, coh[0])


def test_rows_are_independent_and_empty_inputs():
    prob = make_problem(5, 2, 3, 1, 3, seed=12)
    full = oracle.predict(prob)[0]
    rows = np.array([7, 0, 19, 3])
    part = oracle.predict(prob, rows=rows)[0]
    assert np.array_equal(part, full[rows])
    empty = oracle.predict_cluster(prob.freqs, prob.f0, np.zeros((0, 3)), [0.0], [0.0], [1.0], alpha=[0.0])
    assert empty.shape == (0, 3, 4)
    nosrc = oracle.predict_cluster(prob.freqs, prob.f0, prob.uvw, [], [], [], alpha=[])
    assert np.all(nosrc == 0)
