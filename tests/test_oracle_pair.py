"""Pins for the oracle's pair sum (SURVEY.md 8c pin table).

Each test fixes the oracle to something other than itself: hand-derived rationals,
40-digit mpmath brute force written independently here, conservation laws, symmetry.
"""
import os
from fractions import Fraction

import mpmath
import numpy as np
import pytest

from oracle import oracle as O
from paper_2511_22468_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def test_345_triangle_matches_hand_rationals():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "pair_345_triangle.txt"))
            if l.strip() and not l.startswith("#")]
    posm = np.array([[0, 0, 0, 1], [3, 0, 0, 2], [0, 4, 0, 3]], dtype=np.float64)
    acc, S = O.pair_accel(posm, 1.0, 0.0)
    for row in rows:
        i = int(row[0])
        vals = [float(Fraction(int(row[1 + 2 * k]), int(row[2 + 2 * k]))) for k in range(4)]
        np.testing.assert_allclose(acc[i], vals[:3], rtol=0, atol=2e-16)
        assert abs(S[i] - vals[3]) <= 2e-16
    # Newton's third law, exact rationals sum to zero
    assert np.max(np.abs(np.sum(posm[:, 3:4] * acc, axis=0))) <= 1e-16


def test_softened_two_body_closed_form():
    # d = 3, eps = 4 -> (9 + 16)^{3/2} = 125 : a_0 = G m_1 * 3 / 125
    posm = np.array([[0, 0, 0, 5.0], [0, 0, 3.0, 7.0]])
    acc, S = O.pair_accel(posm, 2.0, 4.0)
    np.testing.assert_allclose(acc[0], [0, 0, 2.0 * 7.0 * 3 / 125], rtol=1e-15)
    np.testing.assert_allclose(acc[1], [0, 0, -2.0 * 5.0 * 3 / 125], rtol=1e-15)
    np.testing.assert_allclose(S, [2.0 * 7.0 * 3 / 125, 2.0 * 5.0 * 3 / 125], rtol=1e-15)


def _mp_pair(posm, G, eps):
    mpmath.mp.dps = 40
    n = posm.shape[0]
    P = [[mpmath.mpf(float(v)) for v in row] for row in posm]
    acc = np.zeros((n, 3))
    S = np.zeros(n)
    e2 = mpmath.mpf(float(eps)) ** 2
    for i in range(n):
        s = [mpmath.mpf(0)] * 3
        sn = mpmath.mpf(0)
        for j in range(n):
            if j == i:
                continue
            d = [P[j][k] - P[i][k] for k in range(3)]
            d2 = d[0] ** 2 + d[1] ** 2 + d[2] ** 2
            w = P[j][3] * (d2 + e2) ** mpmath.mpf(-1.5)
            s = [s[k] + w * d[k] for k in range(3)]
            sn += w * mpmath.sqrt(d2)
        acc[i] = [float(mpmath.mpf(float(G)) * v) for v in s]
        S[i] = float(mpmath.mpf(float(G)) * sn)
    return acc, S


@pytest.mark.parametrize("case", ["unit_cloud", "f32_rounded_12kpc"])
def test_bruteforce_mpmath(case):
    if case == "unit_cloud":
        posm, _ = W.random_cloud(48, seed=7)
        G, eps = 1.0, 0.05
    else:
        cfg = W.CONFIGS[1]
        posm, _ = W.make_state(cfg, n=64)
        posm = W.to_f32(posm).astype(np.float64)
        G, eps = float(np.float32(cfg.G)), float(np.float32(cfg.eps))
    acc, S = O.pair_accel(posm, G, eps)
    ref, Sref = _mp_pair(posm, G, eps)
    err = np.linalg.norm(acc - ref, axis=1) / Sref
    assert err.max() <= 1e-15
    np.testing.assert_allclose(S, Sref, rtol=1e-15)


def test_targets_subset_equals_rows_of_full():
    posm, _ = W.random_cloud(200, seed=3)
    full, Sf = O.pair_accel(posm, 1.3, 0.02)
    idx = W.target_subset(200, size=17, seed=5)
    sub, Ss = O.pair_accel(posm, 1.3, 0.02, targets=idx)
    assert np.array_equal(sub, full[idx]) and np.array_equal(Ss, Sf[idx])


def test_newtons_third_law():
    posm, _ = W.random_cloud(256, seed=11)
    acc, _ = O.pair_accel(posm, 1.0, 0.01)
    m = posm[:, 3:4]
    ratio = np.linalg.norm(np.sum(m * acc, axis=0)) / np.sum(m[:, 0] * np.linalg.norm(acc, axis=1))
    assert ratio <= 1e-13


def test_translation_and_permutation_invariance():
    posm, _ = W.random_cloud(128, seed=13)
    acc, S = O.pair_accel(posm, 1.0, 0.03)
    shifted = posm.copy()
    shifted[:, :3] += np.array([4.0, -8.0, 16.0])   # powers of two keep differences nearly exact
    acc_s, _ = O.pair_accel(shifted, 1.0, 0.03)
    assert (np.linalg.norm(acc_s - acc, axis=1) / S).max() <= 1e-13
    perm = np.random.Generator(np.random.PCG64(1)).permutation(128)
    acc_p, S_p = O.pair_accel(posm[perm], 1.0, 0.03)
    assert (np.linalg.norm(acc_p - acc[perm], axis=1) / S[perm]).max() <= 1e-15
    np.testing.assert_allclose(S_p, S[perm], rtol=1e-15)


def test_coincident_particles_contribute_zero_with_softening():
    posm = np.array([[1, 2, 3, 1.0], [1, 2, 3, 5.0], [2, 2, 3, 2.0]])
    acc, S = O.pair_accel(posm, 1.0, 0.5)
    one, _ = O.pair_accel(posm[[0, 2]], 1.0, 0.5)
    np.testing.assert_allclose(acc[0], one[0], rtol=1e-15)


def test_pair_equals_mn_point_mass():
    """MN with a = 0, b = eps, M = m at the origin is a Plummer-softened point mass:
    two independent code paths of the oracle must agree."""
    eps, m, G = 0.3, 2.5, 1.7
    rng = np.random.Generator(np.random.PCG64(2))
    pts = rng.normal(0, 1.0, (20, 3))
    pot = O.Potential.make(mn=(m, 0.0, eps))
    for p in pts:
        posm = np.array([[p[0], p[1], p[2], 1.0], [0, 0, 0, m]])
        a_pair, _ = O.pair_accel(posm, G, eps)
        a_ext = O.ext_accel(posm[:1], G, pot)
        np.testing.assert_allclose(a_pair[0], a_ext[0], rtol=1e-14)


def test_pair_potential_energy_is_consistent_with_force():
    """-dW/dx_k = m_k a_k (central finite difference of the diagnostic)."""
    posm, _ = W.random_cloud(24, seed=17)
    G, eps, h = 1.0, 0.1, 1e-5
    acc, _ = O.pair_accel(posm, G, eps)
    for k, c in [(0, 0), (5, 1), (23, 2)]:
        p, q = posm.copy(), posm.copy()
        p[k, c] += h
        q[k, c] -= h
        f = -(O.pair_potential_energy(p, G, eps) - O.pair_potential_energy(q, G, eps)) / (2 * h)
        assert abs(f - posm[k, 3] * acc[k, c]) <= 1e-8 * abs(posm[k, 3]) * np.linalg.norm(acc[k])


def test_degenerate_sizes():
    a, S = O.pair_accel(np.zeros((0, 4)), 1.0, 0.1)
    assert a.shape == (0, 3)
    a, S = O.pair_accel(np.array([[1.0, 2, 3, 4]]), 1.0, 0.1)
    assert np.all(a == 0) and S[0] == 0
