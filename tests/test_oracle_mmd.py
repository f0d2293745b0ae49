"""Pins for oracle/mmd.py (Fig. 2 step 4, L47: MMD between the simulated and the observed stream as the
loss; reading R20 for the kernel and estimator the paper does not print)."""
import numpy as np
import pytest

from oracle import mmd as M

SIG = np.array([0.5, 0.7, 0.3, 0.02, 0.03, 0.01])


def _cloud(n, seed, shift=0.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = rng.normal(0, 0.4, (n, 3)) + np.array([12.4, 0.0, 1.5]) + shift
    vel = rng.normal(0, 0.02, (n, 3)) + np.array([0.0, 0.21, 0.05])
    return pos, vel


def test_identical_clouds_have_zero_mmd_and_it_is_symmetric_and_non_negative():
    xp, xv = _cloud(40, 1)
    yp, yv = _cloud(55, 2, shift=0.3)
    assert abs(M.mmd2(xp, xv, xp, xv, SIG)) <= 1e-15
    a, b = M.mmd2(xp, xv, yp, yv, SIG), M.mmd2(yp, yv, xp, xv, SIG)
    assert abs(a - b) <= 1e-15 and a > 0.0


def test_one_point_against_one_point_closed_form():
    """X = {a}, Y = {b}: MMD^2 = k(a,a) + k(b,b) - 2 k(a,b) = 2 (1 - exp(-q/2)), q = sum ((a-b)/sigma)^2."""
    a = np.array([[1.0, 2.0, 3.0]]), np.array([[0.1, 0.2, 0.3]])
    b = np.array([[1.5, 2.0, 2.7]]), np.array([[0.1, 0.23, 0.3]])
    q = (0.5 / 0.5) ** 2 + (0.3 / 0.3) ** 2 + (0.03 / 0.03) ** 2                       # = 3
    assert abs(M.mmd2(a[0], a[1], b[0], b[1], SIG) - 2.0 * (1.0 - np.exp(-1.5))) <= 1e-15
    assert abs(q - 3.0) <= 1e-12
    # gradient at a: +2/(n m sigma_d^2) k (a - b)_d  (the xx term vanishes for a single point)
    gp, gv = M.mmd2_grad(a[0], a[1], b[0], b[1], SIG)
    k = np.exp(-1.5)
    np.testing.assert_allclose(gp[0], 2 * k * np.array([-0.5, 0.0, 0.3]) / SIG[:3] ** 2, rtol=1e-13, atol=1e-16)
    np.testing.assert_allclose(gv[0], 2 * k * np.array([0.0, -0.03, 0.0]) / SIG[3:] ** 2, rtol=1e-12, atol=1e-16)


def test_two_points_against_one_hand_expansion():
    """X = {0, e_x sigma_x}, Y = {0} (all other coordinates equal): with t = exp(-1/2),
    sxx = 2 + 2 t, syy = 1, sxy = 1 + t  ->  MMD^2 = (2 + 2t)/4 + 1 - (1 + t) = (1 - t)/2."""
    xp = np.array([[0.0, 0, 0], [SIG[0], 0, 0]])
    z = np.zeros((2, 3))
    val = M.mmd2(xp, z, np.zeros((1, 3)), np.zeros((1, 3)), SIG)
    assert abs(val - (1.0 - np.exp(-0.5)) / 2.0) <= 1e-15


def test_bandwidth_limits():
    xp, xv = _cloud(12, 3)
    yp, yv = _cloud(9, 4, shift=0.2)
    assert abs(M.mmd2(xp, xv, yp, yv, 1e9 * SIG)) <= 1e-14                              # k -> 1 everywhere
    assert abs(M.mmd2(xp, xv, yp, yv, 1e-9 * SIG) - (1.0 / 12 + 1.0 / 9)) <= 1e-15       # only i = i', j = j' survive


def test_translation_and_permutation_invariance():
    xp, xv = _cloud(30, 5)
    yp, yv = _cloud(25, 6, shift=0.1)
    ref = M.mmd2(xp, xv, yp, yv, SIG)
    sp, sv = np.array([3.0, -2.0, 0.5]), np.array([0.1, 0.0, -0.2])
    assert abs(M.mmd2(xp + sp, xv + sv, yp + sp, yv + sv, SIG) - ref) <= 1e-13
    perm = np.random.Generator(np.random.PCG64(7)).permutation(30)
    assert abs(M.mmd2(xp[perm], xv[perm], yp, yv, SIG) - ref) <= 1e-15
    # a 4th column (the state's mass lane) is ignored
    xp4 = np.concatenate([xp, np.full((30, 1), 7.0)], axis=1)
    assert M.mmd2(xp4, xv, yp, yv, SIG) == ref


@pytest.mark.parametrize("n,m", [(1, 1), (5, 3), (9, 11)])
def test_gradient_matches_central_finite_differences_of_the_value(n, m):
    xp, xv = _cloud(n, 10 + n)
    yp, yv = _cloud(m, 20 + m, shift=0.25)
    gp, gv = M.mmd2_grad(xp, xv, yp, yv, SIG)
    scale = max(np.abs(gp).max(), 1e-30), max(np.abs(gv).max(), 1e-30)
    for arr, g, sc, h in ((xp, gp, scale[0], 1e-5), (xv, gv, scale[1], 1e-6)):
        for i in range(n):
            for d in range(3):
                old = arr[i, d]
                arr[i, d] = old + h
                fp = M.mmd2(xp, xv, yp, yv, SIG)
                arr[i, d] = old - h
                fm = M.mmd2(xp, xv, yp, yv, SIG)
                arr[i, d] = old
                assert abs((fp - fm) / (2 * h) - g[i, d]) <= 2e-7 * sc, (i, d)


def test_gradient_sums_to_zero_when_the_other_cloud_moves_along():
    """Translation invariance in differential form: d/dX summed over the points of X equals minus the same sum over Y;
    for Y = X (where MMD^2 = 0 is the minimum) every component of the gradient vanishes."""
    xp, xv = _cloud(15, 30)
    gp, gv = M.mmd2_grad(xp, xv, xp, xv, SIG)
    assert np.abs(gp).max() <= 1e-13 and np.abs(gv).max() <= 1e-11
