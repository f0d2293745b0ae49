"""Pins for the bulge term of the oracle ("we adopt the MWPotential2014 model from galpy"; DESIGN.md
reading R21: MWPotential2014's third component is a spherical power law with exponential cut-off,
rho = A r^-alpha exp(-(r/r_c)^2), alpha = 1.8, r_c = 1.9 kpc, giving 5 % of the radial force at the solar circle)."""
import mpmath as mp
import numpy as np
import pytest
from scipy import special

from oracle import adjoint as A
from oracle import oracle as O

G = 4.4985e-12
MB, ALPHA, RC = 4.5e9, 1.8, 1.9
S = 0.5 * (3.0 - ALPHA)
AMP = MB / (2.0 * np.pi * RC ** (3.0 - ALPHA) * special.gamma(S))      # rho = AMP r^-alpha exp(-(r/rc)^2)
POT = O.Potential.make(bulge=(MB, ALPHA, RC))


def _acc(x):
    return O.ext_accel(np.array([[*x, 1.0]]), G, POT)[0]


def _phi(x):
    return O.ext_potential(np.array([[*x, 1.0]]), G, POT)[0]


@pytest.mark.parametrize("r", [0.01, 0.5, 1.9, 5.0, 12.0, 40.0])
def test_enclosed_mass_matches_40_digit_quadrature_of_the_density(r):
    mp.mp.dps = 40
    rho = lambda q: mp.mpf(AMP) * q ** (-mp.mpf(ALPHA)) * mp.e ** (-(q / mp.mpf(RC)) ** 2)       # noqa: E731
    menc = 4 * mp.pi * mp.quad(lambda q: rho(q) * q * q, [0, r / 10, r])
    x = np.array([0.6 * r, 0.0, 0.8 * r])
    a = _acc(x)
    got = -np.dot(a, x) * r / G                                           # a = -G M(<r) x / r^3  ->  M = -a.x r / G
    assert abs(got - float(menc)) <= 1e-13 * float(menc)
    assert abs(got / MB - special.gammainc(S, (r / RC) ** 2)) <= 1e-14    # the library's regularised incomplete gamma


def test_point_mass_far_field_and_power_law_core():
    x = np.array([30.0, -40.0, 0.0])                                      # r = 50 kpc, t = 692
    np.testing.assert_allclose(_acc(x), -G * MB * x / 50.0 ** 3, rtol=1e-15)
    r = 1e-4                                                              # r << r_c: M(<r) = 4 pi A r^(3-alpha) / (3-alpha)
    a = _acc(np.array([r, 0.0, 0.0]))
    assert abs(-a[0] * r * r / G / (4 * np.pi * AMP * r ** (3 - ALPHA) / (3 - ALPHA)) - 1.0) <= 1e-8
    assert np.array_equal(_acc(np.zeros(3)), np.zeros(3))                 # direction undefined at the centre: 0 (as NFW, R12)


def test_potential_zero_point_centre_and_gradient():
    assert abs(_phi(np.zeros(3)) - (-G * MB * special.gamma(S - 0.5) / (RC * special.gamma(S)))) <= 1e-15 * abs(_phi(np.zeros(3)))
    r = 1e7
    assert abs(_phi(np.array([0.0, r, 0.0])) * r / (-G * MB) - 1.0) <= 1e-15          # Phi -> -G M_b / r: no additive constant
    for x in (np.array([0.3, -0.2, 0.1]), np.array([1.0, 1.5, -0.7]), np.array([8.0, 0.0, 0.5]), np.array([-10.0, -4.0, 6.0])):
        h = 1e-4
        grad = np.array([(_phi(x + h * e) - _phi(x - h * e)) / (2 * h) for e in np.eye(3)])
        np.testing.assert_allclose(-grad, _acc(x), rtol=1e-7)


@pytest.mark.parametrize("x", [(0.3, -0.2, 0.1), (1.0, 1.5, -0.7), (3.0, 0.0, 2.0)])
def test_poisson_equation(x):
    x = np.array(x)
    h = 1e-4
    div = sum((_acc(x + h * e)[k] - _acc(x - h * e)[k]) / (2 * h) for k, e in enumerate(np.eye(3)))
    r = np.linalg.norm(x)
    rho = AMP * r ** -ALPHA * np.exp(-(r / RC) ** 2)
    assert abs(div / (-4 * np.pi * G * rho) - 1.0) <= 1e-6


def test_mwpotential2014_normalisation_five_percent_of_the_force_at_the_solar_circle():
    """galpy's MWPotential2014 gives the bulge 5 % of the radial force at R0 = 8 kpc, v_c = 220 km/s = 0.22499 kpc/Myr:
    M_b = 0.05 v_c^2 R0 / G = 4.50e9 Msun (P(0.6, 17.7) = 1 to 1e-9)."""
    a = _acc(np.array([8.0, 0.0, 0.0]))
    assert abs(-a[0] / (0.22499 ** 2 / 8.0) - 0.05) <= 5e-4


def test_terms_add_and_the_leapfrog_feels_the_bulge():
    nfw, mn = (1.0e12, 16.0), (6.8e10, 3.0, 0.28)
    p = np.array([[3.0, 1.0, -0.5, 2.0]])
    both = O.ext_accel(p, G, O.Potential.make(nfw=nfw, mn=mn, bulge=(MB, ALPHA, RC)))
    parts = O.ext_accel(p, G, O.Potential.make(nfw=nfw, mn=mn)) + O.ext_accel(p, G, POT)
    np.testing.assert_allclose(both, parts, rtol=1e-15)
    v = np.array([[0.0, 0.2, 0.0]])
    x1, _, _ = O.leapfrog_kdk(p, v, G, 0.01, 0.5, 20, O.Potential.make(nfw=nfw, mn=mn, bulge=(MB, ALPHA, RC)))
    x0, _, _ = O.leapfrog_kdk(p, v, G, 0.01, 0.5, 20, O.Potential.make(nfw=nfw, mn=mn))
    assert 1e-4 < np.linalg.norm(x1[0, :3] - x0[0, :3]) < 0.1            # pulled inwards, by the right order of magnitude


def test_adjoint_bulge_terms_match_finite_differences_of_the_forward_oracle():
    rng = np.random.Generator(np.random.PCG64(5))
    n = 6
    posm = np.concatenate([rng.normal(0, 1.5, (n, 3)) + np.array([2.0, 0.5, -0.3]), rng.uniform(1, 2, (n, 1))], axis=1)
    c = rng.normal(size=(n, 3))
    bulge = (MB, ALPHA, RC)
    gx, gp, gG = A.ext_accel_vjp(posm, c, G, bulge=bulge)
    f = lambda p, b: float(np.sum(c * O.ext_accel(p, G, O.Potential.make(bulge=b))))                # noqa: E731
    for i in range(n):
        for d in range(3):
            h = 1e-5
            pp, pm = posm.copy(), posm.copy()
            pp[i, d] += h
            pm[i, d] -= h
            assert abs((f(pp, bulge) - f(pm, bulge)) / (2 * h) - gx[i, d]) <= 1e-7 * np.abs(gx).max()
    h = 1e-4 * MB
    assert abs((f(posm, (MB + h, ALPHA, RC)) - f(posm, (MB - h, ALPHA, RC))) / (2 * h) - gp["M_b"]) <= 1e-9 * abs(gp["M_b"])
    h = 1e-6
    assert abs((f(posm, (MB, ALPHA, RC + h)) - f(posm, (MB, ALPHA, RC - h))) / (2 * h) - gp["r_c"]) <= 1e-7 * abs(gp["r_c"])
    # and through the whole leapfrog: dL/dM_b, dL/dr_c of L = sum of final coordinates
    vel = rng.normal(0, 0.1, (n, 3))
    nfw, mn = (1.0e12, 16.0), (6.8e10, 3.0, 0.28)
    lam = np.ones((n, 3))
    r = A.leapfrog_kdk_vjp(posm, vel, G, 0.05, 0.5, 6, lam, np.zeros((n, 3)), nfw=nfw, mn=mn, bulge=bulge)
    L = lambda b: float(np.sum(O.leapfrog_kdk(posm, vel, G, 0.05, 0.5, 6, O.Potential.make(nfw=nfw, mn=mn, bulge=b))[0][:, :3]))   # noqa: E731
    h = 1e-4 * MB
    assert abs((L((MB + h, ALPHA, RC)) - L((MB - h, ALPHA, RC))) / (2 * h) - r["M_b"]) <= 1e-6 * abs(r["M_b"])
    h = 1e-5
    assert abs((L((MB, ALPHA, RC + h)) - L((MB, ALPHA, RC - h))) / (2 * h) - r["r_c"]) <= 1e-6 * abs(r["r_c"])
