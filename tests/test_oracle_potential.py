"""Pins for the oracle's NFW + Miyamoto-Nagai terms.

The paper names the components but prints no formula; the pins are mathematics:
acceleration = -grad(potential) by central differences, Poisson's equation against the
textbook densities (fixes the NFW normalisation, reading R10), circular speed,
in-plane MN closed form, spherical symmetry / axisymmetry.
"""
import os

import numpy as np
import pytest

from oracle import oracle as O
from paper_2511_22468_b200 import workloads as W

G = W.G_KPC_MSUN_MYR
NFW = O.Potential.make(nfw=W.NFW_MW)
MN = O.Potential.make(mn=W.MN_MW)
BOTH = O.Potential.make(nfw=W.NFW_MW, mn=W.MN_MW)
POINTS = np.array([[12.4, 0.0, 1.5], [-10.0, -4.0, 6.0], [8.0, 0.0, 0.0], [0.3, -0.2, 0.05], [1.0, 2.0, -3.0]])


def _posm(pts):
    pts = np.atleast_2d(np.asarray(pts, dtype=np.float64))
    return np.concatenate([pts, np.ones((pts.shape[0], 1))], axis=1)


def _fd_grad(pot, x, h):
    g = np.zeros(3)
    for k in range(3):
        p, q = np.array(x, dtype=np.float64), np.array(x, dtype=np.float64)
        p[k] += h
        q[k] -= h
        g[k] = (O.ext_potential(_posm(p), G, pot)[0] - O.ext_potential(_posm(q), G, pot)[0]) / (2 * h)
    return g


@pytest.mark.parametrize("pot", [NFW, MN, BOTH], ids=["nfw", "mn", "both"])
def test_acceleration_is_minus_gradient_of_potential(pot):
    for x in POINTS:
        a = O.ext_accel(_posm(x), G, pot)[0]
        g = _fd_grad(pot, x, 1e-5 * np.linalg.norm(x))   # truncation ~1e-10, rounding ~1e-11
        assert np.linalg.norm(a + g) <= 1e-8 * np.linalg.norm(a)


def _fd_div(pot, x, h):
    d = 0.0
    for k in range(3):
        p, q = np.array(x, dtype=np.float64), np.array(x, dtype=np.float64)
        p[k] += h
        q[k] -= h
        d += (O.ext_accel(_posm(p), G, pot)[0][k] - O.ext_accel(_posm(q), G, pot)[0][k]) / (2 * h)
    return d


def test_poisson_nfw_fixes_the_normalisation():
    """div a = -4 pi G rho with rho_NFW = M_s / (4 pi r_s^3) / (c (1+c)^2): M_s = 4 pi rho_0 r_s^3."""
    Ms, rs = W.NFW_MW
    for x in POINTS:
        c = np.linalg.norm(x) / rs
        rho = Ms / (4 * np.pi * rs ** 3) / (c * (1 + c) ** 2)
        assert abs(_fd_div(NFW, x, 1e-4 * np.linalg.norm(x)) + 4 * np.pi * G * rho) <= 1e-6 * 4 * np.pi * G * rho


def test_poisson_mn():
    M, a, b = W.MN_MW
    for x in POINTS:
        R2, B = x[0] ** 2 + x[1] ** 2, np.sqrt(x[2] ** 2 + b * b)
        rho = (b * b * M / (4 * np.pi)) * (a * R2 + (a + 3 * B) * (a + B) ** 2) / ((R2 + (a + B) ** 2) ** 2.5 * B ** 3)
        assert abs(_fd_div(MN, x, 1e-5 * np.linalg.norm(x)) + 4 * np.pi * G * rho) <= 1e-6 * 4 * np.pi * G * rho


def test_nfw_circular_speed_and_symmetry():
    Ms, rs = W.NFW_MW
    r = 12.49
    c = r / rs
    vc2 = G * Ms * (np.log(1 + c) - c / (1 + c)) / r
    assert abs(np.sqrt(vc2) - 0.223399) <= 2e-6         # kpc/Myr (218.44 km/s), SURVEY 8c
    rng = np.random.Generator(np.random.PCG64(4))
    for _ in range(5):
        u = rng.normal(size=3)
        u /= np.linalg.norm(u)
        a = O.ext_accel(_posm(r * u), G, NFW)[0]
        np.testing.assert_allclose(a, -vc2 / r * u, rtol=1e-13, atol=1e-20)


def test_mn_in_plane_closed_form_and_axisymmetry():
    M, a, b = W.MN_MW
    for R in (0.5, 3.0, 8.0, 20.0):
        expect = -G * M * R / (R * R + (a + b) ** 2) ** 1.5
        for phi in (0.0, 0.7, 2.9):
            x = np.array([R * np.cos(phi), R * np.sin(phi), 0.0])
            acc = O.ext_accel(_posm(x), G, MN)[0]
            np.testing.assert_allclose(acc[:2], expect * x[:2] / R, rtol=1e-13, atol=1e-22)
            assert acc[2] == 0.0
    up = O.ext_accel(_posm([3.0, 1.0, 0.4]), G, MN)[0]
    dn = O.ext_accel(_posm([3.0, 1.0, -0.4]), G, MN)[0]
    np.testing.assert_allclose(up * [1, 1, -1], dn, rtol=1e-15)


def test_far_field_is_keplerian_for_mn():
    M, a, b = W.MN_MW
    x = np.array([3.0e4, 4.0e4, 0.0])
    acc = O.ext_accel(_posm(x), G, MN)[0]
    r = np.linalg.norm(x)
    np.testing.assert_allclose(acc, -G * M * x / r ** 3, rtol=1e-7, atol=1e-30)


def test_sum_of_terms_and_disabled_terms():
    p = _posm(POINTS)
    np.testing.assert_allclose(O.ext_accel(p, G, BOTH), O.ext_accel(p, G, NFW) + O.ext_accel(p, G, MN), rtol=1e-15)
    assert np.all(O.ext_accel(p, G, None) == 0)
    assert np.all(O.ext_accel(p, G, O.Potential.make()) == 0)
    assert np.all(O.ext_accel(_posm([0, 0, 0]), G, NFW) == 0)        # reading R12


def test_transcription_crosscheck_against_survey_values():
    rows = [l.split() for l in open(os.path.join(os.path.dirname(__file__), "golden", "ext_accel_mw.txt"))
            if l.strip() and not l.startswith("#")]
    for row in rows:
        v = np.array([float(t) for t in row])
        a_nfw = O.ext_accel(_posm(v[:3]), G, NFW)[0]
        a_mn = O.ext_accel(_posm(v[:3]), G, MN)[0]
        for got, want in ((a_nfw, v[3:6]), (a_mn, v[6:9])):
            ok = ~np.isnan(want)
            np.testing.assert_allclose(got[ok], want[ok], rtol=1e-12, atol=1e-18)


def test_nfw_against_40_digit_evaluation_and_conditioning_at_small_radius():
    """The oracle evaluates ln(1+c) - c/(1+c) as written; at c << 1 the two terms cancel and
    the relative error grows like eps * 2/c.  Pin: exact (mpmath) within that bound everywhere,
    and to 1e-14 at workload radii (r >= 1 kpc)."""
    import mpmath
    mpmath.mp.dps = 40
    Ms, rs = W.NFW_MW
    for r in (1e-4, 1e-2, 0.5, 1.0, 8.0, 12.4, 40.0):
        x = np.array([r * 0.6, 0.0, r * 0.8])
        a = O.ext_accel(_posm(x), G, NFW)[0]
        c = mpmath.mpf(r) / rs
        f = -mpmath.mpf(G) * Ms * (mpmath.log(1 + c) - c / (1 + c)) / mpmath.mpf(r) ** 3
        exact = np.array([float(f * t) for t in x])
        tol = max(1e-14, 4 * 2.2e-16 * 2 * rs / r)
        assert np.linalg.norm(a - exact) <= tol * np.linalg.norm(exact)


# ---- zero point of the potentials (finite differences and Poisson pin only grad Phi) ----------------
# Closed forms: Phi_NFW(r -> 0) = -G M_s / r_s; r Phi_NFW(r) / ln(1 + r/r_s) = -G M_s for every r
# (so Phi -> 0 like ln(r)/r at infinity, no additive constant); Phi_MN(0,0,0) = -G M / (a + b);
# Phi_MN(R,0,z) r -> -G M as r -> infinity.

def test_potential_zero_points_closed_forms():
    G, Ms, rs, Md, a, b = 4.4985e-12, 1e12, 16.0, 6.8e10, 3.0, 0.28
    nfw = O.Potential.make(nfw=(Ms, rs))
    mn = O.Potential.make(mn=(Md, a, b))
    # NFW centre: exact limit at r = 0 and the first-order expansion -G M_s/r_s (1 - c/2) next to it
    assert O.ext_potential(np.array([[0.0, 0.0, 0.0, 1.0]]), G, nfw)[0] == -G * Ms / rs
    r = 1e-6 * rs
    phi = O.ext_potential(np.array([[r, 0.0, 0.0, 1.0]]), G, nfw)[0]
    assert abs(phi / (-G * Ms / rs) - (1 - 0.5e-6)) <= 1e-11
    # NFW far field: r Phi / ln(1 + r/r_s) = -G M_s (an additive constant C would add C r / ln(1+c))
    for c in (1.0, 1e3, 1e6):
        r = c * rs
        phi = O.ext_potential(np.array([[0.0, r / np.sqrt(2), -r / np.sqrt(2), 1.0]]), G, nfw)[0]
        assert abs(phi * r / np.log1p(c) / (-G * Ms) - 1.0) <= 1e-14
    # hand value: c = 1 -> Phi = -G M_s ln 2 / r_s
    phi = O.ext_potential(np.array([[rs, 0.0, 0.0, 1.0]]), G, nfw)[0]
    assert abs(phi - (-G * Ms * 0.6931471805599453 / rs)) <= 1e-15 * abs(phi)
    # MN centre and far field
    assert abs(O.ext_potential(np.array([[0.0, 0.0, 0.0, 1.0]]), G, mn)[0] - (-G * Md / (a + b))) <= 1e-16
    r = 1e9
    phi = O.ext_potential(np.array([[0.6 * r, 0.0, 0.8 * r, 1.0]]), G, mn)[0]
    assert abs(phi * r / (-G * Md) - 1.0) <= 1e-8
    # off-centre value from the definition written out: B = sqrt(z^2 + b^2), D = sqrt(R^2 + (a + B)^2)
    B = np.sqrt(1.0 + b * b); D = np.sqrt(16.0 + (a + B) ** 2)
    phi = O.ext_potential(np.array([[4.0, 0.0, 1.0, 1.0]]), G, mn)[0]
    assert abs(phi - (-G * Md / D)) <= 1e-16
    # the two terms add, and the energy weights by mass: sum m Phi
    both = O.Potential.make(nfw=(Ms, rs), mn=(Md, a, b))
    p = np.array([[8.0, 1.0, -2.0, 3.0]])
    assert abs(O.ext_potential_energy(p, G, both) - 3.0 * (O.ext_potential(p, G, nfw)[0] + O.ext_potential(p, G, mn)[0])) <= 1e-18
