"""Pins of the oracle's reverse-mode derivative (oracle/adjoint.py) against central finite differences of the
already pinned forward oracle, plus closed forms / invariants.  CPU only."""
import numpy as np
import pytest

from oracle import adjoint as A
from oracle import oracle as O

NFW = (1.0e12, 16.0)
MN = (6.8e10, 3.0, 0.28)
G_KPC = 4.4985e-12


def _cloud(n, seed, centre=(12.4, 0.0, 1.5), scale=0.05):
    rng = np.random.Generator(np.random.PCG64(seed))
    posm = np.concatenate([rng.normal(0, scale, (n, 3)) + np.asarray(centre), rng.uniform(0.5, 1.5, (n, 1)) * 1e3], axis=1)
    vel = rng.normal(0, 0.01, (n, 3)) + np.array([0.0, 0.21, 0.05])
    return posm, vel


def _fd(fun, x0, h):
    return (fun(x0 + h) - fun(x0 - h)) / (2 * h)


def test_pair_vjp_matches_finite_differences_of_the_forward_oracle():
    posm, _ = _cloud(7, 1)
    G, eps = 1.3, 0.02
    c = np.random.Generator(np.random.PCG64(2)).normal(size=(7, 3))
    gx, gm, gG, geps = A.pair_accel_vjp(posm, c, G, eps)
    loss = lambda p, G_=G, e_=eps: float(np.sum(c * O.pair_accel(p, G_, e_)[0]))
    for i in range(7):
        for k in range(4):
            def f(t, i=i, k=k):
                p = posm.copy(); p[i, k] = t
                return loss(p)
            h = 1e-6 if k < 3 else 1e-2
            ref = _fd(f, posm[i, k], h)
            got = gx[i, k] if k < 3 else gm[i]
            assert abs(got - ref) <= 1e-7 * max(abs(ref), np.abs(gx).max() if k < 3 else np.abs(gm).max())
    assert abs(gG - _fd(lambda t: loss(posm, G_=t), G, 1e-5)) <= 1e-8 * abs(gG)
    assert abs(geps - _fd(lambda t: loss(posm, e_=t), eps, 1e-7)) <= 1e-6 * abs(geps)


@pytest.mark.parametrize("n,eps", [(2, 0.0), (7, 0.02), (200, 0.003)])
def test_pair_vjp_row_form_equals_the_dense_form_and_finite_differences(n, eps):
    """pair_accel_vjp(targets=...) and pair_accel_vjp_scale(targets=...) evaluate one particle at a time (what lets the
    GPU parity tests reach N = 65,536): all rows == the dense form to rounding, a subset == those rows, the rows'
    gG / geps == the dense totals, and on n = 7 the rows also meet central differences of the forward oracle directly."""
    posm, _ = _cloud(n, 21 + n)
    G = 1.3
    c = np.random.Generator(np.random.PCG64(22 + n)).normal(size=(n, 3))
    gx, gm, gG, geps = A.pair_accel_vjp(posm, c, G, eps)
    rx, rm, rG, reps = A.pair_accel_vjp(posm, c, G, eps, targets=np.arange(n))
    assert np.abs(rx - gx).max() <= 1e-13 * np.abs(gx).max() and np.abs(rm - gm).max() <= 1e-13 * np.abs(gm).max()
    assert abs(rG - gG) <= 1e-12 * np.abs(c).max() * np.abs(O.pair_accel(posm, 1.0, eps)[0]).sum()
    assert abs(reps - geps) <= 1e-12 * max(abs(geps), 1e-300) + (0 if eps else 1e-300)
    sub = np.array([n - 1, 0, n // 2])
    sx, sm, _, _ = A.pair_accel_vjp(posm, c, G, eps, targets=sub)
    assert np.array_equal(sx, rx[sub]) and np.array_equal(sm, rm[sub])
    Sx, Sm = A.pair_accel_vjp_scale(posm, c, G, eps)
    Tx, Tm = A.pair_accel_vjp_scale(posm, c, G, eps, targets=sub)
    assert np.abs(Tx - Sx[sub]).max() <= 1e-13 * Sx.max() and np.abs(Tm - Sm[sub]).max() <= 1e-13 * Sm.max()
    assert np.all(np.linalg.norm(sx, axis=1) <= Tx * (1 + 1e-12)) and np.all(np.abs(sm) <= Tm * (1 + 1e-12))
    if n == 7:
        loss = lambda p: float(np.sum(c * O.pair_accel(p, G, eps)[0]))                  # noqa: E731
        for row, i in enumerate(sub):
            for k in range(4):
                def f(t, i=i, k=k):
                    p = posm.copy(); p[i, k] = t
                    return loss(p)
                ref = _fd(f, posm[i, k], 1e-6 if k < 3 else 1e-2)
                got = sx[row, k] if k < 3 else sm[row]
                assert abs(got - ref) <= 1e-7 * max(abs(ref), np.abs(gx).max() if k < 3 else np.abs(gm).max())


def test_leapfrog_vjp_row_form_equals_the_dense_form():
    n, nsteps = 60, 4
    posm, vel = _cloud(n, 31, scale=0.02)
    rng = np.random.Generator(np.random.PCG64(32))
    lx, lv = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)) * 10.0
    a = A.leapfrog_kdk_vjp(posm, vel, G_KPC, 0.003, 0.7, nsteps, lx, lv, NFW, MN)
    b = A.leapfrog_kdk_vjp(posm, vel, G_KPC, 0.003, 0.7, nsteps, lx, lv, NFW, MN, rowwise=True)
    for key in a:
        scale = np.abs(a[key]).max() if key != "eps" else max(abs(a["eps"]), 1e-300)
        tol = 1e-12 if key not in ("G", "eps") else 1e-9       # totals that cancel between particles
        assert np.abs(np.asarray(a[key]) - np.asarray(b[key])).max() <= tol * scale, key


def test_pair_vjp_invariants_and_two_body_closed_form():
    posm, _ = _cloud(40, 3)
    c = np.tile(np.array([[0.3, -1.0, 2.0]]), (40, 1))
    gx, gm, gG, _ = A.pair_accel_vjp(posm, c, 1.0, 0.01)
    # L = c . sum_i a_i is translation invariant  ->  sum_i dL/dx_i = 0
    assert np.abs(gx.sum(axis=0)).max() <= 1e-12 * np.abs(gx).max()
    # two bodies on the x axis, eps = 0: a_0 = G m_1 / d^2 e_x; dL/dx_0 for L = a_0x is +2 G m_1 / d^3
    p2 = np.array([[0, 0, 0, 2.0], [3.0, 0, 0, 5.0]])
    c2 = np.array([[1.0, 0, 0], [0, 0, 0]])
    g2, m2, _, _ = A.pair_accel_vjp(p2, c2, 1.5, 0.0)
    assert abs(g2[0, 0] - 2 * 1.5 * 5.0 / 27) <= 1e-15 and abs(g2[1, 0] + 2 * 1.5 * 5.0 / 27) <= 1e-15
    assert abs(m2[1] - 1.5 / 9) <= 1e-15 and m2[0] == 0


def test_ext_vjp_matches_finite_differences():
    posm, _ = _cloud(9, 4, scale=3.0)
    c = np.random.Generator(np.random.PCG64(5)).normal(size=(9, 3))

    def loss(p, nfw=NFW, mn=MN, G=G_KPC):
        return float(np.sum(c * O.ext_accel(p, G, O.Potential.make(nfw=nfw, mn=mn))))
    gx, gp, gG = A.ext_accel_vjp(posm, c, G_KPC, NFW, MN)
    for i in range(9):
        for k in range(3):
            def f(t, i=i, k=k):
                p = posm.copy(); p[i, k] = t
                return loss(p)
            assert abs(gx[i, k] - _fd(f, posm[i, k], 1e-5)) <= 1e-7 * np.abs(gx).max()
    refs = {"M_s": _fd(lambda t: loss(posm, nfw=(t, NFW[1])), NFW[0], 1e6),
            "r_s": _fd(lambda t: loss(posm, nfw=(NFW[0], t)), NFW[1], 1e-5),
            "M_d": _fd(lambda t: loss(posm, mn=(t, MN[1], MN[2])), MN[0], 1e5),
            "a": _fd(lambda t: loss(posm, mn=(MN[0], t, MN[2])), MN[1], 1e-5),
            "b": _fd(lambda t: loss(posm, mn=(MN[0], MN[1], t)), MN[2], 1e-6)}
    for name, ref in refs.items():
        assert abs(gp[name] - ref) <= 2e-7 * abs(ref), name
    assert abs(gG - _fd(lambda t: loss(posm, G=t), G_KPC, 1e-17)) <= 1e-7 * abs(gG)


@pytest.mark.parametrize("nsteps", [0, 1, 6])
def test_leapfrog_vjp_matches_finite_differences_of_the_forward_leapfrog(nsteps):
    n = 5
    posm, vel = _cloud(n, 6, scale=0.02)
    posm[:, 3] *= 2.0                                    # self-gravity comparable to the tidal field over a few steps
    G, eps, dt = G_KPC, 0.003, 0.7
    rng = np.random.Generator(np.random.PCG64(7))
    lx, lv = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)) * 10.0

    def loss(p=posm, v=vel, G_=G, e_=eps, dt_=dt, nfw=NFW, mn=MN):
        pf, vf, _ = O.leapfrog_kdk(p, v, G_, e_, dt_, nsteps, O.Potential.make(nfw=nfw, mn=mn))
        return float(np.sum(lx * pf[:, :3]) + np.sum(lv * vf))
    g = A.leapfrog_kdk_vjp(posm, vel, G, eps, dt, nsteps, lx, lv, NFW, MN)
    for i in range(n):
        for k in range(3):
            def fx(t, i=i, k=k):
                p = posm.copy(); p[i, k] = t
                return loss(p=p)
            def fv(t, i=i, k=k):
                v = vel.copy(); v[i, k] = t
                return loss(v=v)
            assert abs(g["x0"][i, k] - _fd(fx, posm[i, k], 1e-6)) <= 1e-6 * np.abs(g["x0"]).max()
            assert abs(g["v0"][i, k] - _fd(fv, vel[i, k], 1e-6)) <= 1e-6 * np.abs(g["v0"]).max()
        def fm(t, i=i):
            p = posm.copy(); p[i, 3] = t
            return loss(p=p)
        if nsteps:
            assert abs(g["m"][i] - _fd(fm, posm[i, 3], 1e-1)) <= 1e-5 * np.abs(g["m"]).max()
    if nsteps == 0:
        assert g["dt"] == 0 and g["M_s"] == 0 and np.all(g["m"] == 0)
        return
    refs = {"M_s": _fd(lambda t: loss(nfw=(t, NFW[1])), NFW[0], 1e6), "r_s": _fd(lambda t: loss(nfw=(NFW[0], t)), NFW[1], 1e-5),
            "M_d": _fd(lambda t: loss(mn=(t, MN[1], MN[2])), MN[0], 1e5), "a": _fd(lambda t: loss(mn=(MN[0], t, MN[2])), MN[1], 1e-5),
            "b": _fd(lambda t: loss(mn=(MN[0], MN[1], t)), MN[2], 1e-6), "dt": _fd(lambda t: loss(dt_=t), dt, 1e-6),
            "G": _fd(lambda t: loss(G_=t), G, 1e-18), "eps": _fd(lambda t: loss(e_=t), eps, 2e-5)}
    for name, ref in refs.items():
        # the loss is O(100) and d loss / d eps O(1e-4): the difference quotient carries ~1e-5 of rounding noise
        assert abs(g[name] - ref) <= (1e-4 if name == "eps" else 2e-6) * abs(ref) + 1e-12 * abs(g["dt"]), name


def test_pair_vjp_scale_bounds_the_gradient_and_is_tight_for_one_aligned_partner():
    """The per-element tolerance denominators: triangle inequality on random inputs, equality for two particles
    whose u = m_0 c_1 - m_1 c_0 is parallel to their separation (closed form: G (f |u| + |g| |d|^2 |u|))."""
    rng = np.random.default_rng(5)
    posm = np.concatenate([rng.normal(size=(17, 3)), rng.uniform(0.5, 2.0, size=(17, 1))], axis=1)
    c = rng.normal(size=(17, 3))
    gx, gm, _, _ = A.pair_accel_vjp(posm, c, 1.3, 0.2)
    Sx, Sm = A.pair_accel_vjp_scale(posm, c, 1.3, 0.2)
    assert np.all(np.linalg.norm(gx, axis=1) <= Sx * (1 + 1e-12)) and np.all(np.abs(gm) <= Sm * (1 + 1e-12))
    assert np.all(Sx > 0) and np.all(Sm > 0)
    two = np.array([[0.0, 0.0, 0.0, 2.0], [3.0, 0.0, 0.0, 5.0]])
    c2 = np.array([[1.0, 0.0, 0.0], [-0.5, 0.0, 0.0]])                  # u_01 = 2 (-0.5) - 5 (1) = -6 along x = along d
    G, eps = 0.7, 4.0
    s = 9.0 + 16.0
    expect = G * (s ** -1.5 * 6.0 + 3.0 * s ** -2.5 * 3.0 * 18.0)
    Sx2, Sm2 = A.pair_accel_vjp_scale(two, c2, G, eps)
    gx2, gm2, _, _ = A.pair_accel_vjp(two, c2, G, eps)
    assert abs(Sx2[0] - expect) <= 1e-15 * expect and abs(Sx2[1] - expect) <= 1e-15 * expect
    # f u and g d (d.u) have opposite signs here, so the gradient is strictly smaller than the scale
    assert abs(gx2[0, 0]) < Sx2[0] and abs(abs(gx2[0, 0]) - G * abs(s ** -1.5 * 6.0 - 3.0 * s ** -2.5 * 54.0)) <= 1e-15
    assert abs(Sm2[0] - G * s ** -1.5 * 1.5) <= 1e-16 and abs(abs(gm2[0]) - Sm2[0]) <= 1e-16
