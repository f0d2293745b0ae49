"""Reverse-mode derivative of the hot path, fp64 numpy -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` leg may import this module; it
imports nothing from the CUDA package and shares no code with it.

What it follows: the paper's simulator is "end-to-end differentiable" with respect to "initial conditions,
integration time, particle masses and potential parameters" (section 1, L21 section 2); its inference
differentiates a loss of the final state with respect to Theta = (t_end, M_Plummer, M_NFW, M_MN) (PAPER.md:L43
Fig. 2 step 5) and takes a Hessian with respect to (M_vir, r_s, M, a, b).  The paper obtains these
with JAX autodiff and prints no formula, so this file writes the vector-Jacobian products of the three pieces
of DESIGN.md section 1 out by hand, in the order reverse-mode differentiation of the KDK loop gives:

  pair   a_i = G sum_j m_j d f,  d = x_j - x_i,  f = (|d|^2 + eps^2)^(-3/2),  g = -3 (|d|^2 + eps^2)^(-5/2)
         (J^T c)_i = G sum_j (f u + g d (d.u)),  u = m_i c_j - m_j c_i
         dL/dm_i   = -G sum_j f (d.c_j)          dL/dG = sum_i c_i.a_i / G
         dL/deps   = eps G sum_i sum_j m_j g (d.c_i)
  ext    analytic Hessians and parameter derivatives of the NFW and Miyamoto-Nagai accelerations
  kdk    Lv_N = lam_v, Lx_N = lam_x + J(x_N)^T (dt/2 Lv_N);
         Lv_k = Lv_{k+1} + dt Lx_{k+1};  Lx_k = Lx_{k+1} + J(x_k)^T (w_k Lv_k),  w_k = dt (0 < k < N), dt/2 (k = 0)
         dL/dtheta = sum_k (da/dtheta (x_k))^T (w_k Lv_k)
         dL/ddt    = sum_k [ Lx_{k+1}.vh_k + (Lv_k.a_k + Lv_{k+1}.a_{k+1}) / 2 ],  vh_k = v_k + dt/2 a_k

Pins (tests/test_oracle_adjoint.py): every output against central finite differences of the already pinned
forward oracle (oracle.pair_accel / ext_accel / leapfrog_kdk) on tiny inputs, the symmetry of the pair Jacobian
(sum_i (J^T c)_i = 0 for equal c), and the closed form of a two-body gradient.  Nothing here is "parity unpinned".

Layouts: posm float64 [n, 4] = {x, y, z, m}; vel, cotangents and gradients float64 [n, 3]; potential given as
(M_s, r_s) and (M, a, b) tuples or None.
"""
from __future__ import annotations

import numpy as np

PARAM_NAMES = ("M_s", "r_s", "M_d", "a", "b")
BULGE_PARAM_NAMES = ("M_b", "r_c")                        # alpha (the shape) is not differentiated


def pair_accel_vjp(posm, c, G, eps, targets=None):
    """(gx [n,3], gm [n], gG, geps) = cotangent c [n,3] pulled back through a_pair(x, m, G, eps).

    targets = index array: only the rows gx[targets], gm[targets] are evaluated, one particle at a time with O(n)
    memory (the dense form below holds [n, n, 3] arrays and stops near n = 3,000); the return value is
    (gx [len(targets), 3], gm [len(targets)], gG, geps) with gG and geps summed over the target rows i only (the
    totals when targets = every particle).  Same formula, term for term; pinned by targets = all particles
    against the dense form and by finite differences of the forward oracle (tests/test_oracle_adjoint.py)."""
    posm = np.asarray(posm, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    if targets is not None:
        x, m = posm[:, :3], posm[:, 3]
        gx = np.zeros((len(targets), 3))
        gm = np.zeros(len(targets))
        gG = geps = 0.0
        for row, i in enumerate(targets):
            d = x - x[i]                                      # d[j] = x_j - x_i
            s = np.einsum("jk,jk->j", d, d) + eps * eps
            with np.errstate(divide="ignore"):
                f = s ** -1.5
                g = -3.0 * s ** -2.5
            f[i] = 0.0                                        # the pair sum skips j == i
            g[i] = 0.0
            u = m[i] * c - m[:, None] * c[i]                  # u[j] = m_i c_j - m_j c_i
            du = np.einsum("jk,jk->j", d, u)
            gx[row] = G * (np.einsum("j,jk->k", f, u) + np.einsum("j,jk->k", g * du, d))
            gm[row] = -G * np.sum(f * np.einsum("jk,jk->j", d, c))
            gG += float(np.dot(c[i], np.einsum("j,jk->k", f * m, d)))             # c_i . a_i / G
            geps += float(eps * G * np.sum(m * g * (d @ c[i])))
        return gx, gm, gG, geps
    x, m = posm[:, :3], posm[:, 3]
    d = x[None, :, :] - x[:, None, :]                     # d[i, j] = x_j - x_i
    s = np.einsum("ijk,ijk->ij", d, d) + eps * eps
    with np.errstate(divide="ignore"):                    # eps = 0: the diagonal is 1/0 before it is zeroed
        f = s ** -1.5
        g = -3.0 * s ** -2.5
    np.fill_diagonal(f, 0.0)                              # the oracle's pair sum skips j == i
    np.fill_diagonal(g, 0.0)
    u = m[:, None, None] * c[None, :, :] - m[None, :, None] * c[:, None, :]       # u[i, j] = m_i c_j - m_j c_i
    du = np.einsum("ijk,ijk->ij", d, u)
    gx = G * (np.einsum("ij,ijk->ik", f, u) + np.einsum("ij,ijk->ik", g * du, d))
    p = np.einsum("ijk,jk->ij", d, c)                     # d . c_j
    q = np.einsum("ijk,ik->ij", d, c)                     # d . c_i
    gm = -G * np.sum(f * p, axis=1)
    a_over_G = np.einsum("ij,ijk->ik", f * m[None, :], d)
    gG = float(np.sum(c * a_over_G))
    geps = float(eps * G * np.sum(m[None, :] * g * q))
    return gx, gm, gG, geps


def pair_accel_vjp_scale(posm, c, G, eps, targets=None):
    """Per-particle sums of the MAGNITUDES of the terms pair_accel_vjp adds, the denominators of the per-element
    gradient tolerance (the analogue of S_i = sum_j |a_ij| of the forward tolerance, reading R6):
      Sx_i = G sum_j (f |u| + |g| |d| |d.u|),   Sm_i = G sum_j f |d.c_j|.
    By the triangle inequality |gx_i| <= Sx_i and |gm_i| <= Sm_i, with equality when a particle has one partner
    and u is parallel to d (tests/test_oracle_adjoint.py).  targets = index array: those rows only, one particle at a
    time with O(n) memory (as in pair_accel_vjp)."""
    posm = np.asarray(posm, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    if targets is not None:
        x, m = posm[:, :3], posm[:, 3]
        Sx = np.zeros(len(targets))
        Sm = np.zeros(len(targets))
        for row, i in enumerate(targets):
            d = x - x[i]
            s = np.einsum("jk,jk->j", d, d) + eps * eps
            with np.errstate(divide="ignore"):
                f = s ** -1.5
                g = 3.0 * s ** -2.5
            f[i] = 0.0
            g[i] = 0.0
            u = m[i] * c - m[:, None] * c[i]
            du = np.abs(np.einsum("jk,jk->j", d, u))
            Sx[row] = G * np.sum(f * np.linalg.norm(u, axis=1) + g * np.linalg.norm(d, axis=1) * du)
            Sm[row] = G * np.sum(f * np.abs(np.einsum("jk,jk->j", d, c)))
        return Sx, Sm
    x, m = posm[:, :3], posm[:, 3]
    d = x[None, :, :] - x[:, None, :]
    s = np.einsum("ijk,ijk->ij", d, d) + eps * eps
    with np.errstate(divide="ignore"):
        f = s ** -1.5
        g = 3.0 * s ** -2.5
    np.fill_diagonal(f, 0.0)
    np.fill_diagonal(g, 0.0)
    u = m[:, None, None] * c[None, :, :] - m[None, :, None] * c[:, None, :]
    du = np.abs(np.einsum("ijk,ijk->ij", d, u))
    Sx = G * np.sum(f * np.linalg.norm(u, axis=2) + g * np.linalg.norm(d, axis=2) * du, axis=1)
    Sm = G * np.sum(f * np.abs(np.einsum("ijk,jk->ij", d, c)), axis=1)
    return Sx, Sm


def _nfw_parts(x, G, Ms, rs):
    r = np.linalg.norm(x, axis=1)
    cc = r / rs
    mu = np.log1p(cc) - cc / (1.0 + cc)
    dmu_dr = cc / (1.0 + cc) ** 2 / rs
    F = mu / r ** 3
    dF_dr = dmu_dr / r ** 3 - 3.0 * mu / r ** 4
    return r, cc, mu, F, dF_dr


def ext_accel_vjp(posm, c, G, nfw=None, mn=None, bulge=None):
    """(gx [n,3], gparams {M_s, r_s, M_d, a, b, M_b, r_c}, gG): cotangent c pulled back through a_NFW + a_MN + a_bulge."""
    x = np.asarray(posm, dtype=np.float64)[:, :3]
    c = np.asarray(c, dtype=np.float64)
    gx = np.zeros_like(x)
    gp = dict.fromkeys(PARAM_NAMES + BULGE_PARAM_NAMES, 0.0)
    gG = 0.0
    if bulge is not None and bulge[0] > 0:
        # a = -G M_b F(r) x,  F = P(s, t)/r^3,  t = (r/r_c)^2,  dP/dt = t^(s-1) e^-t / Gamma(s)
        from scipy import special
        Mb, alpha, rc = bulge
        s_ = 0.5 * (3.0 - alpha)
        r = np.linalg.norm(x, axis=1)
        t = (r / rc) ** 2
        P = special.gammainc(s_, t)
        dP_dt = np.exp((s_ - 1.0) * np.log(t) - t - special.gammaln(s_))
        F = P / r ** 3
        dF_dr = dP_dt * (2.0 * r / rc ** 2) / r ** 3 - 3.0 * P / r ** 4
        xc = np.einsum("ik,ik->i", x, c)
        gx += -G * Mb * (F[:, None] * c + (dF_dr / r * xc)[:, None] * x)
        a = -G * Mb * F[:, None] * x
        gp["M_b"] += float(np.sum(a * c)) / Mb
        gG += float(np.sum(a * c)) / G
        gp["r_c"] += float(np.sum(-G * Mb * (dP_dt * (-2.0 * t / rc)) / r ** 3 * xc))
    if nfw is not None and nfw[0] > 0:
        Ms, rs = nfw
        r, cc, mu, F, dF_dr = _nfw_parts(x, G, Ms, rs)
        xc = np.einsum("ik,ik->i", x, c)
        # a = -G Ms F(r) x ;  da/dx = -G Ms (F I + F'/r x x^T) (symmetric)
        gx += -G * Ms * (F[:, None] * c + (dF_dr / r * xc)[:, None] * x)
        a = -G * Ms * F[:, None] * x
        gp["M_s"] += float(np.sum(a * c)) / Ms
        gG += float(np.sum(a * c)) / G
        dmu_drs = -cc * cc / ((1.0 + cc) ** 2 * rs)
        gp["r_s"] += float(np.sum(-G * Ms * (dmu_drs / r ** 3) * xc))
    if mn is not None and mn[0] > 0:
        Md, aa, bb = mn
        X, Y, Z = x[:, 0], x[:, 1], x[:, 2]
        B = np.sqrt(Z * Z + bb * bb)
        s = aa + B
        D2 = X * X + Y * Y + s * s
        D3, D5 = D2 ** 1.5, D2 ** 2.5
        k = s / B
        a = -G * Md * np.stack([X / D3, Y / D3, Z * k / D3], axis=1)
        gp["M_d"] += float(np.sum(a * c)) / Md
        gG += float(np.sum(a * c)) / G
        # gradient of each component; w = (X, Y, Z k) = 1/2 grad D2, so d(1/D3) = -3 w / D5
        w = np.stack([X, Y, Z * k], axis=1)
        dk_dz = -aa * Z / B ** 3                           # k = 1 + a / B
        dzk_dz = k + Z * dk_dz
        cw = c[:, 0] * X + c[:, 1] * Y + c[:, 2] * Z * k   # c . (numerators)
        diag = np.stack([c[:, 0], c[:, 1], c[:, 2] * dzk_dz], axis=1)
        gx += -G * Md * (diag / D3[:, None] - 3.0 * (cw / D5)[:, None] * w)
        # d/da: s -> s + 1: dk/da = 1/B, dD2/da = 2 s
        gp["a"] += float(np.sum(-G * Md * (c[:, 2] * Z / B / D3 - 3.0 * cw * s / D5)))
        # d/db: dB/db = b/B: ds/db = b/B, dk/db = -a b / B^3, dD2/db = 2 s b / B
        gp["b"] += float(np.sum(-G * Md * (c[:, 2] * Z * (-aa * bb / B ** 3) / D3 - 3.0 * cw * s * (bb / B) / D5)))
    return gx, gp, gG


def _total_accel(posm, G, eps, nfw, mn, bulge=None):
    from oracle import oracle as O
    pot = O.Potential.make(nfw=nfw, mn=mn, bulge=bulge) if (nfw is not None or mn is not None or bulge is not None) else None
    acc, _ = O.pair_accel(posm, G, eps)
    if pot is not None:
        acc = acc + O.ext_accel(posm, G, pot)
    return acc


def accel_vjp(posm, c, G, eps, nfw=None, mn=None, bulge=None, rowwise=False):
    """Cotangent c pulled back through a = a_pair + a_ext: (gx, gm, gparams, gG, geps).  rowwise: the pair part
    particle by particle (pair_accel_vjp with targets = every particle) for n beyond the dense form's memory."""
    gx, gm, gG, geps = pair_accel_vjp(posm, c, G, eps, np.arange(np.asarray(posm).shape[0]) if rowwise else None)
    ex, gp, eG = ext_accel_vjp(posm, c, G, nfw, mn, bulge)
    return gx + ex, gm, gp, gG + eG, geps


def leapfrog_kdk_vjp(posm, vel, G, eps, dt, nsteps, lam_x, lam_v, nfw=None, mn=None, bulge=None, rowwise=False):
    """Reverse-mode derivative of nsteps KDK steps (oracle.leapfrog_kdk) of a loss with final-state cotangents
    lam_x = dL/dx_N, lam_v = dL/dv_N.  Returns a dict: x0, v0 [n,3]; m [n]; M_s, r_s, M_d, a, b, dt, G, eps.
    rowwise: every pair pull-back particle by particle (accel_vjp), same arithmetic, O(n) memory."""
    posm = np.array(posm, dtype=np.float64)
    v = np.array(vel, dtype=np.float64)
    xs, vs, accs = [posm.copy()], [v.copy()], [_total_accel(posm, G, eps, nfw, mn, bulge)]
    for _ in range(nsteps):                               # forward, textbook order, taping (x_k, v_k, a_k)
        vh = vs[-1] + 0.5 * dt * accs[-1]
        p = xs[-1].copy()
        p[:, :3] += dt * vh
        a = _total_accel(p, G, eps, nfw, mn, bulge)
        xs.append(p)
        vs.append(vh + 0.5 * dt * a)
        accs.append(a)
    Lv = np.array(lam_v, dtype=np.float64)
    Lx = np.array(lam_x, dtype=np.float64)
    out = {"m": np.zeros(posm.shape[0]), "dt": 0.0, "G": 0.0, "eps": 0.0}
    out.update(dict.fromkeys(PARAM_NAMES + BULGE_PARAM_NAMES, 0.0))

    def pull(k, w):
        gx, gm, gp, gG, geps = accel_vjp(xs[k], w * Lv, G, eps, nfw, mn, bulge, rowwise)
        out["m"] += gm
        out["G"] += gG
        out["eps"] += geps
        for name in PARAM_NAMES + BULGE_PARAM_NAMES:
            out[name] += gp[name]
        return gx

    if nsteps == 0:
        out["x0"], out["v0"] = Lx, Lv
        return out
    Lx = Lx + pull(nsteps, 0.5 * dt)
    for k in range(nsteps - 1, -1, -1):
        vh = vs[k] + 0.5 * dt * accs[k]
        out["dt"] += float(np.sum(Lx * vh)) + 0.5 * float(np.sum(Lv * accs[k + 1]))
        Lv = Lv + dt * Lx
        out["dt"] += 0.5 * float(np.sum(Lv * accs[k]))
        Lx = Lx + pull(k, dt if k > 0 else 0.5 * dt)
    out["x0"], out["v0"] = Lx, Lv
    return out
