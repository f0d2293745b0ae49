"""torch.autograd faces of the differentiable leapfrog: plumbing around the C ABI, no arithmetic of the method.

The paper's users write a loss of the final particle state and ask JAX for its gradient with respect to the
potential parameters, the integration time, the masses and the initial conditions (PAPER.md:L15, L21, L43
step 5, L63).  With these two Functions the same workflow runs on the CUDA library:

    xf, vf = leapfrog_kdk(posm0, vel0, theta, dt, G, eps, nsteps)      # theta = (M_s, r_s, M_d, a, b)
    loss(xf, vf).backward()                                           # posm0.grad[:, 3] is dL/dm_i, theta.grad, dt.grad

forward  = odisseo_leapfrog_kdk_tape_*           (records the state tape)
backward = odisseo_leapfrog_kdk_vjp_*            (walks it backwards; csrc/adjoint.cu)
and the ensemble pair odisseo_ensemble_leapfrog_kdk_tape_f32 / _vjp_f32 for batches of small simulations.
Inputs are never modified; the tape lives until backward has run (or the graph is freed).
"""
from __future__ import annotations

import torch

from . import binding as B


def _potential(theta) -> B.Potential:
    """theta = (M_s, r_s, M_d, a, b) or, with the bulge of MWPotential2014, (M_s, r_s, M_d, a, b, M_b, alpha, r_c)."""
    t = [float(x) for x in theta.detach().cpu().tolist()]
    return B.Potential.make(nfw=(t[0], t[1]), mn=(t[2], t[3], t[4]), bulge=(t[5], t[6], t[7]) if len(t) == 8 else None)


def _theta_grad(gp, theta):
    """Gradient slots of the C ABI (binding.GRADIENT_FIELDS) re-ordered like theta; the bulge shape alpha gets 0."""
    idx = [0, 1, 2, 3, 4] if theta.shape[-1] == 5 else [0, 1, 2, 3, 4, 8, 8, 9]
    g = gp[..., idx].clone()
    if theta.shape[-1] == 8:
        g[..., 6] = 0
    return g.to(theta.dtype).to(theta.device)


def _check_alpha(theta, freeze_alpha: bool):
    """The C ABI has no gradient slot for the bulge shape alpha (binding.GRADIENT_FIELDS): an 8-parameter theta that
    requires grad would get a silent 0 there.  Refuse unless the caller says that is what they want."""
    if theta.shape[-1] == 8 and theta.requires_grad and not freeze_alpha:
        raise ValueError("theta has 8 entries (with the bulge) and requires grad, but d/d(alpha) is not computed: pass "
                         "freeze_alpha=True to accept a zero gradient for alpha (entry 6), or detach theta")


def _check_observed(yposm, yvel):
    if yposm.requires_grad or yvel.requires_grad:
        raise ValueError("mmd2 differentiates with respect to the simulated clouds only: the observed cloud (yposm, yvel) "
                         "gets no gradient; detach it")


class _LeapfrogKDK(torch.autograd.Function):
    @staticmethod
    def forward(ctx, posm0, vel0, theta, dt, G, eps, nsteps):
        n = posm0.shape[0]
        f64 = posm0.dtype == torch.float64
        posm, vel = posm0.detach().clone().contiguous(), vel0.detach().clone().contiguous()
        acc = torch.empty_like(posm)
        ws = B.alloc_workspace(max(B.workspace_bytes(n, f64), B.vjp_workspace_bytes(n, f64)))
        tape = torch.empty(B.tape_bytes(n, nsteps, f64) // posm.element_size(), dtype=posm.dtype, device=posm.device)
        pot = _potential(theta)
        B.leapfrog_kdk_tape(posm, vel, acc, float(G), float(eps), float(dt), int(nsteps), pot, tape, ws)
        ctx.save_for_backward(tape, theta, dt)
        ctx.meta = (n, float(G), float(eps), int(nsteps), ws)
        return posm, vel

    @staticmethod
    def backward(ctx, g_posm, g_vel):
        tape, theta, dt = ctx.saved_tensors
        n, G, eps, nsteps, ws = ctx.meta
        lx = g_posm.detach().clone().contiguous()
        lv = g_vel.detach().clone().contiguous()
        g_mass_final = lx[:, 3].clone()                    # the final mass lane IS the initial mass lane
        lx[:, 3] = 0
        lv[:, 3] = 0
        gm = torch.empty(n, dtype=torch.float64, device=lx.device)
        gp = torch.empty(B.NGRAD, dtype=torch.float64, device=lx.device)
        B.leapfrog_kdk_vjp(tape, n, G, eps, float(dt), nsteps, _potential(theta), lx, lv, gm, gp, ws)
        g_posm0 = lx
        g_posm0[:, 3] = gm.to(lx.dtype) + g_mass_final
        g_theta = _theta_grad(gp, theta)
        g_dt = gp[7].to(dt.dtype).to(dt.device).reshape(dt.shape)
        return g_posm0, lv, g_theta, g_dt, None, None, None


def leapfrog_kdk(posm0: torch.Tensor, vel0: torch.Tensor, theta: torch.Tensor, dt: torch.Tensor, G: float, eps: float,
                 nsteps: int, freeze_alpha: bool = False):
    """Differentiable nsteps KDK steps.  posm0, vel0: CUDA [n, 4] (float32 or float64); theta: 5 values
    (M_s, r_s, M_d, a, b), a mass <= 0 disables that term, or 8 with the bulge (M_b, alpha, r_c); dt: 0-d tensor.
    Returns (posm_final, vel_final); gradients flow to posm0 (lane 3 = masses), vel0, theta and dt.
    LIMITATION: the bulge shape alpha is not differentiated.  An 8-entry theta that requires grad raises ValueError
    unless freeze_alpha=True, in which case theta.grad[6] is 0 by construction, not by calculus."""
    _check_alpha(theta, freeze_alpha)
    dt = torch.as_tensor(dt)
    return _LeapfrogKDK.apply(posm0, vel0, theta, dt, G, eps, nsteps)


def _ens_params(theta, dt, G, eps):
    dts = dt.detach().cpu().tolist()
    return [(float(G), float(eps), float(dts[k]), _potential(theta[k])) for k in range(len(dts))]


class _EnsembleLeapfrogKDK(torch.autograd.Function):
    """checkpoint_every = K > 0: only the states at the starts of K-step segments are kept; backward re-runs one
    segment at a time with a tape (bit-identical recomputation) and pulls the cotangents back through it, so the
    tape holds K + 1 snapshots instead of nsteps + 1 (48 MB per simulation at N = 1,000 and 1,000 steps otherwise)."""

    @staticmethod
    def forward(ctx, posm0, vel0, theta, dt, G, eps, nsteps, checkpoint_every):
        nsim, n = posm0.shape[:2]
        nsteps = int(nsteps)
        K = int(checkpoint_every) if checkpoint_every else nsteps
        K = max(1, min(K, max(nsteps, 1)))
        posm, vel = posm0.detach().clone().contiguous(), vel0.detach().clone().contiguous()
        ws = B.alloc_workspace(B.ensemble_workspace_bytes(nsim))
        params = _ens_params(theta, dt, G, eps)
        segments, starts, done = [], [], 0
        tape = None
        if K >= nsteps:                                                   # one segment: tape the forward directly
            tape = torch.empty(B.ensemble_tape_bytes(n, nsim, nsteps) // 4, dtype=torch.float32, device=posm.device)
            B.ensemble_leapfrog_kdk_tape(posm, vel, params, nsteps, tape, ws)
            segments = [nsteps]
        else:
            while done < nsteps:
                k = min(K, nsteps - done)
                starts.append((posm.clone(), vel.clone()))
                B.ensemble_leapfrog_kdk(posm, vel, params, k, ws)
                segments.append(k)
                done += k
        ctx.save_for_backward(theta, dt)
        ctx.meta = (nsim, n, params, segments, starts, tape, ws)
        return posm, vel

    @staticmethod
    def backward(ctx, g_posm, g_vel):
        theta, dt = ctx.saved_tensors
        nsim, n, params, segments, starts, tape, ws = ctx.meta
        lx, lv = g_posm.detach().clone().contiguous(), g_vel.detach().clone().contiguous()
        g_mass_final = lx[:, :, 3].clone()
        lx[:, :, 3] = 0
        lv[:, :, 3] = 0
        # the C ABI accumulates the segment gradients itself (accumulate flag): no gradient arithmetic here
        gm_tot = torch.empty(nsim, n, dtype=torch.float64, device=lx.device)
        gp_tot = torch.empty(nsim, B.NGRAD, dtype=torch.float64, device=lx.device)
        for s in range(len(segments) - 1, -1, -1):
            k = segments[s]
            if starts:                                                    # recompute this segment with a tape
                p, v = starts[s][0].clone(), starts[s][1].clone()
                seg_tape = torch.empty(B.ensemble_tape_bytes(n, nsim, k) // 4, dtype=torch.float32, device=lx.device)
                B.ensemble_leapfrog_kdk_tape(p, v, params, k, seg_tape, ws)
            else:
                seg_tape = tape
            B.ensemble_leapfrog_kdk_vjp(seg_tape, params, k, lx, lv, gm_tot, gp_tot, ws, accumulate=s < len(segments) - 1)
        lx[:, :, 3] = gm_tot.to(lx.dtype) + g_mass_final
        return (lx, lv, _theta_grad(gp_tot, theta), gp_tot[:, 7].to(dt.dtype).to(dt.device),
                None, None, None, None)


def ensemble_leapfrog_kdk(posm0: torch.Tensor, vel0: torch.Tensor, theta: torch.Tensor, dt: torch.Tensor, G: float,
                          eps: float, nsteps: int, checkpoint_every: int = 0, freeze_alpha: bool = False):
    """Differentiable batch of small simulations: posm0, vel0 float32 CUDA [nsim, n, 4] (n <= 2,048); theta [nsim, 5]
    (or [nsim, 8] with the bulge); dt [nsim].  Returns (posm_final, vel_final); gradients flow to posm0 (lane 3 =
    masses), vel0, theta and dt.  checkpoint_every = K keeps a K-step tape instead of the whole trajectory (one extra
    forward pass in backward).  LIMITATION: the bulge shape alpha is not differentiated; an 8-entry theta that requires
    grad raises ValueError unless freeze_alpha=True (theta.grad[:, 6] is then 0 by construction)."""
    _check_alpha(theta, freeze_alpha)
    return _EnsembleLeapfrogKDK.apply(posm0, vel0, theta, dt, G, eps, nsteps, checkpoint_every)


class _MMD2(torch.autograd.Function):
    """MMD^2 between simulated clouds and an observed one (odisseo_mmd2_f32).  forward: the value; backward: the same
    kernel again with the upstream gradient as its per-simulation scale, so the cotangents of (posm, vel) come out of
    the C ABI ready for the ensemble pull-back -- no gradient arithmetic in Python."""

    @staticmethod
    def forward(ctx, posm, vel, yposm, yvel, sigma):
        x, v = posm.detach().contiguous(), vel.detach().contiguous()
        single = x.dim() == 2
        nsim, n = (1, x.shape[0]) if single else x.shape[:2]
        m = yposm.shape[-2]
        out = torch.empty(nsim, dtype=torch.float64, device=x.device)
        ws = B.alloc_workspace(B.mmd_workspace_bytes(n, m, nsim))
        B.mmd2(x, v, yposm.detach().contiguous(), yvel.detach().contiguous(), sigma, out, ws)
        ctx.save_for_backward(x, v, yposm.detach().contiguous(), yvel.detach().contiguous())
        ctx.meta = (tuple(float(s) for s in sigma), ws, single)
        return out[0] if single else out

    @staticmethod
    def backward(ctx, g_out):
        x, v, y, yv = ctx.saved_tensors
        sigma, ws, single = ctx.meta
        scale = g_out.detach().to(torch.float64).reshape(-1).contiguous()
        out = torch.empty_like(scale)
        gp, gv = torch.empty_like(x), torch.empty_like(v)
        B.mmd2(x, v, y, yv, sigma, out, ws, gp, gv, scale)
        return gp, gv, None, None, None


def mmd2(posm: torch.Tensor, vel: torch.Tensor, yposm: torch.Tensor, yvel: torch.Tensor, sigma):
    """Differentiable MMD^2 loss (Fig. 2 step 4): posm, vel float32 CUDA [nsim, n, 4] (or [n, 4]) simulated
    clouds, yposm, yvel [m, 4] (shared) or [nsim, m, 4] observed; sigma: 6 kernel scales (x, y, z, vx, vy, vz).  Returns
    [nsim] float64 (or a 0-d tensor); gradients flow to posm and vel ONLY: an observed cloud that requires grad raises
    ValueError (it would silently get none)."""
    _check_observed(yposm, yvel)
    return _MMD2.apply(posm, vel, yposm, yvel, tuple(float(s) for s in sigma))
