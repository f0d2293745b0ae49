"""torch.autograd faces (paper_2511_22468_b200/autograd.py) against the oracle adjoint: a loss of the final state,
`.backward()`, and the gradients land on the initial state (mass lane included), the potential parameters and dt."""
import numpy as np
import pytest
import torch

from oracle import adjoint as A
from paper_2511_22468_b200 import autograd as AG
from paper_2511_22468_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _state(n, seed, dtype):
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.random_cloud(n, seed=seed, scale=0.01, centre=cfg.centre)
    posm64[:, 3] *= cfg.M / n
    vel64 = vel64 * 0.02 + np.asarray(cfg.velocity)
    return cfg, posm64.astype(dtype), W.vel4(vel64.astype(dtype), dtype)


def test_single_simulation_f64_backward_matches_the_oracle_adjoint():
    n, nsteps = 300, 5
    cfg, p, v = _state(n, 21, np.float64)
    rng = np.random.Generator(np.random.PCG64(22))
    wx, wv = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)) * 10.0
    posm0 = torch.from_numpy(p).cuda().requires_grad_()
    vel0 = torch.from_numpy(v).cuda().requires_grad_()
    theta = torch.tensor([cfg.nfw[0], cfg.nfw[1], cfg.mn[0], cfg.mn[1], cfg.mn[2]], dtype=torch.float64, requires_grad=True)
    dt = torch.tensor(cfg.dt, dtype=torch.float64, requires_grad=True)
    xf, vf = AG.leapfrog_kdk(posm0, vel0, theta, dt, cfg.G, cfg.eps, nsteps)
    loss = (torch.from_numpy(wx).cuda() * xf[:, :3]).sum() + (torch.from_numpy(wv).cuda() * vf[:, :3]).sum()
    loss.backward()
    ref = A.leapfrog_kdk_vjp(p, v[:, :3], cfg.G, cfg.eps, cfg.dt, nsteps, wx, wv, cfg.nfw, cfg.mn)
    g = posm0.grad.cpu().numpy()
    assert np.abs(g[:, :3] - ref["x0"]).max() <= 1e-9 * np.abs(ref["x0"]).max()
    assert np.abs(g[:, 3] - ref["m"]).max() <= 1e-9 * np.abs(ref["m"]).max()
    assert np.abs(vel0.grad.cpu().numpy()[:, :3] - ref["v0"]).max() <= 1e-9 * np.abs(ref["v0"]).max()
    for k, name in enumerate(A.PARAM_NAMES):
        assert abs(theta.grad[k].item() - ref[name]) <= 1e-8 * abs(ref[name]), name
    assert abs(dt.grad.item() - ref["dt"]) <= 1e-8 * abs(ref["dt"])
    assert np.array_equal(posm0.detach().cpu().numpy(), p)               # inputs untouched


def test_ensemble_f32_backward_matches_the_oracle_adjoint_per_simulation():
    nsim, n, nsteps = 3, 500, 4
    cfg, p, v = _state(n, 31, np.float32)
    posm = np.repeat(p[None], nsim, axis=0)
    vel = np.repeat(v[None], nsim, axis=0)
    rng = np.random.Generator(np.random.PCG64(32))
    wx = rng.normal(size=(nsim, n, 3)).astype(np.float32)
    scale = np.array([[1.0, 1.0, 1.0, 1.0, 1.0], [0.7, 1.0, 1.3, 1.0, 1.0], [1.2, 1.1, 0.9, 1.0, 1.2]])
    th = scale * np.array([cfg.nfw[0], cfg.nfw[1], cfg.mn[0], cfg.mn[1], cfg.mn[2]])
    dts = np.array([cfg.dt, 0.5 * cfg.dt, -cfg.dt])
    posm0 = torch.from_numpy(posm).cuda().requires_grad_()
    vel0 = torch.from_numpy(vel).cuda().requires_grad_()
    theta = torch.tensor(th, dtype=torch.float64, requires_grad=True)
    dt = torch.tensor(dts, dtype=torch.float64, requires_grad=True)
    xf, vf = AG.ensemble_leapfrog_kdk(posm0, vel0, theta, dt, cfg.G, cfg.eps, nsteps)
    (torch.from_numpy(wx).cuda() * xf[:, :, :3]).sum().backward()
    G, eps = float(np.float32(cfg.G)), float(np.float32(cfg.eps))
    for k in range(nsim):
        ref = A.leapfrog_kdk_vjp(posm[k].astype(np.float64), vel[k, :, :3].astype(np.float64), G, eps, float(np.float32(dts[k])),
                                 nsteps, wx[k].astype(np.float64), np.zeros((n, 3)), (th[k, 0], th[k, 1]), (th[k, 2], th[k, 3], th[k, 4]))
        g = posm0.grad[k].cpu().numpy().astype(np.float64)
        assert np.abs(g[:, :3] - ref["x0"]).max() <= 1e-3 * np.abs(ref["x0"]).max()
        assert np.abs(g[:, 3] - ref["m"]).max() <= 1e-3 * np.abs(ref["m"]).max()
        for j, name in enumerate(A.PARAM_NAMES):
            assert abs(theta.grad[k, j].item() - ref[name]) <= 1e-3 * abs(ref[name]), (k, name)
        assert abs(dt.grad[k].item() - ref["dt"]) <= 1e-3 * abs(ref["dt"])


def test_ensemble_checkpointed_backward_equals_the_full_tape_backward():
    """checkpoint_every = K recomputes K-step segments in backward (bit-identical forward); the gradients agree with the
    full-tape run up to the regrouping of the boundary pulls (dt/2 + dt/2 instead of dt)."""
    nsim, n, nsteps = 4, 700, 7
    cfg, p, v = _state(n, 41, np.float32)
    posm = np.repeat(p[None], nsim, axis=0)
    vel = np.repeat(v[None], nsim, axis=0)
    wx = torch.from_numpy(np.random.Generator(np.random.PCG64(42)).normal(size=(nsim, n, 3)).astype(np.float32)).cuda()
    th = np.tile(np.array([cfg.nfw[0], cfg.nfw[1], cfg.mn[0], cfg.mn[1], cfg.mn[2]]), (nsim, 1)) * np.linspace(0.8, 1.2, nsim)[:, None]
    grads = []
    for K in (0, 3, 1):
        posm0 = torch.from_numpy(posm).cuda().requires_grad_()
        vel0 = torch.from_numpy(vel).cuda().requires_grad_()
        theta = torch.tensor(th, dtype=torch.float64, requires_grad=True)
        dt = torch.full((nsim,), cfg.dt, dtype=torch.float64, requires_grad=True)
        xf, vf = AG.ensemble_leapfrog_kdk(posm0, vel0, theta, dt, cfg.G, cfg.eps, nsteps, checkpoint_every=K)
        (wx * xf[:, :, :3]).sum().backward()
        grads.append((xf.detach().cpu().numpy(), posm0.grad.cpu().numpy(), vel0.grad.cpu().numpy(), theta.grad.numpy(), dt.grad.numpy()))
    for g in grads[1:]:
        assert g[0].tobytes() == grads[0][0].tobytes()                   # same forward, bit for bit
        for a, b in zip(g[1:], grads[0][1:]):
            assert np.abs(a - b).max() <= 2e-5 * np.abs(b).max()


def test_gradient_descent_on_the_halo_mass_recovers_the_mock_value():
    """The paper's use of the gradients in miniature (PAPER.md:L43 steps 4-5): a mock stream is simulated with the true
    halo mass, the same progenitor is re-simulated with a wrong halo mass, and gradient steps on a point-wise loss of the
    final positions (obtained through ensemble autograd) drive the halo mass back to the true value."""
    cfg = W.CONFIGS[1]
    n, nsteps = 500, 60
    _, p, v = _state(n, 51, np.float32)
    posm0 = torch.from_numpy(p[None]).cuda()
    vel0 = torch.from_numpy(v[None]).cuda()
    dt = torch.tensor([cfg.dt], dtype=torch.float64)
    true = torch.tensor([[cfg.nfw[0], cfg.nfw[1], cfg.mn[0], cfg.mn[1], cfg.mn[2]]], dtype=torch.float64)
    with torch.no_grad():
        x_obs, _ = AG.ensemble_leapfrog_kdk(posm0, vel0, true, dt, cfg.G, cfg.eps, nsteps)
    log_m = torch.tensor(np.log(1.3 * cfg.nfw[0]), dtype=torch.float64, requires_grad=True)      # 30 % too heavy
    losses = []
    for _ in range(12):
        theta = torch.stack([torch.exp(log_m), true[0, 1], true[0, 2], true[0, 3], true[0, 4]]).reshape(1, 5)
        xf, _ = AG.ensemble_leapfrog_kdk(posm0, vel0, theta, dt, cfg.G, cfg.eps, nsteps, checkpoint_every=20)
        loss = ((xf[:, :, :3] - x_obs[:, :, :3]).double() ** 2).mean()
        (g,) = torch.autograd.grad(loss, log_m)
        losses.append(loss.item())
        # Gauss-Newton-like step for a one-parameter least-squares problem: loss ~ c (log m - log m*)^2
        with torch.no_grad():
            log_m -= (2.0 * loss.item() / g.item()) if g.item() != 0.0 else 0.0
            log_m.clamp_(np.log(0.5 * cfg.nfw[0]), np.log(2.0 * cfg.nfw[0]))
    m = float(torch.exp(log_m.detach()))
    assert losses[-1] <= 1e-3 * losses[0]
    assert abs(m / cfg.nfw[0] - 1.0) <= 1e-2
