"""GPU parity of odisseo_mmd2_f32 (MMD^2 between simulated and observed 6-D clouds and its gradient; Fig. 2
step 4, L47) against oracle/mmd.py, which is pinned by closed forms and finite differences.
Tolerances: the value is a difference of three means of numbers in [0, 1] evaluated in fp32 (ex2.approx, 2-ulp) with
fp64 tile sums: |delta| <= 2e-6 absolute; gradient components <= 2e-4 of the largest component (fp32 coordinate
differences scaled by 1/sigma, ~1e-6 relative each, summed over up to 2,000 terms with cancellation)."""
import numpy as np
import pytest
import torch

from oracle import mmd as M
from oracle import oracle as O
from paper_2511_22468_b200 import binding as B

pytestmark = pytest.mark.gpu
SIG = np.array([0.5, 0.7, 0.3, 0.02, 0.03, 0.01])


def _cloud(nsim, n, seed, shift=0.0, spread=0.4):
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = np.zeros((nsim, n, 4), dtype=np.float32)
    vel = np.zeros((nsim, n, 4), dtype=np.float32)
    pos[:, :, :3] = rng.normal(0, spread, (nsim, n, 3)) + np.array([12.4, 0.0, 1.5]) + shift
    pos[:, :, 3] = 7.0                                                    # the mass lane must be ignored
    vel[:, :, :3] = rng.normal(0, 0.02, (nsim, n, 3)) + np.array([0.0, 0.21, 0.05])
    vel[:, :, 3] = -3.0
    return pos, vel


def gpu_mmd(xp, xv, yp, yv, sigma, grad=True, scale=None):
    nsim, n = xp.shape[:2]
    m = yp.shape[-2]
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()         # noqa: E731
    out = torch.full((nsim,), float("nan"), dtype=torch.float64, device="cuda")
    gp = torch.full((nsim, n, 4), float("nan"), device="cuda") if grad else None
    gv = torch.full((nsim, n, 4), float("nan"), device="cuda") if grad else None
    ws = B.alloc_workspace(B.mmd_workspace_bytes(n, m, nsim))
    B.mmd2(t(xp), t(xv), t(yp), t(yv), sigma, out, ws, gp, gv, t(scale) if scale is not None else None)
    torch.cuda.synchronize()
    return out.cpu().numpy(), (gp.cpu().numpy() if grad else None), (gv.cpu().numpy() if grad else None)


@pytest.mark.parametrize("n,m", [(1, 1), (5, 7), (255, 257), (300, 1000), (1000, 1000), (1025, 40)])
@pytest.mark.parametrize("shared", [True, False])
def test_mmd_value_and_gradient_match_the_oracle(n, m, shared):
    nsim = 3
    xp, xv = _cloud(nsim, n, 100 + n)
    yp, yv = _cloud(1 if shared else nsim, m, 200 + m, shift=0.25)
    val, gp, gv = gpu_mmd(xp, xv, yp[0] if shared else yp, yv[0] if shared else yv, SIG)
    for s in range(nsim):
        y = (yp[0], yv[0]) if shared else (yp[s], yv[s])
        args = (xp[s].astype(np.float64), xv[s].astype(np.float64), y[0].astype(np.float64), y[1].astype(np.float64), SIG)
        assert abs(val[s] - M.mmd2(*args)) <= 2e-6
        rp, rv = M.mmd2_grad(*args)
        assert np.abs(gp[s, :, :3] - rp).max() <= 2e-4 * np.abs(rp).max() + 1e-9
        assert np.abs(gv[s, :, :3] - rv).max() <= 2e-4 * np.abs(rv).max() + 1e-8
        assert np.all(gp[s, :, 3] == 0) and np.all(gv[s, :, 3] == 0)


def test_mmd_of_a_cloud_with_itself_is_zero_and_the_call_is_bit_reproducible():
    xp, xv = _cloud(2, 777, 5)
    v1, g1, h1 = gpu_mmd(xp, xv, xp, xv, SIG)
    v2, g2, h2 = gpu_mmd(xp, xv, xp, xv, SIG)
    assert np.abs(v1).max() <= 1e-6
    assert v1.tobytes() == v2.tobytes() and g1.tobytes() == g2.tobytes() and h1.tobytes() == h2.tobytes()
    assert np.abs(g1[:, :, :3]).max() <= 1e-6 and np.abs(h1[:, :, :3]).max() <= 1e-4     # the minimum: zero gradient


def test_mmd_value_only_and_gradient_scale():
    xp, xv = _cloud(4, 300, 8)
    yp, yv = _cloud(1, 200, 9, shift=0.1)
    v0, _, _ = gpu_mmd(xp, xv, yp[0], yv[0], SIG, grad=False)
    v1, g1, h1 = gpu_mmd(xp, xv, yp[0], yv[0], SIG)
    assert v0.tobytes() == v1.tobytes()
    scale = np.array([2.0, -1.0, 0.0, 0.5])
    v2, g2, h2 = gpu_mmd(xp, xv, yp[0], yv[0], SIG, scale=scale)
    assert v2.tobytes() == v1.tobytes()
    for s in range(4):
        np.testing.assert_allclose(g2[s], scale[s] * g1[s], rtol=1e-6, atol=1e-12)
        np.testing.assert_allclose(h2[s], scale[s] * h1[s], rtol=1e-6, atol=1e-12)


def test_mmd_separates_streams_by_distance():
    """A loss has to rank candidates: the further the simulated cloud from the observed one, the larger MMD^2."""
    yp, yv = _cloud(1, 500, 11)
    vals = []
    for shift in (0.0, 0.2, 0.8, 3.0):
        xp, xv = _cloud(1, 500, 12, shift=shift)
        vals.append(gpu_mmd(xp, xv, yp[0], yv[0], 4.0 * SIG, grad=False)[0][0])
    assert vals[0] < vals[1] < vals[2] < vals[3] and vals[3] > 20 * vals[0]


def test_mmd_error_codes():
    xp, xv = _cloud(1, 8, 1)
    t = lambda a: torch.from_numpy(a).cuda()                               # noqa: E731
    out = torch.zeros(1, dtype=torch.float64, device="cuda")
    ws = B.alloc_workspace(4096)
    with pytest.raises(B.OdisseoError, match="ERR_ARG"):
        B.mmd2(t(xp), t(xv), t(xp[0]), t(xv[0]), [1, 1, 0, 1, 1, 1], out, ws)          # sigma must be > 0
    with pytest.raises(B.OdisseoError, match="ERR_WORKSPACE"):
        B.mmd2(t(xp), t(xv), t(xp[0]), t(xv[0]), SIG, out, ws[:8])


def test_simulate_then_mmd_then_backward_matches_the_oracle_chain():
    """The paper's loop on the device (PAPER.md:L43 steps 3-5): ensemble forward -> MMD^2 against an observed cloud ->
    backward -> d loss / d (M_NFW, M_MN, dt) of every simulation, against oracle.mmd2_grad pulled back by oracle.adjoint."""
    from oracle import adjoint as A
    from paper_2511_22468_b200 import autograd as AG
    from paper_2511_22468_b200 import workloads as W
    cfg = W.CONFIGS[1]
    nsim, n, nsteps = 2, 200, 5
    p64, v64 = W.make_state(cfg, n=n)
    p32, v32 = W.to_f32(p64), W.vel4(W.to_f32(v64), np.float32)
    posm0 = torch.from_numpy(np.repeat(p32[None], nsim, axis=0)).cuda()
    vel0 = torch.from_numpy(np.repeat(v32[None], nsim, axis=0)).cuda()
    th = np.array([[cfg.nfw[0], cfg.nfw[1], cfg.mn[0], cfg.mn[1], cfg.mn[2]]] * nsim)
    th[1, 0] *= 1.2
    th[1, 2] *= 0.8
    theta = torch.tensor(th, dtype=torch.float64, requires_grad=True)
    dt = torch.tensor([cfg.dt, 0.8 * cfg.dt], dtype=torch.float64, requires_grad=True)
    G, eps = float(np.float32(cfg.G)), float(np.float32(cfg.eps))
    yp, yv = _cloud(1, 150, 33, spread=0.02)
    yp[0, :, :3] += np.array(cfg.centre) - np.array([12.4, 0.0, 1.5]) + np.array(cfg.velocity) * cfg.dt * nsteps
    sigma = [0.05, 0.05, 0.05, 0.05, 0.05, 0.05]
    xf, vf = AG.ensemble_leapfrog_kdk(posm0, vel0, theta, dt, G, eps, nsteps)
    loss = AG.mmd2(xf, vf, torch.from_numpy(yp[0]).cuda(), torch.from_numpy(yv[0]).cuda(), sigma)
    loss.sum().backward()
    torch.cuda.synchronize()
    for s in range(nsim):
        dts = float(np.float32(dt[s].item()))
        pf, vfo, _ = O.leapfrog_kdk(p32.astype(np.float64), v32[:, :3].astype(np.float64), G, eps, dts, nsteps,
                                    O.Potential.make(nfw=(th[s, 0], th[s, 1]), mn=(th[s, 2], th[s, 3], th[s, 4])))
        ref_val = M.mmd2(pf, vfo, yp[0].astype(np.float64), yv[0].astype(np.float64), sigma)
        assert abs(loss[s].item() - ref_val) <= 5e-6
        gp, gv = M.mmd2_grad(pf, vfo, yp[0].astype(np.float64), yv[0].astype(np.float64), sigma)
        r = A.leapfrog_kdk_vjp(p32.astype(np.float64), v32[:, :3].astype(np.float64), G, eps, dts, nsteps, gp, gv,
                               nfw=(th[s, 0], th[s, 1]), mn=(th[s, 2], th[s, 3], th[s, 4]))
        got = theta.grad[s].numpy()
        want = np.array([r[k] for k in A.PARAM_NAMES])
        for k in (0, 2):                                                  # the paper's Theta: M_NFW, M_MN (L43)
            assert abs(got[k] - want[k]) <= 2e-3 * abs(want[k]) + 1e-30, (s, k, got[k], want[k])
        assert abs(dt.grad[s].item() - r["dt"]) <= 2e-3 * abs(r["dt"])
