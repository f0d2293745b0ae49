"""GPU parity of the bulge term of MWPotential2014 (reading R21) through every
entry point that takes a potential: ext_accel, leapfrog, diagnostics, ensembles and the reverse mode, against the oracle
(pinned in tests/test_oracle_bulge.py).  The device evaluates the regularised incomplete gamma function by series /
continued fraction; tolerances: fp64 1e-12, fp32 1e-5 relative."""
import numpy as np
import pytest
import torch

from oracle import adjoint as A
from oracle import oracle as O
from paper_2511_22468_b200 import binding as B
from paper_2511_22468_b200 import workloads as W

pytestmark = pytest.mark.gpu
G = 4.4985e-12
NFW, MN, BULGE = (1.0e12, 16.0), (6.8e10, 3.0, 0.28), (4.5e9, 1.8, 1.9)


def dev(a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def _radii_cloud(n, seed):
    """Points at radii from 1e-3 to 80 kpc: both branches of the incomplete gamma evaluation and the P = 1 plateau."""
    rng = np.random.Generator(np.random.PCG64(seed))
    r = 10.0 ** rng.uniform(-3, np.log10(80.0), n)
    d = rng.normal(size=(n, 3))
    d /= np.linalg.norm(d, axis=1)[:, None]
    return np.concatenate([r[:, None] * d, np.ones((n, 1))], axis=1)


@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-12), (np.float32, 1e-5)])
@pytest.mark.parametrize("bulge", [BULGE, (1.0e9, 0.0, 0.5), (2.0e9, 1.0, 3.0), (1.0e9, 1.95, 1.0)])
def test_ext_accel_with_bulge_matches_the_oracle(dtype, tol, bulge):
    posm64 = _radii_cloud(4000, 3)
    posm64[0, :3] = 0.0                                                   # the centre: acceleration := 0
    p = posm64.astype(dtype)
    posm = dev(p, dtype)
    acc = torch.full_like(posm, float("nan"))
    B.ext_accel(posm, acc, G, B.Potential.make(bulge=bulge))
    torch.cuda.synchronize()
    ref = O.ext_accel(p.astype(np.float64), float(dtype(G)), O.Potential.make(bulge=bulge))
    got = acc.cpu().numpy()[:, :3].astype(np.float64)
    err = np.linalg.norm(got - ref, axis=1) / np.maximum(np.linalg.norm(ref, axis=1), 1e-300)
    assert np.all(got[0] == 0) and err[1:].max() <= tol
    # all three terms together
    B.ext_accel(posm, acc, G, B.Potential.make(nfw=NFW, mn=MN, bulge=bulge))
    torch.cuda.synchronize()
    ref = O.ext_accel(p.astype(np.float64), float(dtype(G)), O.Potential.make(nfw=NFW, mn=MN, bulge=bulge))
    got = acc.cpu().numpy()[:, :3].astype(np.float64)
    err = np.linalg.norm(got - ref, axis=1) / np.maximum(np.linalg.norm(ref, axis=1), 1e-300)
    # r >= 0.1 kpc: below, the fp64 ORACLE's NFW mass function cancels (relative error ~ eps 2 r_s / r, R12; the
    # small-radius NFW branch is tested against 40-digit arithmetic in test_gpu_parity.py)
    far = np.linalg.norm(p[:, :3].astype(np.float64), axis=1) >= 0.1
    assert err[far].max() <= 2 * tol


def test_leapfrog_diagnostics_and_ensemble_with_bulge_match_the_oracle():
    cfg = W.CONFIGS[1]
    n, nsteps = 400, 10
    posm64, vel64 = W.make_state(cfg, n=n)
    posm64[:, :3] += np.array([-9.0, 0.0, -1.0])                          # orbit at r ~ 3.5 kpc: the bulge matters there
    pot = B.Potential.make(nfw=NFW, mn=MN, bulge=BULGE)
    opot = O.Potential.make(nfw=NFW, mn=MN, bulge=BULGE)
    # fp64 trajectory and diagnostics
    posm, vel = dev(posm64, np.float64), dev(W.vel4(vel64, np.float64), np.float64)
    acc = torch.empty_like(posm)
    B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, nsteps, pot, B.alloc_workspace(B.workspace_bytes(n, True)))
    out = torch.empty(16, dtype=torch.float64, device="cuda")
    B.diagnostics(posm, vel, cfg.G, cfg.eps, pot, out, B.alloc_workspace(B.diagnostics_workspace_bytes(n)))
    torch.cuda.synchronize()
    pr, vr, _ = O.leapfrog_kdk(posm64, vel64, cfg.G, cfg.eps, cfg.dt, nsteps, opot)
    assert np.abs(posm.cpu().numpy()[:, :3] - pr[:, :3]).max() <= 1e-10 * 3.5
    assert np.abs(vel.cpu().numpy()[:, :3] - vr).max() <= 1e-10 * 0.21
    e_ext = O.ext_potential_energy(posm.cpu().numpy(), cfg.G, opot)
    assert abs(out[2].item() - e_ext) <= 1e-12 * abs(e_ext)
    # and the bulge is really felt: the same run without it ends elsewhere
    p0, _, _ = O.leapfrog_kdk(posm64, vel64, cfg.G, cfg.eps, cfg.dt, nsteps, O.Potential.make(nfw=NFW, mn=MN))
    assert np.abs(p0[:, :3] - pr[:, :3]).max() > 1e-4
    # fp32 ensemble of two simulations with different bulge masses
    p32, v32 = W.to_f32(posm64), W.vel4(W.to_f32(vel64), np.float32)
    ep = torch.from_numpy(np.repeat(p32[None], 2, axis=0)).cuda()
    ev = torch.from_numpy(np.repeat(v32[None], 2, axis=0)).cuda()
    prm = [(cfg.G, cfg.eps, cfg.dt, B.Potential.make(nfw=NFW, mn=MN, bulge=(mb, 1.8, 1.9))) for mb in (4.5e9, 9.0e9)]
    B.ensemble_leapfrog_kdk(ep, ev, prm, nsteps, B.alloc_workspace(B.ensemble_workspace_bytes(2)))
    torch.cuda.synchronize()
    Gf, ef, df = float(np.float32(cfg.G)), float(np.float32(cfg.eps)), float(np.float32(cfg.dt))
    for s, mb in enumerate((4.5e9, 9.0e9)):
        pr, vr, _ = O.leapfrog_kdk(p32.astype(np.float64), v32[:, :3].astype(np.float64), Gf, ef, df, nsteps,
                                   O.Potential.make(nfw=NFW, mn=MN, bulge=(mb, 1.8, 1.9)))
        assert np.abs(ep[s].cpu().numpy()[:, :3] - pr[:, :3]).max() <= 1e-5 * 3.5
        assert np.abs(ev[s].cpu().numpy()[:, :3] - vr).max() <= 1e-5 * 0.3


@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-9), (np.float32, 2e-4)])
def test_reverse_mode_with_bulge_matches_the_oracle_adjoint(dtype, tol):
    cfg = W.CONFIGS[1]
    n, nsteps = 300, 5
    posm64, vel64 = W.make_state(cfg, n=n)
    posm64[:, :3] += np.array([-9.0, 0.0, -1.0])
    p, v = posm64.astype(dtype), W.vel4(vel64.astype(dtype), dtype)
    Gd, ed, dd = (cfg.G, cfg.eps, cfg.dt) if dtype == np.float64 else tuple(float(np.float32(q)) for q in (cfg.G, cfg.eps, cfg.dt))
    pot = B.Potential.make(nfw=NFW, mn=MN, bulge=BULGE)
    f64 = dtype == np.float64
    posm, vel = dev(p, dtype), dev(v, dtype)
    acc = torch.empty_like(posm)
    ws = B.alloc_workspace(max(B.workspace_bytes(n, f64), B.vjp_workspace_bytes(n, f64)))
    tape = torch.empty(B.tape_bytes(n, nsteps, f64) // posm.element_size(), dtype=posm.dtype, device="cuda")
    B.leapfrog_kdk_tape(posm, vel, acc, Gd, ed, dd, nsteps, pot, tape, ws)
    lx = torch.ones_like(posm)
    lx[:, 3] = 0
    lv = torch.zeros_like(posm)
    gm = torch.empty(n, dtype=torch.float64, device="cuda")
    gp = torch.empty(B.NGRAD, dtype=torch.float64, device="cuda")
    B.leapfrog_kdk_vjp(tape, n, Gd, ed, dd, nsteps, pot, lx, lv, gm, gp, ws)
    torch.cuda.synchronize()
    r = A.leapfrog_kdk_vjp(p.astype(np.float64), v[:, :3].astype(np.float64), Gd, ed, dd, nsteps, np.ones((n, 3)), np.zeros((n, 3)),
                           nfw=NFW, mn=MN, bulge=BULGE)
    gpn = gp.cpu().numpy()
    for k, name in enumerate(B.GRADIENT_FIELDS):
        if name in ("G", "eps"):
            continue
        assert abs(gpn[k] - r[name]) <= tol * abs(r[name]) + 1e-300, name
    assert np.abs(lx.cpu().numpy()[:, :3] - r["x0"]).max() <= tol * np.abs(r["x0"]).max()
    assert np.abs(lv.cpu().numpy()[:, :3] - r["v0"]).max() <= tol * np.abs(r["v0"]).max()


def test_bulge_argument_validation():
    posm = torch.zeros(4, 4, device="cuda")
    acc = torch.zeros(4, 4, device="cuda")
    for bad in ((1e9, 2.0, 1.0), (1e9, -0.1, 1.0), (1e9, 1.8, 0.0), (float("inf"), 1.8, 1.0)):
        with pytest.raises(B.OdisseoError, match="ERR_ARG"):
            B.ext_accel(posm, acc, G, B.Potential.make(bulge=bad))
    B.ext_accel(posm, acc, G, B.Potential.make(bulge=(0.0, 5.0, -1.0)))   # disabled: parameters are not looked at
