"""GPU parity of the batched small-N ensemble call against the fp64 CPU oracle:
every simulation of a batch must match oracle.leapfrog_kdk run on its own inputs and parameters."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2511_22468_b200 import binding as B
from paper_2511_22468_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _f32(x):
    return float(np.float32(x))


def _make_batch(n, sims):
    """sims: list of dicts(seed, M, dt_scale, nfw_scale, mn_scale, unequal, isolated)."""
    cfg = W.CONFIGS[1]
    posm = np.zeros((len(sims), n, 4), dtype=np.float32)
    vel = np.zeros((len(sims), n, 4), dtype=np.float32)
    bparams, oparams = [], []
    for k, s in enumerate(sims):
        if s.get("isolated"):
            c0 = W.CONFIGS[0]
            p64, v64 = W.plummer_sphere(n, c0.G, c0.M, c0.a, s["seed"])
            G, eps, dt, bpot, opot = c0.G, c0.eps, c0.dt, None, None
        else:
            p64, v64 = W.plummer_sphere(n, cfg.G, s["M"], cfg.a, s["seed"])
            p64[:, :3] += np.asarray(cfg.centre)
            v64 += np.asarray(cfg.velocity)
            nfw = (cfg.nfw[0] * s["nfw_scale"], cfg.nfw[1])
            mn = (cfg.mn[0] * s["mn_scale"], cfg.mn[1], cfg.mn[2])
            G, eps, dt = cfg.G, cfg.eps, cfg.dt * s["dt_scale"]
            bpot, opot = B.Potential.make(nfw=nfw, mn=mn), O.Potential.make(nfw=nfw, mn=mn)
        if s.get("unequal"):
            p64[:, 3] *= np.random.Generator(np.random.PCG64(s["seed"])).uniform(0.5, 1.5, n)
        posm[k] = W.to_f32(p64)
        vel[k, :, :3] = W.to_f32(v64)
        bparams.append((G, eps, dt, bpot))
        oparams.append((_f32(G), _f32(eps), _f32(dt), opot))
    return posm, vel, bparams, oparams


def _check_against_oracle(posm0, vel0, posm1, vel1, oparams, nsteps, a_scale):
    for k, (G, eps, dt, opot) in enumerate(oparams):
        pr, vr, _ = O.leapfrog_kdk(posm0[k].astype(np.float64), vel0[k, :, :3].astype(np.float64), G, eps, dt, nsteps, opot)
        _, S = O.pair_accel(pr, G, eps)
        aext = np.linalg.norm(O.ext_accel(pr, G, opot), axis=1) if opot is not None else 0.0
        dx = np.linalg.norm(posm1[k, :, :3] - pr[:, :3], axis=1)
        dv = np.linalg.norm(vel1[k, :, :3] - vr, axis=1)
        # 10-step short-horizon tolerances
        assert np.all(dx <= 1e-5 * np.maximum(np.linalg.norm(pr[:, :3], axis=1), a_scale[k])), "sim %d dx" % k
        assert np.all(dv <= 1e-5 * np.linalg.norm(vr, axis=1) + 1.5e-4 * abs(dt) * (S + aext)), "sim %d dv" % k
        assert np.array_equal(posm1[k, :, 3], posm0[k, :, 3])
        assert np.all(vel1[k, :, 3] == 0)


def _run(posm, vel, bparams, nsteps):
    dp, dv = torch.from_numpy(posm.copy()).cuda(), torch.from_numpy(vel.copy()).cuda()
    ws = B.alloc_workspace(B.ensemble_workspace_bytes(posm.shape[0]))
    B.ensemble_leapfrog_kdk(dp, dv, bparams, nsteps, ws)
    torch.cuda.synchronize()
    return dp.cpu().numpy(), dv.cpu().numpy()


def test_ensemble_per_simulation_parameters_match_the_oracle():
    n = 1000                                                    # the paper's N; ragged vs 1,024
    sims = [dict(seed=11, M=1.0e4, dt_scale=1.0, nfw_scale=1.0, mn_scale=1.0),
            dict(seed=12, M=2.0e4, dt_scale=0.5, nfw_scale=0.7, mn_scale=1.3),
            dict(seed=13, M=0.5e4, dt_scale=-1.0, nfw_scale=1.2, mn_scale=0.0),       # backward, no disk
            dict(seed=14, M=1.0e4, dt_scale=1.0, nfw_scale=0.0, mn_scale=1.0),        # no halo
            dict(seed=15, M=1.0e4, dt_scale=1.0, nfw_scale=1.0, mn_scale=1.0, unequal=True),
            dict(seed=16, isolated=True)]
    posm, vel, bparams, oparams = _make_batch(n, sims)
    p1, v1 = _run(posm, vel, bparams, 10)
    a_scale = [W.CONFIGS[1].a] * 5 + [W.CONFIGS[0].a]
    _check_against_oracle(posm, vel, p1, v1, oparams, 10, a_scale)


@pytest.mark.parametrize("n", [1, 2, 3, 255, 257, 512, 513, 1024, 1025, 1536, 2000, 2048])
def test_ensemble_sizes_and_shared_parameters(n):
    sims = [dict(seed=100 + n + k, M=1.0e4, dt_scale=1.0, nfw_scale=1.0, mn_scale=1.0, unequal=(k == 1)) for k in range(3)]
    posm, vel, bparams, oparams = _make_batch(n, sims)
    p1, v1 = _run(posm, vel, bparams[:1], 4)                    # one shared parameter record
    _check_against_oracle(posm, vel, p1, v1, oparams, 4, [W.CONFIGS[1].a] * 3)


@pytest.mark.parametrize("n", [1, 300])
def test_ensemble_backward_in_time_matches_the_oracle_and_returns(n):
    """dt < 0 in the batched call: Fig. 2 step 2 integrates the centre of mass BACKWARD for t_end as a single
    particle in the external potential (n = 1, orbit mode: no pair loop), then the stream forward.  Every simulation
    against oracle.leapfrog_kdk run with the same negative dt, and forward after backward returns to the start."""
    nsteps = 25
    sims = [dict(seed=300 + n + k, M=1.0e4, dt_scale=-1.0 if k != 1 else -0.37, nfw_scale=1.0, mn_scale=1.0) for k in range(3)]
    posm, vel, bparams, oparams = _make_batch(n, sims)
    p1, v1 = _run(posm, vel, bparams, nsteps)
    assert all(dt < 0 for _, _, dt, _ in oparams)
    _check_against_oracle(posm, vel, p1, v1, oparams, nsteps, [W.CONFIGS[1].a] * 3)
    moved = np.linalg.norm(p1[:, :, :3] - posm[:, :, :3], axis=2)
    assert moved.min() > 0.3                                     # ~0.2 kpc/Myr x 25 x 0.5 Myr (0.37 of it in sim 1)
    forward = [(G, eps, -dt, pot) for G, eps, dt, pot in bparams]
    p2, v2 = _run(p1, v1, forward, nsteps)
    back = np.linalg.norm(p2[:, :, :3] - posm[:, :, :3], axis=2)
    assert back.max() <= 2e-5 * np.linalg.norm(posm[:, :, :3], axis=2).max()            # fp32 KDK is reversible to rounding
    assert np.abs(v2[:, :, :3] - vel[:, :, :3]).max() <= 2e-5 * np.abs(vel[:, :, :3]).max() + 1e-6


def test_ensemble_agrees_with_the_single_simulation_path_and_is_reproducible():
    n = 1000
    sims = [dict(seed=21 + k, M=1.0e4, dt_scale=1.0, nfw_scale=1.0, mn_scale=1.0) for k in range(4)]
    posm, vel, bparams, _ = _make_batch(n, sims)
    p1, v1 = _run(posm, vel, bparams, 20)
    p2, v2 = _run(posm, vel, bparams, 20)
    assert p1.tobytes() == p2.tobytes() and v1.tobytes() == v2.tobytes()
    cfg = W.CONFIGS[1]
    for k in range(4):
        dp, dv = torch.from_numpy(posm[k].copy()).cuda(), torch.from_numpy(vel[k].copy()).cuda()
        acc = torch.empty_like(dp)
        ws = B.alloc_workspace(B.workspace_bytes(n))
        B.leapfrog_kdk(dp, dv, acc, cfg.G, cfg.eps, cfg.dt, 20, bparams[k][3], ws)
        torch.cuda.synchronize()
        rel = np.abs(dp.cpu().numpy()[:, :3] - p1[k, :, :3]).max() / 12.4
        assert rel <= 2e-6


def test_ensemble_zero_steps_many_simulations_and_argument_errors():
    n, nsim = 300, 700                                          # more CTAs than one wave
    cfg = W.CONFIGS[1]
    p64, v64 = W.make_state(cfg, n=n)
    posm = np.repeat(W.to_f32(p64)[None], nsim, axis=0)
    vel = np.repeat(W.vel4(W.to_f32(v64), np.float32)[None], nsim, axis=0)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    p0, v0 = _run(posm, vel, [(cfg.G, cfg.eps, cfg.dt, pot)], 0)
    assert p0.tobytes() == posm.tobytes() and v0.tobytes() == vel.tobytes()
    p1, v1 = _run(posm, vel, [(cfg.G, cfg.eps, cfg.dt, pot)], 3)
    assert all(p1[k].tobytes() == p1[0].tobytes() for k in range(nsim))      # identical inputs, identical outputs
    dp, dv = torch.from_numpy(posm).cuda(), torch.from_numpy(vel).cuda()
    ws = B.alloc_workspace(B.ensemble_workspace_bytes(nsim))
    with pytest.raises(B.OdisseoError, match="ERR_ARG"):
        B.ensemble_leapfrog_kdk(dp, dv, [(cfg.G, cfg.eps, cfg.dt, pot)] * 2, 1, ws)       # 2 records for 700 sims
    with pytest.raises(B.OdisseoError, match="ERR_ARG"):
        B.ensemble_leapfrog_kdk(dp, dv, [(cfg.G, 0.0, cfg.dt, pot)], 1, ws)               # eps must be > 0
    big = torch.zeros(1, 2049, 4, device="cuda")
    with pytest.raises(B.OdisseoError, match="ERR_ARG"):
        B.ensemble_leapfrog_kdk(big, big.clone(), [(cfg.G, cfg.eps, cfg.dt, pot)], 1, ws)


# ---------------------------------------------------------------------------------------------
# reverse-mode derivative of the ensembles (oracle/adjoint.py, pinned by finite differences)
# ---------------------------------------------------------------------------------------------
def _run_vjp(posm, vel, bparams, nsteps, lx, lv, with_eps_G=False):
    nsim, n = posm.shape[:2]
    dp, dv = torch.from_numpy(posm.copy()).cuda(), torch.from_numpy(vel.copy()).cuda()
    ws = B.alloc_workspace(B.ensemble_workspace_bytes(nsim))
    tape = torch.empty(B.ensemble_tape_bytes(n, nsim, nsteps) // 4, dtype=torch.float32, device="cuda")
    B.ensemble_leapfrog_kdk_tape(dp, dv, bparams, nsteps, tape, ws)
    dlx, dlv = torch.from_numpy(lx.copy()).cuda(), torch.from_numpy(lv.copy()).cuda()
    gm = torch.full((nsim, n), float("nan"), dtype=torch.float64, device="cuda")
    gp = torch.full((nsim, B.NGRAD), float("nan"), dtype=torch.float64, device="cuda")
    B.ensemble_leapfrog_kdk_vjp(tape, bparams, nsteps, dlx, dlv, gm, gp, ws, with_eps_G=with_eps_G)
    torch.cuda.synchronize()
    return dp.cpu().numpy(), dv.cpu().numpy(), dlx.cpu().numpy(), dlv.cpu().numpy(), gm.cpu().numpy(), gp.cpu().numpy()


@pytest.mark.parametrize("n,nsteps", [(1000, 5), (300, 3), (1, 2), (1300, 2), (2048, 1)])
def test_ensemble_vjp_matches_the_oracle_adjoint_per_simulation(n, nsteps):
    from oracle import adjoint as A
    sims = [dict(seed=31, M=1.0e4, dt_scale=1.0, nfw_scale=1.0, mn_scale=1.0),
            dict(seed=32, M=2.0e4, dt_scale=0.5, nfw_scale=0.7, mn_scale=1.3),
            dict(seed=33, M=1.0e4, dt_scale=-1.0, nfw_scale=1.2, mn_scale=1.0, unequal=True)]
    posm, vel, bparams, oparams = _make_batch(n, sims)
    rng = np.random.Generator(np.random.PCG64(34))
    lx = np.zeros((3, n, 4), dtype=np.float32)
    lv = np.zeros((3, n, 4), dtype=np.float32)
    lx[:, :, :3] = rng.normal(size=(3, n, 3))
    lv[:, :, :3] = rng.normal(size=(3, n, 3)) * 10.0
    pf, vf, gx0, gv0, gm, gp = _run_vjp(posm, vel, bparams, nsteps, lx, lv)
    # the tape call leaves the same final state as the plain call
    p_plain, v_plain = _run(posm, vel, bparams, nsteps)
    assert pf.tobytes() == p_plain.tobytes() and vf.tobytes() == v_plain.tobytes()
    cfg = W.CONFIGS[1]
    for k, (G, eps, dt, _) in enumerate(oparams):
        s = sims[k]
        nfw = (cfg.nfw[0] * s["nfw_scale"], cfg.nfw[1])
        mn = (cfg.mn[0] * s["mn_scale"], cfg.mn[1], cfg.mn[2])
        ref = A.leapfrog_kdk_vjp(posm[k].astype(np.float64), vel[k, :, :3].astype(np.float64), G, eps, dt, nsteps,
                                 lx[k, :, :3].astype(np.float64), lv[k, :, :3].astype(np.float64), nfw, mn)
        # fp32 pull-back: 1e-3 of the largest component (measured ~3e-4 after 5 steps)
        assert np.abs(gx0[k, :, :3] - ref["x0"]).max() <= 1e-3 * np.abs(ref["x0"]).max(), "sim %d x0" % k
        assert np.abs(gv0[k, :, :3] - ref["v0"]).max() <= 1e-3 * np.abs(ref["v0"]).max(), "sim %d v0" % k
        assert np.abs(gm[k] - ref["m"]).max() <= 1e-3 * max(np.abs(ref["m"]).max(), 1e-300), "sim %d m" % k
        for name in ("M_s", "r_s", "M_d", "a", "b", "dt"):
            kk = B.GRADIENT_FIELDS.index(name)
            assert abs(gp[k, kk] - ref[name]) <= 1e-3 * abs(ref[name]), "sim %d %s" % (k, name)
        assert np.all(gx0[k, :, 3] == 0) and np.all(gv0[k, :, 3] == 0)
        assert gp[k, 5] == 0 and gp[k, 6] == 0                       # eps / G terms not requested
    # with the eps and G terms (general loop for every simulation): same gradients to rounding, slots 5, 6 filled
    _, _, gx1, gv1, gm1, gp1 = _run_vjp(posm, vel, bparams, nsteps, lx, lv, with_eps_G=True)
    for k, (G, eps, dt, _) in enumerate(oparams):
        s = sims[k]
        ref = A.leapfrog_kdk_vjp(posm[k].astype(np.float64), vel[k, :, :3].astype(np.float64), G, eps, dt, nsteps,
                                 lx[k, :, :3].astype(np.float64), lv[k, :, :3].astype(np.float64),
                                 (cfg.nfw[0] * s["nfw_scale"], cfg.nfw[1]), (cfg.mn[0] * s["mn_scale"], cfg.mn[1], cfg.mn[2]))
        assert np.abs(gx1[k, :, :3] - ref["x0"]).max() <= 1e-3 * np.abs(ref["x0"]).max()
        assert abs(gp1[k, 5] - ref["G"]) <= 2e-3 * abs(ref["G"])
        assert abs(gp1[k, 6] - ref["eps"]) <= 2e-2 * abs(ref["eps"]) + 1e-6 * abs(ref["dt"])


def test_ensemble_vjp_zero_steps_is_the_identity_and_is_reproducible():
    sims = [dict(seed=41 + k, M=1.0e4, dt_scale=1.0, nfw_scale=1.0, mn_scale=1.0) for k in range(2)]
    posm, vel, bparams, _ = _make_batch(500, sims)
    lx = np.random.Generator(np.random.PCG64(1)).normal(size=(2, 500, 4)).astype(np.float32)
    lv = np.random.Generator(np.random.PCG64(2)).normal(size=(2, 500, 4)).astype(np.float32)
    lx[:, :, 3] = 0
    lv[:, :, 3] = 0
    _, _, gx0, gv0, gm, gp = _run_vjp(posm, vel, bparams, 0, lx, lv)
    assert gx0.tobytes() == lx.tobytes() and gv0.tobytes() == lv.tobytes() and np.all(gm == 0) and np.all(gp == 0)
    a = _run_vjp(posm, vel, bparams, 6, lx, lv)
    b = _run_vjp(posm, vel, bparams, 6, lx, lv)
    for x, y in zip(a, b):
        assert x.tobytes() == y.tobytes()
