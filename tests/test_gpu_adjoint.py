"""GPU parity of the reverse-mode derivative against oracle/adjoint.py, which is itself
pinned by finite differences of the forward oracle.  fp64: 1e-10 relative to the largest gradient component;
fp32: tolerances derived from fp32 rounding of the pull-back."""
import numpy as np
import pytest
import torch

from oracle import adjoint as A
from oracle import oracle as O
from paper_2511_22468_b200 import binding as B
from paper_2511_22468_b200 import workloads as W

pytestmark = pytest.mark.gpu
NAMES = B.GRADIENT_FIELDS


def dev(a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def pad4(a, dtype):
    out = np.zeros((a.shape[0], 4), dtype=dtype)
    out[:, :3] = a
    return out


def gpu_accel_vjp(posm, c, G, eps, pot, dtype, with_eps_G=True):
    n = posm.shape[0]
    gx = torch.full((n, 4), float("nan"), dtype=torch.float32 if dtype == np.float32 else torch.float64, device="cuda")
    gm = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    gp = torch.full((B.NGRAD,), float("nan"), dtype=torch.float64, device="cuda")
    ws = B.alloc_workspace(B.vjp_workspace_bytes(n, dtype == np.float64))
    B.accel_vjp(dev(posm, dtype), dev(pad4(c, dtype), dtype), G, eps, pot, gx, gm, gp, ws, with_eps_G=with_eps_G)
    torch.cuda.synchronize()
    return gx.cpu().numpy().astype(np.float64), gm.cpu().numpy(), gp.cpu().numpy()


def _inputs(n, seed, dtype, unequal=True):
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.random_cloud(n, seed=seed, scale=0.01, centre=cfg.centre, unequal_mass=unequal)
    posm64[:, 3] *= cfg.M / n
    c = np.random.Generator(np.random.PCG64(seed + 1)).normal(size=(n, 3))
    p = posm64.astype(dtype)
    c = c.astype(dtype)
    G, eps = (float(np.float32(cfg.G)), float(np.float32(cfg.eps))) if dtype == np.float32 else (cfg.G, cfg.eps)
    return cfg, p, vel64.astype(dtype), c, G, eps


@pytest.mark.parametrize("n", [1, 2, 3, 127, 129, 513, 1000, 3001])
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 2e-5)])
def test_accel_vjp_matches_the_oracle(n, dtype, tol):
    cfg, p, _, c, G, eps = _inputs(n, 600 + n, dtype)
    gx, gm, gp = gpu_accel_vjp(p, c, G, eps, B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), dtype)
    p64, c64 = p.astype(np.float64), c.astype(np.float64)
    rx, rm, rp, rG, reps = A.accel_vjp(p64, c64, G, eps, cfg.nfw, cfg.mn)
    # scale of the per-particle sums: sum_j |term| is bounded by the pair part's own magnitude
    px, pm, pG, peps = A.pair_accel_vjp(p64, np.abs(c64), G, eps)
    sx = max(np.abs(rx).max(), 1e-300)
    assert np.abs(gx[:, :3] - rx).max() <= tol * sx and np.all(gx[:, 3] == 0)
    assert np.abs(gm - rm).max() <= tol * max(np.abs(rm).max(), 1e-300)
    ref = [rp[k] for k in A.PARAM_NAMES] + [rG, reps]
    for k, r in enumerate(ref):
        scale = max(abs(r), 1e-300)
        if k >= 5:                                         # G and eps sums cancel heavily between particles
            scale = max(scale, abs(pG) if k == 5 else abs(peps))
        assert abs(gp[k] - r) <= 10 * tol * scale, NAMES[k]
    assert gp[7] == 0
    # without the eps / G terms: same gradients, slots 5 and 6 left 0
    gx2, gm2, gp2 = gpu_accel_vjp(p, c, G, eps, B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), dtype, with_eps_G=False)
    assert gx2.tobytes() == gx.tobytes() and gm2.tobytes() == gm.tobytes()
    assert np.array_equal(gp2[:5], gp[:5]) and gp2[5] == 0 and gp2[6] == 0


@pytest.mark.parametrize("n", [2, 128, 513, 3001])
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-10), (np.float32, 2e-5)])
def test_accel_vjp_equal_masses_take_the_tile_wise_equal_mass_loop(n, dtype, tol):
    """All masses equal: full tiles run the loop without the mass (decided per tile on the device); the padded
    last tile and any tile with a different mass fall back to the general loop.  Same oracle, same tolerance."""
    cfg, p, _, c, G, eps = _inputs(n, 650 + n, dtype, unequal=False)
    gx, gm, gp = gpu_accel_vjp(p, c, G, eps, None, dtype, with_eps_G=False)
    rx, rm, _, _ = A.pair_accel_vjp(p.astype(np.float64), c.astype(np.float64), G, eps)
    assert np.abs(gx[:, :3] - rx).max() <= tol * np.abs(rx).max()
    assert np.abs(gm - rm).max() <= tol * max(np.abs(rm).max(), 1e-300)
    if n > 200:                                          # one odd mass in the middle: its tile goes general
        p2 = p.copy()
        p2[n // 2, 3] *= 3
        gx2, gm2, _ = gpu_accel_vjp(p2, c, G, eps, None, dtype, with_eps_G=False)
        rx2, rm2, _, _ = A.pair_accel_vjp(p2.astype(np.float64), c.astype(np.float64), G, eps)
        assert np.abs(gx2[:, :3] - rx2).max() <= tol * np.abs(rx2).max()
        assert np.abs(gm2 - rm2).max() <= tol * np.abs(rm2).max()


@pytest.mark.parametrize("n", [2, 129, 1000, 3001])
@pytest.mark.parametrize("dtype,tol", [(np.float64, 1e-12), (np.float32, 1e-5)])
@pytest.mark.parametrize("unequal", [True, False])
def test_accel_vjp_per_element_bound(n, dtype, tol, unequal):
    """Every particle's gradient against the sum of the magnitudes of ITS OWN terms (not the largest component of the
    whole array): |gx_i - ref_i| <= tol * G sum_j (f |u| + |g| |d| |d.u|), |gm_i - ref_i| <= tol * G sum_j f |d.c_j| --
    the forward tolerance's form (north_star: |a_gpu,i - a_ref,i| / sum_j |a_ij|) carried to the pull-back."""
    cfg, p, _, c, G, eps = _inputs(n, 900 + n, dtype, unequal=unequal)
    gx, gm, _ = gpu_accel_vjp(p, c, G, eps, None, dtype, with_eps_G=False)
    p64, c64 = p.astype(np.float64), c.astype(np.float64)
    rx, rm, _, _ = A.pair_accel_vjp(p64, c64, G, eps)
    Sx, Sm = A.pair_accel_vjp_scale(p64, c64, G, eps)
    assert np.all(np.linalg.norm(gx[:, :3] - rx, axis=1) <= tol * Sx)
    assert np.all(np.abs(gm - rm) <= tol * Sm)


@pytest.mark.parametrize("n,ntargets,variant", [(16384, 1024, "unequal"), (16384, 1024, "equal"), (16384, 1024, "odd_late"),
                                                (65536, 256, "unequal"), (65536, 256, "odd_late")])
def test_accel_vjp_at_the_benchmarked_sizes_on_seeded_targets(n, ntargets, variant):
    """The pull-back on the path the sizes bench.py times take (cfg1 / cfg2 shape): several tiles per unit (fp64 sums
    across tiles in flush_tile), the 4-stage ring wrapping around, CTAs that walk several units and cross i-blocks
    (N = 65,536: 7 / 13 units per CTA in fp32 / fp64), and -- "odd_late" -- one different mass in a LATE tile of an
    otherwise equal-mass cloud, so that the tile-wise equal-mass decision flips in the middle of a unit.  Oracle: the row
    form of oracle/adjoint.py (O(n) memory) on seeded targets, which always include the particle with the odd mass,
    the first and the last; per-element bound of test_accel_vjp_per_element_bound, fp32 and fp64 on the same
    fp32-rounded inputs."""
    cfg, p32, _, c32, G, eps = _inputs(n, 1200 + n, np.float32, unequal=(variant == "unequal"))
    odd = (7 * n) // 8 + 3
    if variant == "odd_late":
        p32[odd, 3] *= 3
    rng = np.random.Generator(np.random.PCG64(n + 5))
    targets = np.unique(np.concatenate([rng.choice(n, ntargets - 3, replace=False), [0, odd, n - 1]]))
    p64, c64 = p32.astype(np.float64), c32.astype(np.float64)
    rx, rm, _, _ = A.pair_accel_vjp(p64, c64, G, eps, targets=targets)
    Sx, Sm = A.pair_accel_vjp_scale(p64, c64, G, eps, targets=targets)
    assert np.all(Sx > 0) and np.all(Sm > 0)
    for dtype, tol in ((np.float32, 1e-5), (np.float64, 1e-12)):
        gx, gm, _ = gpu_accel_vjp(p32.astype(dtype), c32.astype(dtype), G, eps, None, dtype, with_eps_G=False)
        ex = np.linalg.norm(gx[targets, :3] - rx, axis=1) / Sx
        em = np.abs(gm[targets] - rm) / Sm
        print("n %d %s %s: max err / scale  gx %.2e gm %.2e" % (n, variant, dtype.__name__, ex.max(), em.max()))
        assert ex.max() <= tol and em.max() <= tol
        assert np.all(gx[:, 3] == 0) and np.all(np.isfinite(gx)) and np.all(np.isfinite(gm))


def test_leapfrog_vjp_f64_with_several_tiles_per_unit_matches_the_row_wise_oracle():
    """n = 6,000 x 3 steps in fp64: the pull-back plan gives 12 chunks of 504 records = 4 tiles of 128 per unit (the
    n <= 3,001 cases above are one tile per unit), through the whole tape / KDK reverse loop.  Oracle: leapfrog_kdk_vjp
    with rowwise=True (the dense form would need [n, n, 3] arrays)."""
    n, nsteps = 6000, 3
    cfg, p, v, _, G, eps = _inputs(n, 1300, np.float64)
    v = v * 0.02 + np.asarray(cfg.velocity)
    rng = np.random.Generator(np.random.PCG64(12))
    lx, lv = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)) * 10.0
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    gx0, gv0, gm, gp, _ = gpu_leapfrog_vjp(p, v, G, eps, cfg.dt, nsteps, pot, lx, lv, np.float64)
    ref = A.leapfrog_kdk_vjp(p, v, G, eps, cfg.dt, nsteps, lx, lv, cfg.nfw, cfg.mn, rowwise=True)
    assert np.abs(gx0[:, :3] - ref["x0"]).max() <= 1e-9 * np.abs(ref["x0"]).max()
    assert np.abs(gv0[:, :3] - ref["v0"]).max() <= 1e-9 * np.abs(ref["v0"]).max()
    assert np.abs(gm - ref["m"]).max() <= 1e-9 * np.abs(ref["m"]).max()
    for k, name in enumerate(NAMES):
        assert abs(gp[k] - ref[name]) <= 1e-8 * abs(ref[name]) + 1e-13 * abs(ref["dt"]), name


def test_accel_vjp_without_potential_and_reproducible():
    cfg, p, _, c, G, eps = _inputs(2000, 77, np.float64)
    a = gpu_accel_vjp(p, c, G, eps, None, np.float64)
    b = gpu_accel_vjp(p, c, G, eps, None, np.float64)
    for x, y in zip(a, b):
        assert x.tobytes() == y.tobytes()
    rx, rm, rG, reps = A.pair_accel_vjp(p, c, G, eps)
    assert np.abs(a[0][:, :3] - rx).max() <= 1e-11 * np.abs(rx).max()
    assert np.all(a[2][:5] == 0)


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n,nsteps,unequal", [(1, 2, False), (129, 4, True), (1000, 6, False), (2048, 3, False)])
def test_tape_of_the_flag_in_data_kernel_equals_the_per_step_tape(n, nsteps, unequal, dtype):
    """At small n the forward pass with a tape is ONE launch of the owner-computes kernel (csrc/ll_kdk.cuh), whose owner
    threads store the snapshots {x_k, v_k, pair-only a_k}; tape and final state must equal the per-step launches' bit for bit."""
    cfg, p, v, _, G, eps = _inputs(n, 40 + n, dtype, unequal=unequal)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    dt = float(np.float32(cfg.dt)) if dtype == np.float32 else cfg.dt
    out = []
    try:
        for ll in (6144, 0):
            B.set_ll_max_n(ll)
            posm, vel = dev(p, dtype), dev(W.vel4(v, dtype), dtype)
            acc = torch.empty_like(posm)
            ws = B.alloc_workspace(B.workspace_bytes(n, dtype == np.float64))
            tape = torch.full((B.tape_bytes(n, nsteps, dtype == np.float64) // posm.element_size(),), float("nan"), dtype=posm.dtype, device="cuda")
            c0 = B.launch_count()
            B.leapfrog_kdk_tape(posm, vel, acc, G, eps, dt, nsteps, pot, tape, ws)
            torch.cuda.synchronize()
            assert (B.launch_count() - c0 == 1) == (ll != 0)
            out.append((tape.cpu().numpy(), posm.cpu().numpy(), vel.cpu().numpy(), acc.cpu().numpy()))
    finally:
        B.set_ll_max_n(-1)
    for a, b in zip(*out):
        assert a.tobytes() == b.tobytes()


def gpu_leapfrog_vjp(p, v, G, eps, dt, nsteps, pot, lx, lv, dtype):
    n = p.shape[0]
    posm, vel = dev(p, dtype), dev(W.vel4(v, dtype), dtype)
    acc = torch.empty_like(posm)
    ws = B.alloc_workspace(max(B.workspace_bytes(n, dtype == np.float64), B.vjp_workspace_bytes(n, dtype == np.float64)))
    tape = torch.empty(B.tape_bytes(n, nsteps, dtype == np.float64) // posm.element_size(), dtype=posm.dtype, device="cuda")
    B.leapfrog_kdk_tape(posm, vel, acc, G, eps, dt, nsteps, pot, tape, ws)
    dlx, dlv = dev(pad4(lx, dtype), dtype), dev(pad4(lv, dtype), dtype)
    gm = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda")
    gp = torch.full((B.NGRAD,), float("nan"), dtype=torch.float64, device="cuda")
    B.leapfrog_kdk_vjp(tape, n, G, eps, dt, nsteps, pot, dlx, dlv, gm, gp, ws, with_eps_G=True)
    torch.cuda.synchronize()
    final = (posm.cpu().numpy(), vel.cpu().numpy(), acc.cpu().numpy())
    return dlx.cpu().numpy().astype(np.float64), dlv.cpu().numpy().astype(np.float64), gm.cpu().numpy(), gp.cpu().numpy(), final


@pytest.mark.parametrize("n,nsteps", [(1, 3), (64, 0), (300, 1), (1000, 10)])
def test_leapfrog_vjp_f64_matches_the_oracle_and_the_tape_call_matches_the_plain_call(n, nsteps):
    cfg, p, v, _, G, eps = _inputs(n, 700 + n, np.float64)
    v = v * 0.02 + np.asarray(cfg.velocity)
    rng = np.random.Generator(np.random.PCG64(9))
    lx, lv = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)) * 10.0
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    gx0, gv0, gm, gp, final = gpu_leapfrog_vjp(p, v, G, eps, cfg.dt, nsteps, pot, lx, lv, np.float64)
    ref = A.leapfrog_kdk_vjp(p, v, G, eps, cfg.dt, nsteps, lx, lv, cfg.nfw, cfg.mn)
    assert np.abs(gx0[:, :3] - ref["x0"]).max() <= 1e-9 * np.abs(ref["x0"]).max()
    assert np.abs(gv0[:, :3] - ref["v0"]).max() <= 1e-9 * np.abs(ref["v0"]).max()
    if nsteps:
        assert np.abs(gm - ref["m"]).max() <= 1e-9 * max(np.abs(ref["m"]).max(), 1e-300)
        for k, name in enumerate(NAMES):
            assert abs(gp[k] - ref[name]) <= 1e-8 * abs(ref[name]) + 1e-13 * abs(ref["dt"]), name
    else:
        assert np.all(gm == 0) and np.all(gp == 0)
    # forward with tape == plain forward, bit for bit
    posm, vel = dev(p, np.float64), dev(W.vel4(v, np.float64), np.float64)
    acc = torch.empty_like(posm)
    B.leapfrog_kdk(posm, vel, acc, G, eps, cfg.dt, nsteps, pot, B.alloc_workspace(B.workspace_bytes(n, True)))
    torch.cuda.synchronize()
    for got, want in zip(final, (posm, vel, acc)):
        assert got.tobytes() == want.cpu().numpy().tobytes()


def test_leapfrog_vjp_f32_against_the_fp64_oracle():
    """fp32 state, 5 steps, N = 1,000 (the paper's inference size): gradients agree with the fp64 oracle run on the
    same fp32-rounded inputs to 1e-3 of the largest component (fp32 pull-back through an N-body system amplifies
    rounding by the same Jacobians it propagates; measured ~1e-5)."""
    n, nsteps = 1000, 5
    cfg, p, v, _, G, eps = _inputs(n, 800, np.float32, unequal=False)
    v = (v.astype(np.float64) * 0.02 + np.asarray(cfg.velocity)).astype(np.float32)
    dt = float(np.float32(cfg.dt))
    rng = np.random.Generator(np.random.PCG64(10))
    lx, lv = rng.normal(size=(n, 3)).astype(np.float32), (rng.normal(size=(n, 3)) * 10.0).astype(np.float32)
    gx0, gv0, gm, gp, _ = gpu_leapfrog_vjp(p, v, G, eps, dt, nsteps, B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), lx, lv, np.float32)
    ref = A.leapfrog_kdk_vjp(p.astype(np.float64), v.astype(np.float64), G, eps, dt, nsteps, lx.astype(np.float64),
                             lv.astype(np.float64), cfg.nfw, cfg.mn)
    print("fp32 vjp rel err x0 %.2e v0 %.2e m %.2e" % (np.abs(gx0[:, :3] - ref["x0"]).max() / np.abs(ref["x0"]).max(),
          np.abs(gv0[:, :3] - ref["v0"]).max() / np.abs(ref["v0"]).max(), np.abs(gm - ref["m"]).max() / np.abs(ref["m"]).max()))
    assert np.abs(gx0[:, :3] - ref["x0"]).max() <= 1e-3 * np.abs(ref["x0"]).max()
    assert np.abs(gv0[:, :3] - ref["v0"]).max() <= 1e-3 * np.abs(ref["v0"]).max()
    assert np.abs(gm - ref["m"]).max() <= 1e-3 * np.abs(ref["m"]).max()
    for k, name in enumerate(NAMES[:5] + ("dt",)):
        kk = NAMES.index(name)
        assert abs(gp[kk] - ref[name]) <= 1e-3 * abs(ref[name]), name


def test_gradient_of_the_gpu_forward_by_finite_differences():
    """Independent of the oracle: d(loss)/d(M_NFW) and d(loss)/d(dt) of the GPU fp64 forward by central differences
    reproduce the GPU reverse-mode values (the paper's Theta contains t_end and M_NFW)."""
    n, nsteps = 400, 8
    cfg, p, v, _, G, eps = _inputs(n, 900, np.float64)
    v = v * 0.02 + np.asarray(cfg.velocity)
    rng = np.random.Generator(np.random.PCG64(11))
    lx, lv = rng.normal(size=(n, 3)), rng.normal(size=(n, 3)) * 10.0

    def forward_loss(nfw, dt):
        posm, vel = dev(p, np.float64), dev(W.vel4(v, np.float64), np.float64)
        acc = torch.empty_like(posm)
        B.leapfrog_kdk(posm, vel, acc, G, eps, dt, nsteps, B.Potential.make(nfw=nfw, mn=cfg.mn),
                       B.alloc_workspace(B.workspace_bytes(n, True)))
        torch.cuda.synchronize()
        return float(np.sum(lx * posm.cpu().numpy()[:, :3]) + np.sum(lv * vel.cpu().numpy()[:, :3]))
    _, _, _, gp, _ = gpu_leapfrog_vjp(p, v, G, eps, cfg.dt, nsteps, B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), lx, lv, np.float64)
    hM = 1e6
    fd_M = (forward_loss((cfg.nfw[0] + hM, cfg.nfw[1]), cfg.dt) - forward_loss((cfg.nfw[0] - hM, cfg.nfw[1]), cfg.dt)) / (2 * hM)
    hd = 1e-6
    fd_dt = (forward_loss(cfg.nfw, cfg.dt + hd) - forward_loss(cfg.nfw, cfg.dt - hd)) / (2 * hd)
    assert abs(gp[0] - fd_M) <= 1e-5 * abs(fd_M)
    assert abs(gp[7] - fd_dt) <= 1e-6 * abs(fd_dt)
