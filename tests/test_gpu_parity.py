"""GPU parity: the CUDA path (through the C ABI) against the fp64 CPU oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json north_star's:
  fp32 pair:  |a_gpu,i - a_ref,i| / sum_j |a_ij| <= 1e-5 for every particle
  fp64 pair:  the same ratio <= 1e-12
  config 0, fp64, 10 steps: positions agree to <= 1e-10 relative
fp32 trajectory tolerances are SURVEY.md 8c (iii)/(iv), derived in DESIGN.md.
"""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2511_22468_b200 import binding as B
from paper_2511_22468_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL_F32 = 1e-5
TOL_F64 = 1e-12


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "gpu tests need a B200"
    B.lib()


def dev(a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def gpu_pair(posm_np, G, eps, dtype):
    posm = dev(posm_np, dtype)
    acc = torch.full_like(posm, float("nan"))
    ws = B.alloc_workspace(B.workspace_bytes(posm.shape[0], dtype == np.float64))
    B.pair_accel(posm, acc, G, eps, ws)
    torch.cuda.synchronize()
    return acc.cpu().numpy()


def pair_ratio(acc_gpu, posm64, G, eps, targets=None):
    ref, S = O.pair_accel(posm64, G, eps, targets=targets)
    got = acc_gpu[:, :3].astype(np.float64)
    if targets is not None:
        got = got[targets]
    num = np.linalg.norm(got - ref, axis=1)
    with np.errstate(invalid="ignore", divide="ignore"):
        ratio = np.where(S > 0, num / S, np.where(num == 0, 0.0, np.inf))
    return float(ratio.max()) if ratio.size else 0.0


def f32_inputs(posm64, G, eps):
    """Same seeded inputs for both sides: fp32-rounded state and scalars, promoted to double."""
    p32 = W.to_f32(posm64)
    return p32, p32.astype(np.float64), float(np.float32(G)), float(np.float32(eps))


@pytest.mark.parametrize("n", [1, 2, 3, 31, 127, 129, 1000, 1025, 4096, 4097, 5000, 9001])
def test_pair_f32_ragged_sizes_unequal_masses(n):
    posm64, _ = W.random_cloud(n, seed=100 + n)
    p32, p64, G, eps = f32_inputs(posm64, 1.0, 0.05)
    acc = gpu_pair(p32, G, eps, np.float32)
    assert np.all(acc[:, 3] == 0)
    assert pair_ratio(acc, p64, G, eps) <= TOL_F32


def test_pair_f32_accepted_region_of_tiny_softening_with_unequal_masses():
    """include/odisseo.h: eps >= 1e-12 is accepted in fp32, and with unequal masses the self term m_j eps^-3 must stay below
    FLT_MAX.  Inside the region (m <= 300 at eps = 1.1e-12: 2.3e38) the result meets the usual tolerance; just outside (one
    mass of 500: 3.8e38 = inf, inf * 0 = NaN) the accelerations are NaN, as documented -- not silently wrong numbers."""
    n = 700
    posm64, _ = W.random_cloud(n, seed=4242)
    posm64[:, 3] = np.random.Generator(np.random.PCG64(1)).uniform(100.0, 300.0, n)
    p32, p64, G, eps = f32_inputs(posm64, 1.0, 1.1e-12)       # float32(1e-12) itself rounds below the bound
    acc = gpu_pair(p32, G, eps, np.float32)
    assert np.all(np.isfinite(acc)) and pair_ratio(acc, p64, G, eps) <= TOL_F32
    p32[n // 2, 3] = 500.0
    assert not np.all(np.isfinite(gpu_pair(p32, G, eps, np.float32)[:, :3]))
    p32[:, 3] = 500.0                                    # equal masses: applied in fp64 after the sum, no bound
    acc = gpu_pair(p32, G, eps, np.float32)
    assert np.all(np.isfinite(acc)) and pair_ratio(acc, p32.astype(np.float64), G, eps) <= TOL_F32


@pytest.mark.parametrize("n", [1, 2, 127, 1000, 1025, 4097, 6000])
def test_pair_f64_ragged_sizes_unequal_masses(n):
    posm64, _ = W.random_cloud(n, seed=200 + n)
    acc = gpu_pair(posm64, 1.0, 0.05, np.float64)
    assert pair_ratio(acc, posm64, 1.0, 0.05) <= TOL_F64


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n", [1, 2, 3, 127, 129, 1000, 1025, 4097, 5000])
def test_pair_equal_masses_ragged_sizes_take_the_equal_mass_path(n, dtype):
    """All masses equal: the kernels drop the per-source mass factor from the inner loop (the staging
    kernel's flags decide on the device); ragged tails are padded with far-away zero-mass records."""
    posm64, _ = W.random_cloud(n, seed=300 + n, unequal_mass=False)
    posm64[:, 3] = 0.37
    if dtype == np.float32:
        p, p64, G, eps = f32_inputs(posm64, 1.0, 0.05)
        tol = TOL_F32
    else:
        p, p64, G, eps, tol = posm64, posm64, 1.0, 0.05, TOL_F64
    acc = gpu_pair(p, G, eps, dtype)
    assert np.all(np.isfinite(acc))
    assert pair_ratio(acc, p64, G, eps) <= tol


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n,odd", [(1025, 1024), (5000, 0), (5000, 4999), (9001, 4500)])
def test_pair_one_different_mass_anywhere_selects_the_general_path(n, odd, dtype):
    """A single particle whose mass differs (first, middle or last record, incl. the ragged tail block) must
    switch every CTA to the general kernel; using the equal-mass path would miss a factor 5."""
    posm64, _ = W.random_cloud(n, seed=400 + n, unequal_mass=False)
    posm64[odd, 3] = 5.0
    if dtype == np.float32:
        p, p64, G, eps = f32_inputs(posm64, 1.0, 0.05)
        tol = TOL_F32
    else:
        p, p64, G, eps, tol = posm64, posm64, 1.0, 0.05, TOL_F64
    acc = gpu_pair(p, G, eps, dtype)
    assert pair_ratio(acc, p64, G, eps) <= tol
    # and the decision is re-taken on every call with the same workspace
    posm = dev(p, dtype)
    out = torch.empty_like(posm)
    ws = B.alloc_workspace(B.workspace_bytes(n, dtype == np.float64))
    B.pair_accel(posm, out, G, eps, ws)
    posm[odd, 3] = 1.0
    B.pair_accel(posm, out, G, eps, ws)
    torch.cuda.synchronize()
    p64b = p64.copy()
    p64b[odd, 3] = 1.0
    assert pair_ratio(out.cpu().numpy(), p64b, G, eps) <= tol


@pytest.mark.parametrize("ci", [0, 1, 2])
def test_pair_f32_configs_full(ci):
    """step-0 acceleration parity at FULL N for configs 0-2 (config 2: 4.3e9 oracle
    interactions, ~1 s on the box's cores)."""
    cfg = W.CONFIGS[ci]
    posm64, _ = W.make_state(cfg)
    p32, p64, G, eps = f32_inputs(posm64, cfg.G, cfg.eps)
    acc = gpu_pair(p32, G, eps, np.float32)
    assert pair_ratio(acc, p64, G, eps) <= TOL_F32


def test_pair_f64_config0_full():
    cfg = W.CONFIGS[0]
    posm64, _ = W.make_state(cfg)
    acc = gpu_pair(posm64, cfg.G, cfg.eps, np.float64)
    assert pair_ratio(acc, posm64, cfg.G, cfg.eps) <= TOL_F64


def test_pair_beyond_the_baseline_sizes_ragged_two_million():
    """Twice the largest BASELINE size plus a ragged tail (N = 2^21 + 5, config 4's shape, fp32): 4.4e12 interactions in
    one evaluation, checked on 1,024 seeded targets against all sources (index arithmetic and workspace sizes past 2^31
    bytes of rows and 2^42 interactions)."""
    cfg = W.CONFIGS[4]
    n = (1 << 21) + 5
    posm64, _ = W.make_state(cfg, n=n)
    p, p64, G, eps = f32_inputs(posm64, cfg.G, cfg.eps)
    acc = gpu_pair(p, G, eps, np.float32)
    assert np.all(np.isfinite(acc))
    idx = W.target_subset(n, size=1024)
    assert pair_ratio(acc, p64, G, eps, targets=idx) <= TOL_F32


@pytest.mark.parametrize("ci,dtype", [(2, np.float32), (3, np.float32), (3, np.float64), (4, np.float32)])
def test_pair_full_size_on_seeded_target_subset(ci, dtype):
    """BASELINE.json full sizes in the launch configuration bench.py times; the oracle
    evaluates the seeded 4,096-target subset against all sources."""
    cfg = W.CONFIGS[ci]
    posm64, _ = W.make_state(cfg)
    idx = W.target_subset(cfg.n)
    if dtype == np.float32:
        p, p64, G, eps = f32_inputs(posm64, cfg.G, cfg.eps)
        tol = TOL_F32
    else:
        p, p64, G, eps, tol = posm64, posm64, cfg.G, cfg.eps, TOL_F64
    acc = gpu_pair(p, G, eps, dtype)
    assert np.all(np.isfinite(acc))
    assert pair_ratio(acc, p64, G, eps, targets=idx) <= tol


def test_pair_is_bit_reproducible_and_obeys_newtons_third_law():
    cfg = W.CONFIGS[1]
    posm64, _ = W.make_state(cfg)
    p32, p64, G, eps = f32_inputs(posm64, cfg.G, cfg.eps)
    a1 = gpu_pair(p32, G, eps, np.float32)
    a2 = gpu_pair(p32, G, eps, np.float32)
    assert a1.tobytes() == a2.tobytes()
    m = p64[:, 3:4]
    a = a1[:, :3].astype(np.float64)
    assert np.linalg.norm(np.sum(m * a, axis=0)) / np.sum(m[:, 0] * np.linalg.norm(a, axis=1)) <= 1e-5


def test_pair_coincident_particles_and_self_term_contribute_zero():
    posm = np.array([[1, 2, 3, 1.0], [1, 2, 3, 5.0], [2, 2, 3, 2.0]])
    acc = gpu_pair(posm.astype(np.float32), 1.0, 0.5, np.float32)
    assert pair_ratio(acc, posm, 1.0, 0.5) <= TOL_F32
    one = gpu_pair(np.array([[4.0, 5.0, 6.0, 7.0]], dtype=np.float32), 1.0, 0.5, np.float32)
    assert np.all(one == 0)


def test_pair_soa_matches_aos_bitwise():
    posm64, _ = W.random_cloud(3001, seed=5)
    p32 = W.to_f32(posm64)
    ref = gpu_pair(p32, 1.0, 0.05, np.float32)
    cols = [dev(p32[:, k].copy(), np.float32) for k in range(4)]
    outs = [torch.empty(3001, device="cuda") for _ in range(3)]
    ws = B.alloc_workspace(B.workspace_bytes(3001) + 32 * 3001 + 512)
    B.pair_accel_soa(*cols, *outs, 1.0, 0.05, ws)
    torch.cuda.synchronize()
    for k in range(3):
        assert outs[k].cpu().numpy().tobytes() == np.ascontiguousarray(ref[:, k]).tobytes()


# ---------------------------------------------------------------------------------------------
# external potential
# ---------------------------------------------------------------------------------------------
def _mw(cfg=W.CONFIGS[1]):
    return B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), O.Potential.make(nfw=cfg.nfw, mn=cfg.mn)


@pytest.mark.parametrize("dtype,tol", [(np.float32, 2e-6), (np.float64, 1e-13)])
def test_ext_accel_workload_radii(dtype, tol):
    cfg = W.CONFIGS[2]
    posm64, _ = W.make_state(cfg, n=5000)
    posm64[:2000, :3] = np.random.Generator(np.random.PCG64(3)).uniform(-25, 25, (2000, 3))   # whole galaxy
    bpot, opot = _mw(cfg)
    if dtype == np.float32:
        p = W.to_f32(posm64)
        p64, G = p.astype(np.float64), float(np.float32(cfg.G))
    else:
        p, p64, G = posm64, posm64, cfg.G
    posm = dev(p, dtype)
    acc = torch.full_like(posm, float("nan"))
    B.ext_accel(posm, acc, G, bpot)
    ref = O.ext_accel(p64, G, opot)
    got = acc.cpu().numpy()[:, :3].astype(np.float64)
    rel = np.linalg.norm(got - ref, axis=1) / np.linalg.norm(ref, axis=1)
    assert rel.max() <= tol
    B.ext_accel(posm, acc, G, bpot, accumulate=True)                # acc.xyz += a_ext
    got2 = acc.cpu().numpy()[:, :3].astype(np.float64)
    assert np.abs(got2 - 2 * got).max() <= 1e-6 * np.abs(got).max()
    B.ext_accel(posm, acc, G, None)
    assert np.all(acc.cpu().numpy() == 0)


def _nfw_accel_mpmath(pts, G, Ms, rs):
    """40-digit evaluation of the NFW formula (include/odisseo.h): the fp64 oracle itself loses
    ~eps * 2 r_s / r to cancellation at r << r_s, so small radii are checked against this."""
    import mpmath
    mpmath.mp.dps = 40
    out = np.zeros((len(pts), 3))
    for k, p in enumerate(pts):
        x = [mpmath.mpf(float(t)) for t in p]
        r = mpmath.sqrt(x[0] ** 2 + x[1] ** 2 + x[2] ** 2)
        c = r / mpmath.mpf(rs)
        f = -mpmath.mpf(G) * mpmath.mpf(Ms) * (mpmath.log(1 + c) - c / (1 + c)) / r ** 3
        out[k] = [float(f * t) for t in x]
    return out


@pytest.mark.parametrize("dtype,tol", [(np.float32, 3e-6), (np.float64, 1e-13)])
def test_ext_accel_small_radii_series_branch_and_origin(dtype, tol):
    r = np.geomspace(1e-4, 5.0, 400)
    dirs = np.random.Generator(np.random.PCG64(8)).normal(size=(400, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    posm64 = np.concatenate([r[:, None] * dirs, np.ones((400, 1))], axis=1)
    posm64 = np.concatenate([posm64, [[0, 0, 0, 1.0]]])
    p = posm64.astype(dtype)
    nfw_b = B.Potential.make(nfw=W.NFW_MW)
    G = float(np.float32(W.G_KPC_MSUN_MYR)) if dtype == np.float32 else W.G_KPC_MSUN_MYR
    posm = dev(p, dtype)
    acc = torch.empty_like(posm)
    B.ext_accel(posm, acc, G, nfw_b)
    got = acc.cpu().numpy()[:, :3].astype(np.float64)
    ref = _nfw_accel_mpmath(p[:-1, :3].astype(np.float64), G, *W.NFW_MW)
    assert np.all(got[-1] == 0)
    rel = np.linalg.norm(got[:-1] - ref, axis=1) / np.linalg.norm(ref, axis=1)
    assert rel.max() <= tol
    # where the oracle is well conditioned (r >= 1 kpc) the two references agree
    far = r >= 1.0
    oref = O.ext_accel(p[:-1].astype(np.float64), G, O.Potential.make(nfw=W.NFW_MW))
    assert (np.linalg.norm(oref[far] - ref[far], axis=1) / np.linalg.norm(ref[far], axis=1)).max() <= 1e-14


# ---------------------------------------------------------------------------------------------
# leapfrog
# ---------------------------------------------------------------------------------------------
def gpu_leapfrog(posm_np, vel_np, G, eps, dt, nsteps, pot, dtype, acc_valid=False, acc_np=None, chunks=None):
    posm = dev(posm_np, dtype)
    vel = dev(W.vel4(vel_np, dtype) if vel_np.shape[1] == 3 else vel_np, dtype)
    acc = dev(acc_np, dtype) if acc_np is not None else torch.full_like(posm, float("nan"))
    ws = B.alloc_workspace(B.workspace_bytes(posm.shape[0], dtype == np.float64))
    valid = acc_valid
    for k in (chunks or [nsteps]):
        B.leapfrog_kdk(posm, vel, acc, G, eps, dt, k, pot, ws, acc_valid=valid)
        valid = True
    torch.cuda.synchronize()
    return posm.cpu().numpy(), vel.cpu().numpy(), acc.cpu().numpy()


def test_leapfrog_f64_config0_ten_steps_matches_oracle_to_1e10():
    cfg = W.CONFIGS[0]
    posm64, vel64 = W.make_state(cfg)
    p, v, a = gpu_leapfrog(posm64, vel64, cfg.G, cfg.eps, cfg.dt, cfg.nsteps, None, np.float64)
    pr, vr, _ = O.leapfrog_kdk(posm64, vel64, cfg.G, cfg.eps, cfg.dt, cfg.nsteps)
    dx = np.linalg.norm(p[:, :3] - pr[:, :3], axis=1) / np.maximum(np.linalg.norm(pr[:, :3], axis=1), cfg.a)
    dv = np.linalg.norm(v[:, :3] - vr, axis=1) / np.maximum(np.linalg.norm(vr, axis=1), np.sqrt(cfg.G * cfg.M / cfg.a))
    assert dx.max() <= 1e-10 and dv.max() <= 1e-10
    assert np.array_equal(p[:, 3], posm64[:, 3])                       # masses preserved
    assert pair_ratio(a, p, cfg.G, cfg.eps) <= TOL_F64                 # acc == a_pair(x_final)


@pytest.mark.parametrize("ci,n", [(0, None), (1, 4096), (1, None)])
def test_leapfrog_f32_ten_steps_short_horizon_parity(ci, n):
    """10 fp32 steps against the fp64 oracle from the same fp32-rounded state:
    |dx| <= 1e-5 max(|x|, a),  |dv| <= 1e-5 |v| + 1.5e-4 |dt| (S_i + |a_ext,i|)."""
    cfg = W.CONFIGS[ci]
    posm64, vel64 = W.make_state(cfg, n=n)
    p32, v32 = W.to_f32(posm64), W.to_f32(vel64)
    G, eps, dt = (float(np.float32(t)) for t in (cfg.G, cfg.eps, cfg.dt))
    bpot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
    opot = O.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
    p, v, a = gpu_leapfrog(p32, v32, G, eps, dt, 10, bpot, np.float32)
    pr, vr, _ = O.leapfrog_kdk(p32.astype(np.float64), v32.astype(np.float64), G, eps, dt, 10, opot)
    _, S = O.pair_accel(pr, G, eps)
    aext = np.linalg.norm(O.ext_accel(pr, G, opot), axis=1)
    dx = np.linalg.norm(p[:, :3] - pr[:, :3], axis=1)
    dv = np.linalg.norm(v[:, :3] - vr, axis=1)
    assert np.all(dx <= 1e-5 * np.maximum(np.linalg.norm(pr[:, :3], axis=1), cfg.a))
    assert np.all(dv <= 1e-5 * np.linalg.norm(vr, axis=1) + 1.5e-4 * abs(dt) * (S + aext))
    # re-synchronised parity (8c ii): acc left by the call is a_pair of the GPU's own final state
    assert pair_ratio(a, p.astype(np.float64), G, eps) <= TOL_F32


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_leapfrog_chained_calls_are_bit_identical_to_one_call(dtype):
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.make_state(cfg, n=3000)
    p0, v0 = posm64.astype(dtype), vel64.astype(dtype)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    one = gpu_leapfrog(p0, v0, cfg.G, cfg.eps, cfg.dt, 23, pot, dtype)
    chained = gpu_leapfrog(p0, v0, cfg.G, cfg.eps, cfg.dt, 23, pot, dtype, chunks=[1, 0, 2, 19, 1])
    again = gpu_leapfrog(p0, v0, cfg.G, cfg.eps, cfg.dt, 23, pot, dtype)
    for x, y, z in zip(one, chained, again):
        assert x.tobytes() == y.tobytes() == z.tobytes()


def test_leapfrog_zero_steps_evaluates_acc_only_and_negative_dt_reverses():
    cfg = W.CONFIGS[0]
    posm64, vel64 = W.make_state(cfg)
    p, v, a = gpu_leapfrog(posm64, vel64, cfg.G, cfg.eps, cfg.dt, 0, None, np.float64)
    assert np.array_equal(p, posm64) and np.array_equal(v[:, :3], vel64)
    assert pair_ratio(a, posm64, cfg.G, cfg.eps) <= TOL_F64
    pf, vf, af = gpu_leapfrog(posm64, vel64, cfg.G, cfg.eps, cfg.dt, 20, None, np.float64)
    pb, vb, _ = gpu_leapfrog(pf, vf, cfg.G, cfg.eps, -cfg.dt, 20, None, np.float64, acc_valid=True, acc_np=af)
    assert np.abs(pb[:, :3] - posm64[:, :3]).max() <= 1e-12 and np.abs(vb[:, :3] - vel64).max() <= 1e-12


def test_leapfrog_host_face_matches_device_face_bitwise():
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.make_state(cfg, n=5000)
    p32, v32 = W.to_f32(posm64), W.vel4(W.to_f32(vel64), np.float32)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    ref = gpu_leapfrog(p32, v32, cfg.G, cfg.eps, cfg.dt, 7, pot, np.float32)
    hp = torch.from_numpy(p32.copy()).pin_memory()
    hv = torch.from_numpy(v32.copy()).pin_memory()
    ha = torch.empty_like(hp).pin_memory()
    ws = B.alloc_workspace(B.host_workspace_bytes(5000))
    B.leapfrog_kdk_host(hp, hv, ha, cfg.G, cfg.eps, cfg.dt, 7, pot, ws)
    torch.cuda.synchronize()
    assert hp.numpy().tobytes() == ref[0].tobytes()
    assert hv.numpy().tobytes() == ref[1].tobytes()
    assert ha.numpy().tobytes() == ref[2].tobytes()
    # chained host calls re-upload the pair-only acceleration (acc_valid) and stay bit-identical
    hp2 = torch.from_numpy(p32.copy()).pin_memory()
    hv2 = torch.from_numpy(v32.copy()).pin_memory()
    ha2 = torch.empty_like(hp2).pin_memory()
    B.leapfrog_kdk_host(hp2, hv2, ha2, cfg.G, cfg.eps, cfg.dt, 3, pot, ws)
    torch.cuda.synchronize()
    B.leapfrog_kdk_host(hp2, hv2, ha2, cfg.G, cfg.eps, cfg.dt, 4, pot, ws, acc_valid=True)
    torch.cuda.synchronize()
    assert hp2.numpy().tobytes() == ref[0].tobytes()
    assert hv2.numpy().tobytes() == ref[1].tobytes()
    assert ha2.numpy().tobytes() == ref[2].tobytes()


def test_launch_count_and_pair_kernel_profile():
    """Instrumentation used by bench.py: the launch counter counts graph-replayed kernels, and a
    profile brackets exactly the pair-kernel launches without changing results."""
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.make_state(cfg, n=6000)                                     # above the whole-loop kernel's range
    p32, v32 = W.to_f32(posm64), W.to_f32(vel64)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    c0 = B.launch_count()
    ref = gpu_leapfrog(p32, v32, cfg.G, cfg.eps, cfg.dt, 40, pot, np.float32)     # graph replay inside
    c1 = B.launch_count()
    # pack + pair + open, then 40 x (pair + step)
    assert c1 - c0 == 3 + 2 * 40
    B.profile_begin()
    got = gpu_leapfrog(p32, v32, cfg.G, cfg.eps, cfg.dt, 40, pot, np.float32)     # no graph while profiling
    ms, timed, dropped = B.profile_end()
    assert B.launch_count() - c1 == 3 + 2 * 40
    assert timed == 41 and dropped == 0 and ms > 0
    for x, y in zip(ref, got):
        assert x.tobytes() == y.tobytes()
    with pytest.raises(B.OdisseoError):
        B.profile_end()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n,ci", [(1, 1), (2, 0), (129, 1), (1000, 0), (1024, 0), (3000, 1), (4096, 1), (5000, 1), (16384, 1)])
def test_whole_loop_kernel_is_bit_identical_to_the_per_step_launches(n, ci, dtype):
    """Small and mid N run all steps in ONE cooperative launch (csrc/fused_step.cuh: pair phase, grid barrier, integrate
    phase, grid barrier); it executes the same code on the same plan as the {pair, step} launch sequence, so state
    and acc must agree bit for bit -- with and without acc_valid, and chained."""
    cfg = W.CONFIGS[ci]
    posm64, vel64 = W.make_state(cfg, n=n)
    if n == 129:
        posm64[7, 3] *= 1.5                                                      # general-mass loop
    p, v = posm64.astype(dtype), vel64.astype(dtype)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
    old = B.set_fused_max_n(16384)
    B.set_cluster_max_n(0)                                                        # the other whole-loop kernels have their own tests
    B.set_ll_max_n(0)
    try:
        fused = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, 7, pot, dtype)
        c0 = B.launch_count()
        gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, 7, pot, dtype)
        assert B.launch_count() - c0 == 1                                         # one launch for the whole call
        # chained: 3 steps, then 4 more with acc_valid
        posm, vel = dev(p, dtype), dev(W.vel4(v, dtype), dtype)
        acc = torch.empty_like(posm)
        ws = B.alloc_workspace(B.workspace_bytes(n, dtype == np.float64))
        B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, 3, pot, ws)
        B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, 4, pot, ws, acc_valid=True)
        torch.cuda.synchronize()
        chained = (posm.cpu().numpy(), vel.cpu().numpy(), acc.cpu().numpy())
        B.set_fused_max_n(0)
        plain = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, 7, pot, dtype)
    finally:
        B.set_fused_max_n(-1)
        B.set_cluster_max_n(-1)
        B.set_ll_max_n(-1)
    for a, b, c in zip(fused, plain, chained):
        assert a.tobytes() == b.tobytes() and a.tobytes() == c.tobytes()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n,ci,nsteps", [(1, 1, 3), (2, 0, 3), (3, 1, 1), (63, 0, 5), (65, 1, 5), (129, 1, 7), (1000, 0, 7), (1024, 0, 10),
                                         (1025, 1, 4), (1536, 1, 3)])
def test_cluster_kernel_is_bit_identical_to_the_per_step_launches(n, ci, nsteps, dtype):
    """Small N runs the whole call on one thread-block cluster (csrc/cluster_kdk.cuh: every position in the shared memory of
    each CTA, moved records pushed through distributed shared memory, one cluster barrier per step).  It follows the
    canonical summation order, so state and acc must agree bit for bit with the {pair, step} launch sequence -- with and
    without acc_valid, chained, equal and general masses, with and without the external potential."""
    cfg = W.CONFIGS[ci]
    posm64, vel64 = W.make_state(cfg, n=n)
    if n == 129:
        posm64[7, 3] *= 1.5                                                      # general-mass loop
    p, v = posm64.astype(dtype), vel64.astype(dtype)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
    B.set_fused_max_n(0)
    B.set_ll_max_n(0)
    B.set_cluster_max_n(4096)
    try:
        clustered = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype)
        c0 = B.launch_count()
        gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype)
        assert B.launch_count() - c0 == 1                                         # one launch for the whole call
        posm, vel = dev(p, dtype), dev(W.vel4(v, dtype), dtype)
        acc = torch.empty_like(posm)
        ws = B.alloc_workspace(B.workspace_bytes(n, dtype == np.float64))
        k1 = max(1, nsteps // 2)
        B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, k1, pot, ws)
        if nsteps > k1:
            B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, nsteps - k1, pot, ws, acc_valid=True)
        torch.cuda.synchronize()
        chained = (posm.cpu().numpy(), vel.cpu().numpy(), acc.cpu().numpy())
        B.set_cluster_max_n(0)
        plain = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype)
        assert B.launch_count() - c0 > 3
    finally:
        B.set_cluster_max_n(-1)
        B.set_fused_max_n(-1)
        B.set_ll_max_n(-1)
    for a, b, c in zip(clustered, plain, chained):
        assert a.tobytes() == b.tobytes() and a.tobytes() == c.tobytes()


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("n,ci,nsteps", [(1, 1, 3), (2, 0, 3), (3, 1, 1), (63, 0, 5), (65, 1, 5), (129, 1, 7), (1000, 0, 7), (1024, 0, 10),
                                         (1025, 1, 4), (2047, 0, 3), (4096, 1, 3)])
def test_flag_in_data_kernel_is_bit_identical_to_the_per_step_launches(n, ci, nsteps, dtype):
    """Small N runs the whole call as one cooperative launch of the owner-computes kernel (csrc/ll_kdk.cuh: every CTA holds
    all sources in shared memory and owns a few targets; moved positions are exchanged as {value, step tag} words that
    every CTA polls).  It follows the canonical summation order, so state and acc must agree bit for bit with the
    {pair, step} launch sequence -- with and without acc_valid, chained, equal and general masses, with and without
    the external potential."""
    cfg = W.CONFIGS[ci]
    posm64, vel64 = W.make_state(cfg, n=n)
    if n == 129:
        posm64[7, 3] *= 1.5                                                      # general-mass loop
    p, v = posm64.astype(dtype), vel64.astype(dtype)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
    B.set_fused_max_n(0)
    B.set_cluster_max_n(0)
    B.set_ll_max_n(6144)
    try:
        ll = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype)
        c0 = B.launch_count()
        gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype)
        assert B.launch_count() - c0 == 1                                         # one launch for the whole call
        posm, vel = dev(p, dtype), dev(W.vel4(v, dtype), dtype)
        acc = torch.empty_like(posm)
        ws = B.alloc_workspace(B.workspace_bytes(n, dtype == np.float64))
        k1 = max(1, nsteps // 2)
        B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, k1, pot, ws)
        if nsteps > k1:
            B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, nsteps - k1, pot, ws, acc_valid=True)
        torch.cuda.synchronize()
        chained = (posm.cpu().numpy(), vel.cpu().numpy(), acc.cpu().numpy())
        B.set_ll_max_n(0)
        plain = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype)
        assert B.launch_count() - c0 > 3
    finally:
        B.set_cluster_max_n(-1)
        B.set_fused_max_n(-1)
        B.set_ll_max_n(-1)
    for a, b, c in zip(ll, plain, chained):
        assert a.tobytes() == b.tobytes() and a.tobytes() == c.tobytes()


def test_leapfrog_conserves_lz_and_tracks_single_particle_orbit_f32():
    """invariants of a GPU trajectory measured with the oracle's diagnostics."""
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.make_state(cfg, n=4096)
    p32, v32 = W.to_f32(posm64), W.to_f32(vel64)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    p, v, _ = gpu_leapfrog(p32, v32, cfg.G, cfg.eps, cfg.dt, 400, pot, np.float32)
    L0 = O.angular_momentum(p32, v32)[2]
    L1 = O.angular_momentum(p, v[:, :3])[2]
    assert abs(L1 - L0) <= 2e-5 * abs(L0)
    opot = O.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    one, _, _ = O.leapfrog_kdk(np.array([[*cfg.centre, cfg.M]]), np.array([cfg.velocity]), cfg.G, cfg.eps, cfg.dt, 400, opot)
    assert np.linalg.norm(O.centre_of_mass(p) - one[0, :3]) <= 5e-3


def test_workspace_too_small_and_bad_alignment_are_reported():
    posm = torch.zeros(5000, 4, device="cuda")
    acc = torch.zeros_like(posm)
    with pytest.raises(B.OdisseoError, match="ERR_WORKSPACE"):
        B.pair_accel(posm, acc, 1.0, 0.1, B.alloc_workspace(1024))
    ws = B.alloc_workspace(B.workspace_bytes(5000) + 64)
    with pytest.raises(B.OdisseoError, match="ERR_ALIGN"):
        B.pair_accel(posm, acc, 1.0, 0.1, ws[16:])
    with pytest.raises(B.OdisseoError, match="ERR_ARG"):
        B.pair_accel(posm, posm, 1.0, 0.1, ws)


@pytest.mark.parametrize("ci,dtype", [(3, np.float32), (4, np.float32), (3, np.float64)])
def test_full_size_step_resynchronised_parity_and_one_step_shadowing(ci, dtype):
    """SURVEY.md 8c (ii)+(iii) at BASELINE.json's full sizes, in the launch configuration bench.py times
    (one odisseo_leapfrog_kdk call per step, acc_valid = 1).  From the GPU's own state at step k the
    oracle advances the seeded 4,096 targets one KDK step in fp64 (all sources); the GPU state at k+1
    must agree to |dx| <= 1e-6 |x| and |dv| <= 1e-6 |v| + 1.5e-5 |dt| (S_i + |a_ext,i|) in fp32
    (1e-12 / 1e-12 + 1e-11 in fp64), and the acc the call leaves is a_pair of its own final state."""
    cfg = W.CONFIGS[ci]
    posm64, vel64 = W.make_state(cfg)
    f32 = dtype == np.float32
    p0, v0 = posm64.astype(dtype), vel64.astype(dtype)
    G, eps, dt = ((float(np.float32(t)) for t in (cfg.G, cfg.eps, cfg.dt)) if f32 else (cfg.G, cfg.eps, cfg.dt))
    bpot, opot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), O.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    posm, vel = dev(p0, dtype), dev(W.vel4(v0, dtype), dtype)
    acc = torch.full_like(posm, float("nan"))
    ws = B.alloc_workspace(B.workspace_bytes(cfg.n, not f32))
    B.leapfrog_kdk(posm, vel, acc, G, eps, dt, 0, bpot, ws)                      # a_pair(x0)
    B.leapfrog_kdk(posm, vel, acc, G, eps, dt, 1, bpot, ws, acc_valid=True)      # step 1
    torch.cuda.synchronize()
    pk, vk, ak = (t.cpu().numpy().astype(np.float64) for t in (posm, vel, acc))
    B.leapfrog_kdk(posm, vel, acc, G, eps, dt, 1, bpot, ws, acc_valid=True)      # step 2 = k -> k+1
    torch.cuda.synchronize()
    p1, v1, a1 = (t.cpu().numpy().astype(np.float64) for t in (posm, vel, acc))
    assert np.array_equal(p1[:, 3], p0[:, 3].astype(np.float64))                 # masses preserved

    idx = W.target_subset(cfg.n)
    tol_a = TOL_F32 if f32 else TOL_F64
    # (ii) re-synchronised: acc == a_pair(own state), at k and at k+1
    assert pair_ratio(ak, pk, G, eps, targets=idx) <= tol_a
    assert pair_ratio(a1, p1, G, eps, targets=idx) <= tol_a
    # (iii) one oracle KDK step for the targets, from the GPU state at k
    a_pair_k, S_k = O.pair_accel(pk, G, eps, targets=idx)
    a_k = a_pair_k + O.ext_accel(pk[idx], G, opot)
    v_half = vk[idx, :3] + 0.5 * dt * a_k
    x_new = pk[idx, :3] + dt * v_half
    src = p1.copy()
    src[idx, :3] = x_new                                                          # targets at the oracle's x(k+1)
    a_pair_1, S_1 = O.pair_accel(src, G, eps, targets=idx)
    a_1 = a_pair_1 + O.ext_accel(src[idx], G, opot)
    v_new = v_half + 0.5 * dt * a_1
    dx = np.linalg.norm(p1[idx, :3] - x_new, axis=1)
    dv = np.linalg.norm(v1[idx, :3] - v_new, axis=1)
    aext = np.linalg.norm(a_1 - a_pair_1, axis=1)
    rx, rv, ra = (1e-6, 1e-6, 1.5e-5) if f32 else (1e-12, 1e-12, 1e-11)
    assert np.all(dx <= rx * np.linalg.norm(x_new, axis=1))
    assert np.all(dv <= rv * np.linalg.norm(v_new, axis=1) + ra * abs(dt) * (np.maximum(S_k, S_1) + aext))


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_kick_drift_composes_to_the_leapfrog_bitwise(dtype):
    """odisseo_kick_drift (the integrator kernel alone) + odisseo_pair_accel reproduce
    odisseo_leapfrog_kdk bit for bit: a0 = pair(x0); [open]; a1 = pair(x1); [close+open]; a2; [close]."""
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.make_state(cfg, n=3001)
    p0, v0 = posm64.astype(dtype), vel64.astype(dtype)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    ref = gpu_leapfrog(p0, v0, cfg.G, cfg.eps, cfg.dt, 2, pot, dtype)
    posm, vel = dev(p0, dtype), dev(W.vel4(v0, dtype), dtype)
    acc = torch.empty_like(posm)
    ws = B.alloc_workspace(B.workspace_bytes(3001, dtype == np.float64))
    B.pair_accel(posm, acc, cfg.G, cfg.eps, ws)
    B.kick_drift(posm, vel, acc, cfg.G, cfg.dt, pot, 2, ws)
    B.pair_accel(posm, acc, cfg.G, cfg.eps, ws)
    B.kick_drift(posm, vel, acc, cfg.G, cfg.dt, pot, 3, ws)
    B.pair_accel(posm, acc, cfg.G, cfg.eps, ws)
    B.kick_drift(posm, vel, acc, cfg.G, cfg.dt, pot, 1, ws)
    torch.cuda.synchronize()
    for got, want in zip((posm, vel, acc), ref):
        assert got.cpu().numpy().tobytes() == want.tobytes()
    with pytest.raises(B.OdisseoError, match="ERR_ARG"):
        B.kick_drift(posm, vel, acc, cfg.G, cfg.dt, pot, 0, ws)


def test_flag_in_data_kernel_random_sizes_steps_and_splits():
    """Sixty seeded random cases (n = 1 ... 4,096, 1 ... 40 steps, both precisions, with / without the potential, an odd
    mass now and then, the call cut in two at a random step): the one-launch form and the per-step launches agree bit for
    bit.  Guards the two-buffer exchange of csrc/ll_kdk.cuh (a CTA that runs ahead must never overwrite a record another
    CTA still waits for)."""
    rng = np.random.default_rng(2511)
    try:
        for _ in range(60):
            dtype = np.float32 if rng.random() < 0.6 else np.float64
            top = 4097 if dtype == np.float32 else 2049
            n = int(rng.choice([rng.integers(1, 64), rng.integers(64, 1100), rng.integers(1100, top)]))
            nsteps = int(rng.integers(1, 41))
            cfg = W.CONFIGS[int(rng.integers(0, 2))]
            posm64, vel64 = W.make_state(cfg, n=n, seed=int(rng.integers(1, 10 ** 6)))
            if n > 3 and rng.random() < 0.3:
                posm64[int(rng.integers(0, n)), 3] *= 1.7
            p, v = posm64.astype(dtype), vel64.astype(dtype)
            pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
            k1 = int(rng.integers(1, nsteps + 1))
            B.set_fused_max_n(0)
            B.set_cluster_max_n(0)
            B.set_ll_max_n(6144)
            one = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype, chunks=[k1] + ([nsteps - k1] if nsteps > k1 else []))
            B.set_ll_max_n(0)
            ref = gpu_leapfrog(p, v, cfg.G, cfg.eps, cfg.dt, nsteps, pot, dtype)
            for a, b in zip(one, ref):
                assert a.tobytes() == b.tobytes(), (dtype.__name__, n, nsteps, k1)
    finally:
        B.set_ll_max_n(-1)
        B.set_cluster_max_n(-1)
        B.set_fused_max_n(-1)
