"""GPU parity of odisseo_diagnostics_* (energies, momenta, centre of mass in fp64) against the oracle's
pinned definitions (oracle.kinetic_energy, pair_potential_energy, ext_potential_energy, ...)."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2511_22468_b200 import binding as B
from paper_2511_22468_b200 import workloads as W

pytestmark = pytest.mark.gpu


def gpu_diag(posm_np, vel_np, G, eps, pot, dtype, want_phi=False):
    posm = torch.from_numpy(np.ascontiguousarray(posm_np, dtype=dtype)).cuda()
    vel = torch.from_numpy(W.vel4(np.ascontiguousarray(vel_np, dtype=dtype), dtype)).cuda()
    n = posm.shape[0]
    out = torch.full((16,), float("nan"), dtype=torch.float64, device="cuda")
    phi = torch.full((n,), float("nan"), dtype=torch.float64, device="cuda") if want_phi else None
    ws = B.alloc_workspace(B.diagnostics_workspace_bytes(n))
    B.diagnostics(posm, vel, G, eps, pot, out, ws, phi=phi)
    torch.cuda.synchronize()
    return out.cpu().numpy(), (phi.cpu().numpy() if want_phi else None)


def oracle_diag(p64, v64, G, eps, opot):
    K = O.kinetic_energy(p64, v64)
    Wp = O.pair_potential_energy(p64, G, eps)
    E = O.ext_potential_energy(p64, G, opot) if opot is not None else 0.0
    return K, Wp, E, O.linear_momentum(p64, v64), O.angular_momentum(p64, v64), O.centre_of_mass(p64), p64[:, 3].sum()


def check(out, ref, rtol, self_energy):
    """self_energy = 1/2 G sum m_i^2 / eps: the kernel sums the self term m_i / eps with the others and removes
    it afterwards, which leaves its rounding (a few ulp of the self energy) in W."""
    K, Wp, E, P, L, C, M = ref
    assert abs(out[0] - K) <= rtol * abs(K)
    assert abs(out[1] - Wp) <= rtol * abs(Wp) + 4e-16 * self_energy
    assert abs(out[2] - E) <= rtol * max(abs(E), 1e-300)
    scale_p = np.abs(P).max() + 1e-300
    # momenta are sums with cancellation: compare against the sum of magnitudes
    assert np.abs(out[3:6] - P).max() <= 1e-11 * max(scale_p, abs(K) ** 0.5 * M ** 0.5)
    assert np.abs(out[6:9] - L).max() <= 1e-11 * max(np.abs(L).max(), 1e-300) + 1e-11 * np.linalg.norm(C) * max(scale_p, abs(K) ** 0.5 * M ** 0.5)
    assert np.abs(out[9:12] - C).max() <= 1e-12 * max(np.linalg.norm(C), 1.0)
    assert abs(out[12] - M) <= 1e-13 * M
    assert abs(out[13] - (out[0] + out[1] + out[2])) <= 1e-15 * (abs(out[0]) + abs(out[1]) + abs(out[2]))
    assert out[14] == 0 and out[15] == 0


@pytest.mark.parametrize("n", [1, 2, 3, 255, 257, 1000, 4097, 6000])
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_diagnostics_ragged_sizes_unequal_masses(n, dtype):
    cfg = W.CONFIGS[1]
    posm64, vel64 = W.random_cloud(n, seed=500 + n, scale=0.01, centre=cfg.centre)
    posm64[:, 3] *= cfg.M / n
    p = posm64.astype(dtype)
    v = (vel64 * 0.02 + np.asarray(cfg.velocity)).astype(dtype)
    G, eps = (float(np.float32(cfg.G)), float(np.float32(cfg.eps))) if dtype == np.float32 else (cfg.G, cfg.eps)
    bpot, opot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), O.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    out, phi = gpu_diag(p, v, G, eps, bpot, dtype, want_phi=True)
    p64, v64 = p.astype(np.float64), v.astype(np.float64)
    check(out, oracle_diag(p64, v64, G, eps, opot), 1e-12, 0.5 * G * np.sum(p64[:, 3] ** 2) / eps)
    # per-particle potential: W = 1/2 sum m_i phi_i
    assert abs(0.5 * np.sum(p64[:, 3] * phi) - out[1]) <= 1e-13 * abs(out[1]) + 1e-300 + 4e-16 * 0.5 * G * np.sum(p64[:, 3] ** 2) / eps


@pytest.mark.parametrize("ci,dtype", [(0, np.float64), (0, np.float32), (1, np.float32), (2, np.float32)])
def test_diagnostics_configs_equal_masses(ci, dtype):
    cfg = W.CONFIGS[ci]
    posm64, vel64 = W.make_state(cfg)
    p, v = posm64.astype(dtype), vel64.astype(dtype)
    G, eps = (float(np.float32(cfg.G)), float(np.float32(cfg.eps))) if dtype == np.float32 else (cfg.G, cfg.eps)
    bpot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
    opot = O.Potential.make(nfw=cfg.nfw, mn=cfg.mn) if cfg.nfw else None
    out, _ = gpu_diag(p, v, G, eps, bpot, dtype)
    check(out, oracle_diag(p.astype(np.float64), v.astype(np.float64), G, eps, opot), 1e-12,
          0.5 * G * np.sum(p.astype(np.float64)[:, 3] ** 2) / eps)
    again, _ = gpu_diag(p, v, G, eps, bpot, dtype)
    assert out.tobytes() == again.tobytes()                              # fixed-order reductions


def test_diagnostics_plummer_energy_closed_form_and_energy_conservation_of_the_gpu_leapfrog():
    """Pins through the GPU path itself: W of a sampled Plummer sphere -> -3 pi G M^2 / (32 a) (north_star), and the
    energy error of the GPU fp64 leapfrog falls 4x when dt halves (second order)."""
    cfg = W.CONFIGS[0]
    posm64, vel64 = W.plummer_sphere(16384, cfg.G, cfg.M, cfg.a, seed=77)
    out, _ = gpu_diag(posm64, vel64, cfg.G, cfg.eps, None, np.float64)
    assert abs(out[1] / (-3 * np.pi / 32) - 1) <= 0.022                  # 5 sigma at N = 16,384
    assert abs(2 * out[0] / abs(out[1]) - 1) <= 0.02                     # virial equilibrium
    posm64, vel64 = W.make_state(cfg, n=512)
    e0 = gpu_diag(posm64, vel64, cfg.G, cfg.eps, None, np.float64)[0][13]
    errs = []
    for nsteps in (50, 100, 200):
        posm = torch.from_numpy(posm64).cuda()
        vel = torch.from_numpy(W.vel4(vel64, np.float64)).cuda()
        acc = torch.empty_like(posm)
        ws = B.alloc_workspace(B.workspace_bytes(512, True))
        B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, 0.1 / nsteps, nsteps, None, ws)
        out = torch.empty(16, dtype=torch.float64, device="cuda")
        B.diagnostics(posm, vel, cfg.G, cfg.eps, None, out, B.alloc_workspace(B.diagnostics_workspace_bytes(512)))
        torch.cuda.synchronize()
        errs.append(abs(out[13].item() - e0) / abs(e0))
    assert 3.5 <= errs[0] / errs[1] <= 4.5 and 3.5 <= errs[1] / errs[2] <= 4.5


def test_diagnostics_full_size_config3_against_sampled_oracle_potential():
    """N = 262,144 (fp32 state): the oracle cannot afford the full W, so the per-particle potential phi_i is
    checked on the seeded 4,096-target subset against a direct fp64 numpy sum."""
    cfg = W.CONFIGS[3]
    posm64, vel64 = W.make_state(cfg)
    p32, v32 = W.to_f32(posm64), W.to_f32(vel64)
    G, eps = float(np.float32(cfg.G)), float(np.float32(cfg.eps))
    out, phi = gpu_diag(p32, v32, G, eps, B.Potential.make(nfw=cfg.nfw, mn=cfg.mn), np.float32, want_phi=True)
    p64 = p32.astype(np.float64)
    idx = W.target_subset(cfg.n, size=256)
    for i in idx:
        d = p64[:, :3] - p64[i, :3]
        inv = 1.0 / np.sqrt(np.einsum("ij,ij->i", d, d) + eps * eps)
        inv[i] = 0.0
        ref = -G * np.sum(p64[:, 3] * inv)
        assert abs(phi[i] - ref) <= 1e-12 * abs(ref)
    assert abs(out[0] - O.kinetic_energy(p64, v32.astype(np.float64))) <= 1e-12 * out[0]
    assert abs(out[2] - O.ext_potential_energy(p64, G, O.Potential.make(nfw=cfg.nfw, mn=cfg.mn))) <= 1e-12 * abs(out[2])


@pytest.mark.parametrize("ci", [1, 2, 3, 4])
def test_full_length_fp32_runs_keep_the_invariants(ci):
    """SURVEY.md 8c (ii) and (v) at BASELINE.json's sizes AND step counts (config 1: 1,000 steps, config 2: 3,000,
    config 3: 200, config 4: 20): the fp32 GPU trajectory conserves L_z (exact for KDK in an axisymmetric potential),
    keeps the energy error bounded, the cluster's centre of mass follows the single-particle orbit the oracle
    integrates from the same start (PAPER.md:L43 steps 2-3), and the `acc` the call leaves is the oracle's pair
    acceleration of the GPU's own FINAL state on the seeded 4,096 targets (re-synchronised parity, <= 1e-5)."""
    cfg = W.CONFIGS[ci]
    nsteps = cfg.nsteps
    posm64, vel64 = W.make_state(cfg)
    posm = torch.from_numpy(W.to_f32(posm64)).cuda()
    vel = torch.from_numpy(W.vel4(W.to_f32(vel64), np.float32)).cuda()
    acc = torch.empty_like(posm)
    pot = B.Potential.make(nfw=cfg.nfw, mn=cfg.mn)
    ws = B.alloc_workspace(B.workspace_bytes(cfg.n))
    wd = B.alloc_workspace(B.diagnostics_workspace_bytes(cfg.n))
    d0 = torch.empty(16, dtype=torch.float64, device="cuda")
    d1 = torch.empty(16, dtype=torch.float64, device="cuda")
    B.diagnostics(posm, vel, cfg.G, cfg.eps, pot, d0, wd)
    # the centre of mass is compared after at most 600 steps: once the stream wraps a good part of the orbit (config 2
    # covers ~10 orbits) the centre of mass of a curved stream is no longer a point of the orbit (measured 1.2 kpc off)
    ncom = min(nsteps, 600)
    dc = torch.empty(16, dtype=torch.float64, device="cuda")
    B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, ncom, pot, ws)
    B.diagnostics(posm, vel, cfg.G, cfg.eps, pot, dc, wd)
    if nsteps > ncom:
        B.leapfrog_kdk(posm, vel, acc, cfg.G, cfg.eps, cfg.dt, nsteps - ncom, pot, ws, acc_valid=True)
    B.diagnostics(posm, vel, cfg.G, cfg.eps, pot, d1, wd)
    torch.cuda.synchronize()
    d0, d1, dc = d0.cpu().numpy(), d1.cpu().numpy(), dc.cpu().numpy()
    one, _, _ = O.leapfrog_kdk(np.array([[*cfg.centre, cfg.M]]), np.array([cfg.velocity]), cfg.G, cfg.eps, cfg.dt,
                               ncom, O.Potential.make(nfw=cfg.nfw, mn=cfg.mn))
    com_off = float(np.linalg.norm(dc[9:12] - one[0, :3]))
    print("cfg%d %d steps: dLz/Lz %.2e dE/E %.2e CoM offset %.4f kpc" % (
        ci, nsteps, abs(d1[8] - d0[8]) / abs(d0[8]), abs(d1[13] - d0[13]) / abs(d0[13]), com_off))
    assert abs(d1[8] - d0[8]) <= 1e-6 * abs(d0[8])                        # L_z
    assert abs(d1[13] - d0[13]) <= 1e-4 * abs(d0[13])                     # total energy
    assert d1[12] == d0[12]                                               # masses untouched
    assert com_off <= 0.05                                                # kpc, on a ~12 kpc orbit
    # re-synchronised acceleration parity on the final state
    pf = posm.cpu().numpy().astype(np.float64)
    idx = W.target_subset(cfg.n)
    G, eps = float(np.float32(cfg.G)), float(np.float32(cfg.eps))
    ref, S = O.pair_accel(pf, G, eps, targets=idx)
    got = acc.cpu().numpy()[idx, :3].astype(np.float64)
    assert float((np.linalg.norm(got - ref, axis=1) / S).max()) <= 1e-5
