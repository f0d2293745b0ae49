"""Pins for the seeded Plummer workload generator (PAPER.md:L43 step 3 "Plummer sphere in
equilibrium"; BASELINE.json configs[0] recipe), measured with the oracle's diagnostics."""
import numpy as np

from oracle import oracle as O
from paper_2511_22468_b200 import workloads as W


def test_plummer_potential_energy_virial_ratio_and_half_mass_radius():
    n, G, M, a = 16384, 1.0, 1.0, 1.0
    posm, vel = W.plummer_sphere(n, G, M, a, seed=1000)
    Wexact = -3 * np.pi * G * M * M / (32 * a)           # closed form, north_star
    Wpot = O.pair_potential_energy(posm, G, 0.0)
    assert abs(Wpot / Wexact - 1) <= 0.022               # 5 sigma at N = 16,384
    K = O.kinetic_energy(posm, vel)
    assert abs(2 * K / abs(Wpot) - 1) <= 0.02            # equilibrium: virial ratio 1
    r = np.sort(np.linalg.norm(posm[:, :3], axis=1))
    assert abs(r[n // 2] / (1.30477 * a) - 1) <= 0.03    # half-mass radius (2^{2/3}-1)^{-1/2} a
    assert abs(posm[:, 3].sum() - M) <= 1e-12
    assert np.abs(O.centre_of_mass(posm)).max() <= 1e-12 and np.abs(O.linear_momentum(posm, vel)).max() <= 1e-12


def test_plummer_scales_with_units_and_is_bound():
    cfg = W.CONFIGS[1]
    posm, vel = W.plummer_sphere(4096, cfg.G, cfg.M, cfg.a, seed=5)
    Wexact = -3 * np.pi * cfg.G * cfg.M ** 2 / (32 * cfg.a)
    assert abs(O.pair_potential_energy(posm, cfg.G, 0.0) / Wexact - 1) <= 0.05
    r = np.linalg.norm(posm[:, :3], axis=1)
    v = np.linalg.norm(vel, axis=1)
    vesc = np.sqrt(2 * cfg.G * cfg.M / cfg.a) * (1 + (r / cfg.a) ** 2) ** -0.25
    assert np.all(v <= vesc * 1.05)                      # recentring moves speeds by ~1/sqrt(N)


def test_seeded_and_shifted():
    cfg = W.CONFIGS[2]
    p1, v1 = W.make_state(cfg, n=512)
    p2, v2 = W.make_state(cfg, n=512)
    assert np.array_equal(p1, p2) and np.array_equal(v1, v2)
    p3, _ = W.make_state(cfg, n=512, seed=7)
    assert not np.array_equal(p1, p3)
    np.testing.assert_allclose(O.centre_of_mass(p1), cfg.centre, atol=1e-12)
    np.testing.assert_allclose(O.linear_momentum(p1, v1) / cfg.M, cfg.velocity, atol=1e-12)
    idx = W.target_subset(1 << 20)
    assert idx.shape == (4096,) and np.all(np.diff(idx) > 0) and idx.max() < (1 << 20)
    assert np.array_equal(idx, W.target_subset(1 << 20))


def test_config_table_restates_baseline_json():
    ns = [c.n for c in W.CONFIGS]
    assert ns == [1024, 16384, 65536, 262144, 1048576]
    assert [c.nsteps for c in W.CONFIGS] == [10, 1000, 3000, 200, 20]
    assert W.CONFIGS[0].nfw is None and W.CONFIGS[3].precisions == ("f32", "f64")
