"""Host logic of the sharded (one simulation over several ranks) form, on CPU: world_size 2
over gloo with an oracle-backed compute object.  The sharded driver must reproduce oracle.leapfrog_kdk exactly
(the oracle sums each target in source order, so slicing the targets changes nothing)."""
import os
import sys

import numpy as np
import torch
import torch.multiprocessing as mp

from paper_2511_22468_b200 import sharded as S

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
NFW, MN, G, EPS, DT = (1.0e12, 16.0), (6.8e10, 3.0, 0.28), 4.4985e-12, 0.001, 0.5


class OracleCompute:
    """Test stand-in for CudaCompute: the same calls, evaluated by the fp64 oracle on numpy views of torch CPU
    tensors (tests may import the oracle; the product module does not).  Its "staged records" are plain {x, y, z, m}
    rows in an array padded to world * L rows, which is what the exchange all-gathers."""

    def __init__(self, n, world):
        from oracle import oracle as O
        self.O, self.pot, self.n = O, O.Potential.make(nfw=NFW, mn=MN), n
        L, _ = S.aligned_slices(n, world)
        self.rec = torch.zeros(world * L, 4, dtype=torch.float64)

    def stage_all(self, posm_all):
        self.rec[:self.n] = posm_all

    def records(self):
        return self.rec

    def accel(self, targets, acc):
        nt, n = targets.shape[0], self.n
        both = np.concatenate([self.rec[:n].numpy(), targets.numpy()], axis=0).copy()
        both[n:, 3] = 0.0                                                 # targets act as massless tracers
        a, _ = self.O.pair_accel(both, G, EPS, targets=np.arange(n, n + nt))
        acc[:, :3] = torch.from_numpy(a)
        acc[:, 3] = 0

    def kick_drift(self, posm_all, vel, acc, lo, hi, mode):
        posm = posm_all[lo:hi]
        a = acc[:, :3].numpy() + self.O.ext_accel(posm.numpy(), G, self.pot)
        if mode & 1:
            vel[:, :3] += torch.from_numpy(0.5 * DT * a)
        if mode & 2:
            vel[:, :3] += torch.from_numpy(0.5 * DT * a)
            posm[:, :3] += DT * vel[:, :3]
            self.rec[lo:hi] = posm


def _state(n):
    rng = np.random.Generator(np.random.PCG64(3))
    posm = np.concatenate([rng.normal(0, 0.01, (n, 3)) + np.array([12.4, 0, 1.5]), rng.uniform(5, 15, (n, 1))], axis=1)
    vel = np.zeros((n, 4))
    vel[:, :3] = rng.normal(0, 0.002, (n, 3)) + np.array([0, 0.21, 0.05])
    return posm, vel


def _worker(rank, world, port, n, nsteps, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    dist.init_process_group(backend="gloo")
    try:
        posm, vel = _state(n)
        _, bounds = S.aligned_slices(n, world)
        lo, hi = bounds[rank]
        posm_all = torch.from_numpy(posm.copy())
        vel_slice = torch.from_numpy(vel[lo:hi].copy())
        acc_slice = torch.zeros(hi - lo, 4, dtype=torch.float64)
        ex = S.DistExchange(dist, n, world, rank)
        S.sharded_leapfrog_kdk(OracleCompute(n, world), ex, posm_all, vel_slice, acc_slice, lo, hi, nsteps)
        ex.positions(posm_all)
        out.put((rank, lo, hi, posm_all.numpy().copy(), vel_slice.numpy().copy(), acc_slice.numpy().copy()))
    finally:
        dist.destroy_process_group()


def test_slice_bounds_cover_every_particle_once():
    for n in (0, 1, 7, 1000, 1001, 262144):
        for world in (1, 2, 3, 5, 8):
            b = S.slice_bounds(n, world)
            assert len(b) == world and b[0][0] == 0 and b[-1][1] == n
            assert all(b[k][1] == b[k + 1][0] for k in range(world - 1))
            sizes = [hi - lo for lo, hi in b]
            assert max(sizes) - min(sizes) <= 1


def test_aligned_slices_put_every_record_at_its_global_index():
    for n in (0, 1, 7, 8, 9, 1000, 1001, 262144):
        for world in (1, 2, 3, 5, 8):
            L, b = S.aligned_slices(n, world)
            assert L % 8 == 0 and L > 0 and world * L >= n and len(b) == world
            assert b[0][0] == 0 and b[-1][1] == n
            for r, (lo, hi) in enumerate(b):
                assert lo == min(r * L, n) and hi == min((r + 1) * L, n) and 0 <= hi - lo <= L
            assert world * L - n < 8 * world + 8                          # fits the staged array's 1,024-record slack


def test_two_ranks_reproduce_the_single_process_oracle_trajectory():
    from oracle import oracle as O
    n, nsteps = 101, 4                                                    # odd n: slices of 56 and 45
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29600 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, nsteps, out)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted((out.get(timeout=300) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    posm, vel = _state(n)
    pr, vr, _ = O.leapfrog_kdk(posm, vel[:, :3], G, EPS, DT, nsteps, O.Potential.make(nfw=NFW, mn=MN))
    ar, _ = O.pair_accel(pr, G, EPS)
    for rank, lo, hi, p_all, v_slice, a_slice in got:
        assert np.abs(p_all - pr).max() <= 1e-13 * 12.4                  # every rank ends with every slice
        assert np.abs(v_slice[:, :3] - vr[lo:hi]).max() <= 1e-13 * 0.21
        assert np.abs(a_slice[:, :3] - ar[lo:hi]).max() <= 1e-12 * np.abs(ar).max()   # acc = a_pair(x_final) of the slice
