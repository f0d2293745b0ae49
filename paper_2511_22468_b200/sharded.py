"""One simulation spread over several GPUs: plumbing around the C ABI.

The paper's only performance experiment distributes a single simulation over 1-5 A100s "without modifying the
simulation code" and reports near-linear speed-up for N > 10^4 (section 2.1, Fig. 1).  The direct sum
shards naturally over TARGETS: rank r owns the contiguous slice [lo_r, hi_r) of particles, keeps the positions
of ALL particles, and per KDK step

    kick + drift its slice            (odisseo_kick_drift on views of its slice)
    exchange the moved slices         (one broadcast per rank: 16 N bytes in total per step)
    a_pair(slice) from all sources    (odisseo_pair_accel_cross: targets = my slice, sources = all)

Compute per rank is N^2 / R, traffic 16 N bytes per step: at N = 262,144 on 8 GPUs ~3 ms of arithmetic against
microseconds on NVLink, which is the near-linear behaviour the paper reports.

north_star fixes this build to ONE GPU with no collectives, and nothing in this run can execute more than one, so
`bench.py --gpus N` stays "replicas only"; this module is the host logic of the sharded form,
exercised (a) on CPU with world_size 2 over gloo and an oracle-backed compute object, (b) on one GPU with R
emulated ranks run one after another.  The compute object is injected so that neither this module nor the
product path ever imports the oracle.

No arithmetic of the method lives here: slicing, the exchange, and the order of the three calls above.
"""
from __future__ import annotations

from typing import List, Tuple


def slice_bounds(n: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous, balanced (+-1) target slices, one per rank, covering [0, n) exactly once."""
    if n < 0 or world < 1:
        raise ValueError("n >= 0 and world >= 1 required")
    base, extra = divmod(n, world)
    bounds, lo = [], 0
    for r in range(world):
        hi = lo + base + (1 if r < extra else 0)
        bounds.append((lo, hi))
        lo = hi
    return bounds


class CudaCompute:
    """The product path: every call goes through the C ABI (binding.py).  Buffers are torch CUDA tensors."""

    def __init__(self, n: int, n_slice: int, is_f64: bool, G: float, eps: float, dt: float, pot):
        from . import binding as B
        self.B, self.G, self.eps, self.dt, self.pot = B, G, eps, dt, pot
        self.ws_cross = B.alloc_workspace(B.cross_workspace_bytes(max(n_slice, 1), max(n, 1), is_f64))
        self.ws_step = B.alloc_workspace(B.workspace_bytes(max(n_slice, 1), is_f64))

    def cross(self, targets, sources, acc):
        self.B.pair_accel_cross(targets, sources, acc, self.G, self.eps, self.ws_cross)

    def kick_drift(self, posm, vel, acc, mode: int):
        if posm.shape[0]:
            self.B.kick_drift(posm, vel, acc, self.G, self.dt, self.pot, mode, self.ws_step)


class DistExchange:
    """Exchange of the moved slices over a torch.distributed group: one broadcast per rank (NCCL on GPUs, gloo on
    CPU).  Slices may differ in length by one record, which all_gather does not allow."""

    def __init__(self, dist, bounds):
        self.dist, self.bounds = dist, bounds

    def __call__(self, posm_all):
        for src, (lo, hi) in enumerate(self.bounds):
            if hi > lo:
                self.dist.broadcast(posm_all[lo:hi], src=src)


def sharded_leapfrog_kdk(compute, exchange, posm_all, vel_slice, acc_slice, lo: int, hi: int, nsteps: int,
                         acc_valid: bool = False):
    """nsteps KDK steps of the slice [lo, hi) of one simulation whose positions `posm_all` every rank holds.

    posm_all [n, 4] (all particles; rows [lo, hi) are advanced here, the others are refreshed by `exchange`),
    vel_slice, acc_slice [hi - lo, 4].  acc_slice holds the pair-only acceleration of the slice, as in
    odisseo_leapfrog_kdk.  `exchange(posm_all)` must leave every rank with every rank's current slice.
    """
    mine = posm_all[lo:hi]
    if not acc_valid:
        compute.cross(mine, posm_all, acc_slice)
    for step in range(nsteps):
        # closing half kick of the previous step (not before the first) fused with opening half kick + drift
        compute.kick_drift(mine, vel_slice, acc_slice, 2 if step == 0 else 3)
        exchange(posm_all)
        compute.cross(mine, posm_all, acc_slice)
    if nsteps > 0:
        compute.kick_drift(mine, vel_slice, acc_slice, 1)
