"""One simulation spread over several GPUs: plumbing around the C ABI.

The paper's only performance experiment distributes a single simulation over 1-5 A100s "without modifying the
simulation code" and reports near-linear speed-up for N > 10^4 (section 2.1, Fig. 1).  The direct sum
shards naturally over TARGETS: rank r owns the contiguous slice [lo_r, hi_r) of particles, holds the staged source
records of ALL particles, and per KDK step

    kick + drift its slice            odisseo_kick_drift_slice: also re-stages the slice's records in place
    exchange                          ONE in-place all-gather of the record array (16 N bytes in total per step in fp32, 32 N in fp64)
    a_pair(slice) from all sources    odisseo_pair_accel_staged: no re-packing of the N sources

Slices are equal and 8-aligned (the last one shorter), so rank r's records sit at [r L, (r+1) L) of the record array
and the all-gather lands every rank's records at their global index.  The order in which a target's partial sums
are added depends on N only (include/odisseo.h), so any number of ranks -- 1 included -- is BIT-IDENTICAL to
odisseo_leapfrog_kdk on one GPU.  Compute per rank is N^2 / R, traffic 16 N bytes per step (fp32): at N = 262,144 on 8 GPUs
~3 ms of arithmetic against microseconds on NVLink, the near-linear behaviour the paper reports.

north_star fixes this build to ONE GPU, and nothing in this run can execute more than one: `bench.py --mode sharded`
runs this driver under torchrun (strong scaling) but has only ever been run with world size 1 on hardware; the
multi-rank logic is exercised (a) on CPU with world_size 2 over gloo and an oracle-backed compute object, (b) on one
GPU with R emulated ranks run side by side.  The compute object is injected so that neither this module nor the
product path ever imports the oracle.

No arithmetic of the method lives here: slicing, the exchange, and the order of the calls above.
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


def aligned_slices(n: int, world: int) -> Tuple[int, List[Tuple[int, int]]]:
    """(L, bounds): equal slices of L = 8 ceil(ceil(n / world) / 8) particles, rank r owning [r L, min((r+1) L, n))
    (possibly empty at the end), so that an all-gather of L-record blocks puts every record at its global index."""
    if n < 0 or world < 1:
        raise ValueError("n >= 0 and world >= 1 required")
    per = -(-n // world)
    L = 8 * (-(-per // 8)) if n > 0 else 8
    return L, [(min(r * L, n), min((r + 1) * L, n)) for r in range(world)]


class CudaCompute:
    """The product path: every call goes through the C ABI (binding.py).  Buffers are torch CUDA tensors."""

    def __init__(self, n: int, n_slice: int, is_f64: bool, G: float, eps: float, dt: float, pot, world: int = 1):
        import torch
        from . import binding as B
        self.B, self.n, self.G, self.eps, self.dt, self.pot = B, n, G, eps, dt, pot
        self.ws = B.alloc_workspace(B.cross_workspace_bytes(max(n_slice, 1), max(n, 1), is_f64))
        off, rec, cap = B.staged_sources_layout(max(n, 1), is_f64)
        L, _ = aligned_slices(n, world)
        if world * L > cap:
            raise ValueError("too many ranks for the staged array's slack (%d records for %d x %d)" % (cap, world, L))
        dtype = torch.float64 if is_f64 else torch.float32
        self._records = self.ws[off:off + cap * rec].view(dtype).view(cap, -1)

    def stage_all(self, posm_all):
        self.B.stage_sources(posm_all, self.ws)

    def records(self):
        """The staged record array [capacity, scalars per record]: what the exchange all-gathers in place."""
        return self._records

    def accel(self, targets, acc):
        self.B.pair_accel_staged(targets, self.n, acc, self.G, self.eps, self.ws)

    def kick_drift(self, posm_all, vel, acc, lo: int, hi: int, mode: int):
        self.B.kick_drift_slice(posm_all[lo:hi], vel, acc, self.n, lo, self.G, self.dt, self.pot, mode, self.ws)


class DistExchange:
    """One collective per step over a torch.distributed group (NCCL on GPUs, gloo on CPU): the in-place all-gather of
    the L-record blocks of a [world * L, k] array; `positions` does the same for posm at the end of a run."""

    def __init__(self, dist, n: int, world: int, rank: int):
        self.dist, self.n, self.world, self.rank = dist, n, world, rank
        self.L, self.bounds = aligned_slices(n, world)

    def __call__(self, records):
        L, r = self.L, self.rank
        self.dist.all_gather_into_tensor(records[:self.world * L], records[r * L:(r + 1) * L])

    def positions(self, posm_all):
        """Leave every rank with every rank's final slice of posm (once, after the last step)."""
        L, n = self.L, self.n
        if self.world * L == n:
            self.dist.all_gather_into_tensor(posm_all, posm_all[self.rank * L:(self.rank + 1) * L])
            return
        pad = posm_all.new_zeros((self.world * L, posm_all.shape[1]))
        lo, hi = self.bounds[self.rank]
        pad[lo:hi] = posm_all[lo:hi]
        self.dist.all_gather_into_tensor(pad, pad[self.rank * L:(self.rank + 1) * L].clone())
        posm_all.copy_(pad[:n])


def sharded_leapfrog_kdk(compute, exchange, posm_all, vel_slice, acc_slice, lo: int, hi: int, nsteps: int,
                         acc_valid: bool = False):
    """nsteps KDK steps of the slice [lo, hi) of one simulation.

    posm_all [n, 4]: all particles at the start; rows [lo, hi) are advanced here, the other rows are NOT refreshed
    during the run (only their staged records are) -- call `exchange.positions(posm_all)` afterwards for that.
    vel_slice, acc_slice [hi - lo, 4].  acc_slice holds the pair-only acceleration of the slice, as in
    odisseo_leapfrog_kdk.  `exchange(records)` must leave every rank with every rank's current records.
    """
    mine = posm_all[lo:hi]
    compute.stage_all(posm_all)
    if not acc_valid:
        compute.accel(mine, acc_slice)
    for step in range(nsteps):
        # closing half kick of the previous step (not before the first) fused with opening half kick + drift
        compute.kick_drift(posm_all, vel_slice, acc_slice, lo, hi, 2 if step == 0 else 3)
        exchange(compute.records())
        compute.accel(mine, acc_slice)
    if nsteps > 0:
        compute.kick_drift(posm_all, vel_slice, acc_slice, lo, hi, 1)
