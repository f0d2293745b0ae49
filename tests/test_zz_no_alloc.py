"""odisseo_mmd2_static_f32: the MMD^2 loss and gradient for callers that cannot allocate device memory.

Who that is: a loss called from inside a process whose own memory pool took the HBM at start-up (the paper's code is a
JAX program, and JAX does exactly that), where a cudaMalloc beside the pool can fail; and code in a loop or plug-in
where cudaMalloc is ruled out because it stalls every stream of the device.  They hold their inputs and outputs
already but have nowhere to get the workspace odisseo_mmd2_f32 wants, so the library keeps the per-block sums in a
fixed 1 MiB array of its own.

What is checked here: the new entry point runs the same two kernels as odisseo_mmd2_f32 (itself compared with the
oracle in test_gpu_mmd.py), so value and gradient must agree BIT FOR BIT with it -- the bound the MMD reproducibility
test uses -- on two calls in a row.  The second call has other inputs and a smaller grid than the first, so sums the
first call left in the shared array would show up if any of them were read.  The limit is checked too: one
cloud-block beyond the array is refused with ERR_STATIC_LIMIT and the outputs are not touched.

The file sorts last on purpose (pytest -x stops at the first failure, and a failure here must not hide the parity
tests); it passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

from paper_2511_22468_b200 import binding as B

pytestmark = pytest.mark.gpu
SIG = np.array([0.5, 0.7, 0.3, 0.02, 0.03, 0.01])


def _cloud(nsim, n, seed, shift=0.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    pos = np.zeros((nsim, n, 4), dtype=np.float32)
    vel = np.zeros((nsim, n, 4), dtype=np.float32)
    pos[:, :, :3] = rng.normal(0, 0.4, (nsim, n, 3)) + np.array([12.4, 0.0, 1.5]) + shift
    vel[:, :, :3] = rng.normal(0, 0.02, (nsim, n, 3)) + np.array([0.0, 0.21, 0.05])
    return torch.from_numpy(pos).cuda(), torch.from_numpy(vel).cuda()


def _outputs(nsim, n):
    nan = float("nan")
    return (torch.full((nsim,), nan, dtype=torch.float64, device="cuda"), torch.full((nsim, n, 4), nan, device="cuda"),
            torch.full((nsim, n, 4), nan, device="cuda"))


def _both_paths(nsim, n, m, seed, shared):
    xp, xv = _cloud(nsim, n, seed)
    yp, yv = _cloud(1 if shared else nsim, m, seed + 1, shift=0.25)
    if shared:
        yp, yv = yp[0], yv[0]
    scale = torch.linspace(-1.0, 2.0, nsim, dtype=torch.float64, device="cuda")
    ref, rgp, rgv = _outputs(nsim, n)
    B.mmd2(xp, xv, yp, yv, SIG, ref, B.alloc_workspace(B.mmd_workspace_bytes(n, m, nsim)), rgp, rgv, scale)
    out, gp, gv = _outputs(nsim, n)
    B.mmd2_static(xp, xv, yp, yv, SIG, out, gp, gv, scale)
    torch.cuda.synchronize()
    return (ref, rgp, rgv), (out, gp, gv)


def test_two_calls_in_a_row_match_the_workspace_path_bit_for_bit():
    # first call: 37 clouds x 3 blocks (n = 1,100 > 2 x 512) fill 111 slots of the shared array
    # second call: 5 clouds x 1 block, other data, per-cloud observed streams: reads 5 slots, all of them rewritten
    for nsim, n, m, seed, shared in ((37, 1100, 1000, 11, True), (5, 300, 257, 23, False)):
        want, got = _both_paths(nsim, n, m, seed, shared)
        assert torch.isfinite(got[0]).all() and float(got[0].abs().max()) > 1e-4       # a real, non-trivial loss
        for w, g in zip(want, got):
            assert torch.equal(w, g)


def test_value_only_call_and_the_size_limit():
    xp, xv = _cloud(3, 200, 31)
    yp, yv = _cloud(1, 150, 32, shift=0.1)
    ref, _, _ = _outputs(3, 200)
    out, _, _ = _outputs(3, 200)
    B.mmd2(xp, xv, yp[0], yv[0], SIG, ref, B.alloc_workspace(B.mmd_workspace_bytes(200, 150, 3)))
    B.mmd2_static(xp, xv, yp[0], yv[0], SIG, out)
    torch.cuda.synchronize()
    assert torch.equal(ref, out)

    limit = B.mmd2_static_scratch_bytes()
    assert limit == 1 << 20
    nsim = limit // 24 + 1                                    # one-block clouds: 24 bytes each, one too many
    assert B.mmd_workspace_bytes(8, 8, nsim - 1) <= limit < B.mmd_workspace_bytes(8, 8, nsim)
    xp, xv = _cloud(nsim, 8, 33)
    big = torch.full((nsim,), -7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(B.OdisseoError) as err:
        B.mmd2_static(xp, xv, xp[0], xv[0], SIG, big)
    assert err.value.status == 7 and "scratch" in str(err.value)
    torch.cuda.synchronize()
    assert bool((big == -7.0).all())                          # refused before anything was launched
    B.mmd2_static(xp[:nsim - 1], xv[:nsim - 1], xp[0], xv[0], SIG, big[:nsim - 1])     # the largest size that fits
    ok = torch.empty(nsim - 1, dtype=torch.float64, device="cuda")
    B.mmd2(xp[:nsim - 1], xv[:nsim - 1], xp[0], xv[0], SIG, ok, B.alloc_workspace(B.mmd_workspace_bytes(8, 8, nsim - 1)))
    torch.cuda.synchronize()
    assert torch.equal(ok, big[:nsim - 1])
