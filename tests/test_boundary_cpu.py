"""CPU-side checks of the C-ABI boundary: the library builds and loads, exports every symbol
include/odisseo.h declares, validates arguments before touching a device, and its stream-K
bookkeeping (SURVEY.md 8a row a1': fixed-order partial sums) is consistent by brute force.
No compute call is made here."""
import ctypes
import os
import re

import pytest

from paper_2511_22468_b200 import binding as B
from paper_2511_22468_b200 import build as build_mod

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build_mod.build()
    return B.lib()


def test_exports_every_declared_symbol(lib):
    header = open(os.path.join(ROOT, "include", "odisseo.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(odisseo_[a-z0-9_]+)\s*\(", header))
    assert declared, "no declarations parsed"
    assert declared == set(B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert b"sm_100a" in lib.odisseo_version()


def test_status_strings(lib):
    for code in range(8):
        assert lib.odisseo_status_string(code)
    assert lib.odisseo_last_cuda_error() == 0


def test_workspace_bytes_is_monotone_and_bounds_every_plan(lib):
    assert B.workspace_bytes(0) == 0 and B.workspace_bytes(-5) == 0
    prev = 0
    for n in (1, 2, 127, 1024, 4096, 4097, 16384, 65536, 262144, 1048576):
        for f64 in (False, True):
            w = B.workspace_bytes(n, f64)
            for sms in (64, 132, 148, 160, 192):
                p = B.describe_plan(n, f64, sms)
                ib = p["i_bodies_per_thread"] * (p["threads_per_cta"] - 32)
                npad = 8 * -(-n // 8)
                rec = 32 if f64 else 16                                      # staged records are plain {x, y, z, m}
                need = (((-(-npad // 256) + 1) * 4 + 255) // 256) * 256 + (npad + 1024) * rec + p["partial_rows"] * 3 * ib * 8
                assert need <= w, (n, f64, sms)
        assert B.workspace_bytes(n) >= prev
        prev = B.workspace_bytes(n)
    assert B.workspace_bytes(1048576) < 4 << 30


@pytest.mark.parametrize("n,sms", [(1, 148), (33, 148), (1000, 148), (1024, 148), (4097, 148), (16384, 148),
                                   (65536, 148), (100003, 7), (262144, 148)])
@pytest.mark.parametrize("f64", [False, True])
def test_unit_ranges_partition_the_work_and_chunks_partition_the_sources(n, sms, f64):
    p = B.describe_plan(n, f64, sms)
    P, nb, S, T = p["persistent_ctas"], p["i_blocks"], p["source_chunks"], p["max_tile_records"]
    U = nb * S
    ib = p["i_bodies_per_thread"] * (p["threads_per_cta"] - 32)
    assert nb == -(-n // ib) and 1 <= P <= U and p["partial_rows"] == U
    # CTA ranges tile [0, U) in order, sizes differ by at most one
    prev_end, sizes = 0, []
    step = max(1, P // 97)
    cs = sorted(set(list(range(0, P, step)) + [0, P - 1]))
    for c in range(P) if P <= 600 else cs:
        _, s, e, _, _ = B.plan_probe(n, f64, sms, 0, c)
        assert s <= e
        if P <= 600:
            assert s == prev_end
            prev_end = e
        sizes.append(e - s)
    if P <= 600:
        assert prev_end == U
    assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1
    # owner(u) is the CTA whose range holds u
    us = range(U) if U <= 3000 else list(range(0, U, max(1, U // 1500))) + [U - 1]
    for u in us:
        c = B.plan_probe(n, f64, sms, u, 0)[0]
        _, s, e, _, _ = B.plan_probe(n, f64, sms, u, c)
        assert s <= u < e
    # the S chunks of an i-block partition the staged sources [0, 8 ceil(n/8)) in order, on multiples of 8,
    # with sizes equal up to one octet; every chunk is non-empty
    end = 0
    lens = []
    for s in range(S):
        _, _, _, lo, hi = B.plan_probe(n, f64, sms, s, 0)
        assert lo == end and hi > lo and lo % 8 == 0 and hi % 8 == 0
        lens.append(hi - lo)
        end = hi
    assert end == 8 * -(-n // 8)
    assert max(lens) - min(lens) <= 8
    assert T in (256, 512)


@pytest.mark.parametrize("n", [1000, 4096, 4097, 16384, 262144])
@pytest.mark.parametrize("f64", [False, True])
def test_summation_grouping_depends_on_the_source_count_only(n, f64):
    """SURVEY 8f NEXT-1 ("same fixed reduction order per i"): tile length and chunk boundaries -- everything that fixes which
    numbers are added in which grouping -- are the same whatever the number of targets (a rank's slice, a tracer set)."""
    ref = B.describe_plan(n, f64, 148)
    chunks = [B.plan_probe(n, f64, 148, s, 0)[3:] for s in range(ref["source_chunks"])]
    for nt in (1, 7, n // 8 + 1, n // 3, n // 2, n, 3 * n):
        p = B.describe_plan(n, f64, 148, nt=nt)
        assert p["source_chunks"] == ref["source_chunks"] and p["max_tile_records"] == ref["max_tile_records"]
        assert [B.plan_probe(n, f64, 148, s, 0, nt=nt)[3:] for s in range(p["source_chunks"])] == chunks


@pytest.mark.parametrize("n", [65536, 262144, 1048576])
def test_large_plans_have_no_wave_quantisation_tail(n):
    """The chunk count is chosen so that the busiest CTA walks at most 1 % more units than the average
    (N = 262,144 on 148 SMs: 128 i-blocks x 15 chunks = 1,920 units, 13 on the busiest CTA against 12.97)."""
    p = B.describe_plan(n, False, 148)
    U = p["i_blocks"] * p["source_chunks"]
    assert p["persistent_ctas"] == 148
    assert -(-U // 148) <= 1.01 * U / 148


def test_argument_validation_happens_before_any_device_work(lib):
    buf = (ctypes.c_float * 64)()
    addr = ctypes.addressof(buf)
    addr16 = (addr + 15) & ~15
    ws = ctypes.c_void_p(256)
    f = lib.odisseo_pair_accel_f32
    assert f(None, None, 0, 1.0, 0.1, None, 0, None) == 0                       # n == 0: no-op
    assert f(None, None, -1, 1.0, 0.1, None, 0, None) == 3                      # n < 0
    assert f(None, addr16, 4, 1.0, 0.1, ws, 1 << 20, None) == 1                 # NULL
    assert f(addr16 + 4, addr16 + 128, 4, 1.0, 0.1, ws, 1 << 20, None) == 2     # misaligned
    assert f(addr16, addr16 + 16, 4, 1.0, 0.1, ws, 1 << 20, None) == 3          # overlap
    assert f(addr16, addr16 + 128, 4, 1.0, 0.0, ws, 1 << 20, None) == 3         # eps <= 0
    assert f(addr16, addr16 + 128, 4, 1.0, 1e-13, ws, 1 << 20, None) == 3       # fp32: eps^-3 would overflow
    v = lib.odisseo_accel_vjp_f32
    dbl = (ctypes.c_double * 64)()
    a8 = ctypes.addressof(dbl)
    # fp32 pull-back forms 3 eps^-5: eps = 1e-8 is refused before any device work, eps = 1e-6 passes validation
    assert v(addr16, addr16 + 64, 4, 1.0, 1e-8, None, 0, addr16 + 128, a8, a8 + 256, ws, 1 << 20, None) == 3
    assert f(addr16, addr16 + 128, 4, float("nan"), 0.1, ws, 1 << 20, None) == 3
    g = lib.odisseo_leapfrog_kdk_f32
    assert g(addr16, addr16 + 64, addr16 + 128, 0, 4, 1.0, 0.1, 0.1, -1, None, ws, 1 << 20, None) == 3
    assert g(addr16, addr16 + 64, addr16 + 128, 1, 4, 1.0, 0.1, 0.1, 0, None, ws, 1 << 20, None) == 0
    bad = B.Potential.make(mn=(1.0, 1.0, 0.0))                                   # MN with b = 0
    e = lib.odisseo_ext_accel_f32
    assert e(addr16, addr16 + 128, 4, 1.0, ctypes.cast(ctypes.pointer(bad), ctypes.c_void_p), 0, None) == 3


def test_product_path_fails_loudly_without_gpu_or_library(monkeypatch):
    import torch
    if not torch.cuda.is_available():
        with pytest.raises(ValueError, match="CUDA tensor"):
            B.pair_accel(torch.zeros(4, 4), torch.zeros(4, 4), 1.0, 0.1, torch.zeros(256, dtype=torch.uint8))
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", "/nonexistent/libodisseo_b200.so")
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        B.lib()


def test_staged_sources_layout_plain_records(lib):
    """The staged source array of the sharded form holds plain {x, y, z, m} records (16 B fp32, 32 B fp64) behind the
    flag block, with room for the 8-aligned padding plus 1,024 records of slack for the in-place all-gather."""
    for n in (1, 7, 8, 1000, 262144):
        for f64, rec in ((False, 16), (True, 32)):
            off, rec_bytes, cap = B.staged_sources_layout(n, f64)
            assert rec_bytes == rec and off % 256 == 0 and off >= 256
            assert cap == 8 * -(-n // 8) + 1024
            assert off + cap * rec_bytes <= B.workspace_bytes(n, f64)


def test_autograd_faces_refuse_gradients_they_do_not_compute():
    """No silent zeros: the bulge shape alpha has no gradient slot in the C ABI, and the MMD loss is differentiated with
    respect to the simulated clouds only.  Checked before any CUDA call, so this runs without a GPU."""
    import torch
    from paper_2511_22468_b200 import autograd as AG
    posm = torch.zeros(4, 4)
    theta8 = torch.ones(8, requires_grad=True)
    with pytest.raises(ValueError, match="alpha"):
        AG.leapfrog_kdk(posm, posm, theta8, torch.tensor(0.1), 1.0, 0.1, 1)
    with pytest.raises(ValueError, match="alpha"):
        AG.ensemble_leapfrog_kdk(posm[None], posm[None], theta8[None].detach().requires_grad_(), torch.ones(1), 1.0, 0.1, 1)
    y = torch.zeros(3, 4, requires_grad=True)
    with pytest.raises(ValueError, match="observed"):
        AG.mmd2(posm, posm, y, y, (1,) * 6)
