"""Thin ctypes binding of include/odisseo.h: argument marshalling only.

Every step of the path runs in the CUDA library; PyTorch supplies device memory and
streams.  There is no CPU fallback: a missing library or a non-zero status raises.
Function names mirror the C ABI without the ``odisseo_`` prefix and precision suffix
(the dtype of the tensors selects ``_f32`` / ``_f64``).
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libodisseo_b200.so")
_lib = None

STATUS = {0: "OK", 1: "ERR_NULL", 2: "ERR_ALIGN", 3: "ERR_ARG", 4: "ERR_WORKSPACE", 5: "ERR_ARCH", 6: "ERR_CUDA",
          7: "ERR_STATIC_LIMIT"}

EXPORTS = [
    "odisseo_version", "odisseo_status_string", "odisseo_last_cuda_error", "odisseo_workspace_bytes",
    "odisseo_pair_accel_f32", "odisseo_pair_accel_f64", "odisseo_pair_accel_soa_f32",
    "odisseo_ext_accel_f32", "odisseo_ext_accel_f64", "odisseo_leapfrog_kdk_f32", "odisseo_leapfrog_kdk_f64",
    "odisseo_leapfrog_kdk_host_f32", "odisseo_leapfrog_kdk_host_f64", "odisseo_describe_plan",
    "odisseo_describe_plan_for", "odisseo_describe_cross_plan_for", "odisseo_plan_probe", "odisseo_launch_count", "odisseo_pair_kernel_name", "odisseo_profile_begin",
    "odisseo_profile_end", "odisseo_profile_times", "odisseo_shutdown", "odisseo_set_fused_max_n", "odisseo_set_cluster_max_n", "odisseo_set_ll_max_n", "odisseo_kick_drift_f32", "odisseo_kick_drift_f64",
    "odisseo_ensemble_workspace_bytes", "odisseo_ensemble_leapfrog_kdk_f32",
    "odisseo_diagnostics_workspace_bytes", "odisseo_diagnostics_f32", "odisseo_diagnostics_f64",
    "odisseo_vjp_workspace_bytes", "odisseo_tape_bytes", "odisseo_accel_vjp_f32", "odisseo_accel_vjp_f64",
    "odisseo_leapfrog_kdk_tape_f32", "odisseo_leapfrog_kdk_tape_f64", "odisseo_leapfrog_kdk_vjp_f32",
    "odisseo_leapfrog_kdk_vjp_f64", "odisseo_ensemble_tape_bytes", "odisseo_ensemble_leapfrog_kdk_tape_f32",
    "odisseo_ensemble_leapfrog_kdk_vjp_f32", "odisseo_cross_workspace_bytes", "odisseo_pair_accel_cross_f32",
    "odisseo_pair_accel_cross_f64", "odisseo_staged_sources_layout", "odisseo_stage_sources_f32", "odisseo_stage_sources_f64",
    "odisseo_pair_accel_staged_f32", "odisseo_pair_accel_staged_f64", "odisseo_kick_drift_slice_f32",
    "odisseo_kick_drift_slice_f64", "odisseo_mmd_workspace_bytes", "odisseo_mmd2_f32",
    "odisseo_mmd2_static_scratch_bytes", "odisseo_mmd2_static_f32", "odisseo_ubench_kinds", "odisseo_ubench_name", "odisseo_ubench_run",
]


class OdisseoError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        lib = _lib
        detail = lib.odisseo_status_string(status).decode() if lib else "?"
        cuda = lib.odisseo_last_cuda_error() if (lib and status == 6) else 0
        super().__init__("%s failed: %s (%s)%s" % (where, STATUS.get(status, status), detail,
                                                    " cudaError=%d" % cuda if cuda else ""))


class _NFW(ctypes.Structure):
    _fields_ = [("M_s", ctypes.c_double), ("r_s", ctypes.c_double)]


class _MN(ctypes.Structure):
    _fields_ = [("M", ctypes.c_double), ("a", ctypes.c_double), ("b", ctypes.c_double)]


class _Bulge(ctypes.Structure):
    _fields_ = [("M_b", ctypes.c_double), ("alpha", ctypes.c_double), ("r_c", ctypes.c_double)]


class Potential(ctypes.Structure):
    """odisseo_potential: NFW{M_s, r_s} + MN{M, a, b} + bulge{M_b, alpha, r_c}; a mass <= 0 disables the term."""
    _fields_ = [("nfw", _NFW), ("mn", _MN), ("bulge", _Bulge)]

    @classmethod
    def make(cls, nfw: Optional[Sequence[float]] = None, mn: Optional[Sequence[float]] = None,
             bulge: Optional[Sequence[float]] = None):
        p = cls()
        p.nfw = _NFW(*(nfw if nfw else (0.0, 1.0)))
        p.mn = _MN(*(mn if mn else (0.0, 1.0, 1.0)))
        p.bulge = _Bulge(*(bulge if bulge else (0.0, 1.8, 1.0)))
        return p


class SimParams(ctypes.Structure):
    """odisseo_sim_params: per-simulation G, eps, dt and potential of the ensemble call."""
    _fields_ = [("G", ctypes.c_double), ("eps", ctypes.c_double), ("dt", ctypes.c_double), ("pot", Potential)]


def lib():
    """Load the C-ABI library; fail loudly when it has not been built."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("CUDA library %s is missing: run `python -m paper_2511_22468_b200.build` "
                               "(there is no CPU fallback)" % LIB_PATH)
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, sz, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t, ctypes.c_int
        f, d = ctypes.c_float, ctypes.c_double
        L.odisseo_version.restype = ctypes.c_char_p
        L.odisseo_status_string.restype = ctypes.c_char_p
        L.odisseo_status_string.argtypes = [ci]
        L.odisseo_last_cuda_error.restype = ci
        L.odisseo_workspace_bytes.restype = sz
        L.odisseo_workspace_bytes.argtypes = [i64, ci]
        for suffix, sc in (("f32", f), ("f64", d)):
            getattr(L, "odisseo_pair_accel_" + suffix).argtypes = [vp, vp, i64, sc, sc, vp, sz, vp]
            getattr(L, "odisseo_pair_accel_cross_" + suffix).argtypes = [vp, i64, vp, i64, vp, sc, sc, vp, sz, vp]
            getattr(L, "odisseo_ext_accel_" + suffix).argtypes = [vp, vp, i64, sc, vp, ci, vp]
            getattr(L, "odisseo_leapfrog_kdk_" + suffix).argtypes = [vp, vp, vp, ci, i64, sc, sc, sc, i64, vp, vp, sz, vp]
            getattr(L, "odisseo_accel_vjp_" + suffix).argtypes = [vp, vp, i64, sc, sc, vp, ci, vp, vp, vp, vp, sz, vp]
            getattr(L, "odisseo_leapfrog_kdk_tape_" + suffix).argtypes = [vp, vp, vp, i64, sc, sc, sc, i64, vp, vp, sz, vp, sz, vp]
            getattr(L, "odisseo_leapfrog_kdk_vjp_" + suffix).argtypes = [vp, i64, sc, sc, sc, i64, vp, ci, vp, vp, vp, vp, vp, sz, vp]
            getattr(L, "odisseo_diagnostics_" + suffix).argtypes = [vp, vp, i64, sc, sc, vp, vp, vp, vp, sz, vp]
            getattr(L, "odisseo_kick_drift_" + suffix).argtypes = [vp, vp, vp, i64, sc, sc, vp, ci, vp, sz, vp]
            getattr(L, "odisseo_leapfrog_kdk_host_" + suffix).argtypes = [vp, vp, vp, ci, i64, sc, sc, sc, i64, vp, vp, sz, vp]
            getattr(L, "odisseo_stage_sources_" + suffix).argtypes = [vp, i64, vp, sz, vp]
            getattr(L, "odisseo_pair_accel_staged_" + suffix).argtypes = [vp, i64, i64, vp, sc, sc, vp, sz, vp]
            getattr(L, "odisseo_kick_drift_slice_" + suffix).argtypes = [vp, vp, vp, i64, i64, i64, sc, sc, vp, ci, vp, sz, vp]
        L.odisseo_staged_sources_layout.argtypes = [i64, ci, vp]
        L.odisseo_mmd_workspace_bytes.restype = sz
        L.odisseo_mmd_workspace_bytes.argtypes = [i64, i64, i64]
        L.odisseo_mmd2_f32.argtypes = [vp, vp, i64, vp, vp, i64, i64, ci, vp, vp, vp, vp, vp, vp, sz, vp]
        L.odisseo_pair_kernel_name.restype = ctypes.c_char_p
        L.odisseo_pair_kernel_name.argtypes = [i64, ci]
        L.odisseo_mmd2_static_scratch_bytes.restype = sz
        L.odisseo_mmd2_static_scratch_bytes.argtypes = []
        L.odisseo_mmd2_static_f32.argtypes = [vp, vp, i64, vp, vp, i64, i64, ci, vp, vp, vp, vp, vp, vp]
        L.odisseo_cross_workspace_bytes.restype = sz
        L.odisseo_cross_workspace_bytes.argtypes = [i64, i64, ci]
        L.odisseo_pair_accel_soa_f32.argtypes = [vp] * 7 + [i64, f, f, vp, sz, vp]
        L.odisseo_describe_plan.argtypes = [i64, ci, vp]
        L.odisseo_describe_plan_for.argtypes = [i64, ci, ci, vp]
        L.odisseo_describe_cross_plan_for.argtypes = [i64, i64, ci, ci, vp]
        L.odisseo_plan_probe.argtypes = [i64, i64, ci, ci, i64, i64, vp]
        L.odisseo_vjp_workspace_bytes.restype = sz
        L.odisseo_vjp_workspace_bytes.argtypes = [i64, ci]
        L.odisseo_tape_bytes.restype = sz
        L.odisseo_tape_bytes.argtypes = [i64, i64, ci]
        L.odisseo_diagnostics_workspace_bytes.restype = sz
        L.odisseo_diagnostics_workspace_bytes.argtypes = [i64]
        L.odisseo_ensemble_workspace_bytes.restype = sz
        L.odisseo_ensemble_workspace_bytes.argtypes = [i64]
        L.odisseo_ensemble_leapfrog_kdk_f32.argtypes = [vp, vp, i64, i64, vp, i64, i64, vp, sz, vp]
        L.odisseo_ensemble_tape_bytes.restype = sz
        L.odisseo_ensemble_tape_bytes.argtypes = [i64, i64, i64]
        L.odisseo_ensemble_leapfrog_kdk_tape_f32.argtypes = [vp, vp, i64, i64, vp, i64, i64, vp, sz, vp, sz, vp]
        L.odisseo_ensemble_leapfrog_kdk_vjp_f32.argtypes = [vp, i64, i64, vp, i64, i64, ci, ci, vp, vp, vp, vp, vp, sz, vp]
        L.odisseo_launch_count.restype = i64
        L.odisseo_launch_count.argtypes = []
        L.odisseo_profile_begin.argtypes = []
        L.odisseo_profile_end.argtypes = [vp, vp, vp]
        L.odisseo_profile_times.argtypes = [vp, i64, vp]
        L.odisseo_shutdown.argtypes = []
        L.odisseo_set_fused_max_n.restype = i64
        L.odisseo_set_fused_max_n.argtypes = [i64]
        L.odisseo_set_cluster_max_n.restype = i64
        L.odisseo_set_cluster_max_n.argtypes = [i64]
        L.odisseo_set_ll_max_n.restype = i64
        L.odisseo_set_ll_max_n.argtypes = [i64]
        L.odisseo_ubench_kinds.argtypes = []
        L.odisseo_ubench_name.restype = ctypes.c_char_p
        L.odisseo_ubench_name.argtypes = [ci]
        L.odisseo_ubench_run.argtypes = [ci, ci, ci, i64, vp, vp]
        _lib = L
    return _lib


def _on_device(fn):
    """The C library works on the CURRENT CUDA device and the stream passed in.  Every CUDA tensor argument must live
    on one device; that device is made current for the call (so tensors on cuda:1 never launch on GPU 0) and the
    default stream argument resolves to ITS current stream."""
    import functools

    @functools.wraps(fn)
    def wrapper(*args, **kwargs):
        devs = {t.device for t in list(args) + list(kwargs.values()) if isinstance(t, torch.Tensor) and t.is_cuda}
        if len(devs) > 1:
            raise ValueError("%s: tensors live on different devices %s" % (fn.__name__, sorted(str(d) for d in devs)))
        if not devs:
            return fn(*args, **kwargs)
        with torch.cuda.device(next(iter(devs))):
            return fn(*args, **kwargs)
    return wrapper


def _check(status: int, where: str):
    if status != 0:
        raise OdisseoError(status, where)


def _suffix(t: torch.Tensor) -> str:
    if t.dtype == torch.float32:
        return "f32"
    if t.dtype == torch.float64:
        return "f64"
    raise TypeError("expected float32 or float64 tensors, got %s" % t.dtype)


def _rec(t: torch.Tensor, name: str, n: Optional[int] = None, cuda: bool = True) -> int:
    if t.dim() != 2 or t.shape[1] != 4 or not t.is_contiguous():
        raise ValueError("%s must be a contiguous [n, 4] tensor" % name)
    if cuda and not t.is_cuda:
        raise ValueError("%s must be a CUDA tensor (no CPU fallback)" % name)
    if n is not None and t.shape[0] != n:
        raise ValueError("%s has %d records, expected %d" % (name, t.shape[0], n))
    return t.shape[0]


def _stream(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _pot(pot: Optional[Potential]):
    return ctypes.cast(ctypes.pointer(pot), ctypes.c_void_p) if pot is not None else None


def version() -> str:
    return lib().odisseo_version().decode()


def workspace_bytes(n: int, is_f64: bool = False) -> int:
    return int(lib().odisseo_workspace_bytes(int(n), int(bool(is_f64))))


def host_workspace_bytes(n: int, is_f64: bool = False) -> int:
    """Workspace for leapfrog_kdk_host: scratch + three device state arrays."""
    return workspace_bytes(n, is_f64) + 3 * n * (32 if is_f64 else 16) + 768


def alloc_workspace(nbytes: int, device="cuda") -> torch.Tensor:
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


_PLAN_KEYS = ["i_bodies_per_thread", "threads_per_cta", "max_tile_records", "persistent_ctas", "i_blocks", "source_chunks",
              "partial_rows", "kernels_per_step"]


def describe_plan(n: int, is_f64: bool = False, num_sms: Optional[int] = None, nt: Optional[int] = None) -> dict:
    """Launch plan for n sources (and nt targets, default n) on the current device or one with num_sms SMs."""
    out = (ctypes.c_int64 * 8)()
    if num_sms is None:
        _check(lib().odisseo_describe_plan(int(n), int(is_f64), out), "describe_plan")
    else:
        _check(lib().odisseo_describe_cross_plan_for(int(n if nt is None else nt), int(n), int(is_f64), int(num_sms), out),
               "describe_cross_plan_for")
    return dict(zip(_PLAN_KEYS, [int(v) for v in out]))


def plan_probe(n: int, is_f64: bool, num_sms: int, u: int, c: int, nt: Optional[int] = None):
    """(owner CTA of unit u, first unit of CTA c, end unit of CTA c, first source of u's chunk, end source)."""
    out = (ctypes.c_int64 * 5)()
    _check(lib().odisseo_plan_probe(int(n if nt is None else nt), int(n), int(is_f64), int(num_sms), int(u), int(c), out),
           "plan_probe")
    return tuple(int(v) for v in out)


@_on_device
def pair_accel(posm: torch.Tensor, acc: torch.Tensor, G: float, eps: float, workspace: torch.Tensor, stream=None):
    """acc[n,4] = pair acceleration of posm[n,4] (odisseo_pair_accel_f32/_f64)."""
    n = _rec(posm, "posm")
    _rec(acc, "acc", n)
    sfx = _suffix(posm)
    if acc.dtype != posm.dtype:
        raise TypeError("posm and acc dtypes differ")
    fn = getattr(lib(), "odisseo_pair_accel_" + sfx)
    _check(fn(posm.data_ptr(), acc.data_ptr(), n, G, eps, workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "pair_accel_" + sfx)
    return acc


def cross_workspace_bytes(nt: int, n: int, is_f64: bool = False) -> int:
    return int(lib().odisseo_cross_workspace_bytes(int(nt), int(n), int(bool(is_f64))))


@_on_device
def pair_accel_cross(targets: torch.Tensor, sources: torch.Tensor, acc: torch.Tensor, G: float, eps: float,
                     workspace: torch.Tensor, stream=None):
    """acc[nt,4] = acceleration at targets[nt,4] due to sources[n,4] (odisseo_pair_accel_cross_f32/_f64)."""
    nt = _rec(targets, "targets")
    n = _rec(sources, "sources")
    _rec(acc, "acc", nt)
    sfx = _suffix(targets)
    if sources.dtype != targets.dtype or acc.dtype != targets.dtype:
        raise TypeError("targets, sources and acc dtypes differ")
    fn = getattr(lib(), "odisseo_pair_accel_cross_" + sfx)
    _check(fn(targets.data_ptr(), nt, sources.data_ptr(), n, acc.data_ptr(), G, eps, workspace.data_ptr(),
              workspace.numel(), _stream(stream)), "pair_accel_cross_" + sfx)
    return acc


@_on_device
def pair_accel_soa(x, y, z, m, ax, ay, az, G: float, eps: float, workspace: torch.Tensor, stream=None):
    n = x.numel()
    for t in (x, y, z, m, ax, ay, az):
        if t.dtype != torch.float32 or not t.is_cuda or not t.is_contiguous() or t.numel() != n:
            raise ValueError("SoA arguments must be contiguous float32 CUDA vectors of equal length")
    _check(lib().odisseo_pair_accel_soa_f32(x.data_ptr(), y.data_ptr(), z.data_ptr(), m.data_ptr(), ax.data_ptr(),
                                            ay.data_ptr(), az.data_ptr(), n, G, eps, workspace.data_ptr(),
                                            workspace.numel(), _stream(stream)), "pair_accel_soa_f32")


@_on_device
def ext_accel(posm: torch.Tensor, acc: torch.Tensor, G: float, pot: Optional[Potential], accumulate: bool = False,
              stream=None):
    n = _rec(posm, "posm")
    _rec(acc, "acc", n)
    sfx = _suffix(posm)
    fn = getattr(lib(), "odisseo_ext_accel_" + sfx)
    _check(fn(posm.data_ptr(), acc.data_ptr(), n, G, _pot(pot), int(bool(accumulate)), _stream(stream)),
           "ext_accel_" + sfx)
    return acc


@_on_device
def leapfrog_kdk(posm: torch.Tensor, vel: torch.Tensor, acc: torch.Tensor, G: float, eps: float, dt: float,
                 nsteps: int, pot: Optional[Potential], workspace: torch.Tensor, acc_valid: bool = False, stream=None):
    """nsteps KDK steps in place on device tensors (odisseo_leapfrog_kdk_f32/_f64)."""
    n = _rec(posm, "posm")
    _rec(vel, "vel", n)
    _rec(acc, "acc", n)
    sfx = _suffix(posm)
    fn = getattr(lib(), "odisseo_leapfrog_kdk_" + sfx)
    _check(fn(posm.data_ptr(), vel.data_ptr(), acc.data_ptr(), int(bool(acc_valid)), n, G, eps, dt, int(nsteps),
              _pot(pot), workspace.data_ptr(), workspace.numel(), _stream(stream)), "leapfrog_kdk_" + sfx)


@_on_device
def kick_drift(posm: torch.Tensor, vel: torch.Tensor, acc: torch.Tensor, G: float, dt: float,
               pot: Optional[Potential], mode: int, workspace: torch.Tensor, stream=None):
    """The O(N) integrator kernel alone (odisseo_kick_drift_f32/_f64): mode 1 = closing half kick,
    2 = opening half kick + drift (+ staging of the moved sources), 3 = both."""
    n = _rec(posm, "posm")
    _rec(vel, "vel", n)
    _rec(acc, "acc", n)
    sfx = _suffix(posm)
    fn = getattr(lib(), "odisseo_kick_drift_" + sfx)
    _check(fn(posm.data_ptr(), vel.data_ptr(), acc.data_ptr(), n, G, dt, _pot(pot), int(mode), workspace.data_ptr(),
              workspace.numel(), _stream(stream)), "kick_drift_" + sfx)


def leapfrog_kdk_host(posm: torch.Tensor, vel: torch.Tensor, acc: Optional[torch.Tensor], G: float, eps: float,
                      dt: float, nsteps: int, pot: Optional[Potential], workspace: torch.Tensor,
                      acc_valid: bool = False, stream=None):
    """Host-buffer face: posm/vel/acc are (pinned) CPU tensors updated in place after a stream sync."""
    n = _rec(posm, "posm", cuda=False)
    _rec(vel, "vel", n, cuda=False)
    if posm.is_cuda or vel.is_cuda:
        raise ValueError("leapfrog_kdk_host takes host tensors")
    if acc is not None:
        _rec(acc, "acc", n, cuda=False)
    sfx = _suffix(posm)
    fn = getattr(lib(), "odisseo_leapfrog_kdk_host_" + sfx)
    _check(fn(posm.data_ptr(), vel.data_ptr(), acc.data_ptr() if acc is not None else None, int(bool(acc_valid)),
              n, G, eps, dt,
              int(nsteps), _pot(pot), workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "leapfrog_kdk_host_" + sfx)


GRADIENT_FIELDS = ("M_s", "r_s", "M_d", "a", "b", "G", "eps", "dt", "M_b", "r_c")
NGRAD = len(GRADIENT_FIELDS)


def vjp_workspace_bytes(n: int, is_f64: bool = False) -> int:
    return int(lib().odisseo_vjp_workspace_bytes(int(n), int(bool(is_f64))))


def tape_bytes(n: int, nsteps: int, is_f64: bool = False) -> int:
    return int(lib().odisseo_tape_bytes(int(n), int(nsteps), int(bool(is_f64))))


def _f64vec(t: torch.Tensor, name: str, numel: int):
    if t.dtype != torch.float64 or t.numel() < numel or not t.is_cuda or not t.is_contiguous():
        raise ValueError("%s must be a contiguous float64 CUDA tensor of %d values" % (name, numel))


@_on_device
def accel_vjp(posm: torch.Tensor, cot: torch.Tensor, G: float, eps: float, pot: Optional[Potential], gx: torch.Tensor,
              gm: torch.Tensor, gparams: torch.Tensor, workspace: torch.Tensor, with_eps_G: bool = False, stream=None):
    """Cotangent cot [n,4] pulled back through a = a_pair + a_ext (odisseo_accel_vjp_f32/_f64)."""
    n = _rec(posm, "posm")
    _rec(cot, "cot", n)
    _rec(gx, "gx", n)
    _f64vec(gm, "gm", n)
    _f64vec(gparams, "gparams", NGRAD)
    sfx = _suffix(posm)
    fn = getattr(lib(), "odisseo_accel_vjp_" + sfx)
    _check(fn(posm.data_ptr(), cot.data_ptr(), n, G, eps, _pot(pot), int(bool(with_eps_G)), gx.data_ptr(), gm.data_ptr(),
              gparams.data_ptr(),
              workspace.data_ptr(), workspace.numel(), _stream(stream)), "accel_vjp_" + sfx)


@_on_device
def leapfrog_kdk_tape(posm: torch.Tensor, vel: torch.Tensor, acc: torch.Tensor, G: float, eps: float, dt: float,
                      nsteps: int, pot: Optional[Potential], tape: torch.Tensor, workspace: torch.Tensor, stream=None):
    """leapfrog_kdk that also records the nsteps + 1 snapshots {posm, vel, pair-only acc} into tape
    (same dtype, at least 3 * (nsteps + 1) * n * 4 scalars)."""
    n = _rec(posm, "posm")
    _rec(vel, "vel", n)
    _rec(acc, "acc", n)
    sfx = _suffix(posm)
    if tape.dtype != posm.dtype or not tape.is_cuda or not tape.is_contiguous():
        raise ValueError("tape must be a contiguous CUDA tensor of the state's dtype")
    fn = getattr(lib(), "odisseo_leapfrog_kdk_tape_" + sfx)
    _check(fn(posm.data_ptr(), vel.data_ptr(), acc.data_ptr(), n, G, eps, dt, int(nsteps), _pot(pot), tape.data_ptr(),
              tape.numel() * tape.element_size(), workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "leapfrog_kdk_tape_" + sfx)


@_on_device
def leapfrog_kdk_vjp(tape: torch.Tensor, n: int, G: float, eps: float, dt: float, nsteps: int, pot: Optional[Potential],
                     lx: torch.Tensor, lv: torch.Tensor, gm: torch.Tensor, gparams: torch.Tensor,
                     workspace: torch.Tensor, with_eps_G: bool = False, stream=None):
    """Reverse-mode derivative of nsteps KDK steps from the tape: lx, lv [n,4] hold dL/dx_N, dL/dv_N on entry and
    dL/dx_0, dL/dv_0 on exit; gm [n] and gparams [10] (GRADIENT_FIELDS) are float64 outputs."""
    _rec(lx, "lx", n)
    _rec(lv, "lv", n)
    _f64vec(gm, "gm", n)
    _f64vec(gparams, "gparams", NGRAD)
    sfx = _suffix(lx)
    if tape.dtype != lx.dtype or not tape.is_cuda or tape.numel() < 12 * n * (nsteps + 1):
        raise ValueError("tape does not hold nsteps + 1 snapshots of the state's dtype")
    fn = getattr(lib(), "odisseo_leapfrog_kdk_vjp_" + sfx)
    _check(fn(tape.data_ptr(), n, G, eps, dt, int(nsteps), _pot(pot), int(bool(with_eps_G)), lx.data_ptr(), lv.data_ptr(),
              gm.data_ptr(),
              gparams.data_ptr(), workspace.data_ptr(), workspace.numel(), _stream(stream)), "leapfrog_kdk_vjp_" + sfx)


DIAGNOSTIC_FIELDS = ("kinetic", "pair_potential", "ext_potential", "px", "py", "pz", "lx", "ly", "lz",
                     "com_x", "com_y", "com_z", "mass", "energy")


def diagnostics_workspace_bytes(n: int) -> int:
    return int(lib().odisseo_diagnostics_workspace_bytes(int(n)))


@_on_device
def diagnostics(posm: torch.Tensor, vel: torch.Tensor, G: float, eps: float, pot: Optional[Potential],
                out: torch.Tensor, workspace: torch.Tensor, phi: Optional[torch.Tensor] = None, stream=None):
    """Energies, momenta and centre of mass of a state in fp64 (odisseo_diagnostics_f32/_f64).
    out: float64 CUDA tensor of 16 values (DIAGNOSTIC_FIELDS name the first 14); phi: optional float64 [n]."""
    n = _rec(posm, "posm")
    _rec(vel, "vel", n)
    sfx = _suffix(posm)
    if out.dtype != torch.float64 or out.numel() < 16 or not out.is_cuda or not out.is_contiguous():
        raise ValueError("out must be a contiguous float64 CUDA tensor of at least 16 values")
    if phi is not None and (phi.dtype != torch.float64 or phi.numel() != n or not phi.is_cuda or not phi.is_contiguous()):
        raise ValueError("phi must be a contiguous float64 CUDA tensor of n values")
    fn = getattr(lib(), "odisseo_diagnostics_" + sfx)
    _check(fn(posm.data_ptr(), vel.data_ptr(), n, G, eps, _pot(pot), out.data_ptr(),
              phi.data_ptr() if phi is not None else None, workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "diagnostics_" + sfx)
    return out


def ensemble_workspace_bytes(nsim: int) -> int:
    return int(lib().odisseo_ensemble_workspace_bytes(int(nsim)))


def _sim_params(params):
    arr = (SimParams * len(params))()
    for k, (G, eps, dt, pot) in enumerate(params):
        arr[k].G, arr[k].eps, arr[k].dt = float(G), float(eps), float(dt)
        arr[k].pot = pot if pot is not None else Potential.make()
    return arr


def _ens_state(posm, vel, names="posm and vel"):
    if posm.dim() != 3 or posm.shape[2] != 4 or posm.shape != vel.shape or not posm.is_contiguous() \
            or not vel.is_contiguous() or posm.dtype != torch.float32 or vel.dtype != torch.float32:
        raise ValueError("%s must be contiguous float32 [nsim, n, 4] tensors" % names)
    if not (posm.is_cuda and vel.is_cuda):
        raise ValueError("%s must be CUDA tensors (no CPU fallback)" % names)
    return int(posm.shape[0]), int(posm.shape[1])


def ensemble_tape_bytes(n: int, nsim: int, nsteps: int) -> int:
    return int(lib().odisseo_ensemble_tape_bytes(int(n), int(nsim), int(nsteps)))


@_on_device
def ensemble_leapfrog_kdk_tape(posm: torch.Tensor, vel: torch.Tensor, params, nsteps: int, tape: torch.Tensor,
                               workspace: torch.Tensor, stream=None):
    """ensemble_leapfrog_kdk that also records {posm, vel, total acc} per simulation and step into tape (float32)."""
    nsim, n = _ens_state(posm, vel)
    if tape.dtype != torch.float32 or not tape.is_cuda or not tape.is_contiguous():
        raise ValueError("tape must be a contiguous float32 CUDA tensor")
    arr = _sim_params(params)
    _check(lib().odisseo_ensemble_leapfrog_kdk_tape_f32(posm.data_ptr(), vel.data_ptr(), n, nsim,
                                                        ctypes.cast(arr, ctypes.c_void_p), len(params), int(nsteps),
                                                        tape.data_ptr(), tape.numel() * 4, workspace.data_ptr(),
                                                        workspace.numel(), _stream(stream)),
           "ensemble_leapfrog_kdk_tape_f32")


@_on_device
def ensemble_leapfrog_kdk_vjp(tape: torch.Tensor, params, nsteps: int, lx: torch.Tensor, lv: torch.Tensor,
                              gm: torch.Tensor, gparams: torch.Tensor, workspace: torch.Tensor,
                              with_eps_G: bool = False, accumulate: bool = False, stream=None):
    """Gradients of every simulation of a batch from its tape: lx, lv [nsim, n, 4] in/out; gm float64 [nsim, n];
    gparams float64 [nsim, 10] (GRADIENT_FIELDS); accumulate adds to gm and gparams instead of overwriting them."""
    nsim, n = _ens_state(lx, lv, "lx and lv")
    _f64vec(gm, "gm", nsim * n)
    _f64vec(gparams, "gparams", nsim * NGRAD)
    if tape.dtype != torch.float32 or not tape.is_cuda or tape.numel() * 4 < ensemble_tape_bytes(n, nsim, nsteps):
        raise ValueError("tape does not hold nsteps + 1 snapshots of every simulation")
    arr = _sim_params(params)
    _check(lib().odisseo_ensemble_leapfrog_kdk_vjp_f32(tape.data_ptr(), n, nsim, ctypes.cast(arr, ctypes.c_void_p),
                                                       len(params), int(nsteps), int(bool(with_eps_G)), int(bool(accumulate)),
                                                       lx.data_ptr(), lv.data_ptr(), gm.data_ptr(), gparams.data_ptr(),
                                                       workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "ensemble_leapfrog_kdk_vjp_f32")


@_on_device
def ensemble_leapfrog_kdk(posm: torch.Tensor, vel: torch.Tensor, params, nsteps: int, workspace: torch.Tensor,
                          stream=None):
    """nsim independent small-N simulations in one launch (odisseo_ensemble_leapfrog_kdk_f32).

    posm, vel: contiguous float32 CUDA tensors [nsim, n, 4]; params: a list of (G, eps, dt, Potential-or-None)
    tuples, one per simulation or a single one shared by all."""
    if posm.dim() != 3 or posm.shape[2] != 4 or posm.shape != vel.shape or not posm.is_contiguous() \
            or not vel.is_contiguous() or posm.dtype != torch.float32 or vel.dtype != torch.float32:
        raise ValueError("posm and vel must be contiguous float32 [nsim, n, 4] tensors")
    if not (posm.is_cuda and vel.is_cuda):
        raise ValueError("posm and vel must be CUDA tensors (no CPU fallback)")
    nsim, n = int(posm.shape[0]), int(posm.shape[1])
    arr = (SimParams * len(params))()
    for k, (G, eps, dt, pot) in enumerate(params):
        arr[k].G, arr[k].eps, arr[k].dt = float(G), float(eps), float(dt)
        arr[k].pot = pot if pot is not None else Potential.make()
    _check(lib().odisseo_ensemble_leapfrog_kdk_f32(posm.data_ptr(), vel.data_ptr(), n, nsim,
                                                   ctypes.cast(arr, ctypes.c_void_p), len(params), int(nsteps),
                                                   workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "ensemble_leapfrog_kdk_f32")


def launch_count() -> int:
    """Kernels launched by the library in this process so far (odisseo_launch_count)."""
    return int(lib().odisseo_launch_count())


def profile_begin():
    """Start bracketing every pair-kernel launch with CUDA events (odisseo_profile_begin)."""
    _check(lib().odisseo_profile_begin(), "profile_begin")


def profile_end():
    """(total ms of the timed pair-kernel launches, launches timed, launches dropped)."""
    ms, nl, nd = ctypes.c_double(0.0), ctypes.c_int64(0), ctypes.c_int64(0)
    _check(lib().odisseo_profile_end(ctypes.byref(ms), ctypes.byref(nl), ctypes.byref(nd)), "profile_end")
    return float(ms.value), int(nl.value), int(nd.value)


def pair_kernel_name(n: int, is_f64: bool = False) -> str:
    """The pair-kernel instantiation pair_accel / leapfrog_kdk launch for n particles (odisseo_pair_kernel_name)."""
    return lib().odisseo_pair_kernel_name(int(n), int(bool(is_f64))).decode()


def mmd_workspace_bytes(n: int, m: int, nsim: int = 1) -> int:
    return int(lib().odisseo_mmd_workspace_bytes(int(n), int(m), int(nsim)))


@_on_device
def mmd2(xpos: torch.Tensor, xvel: torch.Tensor, ypos: torch.Tensor, yvel: torch.Tensor, sigma: Sequence[float], out: torch.Tensor,
         workspace: torch.Tensor, gpos: Optional[torch.Tensor] = None, gvel: Optional[torch.Tensor] = None,
         grad_scale: Optional[torch.Tensor] = None, stream=None):
    """MMD^2 between simulated clouds xpos/xvel [nsim, n, 4] (or [n, 4]) and observed ypos/yvel ([m, 4] shared, or
    [nsim, m, 4]) into out [nsim] float64; with gpos/gvel also grad_scale * dMMD^2/d(xpos, xvel) (odisseo_mmd2_f32)."""
    if xpos.dim() == 2:
        xpos, xvel = xpos.unsqueeze(0), xvel.unsqueeze(0)
        if gpos is not None:
            gpos, gvel = gpos.unsqueeze(0), gvel.unsqueeze(0)
    nsim, n = _ens_state(xpos, xvel, "xpos and xvel")
    shared = ypos.dim() == 2
    if shared:
        m = _rec(ypos, "ypos")
        _rec(yvel, "yvel", m)
        if ypos.dtype != torch.float32 or yvel.dtype != torch.float32:
            raise TypeError("mmd2 is float32")
    else:
        ns2, m = _ens_state(ypos, yvel, "ypos and yvel")
        if ns2 != nsim:
            raise ValueError("ypos holds %d clouds, expected 1 shared or %d" % (ns2, nsim))
    _f64vec(out, "out", nsim)
    if (gpos is None) != (gvel is None):
        raise ValueError("gpos and gvel go together")
    if gpos is not None:
        ng, nn = _ens_state(gpos, gvel, "gpos and gvel")
        if (ng, nn) != (nsim, n):
            raise ValueError("gpos/gvel must match xpos/xvel")
    if grad_scale is not None:
        _f64vec(grad_scale, "grad_scale", nsim)
    sig = (ctypes.c_double * 6)(*[float(v) for v in sigma])
    _check(lib().odisseo_mmd2_f32(xpos.data_ptr(), xvel.data_ptr(), n, ypos.data_ptr(), yvel.data_ptr(), m, nsim, int(shared), sig,
                                  grad_scale.data_ptr() if grad_scale is not None else None, out.data_ptr(),
                                  gpos.data_ptr() if gpos is not None else None, gvel.data_ptr() if gvel is not None else None,
                                  workspace.data_ptr(), workspace.numel(), _stream(stream)), "mmd2_f32")


def mmd2_static_scratch_bytes() -> int:
    """Size of the library's built-in scratch array; mmd2_static refuses calls whose mmd_workspace_bytes exceed it."""
    return int(lib().odisseo_mmd2_static_scratch_bytes())


@_on_device
def mmd2_static(xpos: torch.Tensor, xvel: torch.Tensor, ypos: torch.Tensor, yvel: torch.Tensor, sigma: Sequence[float],
                out: torch.Tensor, gpos: Optional[torch.Tensor] = None, gvel: Optional[torch.Tensor] = None,
                grad_scale: Optional[torch.Tensor] = None, stream=None):
    """mmd2 without a workspace tensor (odisseo_mmd2_static_f32), for callers that must not allocate device memory:
    a loss evaluated inside a process whose memory pool already owns the HBM, or inside a loop where the stall of a
    cudaMalloc is not acceptable.  You pass inputs and outputs you already hold; the per-block sums go to a 1 MiB
    array built into the library, and neither this wrapper nor the call under it allocates on the device.  Same
    arguments and bit-identical results as mmd2.  Raises OdisseoError (ERR_STATIC_LIMIT) when
    mmd_workspace_bytes(n, m, nsim) > mmd2_static_scratch_bytes().  The first call on a device also looks up the
    array's address: make it before any stream capture.  All calls on a device share the array, so calls that
    overlap on the GPU (two streams with no ordering between them) corrupt each other; calls on one stream are fine."""
    if xpos.dim() == 2:
        xpos, xvel = xpos.unsqueeze(0), xvel.unsqueeze(0)
        if gpos is not None:
            gpos, gvel = gpos.unsqueeze(0), gvel.unsqueeze(0)
    nsim, n = _ens_state(xpos, xvel, "xpos and xvel")
    shared = ypos.dim() == 2
    if shared:
        m = _rec(ypos, "ypos")
        _rec(yvel, "yvel", m)
        if ypos.dtype != torch.float32 or yvel.dtype != torch.float32:
            raise TypeError("mmd2_static is float32")
    else:
        ns2, m = _ens_state(ypos, yvel, "ypos and yvel")
        if ns2 != nsim:
            raise ValueError("ypos holds %d clouds, expected 1 shared or %d" % (ns2, nsim))
    _f64vec(out, "out", nsim)
    if (gpos is None) != (gvel is None):
        raise ValueError("gpos and gvel go together")
    if gpos is not None:
        ng, nn = _ens_state(gpos, gvel, "gpos and gvel")
        if (ng, nn) != (nsim, n):
            raise ValueError("gpos/gvel must match xpos/xvel")
    if grad_scale is not None:
        _f64vec(grad_scale, "grad_scale", nsim)
    sig = (ctypes.c_double * 6)(*[float(v) for v in sigma])
    _check(lib().odisseo_mmd2_static_f32(xpos.data_ptr(), xvel.data_ptr(), n, ypos.data_ptr(), yvel.data_ptr(), m, nsim,
                                         int(shared), sig, grad_scale.data_ptr() if grad_scale is not None else None,
                                         out.data_ptr(), gpos.data_ptr() if gpos is not None else None,
                                         gvel.data_ptr() if gvel is not None else None, _stream(stream)), "mmd2_static_f32")


def set_fused_max_n(n: int) -> int:
    """Largest n leapfrog_kdk runs as one cooperative whole-loop launch (0 = never); returns the previous value."""
    return int(lib().odisseo_set_fused_max_n(int(n)))


def set_ll_max_n(n: int) -> int:
    """Largest n leapfrog_kdk runs as the owner-computes whole-loop kernel with the flag-in-data exchange (0 = never,
    negative = defaults); returns the previous fp32 value."""
    return int(lib().odisseo_set_ll_max_n(int(n)))


def set_cluster_max_n(n: int) -> int:
    """Largest n leapfrog_kdk runs on one thread-block cluster (0 = never, negative = defaults); returns the previous fp32 value."""
    return int(lib().odisseo_set_cluster_max_n(int(n)))


def shutdown():
    """Release the cached graph executables and profile events (odisseo_shutdown)."""
    _check(lib().odisseo_shutdown(), "shutdown")


def profile_times():
    """Durations (ms) of the pair-kernel launches the last profile timed, in launch order."""
    cnt = ctypes.c_int64(0)
    _check(lib().odisseo_profile_times(None, 0, ctypes.byref(cnt)), "profile_times")
    buf = (ctypes.c_double * max(int(cnt.value), 1))()
    _check(lib().odisseo_profile_times(buf, int(cnt.value), ctypes.byref(cnt)), "profile_times")
    return [float(buf[k]) for k in range(int(cnt.value))]


def staged_sources_layout(n: int, is_f64: bool = False):
    """(byte offset of record 0 in a workspace, bytes per record, records the array has room for)."""
    out = (ctypes.c_int64 * 3)()
    _check(lib().odisseo_staged_sources_layout(int(n), int(bool(is_f64)), out), "staged_sources_layout")
    return int(out[0]), int(out[1]), int(out[2])


@_on_device
def stage_sources(posm: torch.Tensor, workspace: torch.Tensor, stream=None):
    """Stage all n sources (records, padding, equal-mass flags) into the workspace (odisseo_stage_sources_*)."""
    n = _rec(posm, "posm")
    sfx = _suffix(posm)
    _check(getattr(lib(), "odisseo_stage_sources_" + sfx)(posm.data_ptr(), n, workspace.data_ptr(), workspace.numel(), _stream(stream)),
           "stage_sources_" + sfx)


@_on_device
def pair_accel_staged(targets: torch.Tensor, n: int, acc: torch.Tensor, G: float, eps: float, workspace: torch.Tensor, stream=None):
    """acc[nt,4] = pair acceleration at targets[nt,4] due to the n sources already staged in the workspace."""
    nt = _rec(targets, "targets")
    _rec(acc, "acc", nt)
    sfx = _suffix(targets)
    _check(getattr(lib(), "odisseo_pair_accel_staged_" + sfx)(targets.data_ptr(), nt, int(n), acc.data_ptr(), G, eps, workspace.data_ptr(),
                                                             workspace.numel(), _stream(stream)), "pair_accel_staged_" + sfx)


@_on_device
def kick_drift_slice(posm_slice: torch.Tensor, vel: torch.Tensor, acc: torch.Tensor, n: int, lo: int, G: float, dt: float,
                     pot: Optional[Potential], mode: int, workspace: torch.Tensor, stream=None):
    """odisseo_kick_drift_slice_*: kick/drift the slice [lo, lo + count) of n particles and re-stage its records."""
    count = _rec(posm_slice, "posm_slice")
    _rec(vel, "vel", count)
    _rec(acc, "acc", count)
    sfx = _suffix(posm_slice)
    _check(getattr(lib(), "odisseo_kick_drift_slice_" + sfx)(posm_slice.data_ptr(), vel.data_ptr(), acc.data_ptr(), int(n), int(lo), count,
                                                            G, dt, _pot(pot), int(mode), workspace.data_ptr(), workspace.numel(),
                                                            _stream(stream)), "kick_drift_slice_" + sfx)


def ubench_kinds():
    """Names of the pipe-rate micro-benchmarks, indexed by kind."""
    L = lib()
    return [L.odisseo_ubench_name(k).decode() for k in range(L.odisseo_ubench_kinds())]


def ubench_run(kind: int, ctas_per_sm: int = 2, threads: int = 1024, iters: int = 1 << 14, stream=None):
    """One micro-benchmark: dict(ms, fp32_lane_ops, mufu, fp64_ops, lds, sms) as counted by the library."""
    out = (ctypes.c_double * 6)()
    _check(lib().odisseo_ubench_run(int(kind), int(ctas_per_sm), int(threads), int(iters), out, _stream(stream)), "ubench_run")
    return {"ms": out[0], "fp32_lane_ops": out[1], "mufu": out[2], "fp64_ops": out[3], "lds": out[4], "sms": int(out[5])}
