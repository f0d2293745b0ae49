"""Python face of the fp64 CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It builds and loads
``oracle/odisseo_oracle.c`` (plain C, gcc -O2 -fopenmp, no -ffast-math) and adds
the O(N) diagnostics as plain numpy definitions.  It imports nothing from the
CUDA package ``paper_2511_22468_b200`` and shares no code with it.

Citations: PAPER.md:L15-17 (direct softened pair force), L9/L45/L63 (NFW + MN),
L47 (Velocity-Verlet, fixed steps); formulas from BASELINE.json north_star and
DESIGN.md readings R1-R14.  No function is "parity unpinned": see the pin list
in the header of odisseo_oracle.c; the O(N) diagnostics below (kinetic energy, momenta, centre of
mass) are pinned by hand values in tests/test_oracle_leapfrog.py (single particle on each axis,
hand-expanded cross product, unequal-mass binary L_z = mu omega d^2) and the zero point of the
potentials by closed forms in tests/test_oracle_potential.py (Phi_NFW(0) = -G M_s/r_s,
r Phi_NFW / ln(1+r/r_s) = -G M_s, Phi_MN(0) = -G M/(a+b)).

Layouts: ``posm`` float64 [n, 4] = {x, y, z, m}; ``vel`` / ``acc`` float64 [n, 3].
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "odisseo_oracle.c")
_LIB = os.path.join(_HERE, "libodisseo_oracle.so")
_lock = threading.Lock()
_lib = None


class NFW(ctypes.Structure):
    _fields_ = [("M_s", ctypes.c_double), ("r_s", ctypes.c_double)]


class MN(ctypes.Structure):
    _fields_ = [("M", ctypes.c_double), ("a", ctypes.c_double), ("b", ctypes.c_double)]


class Bulge(ctypes.Structure):
    _fields_ = [("M_b", ctypes.c_double), ("alpha", ctypes.c_double), ("r_c", ctypes.c_double)]


class Potential(ctypes.Structure):
    """NFW{M_s, r_s} + MN{M, a, b} + bulge{M_b, alpha, r_c}; a mass <= 0 disables that term."""
    _fields_ = [("nfw", NFW), ("mn", MN), ("bulge", Bulge)]

    @classmethod
    def make(cls, nfw=None, mn=None, bulge=None):
        p = cls()
        p.nfw = NFW(*(nfw if nfw else (0.0, 1.0)))
        p.mn = MN(*(mn if mn else (0.0, 1.0, 1.0)))
        p.bulge = Bulge(*(bulge if bulge else (0.0, 1.8, 1.0)))
        return p


def build(force: bool = False) -> str:
    """Compile the oracle's C file (building the checker is not using it)."""
    with _lock:
        stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC)
        if force or stale:
            tmp = _LIB + ".tmp.%d" % os.getpid()
            subprocess.check_call(
                ["gcc", "-O2", "-fopenmp", "-std=c11", "-shared", "-fPIC", "-o", tmp, _SRC, "-lm"])
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        d, i64, p = ctypes.c_double, ctypes.c_int64, ctypes.c_void_p
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_pair_accel.argtypes = [i64, p, d, d, i64, p, p, p]
        lib.oracle_pair_accel.restype = None
        lib.oracle_pair_potential_energy.argtypes = [i64, p, d, d]
        lib.oracle_pair_potential_energy.restype = d
        lib.oracle_ext_accel.argtypes = [i64, p, d, p, p]
        lib.oracle_ext_accel.restype = None
        lib.oracle_ext_potential.argtypes = [i64, p, d, p, p]
        lib.oracle_ext_potential.restype = None
        lib.oracle_total_accel.argtypes = [i64, p, d, d, p, p]
        lib.oracle_total_accel.restype = None
        lib.oracle_leapfrog_kdk.argtypes = [i64, p, p, d, d, d, i64, p, p]
        lib.oracle_leapfrog_kdk.restype = None
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def _f64(a, cols):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.ndim != 2 or a.shape[1] != cols:
        raise ValueError("expected [n, %d] array, got %r" % (cols, a.shape))
    return a


def _ptr(a):
    return a.ctypes.data_as(ctypes.c_void_p)


def _potptr(pot):
    return ctypes.cast(ctypes.pointer(pot), ctypes.c_void_p) if pot is not None else None


def pair_accel(posm, G, eps, targets=None):
    """(acc [nt,3], S [nt]): softened all-pairs acceleration and S_i = sum_j |a_ij|."""
    posm = _f64(posm, 4)
    n = posm.shape[0]
    if targets is None:
        nt, tptr = n, None
    else:
        targets = np.ascontiguousarray(targets, dtype=np.int64)
        nt, tptr = targets.shape[0], _ptr(targets)
    acc = np.zeros((nt, 3), dtype=np.float64)
    S = np.zeros(nt, dtype=np.float64)
    _load().oracle_pair_accel(n, _ptr(posm), float(G), float(eps), nt, tptr, _ptr(acc), _ptr(S))
    return acc, S


def pair_potential_energy(posm, G, eps):
    posm = _f64(posm, 4)
    return float(_load().oracle_pair_potential_energy(posm.shape[0], _ptr(posm), float(G), float(eps)))


def ext_accel(posm, G, pot):
    posm = _f64(posm, 4)
    acc = np.zeros((posm.shape[0], 3), dtype=np.float64)
    _load().oracle_ext_accel(posm.shape[0], _ptr(posm), float(G), _potptr(pot), _ptr(acc))
    return acc


def ext_potential(posm, G, pot):
    posm = _f64(posm, 4)
    phi = np.zeros(posm.shape[0], dtype=np.float64)
    _load().oracle_ext_potential(posm.shape[0], _ptr(posm), float(G), _potptr(pot), _ptr(phi))
    return phi


def total_accel(posm, G, eps, pot):
    posm = _f64(posm, 4)
    acc = np.zeros((posm.shape[0], 3), dtype=np.float64)
    _load().oracle_total_accel(posm.shape[0], _ptr(posm), float(G), float(eps), _potptr(pot), _ptr(acc))
    return acc


def leapfrog_kdk(posm, vel, G, eps, dt, nsteps, pot=None):
    """Advance copies of (posm, vel) by nsteps KDK steps; returns (posm, vel, acc_total)."""
    posm = _f64(posm, 4).copy()
    vel = _f64(vel, 3).copy()
    acc = np.zeros((posm.shape[0], 3), dtype=np.float64)
    _load().oracle_leapfrog_kdk(posm.shape[0], _ptr(posm), _ptr(vel), float(G), float(eps),
                                float(dt), int(nsteps), _potptr(pot), _ptr(acc))
    return posm, vel, acc


# ---- O(N) diagnostics: plain definitions -----------------

def kinetic_energy(posm, vel):
    posm, vel = _f64(posm, 4), _f64(vel, 3)
    return float(0.5 * np.sum(posm[:, 3] * np.sum(vel * vel, axis=1)))


def ext_potential_energy(posm, G, pot):
    posm = _f64(posm, 4)
    return float(np.sum(posm[:, 3] * ext_potential(posm, G, pot)))


def total_energy(posm, vel, G, eps, pot=None):
    e = kinetic_energy(posm, vel) + pair_potential_energy(posm, G, eps)
    if pot is not None:
        e += ext_potential_energy(posm, G, pot)
    return e


def linear_momentum(posm, vel):
    posm, vel = _f64(posm, 4), _f64(vel, 3)
    return np.sum(posm[:, 3:4] * vel, axis=0)


def angular_momentum(posm, vel):
    posm, vel = _f64(posm, 4), _f64(vel, 3)
    return np.sum(posm[:, 3:4] * np.cross(posm[:, :3], vel), axis=0)


def centre_of_mass(posm):
    posm = _f64(posm, 4)
    return np.sum(posm[:, 3:4] * posm[:, :3], axis=0) / np.sum(posm[:, 3])
