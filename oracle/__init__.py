"""CPU oracle for the Lomb-Scargle hot path — TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import
this package.  It never imports the CUDA package (paper_2409_08090_b200) and shares no code with it.
The arithmetic lives in ls_oracle.c (plain C, fp64, OpenMP over frequencies); this file is the
ctypes marshalling around it.  See ls_oracle.c for the passage each function follows
(Eq. 1, PAPER.md:75 phase winding, BASELINE.json north_star for the assembly).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from .build import build as _build

__all__ = ["direct", "chi2", "winding", "stats", "assemble", "num_threads"]

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int64)
        lib.ls_oracle_direct.argtypes = [C.c_int64, dp, dp, dp, C.c_double, C.c_double, C.c_int64, ip, C.c_int, dp, dp, dp]
        lib.ls_oracle_chi2.argtypes = [C.c_int64, dp, dp, dp, C.c_double, C.c_double, C.c_int64, ip, dp]
        lib.ls_oracle_winding.argtypes = [C.c_int64, dp, dp, dp, C.c_double, C.c_double, C.c_int64, C.c_int64, C.c_int, dp]
        lib.ls_oracle_stats.argtypes = [C.c_int64, dp, dp, dp]
        lib.ls_oracle_assemble.argtypes = [C.c_int64, dp, C.c_double, dp, dp]
        for f in (lib.ls_oracle_direct, lib.ls_oracle_chi2, lib.ls_oracle_winding, lib.ls_oracle_stats,
                  lib.ls_oracle_assemble, lib.ls_oracle_num_threads):
            f.restype = C.c_int
        _lib = lib
    return _lib


def _d(a):
    """Promote to contiguous float64 (exact for float32 inputs)."""
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _series(t, y, dy):
    t, y, dy = _d(t), _d(y), _d(dy)
    if t.ndim != 1 or y.shape != t.shape or dy.shape != t.shape:
        raise ValueError("oracle takes one series: t, y, dy of equal 1-D shape")
    return t, y, dy


def _kidx(Nf, k):
    if k is None:
        return int(Nf), None, None
    k = np.ascontiguousarray(k, dtype=np.int64)
    return int(k.size), k, k.ctypes.data_as(C.POINTER(C.c_int64))


def num_threads() -> int:
    return int(_load().ls_oracle_num_threads())


def direct(t, y, dy, f0, df, Nf, k=None, variant="strict", return_sums=False):
    """P at f0 + k*df for k in `k` (default 0..Nf-1).  With return_sums: (P, sums[K,6], aux[K,2]),
    sums = (Sh, Ch, S, C, S2, C2), aux = (tan 2 omega tau, tau-free P)."""
    t, y, dy = _series(t, y, dy)
    K, keep, kp = _kidx(Nf, k)
    P = np.empty(K)
    sums = np.empty((K, 6)) if return_sums else None
    aux = np.empty((K, 2)) if return_sums else None
    rc = _load().ls_oracle_direct(t.size, _p(t), _p(y), _p(dy), float(f0), float(df), K, kp,
                                  {"strict": 0, "double-angle": 1}[variant], _p(P),
                                  _p(sums) if return_sums else None, _p(aux) if return_sums else None)
    if rc:
        raise RuntimeError(f"ls_oracle_direct failed: {rc}")
    return (P, sums, aux) if return_sums else P


def chi2(t, y, dy, f0, df, Nf, k=None):
    """1 - chi2_min/chi2_0 of the 3-parameter weighted least-squares fit (the definition)."""
    t, y, dy = _series(t, y, dy)
    K, keep, kp = _kidx(Nf, k)
    P = np.empty(K)
    rc = _load().ls_oracle_chi2(t.size, _p(t), _p(y), _p(dy), float(f0), float(df), K, kp, _p(P))
    if rc:
        raise RuntimeError(f"ls_oracle_chi2 failed: {rc}")
    return P


def winding(t, y, dy, f0, df, k0, K, reseed=64):
    """Phase-winding evaluation of k = k0..k0+K-1."""
    t, y, dy = _series(t, y, dy)
    P = np.empty(int(K))
    rc = _load().ls_oracle_winding(t.size, _p(t), _p(y), _p(dy), float(f0), float(df), int(k0), int(K), int(reseed), _p(P))
    if rc:
        raise RuntimeError(f"ls_oracle_winding failed: {rc}")
    return P


def stats(y, dy):
    """(W = sum dy^-2, weighted mean, YY = sum w (y - mean)^2)."""
    y, dy = _d(y), _d(dy)
    out = np.empty(3)
    rc = _load().ls_oracle_stats(y.size, _p(y), _p(dy), _p(out))
    if rc:
        raise RuntimeError(f"ls_oracle_stats failed: {rc}")
    return tuple(out)


def assemble(sums, YY):
    """Assembly (O6) alone from sums[K,6]: returns (P, aux[K,2])."""
    sums = _d(sums).reshape(-1, 6)
    P, aux = np.empty(sums.shape[0]), np.empty((sums.shape[0], 2))
    _load().ls_oracle_assemble(sums.shape[0], _p(sums), float(YY), _p(P), _p(aux))
    return P, aux
