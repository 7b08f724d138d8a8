"""ORACLE (test infrastructure, not product code): ctypes access to oracle/phi4_oracle.c, the serial statement of the
Wolff-type embedded cluster update for the O(4) phi^4 theory in four dimensions (section 3, Eq. 2-3;
SURVEY.md 8(f) NEXT-4).  See the header of phi4_oracle.c for the readings and the pins.  Shares nothing with the CUDA path.
"""
from __future__ import annotations

import ctypes
from typing import Optional, Tuple

import numpy as np

from . import lib as _lib

_ready = False


def lib() -> ctypes.CDLL:
    global _ready
    L = _lib()
    if not _ready:
        c = ctypes
        dp, u8p, i32p, i64p = c.POINTER(c.c_double), c.POINTER(c.c_uint8), c.POINTER(c.c_int32), c.POINTER(c.c_int64)
        L.orc4_init.argtypes = [c.c_int32, c.c_uint64, dp]; L.orc4_init.restype = None
        L.orc4_direction.argtypes = [c.c_uint64, c.c_uint64, dp]; L.orc4_direction.restype = c.c_int
        L.orc4_threshold.argtypes = [c.c_double, c.c_double, c.c_double]; L.orc4_threshold.restype = c.c_uint32
        L.orc4_bonds.argtypes = [c.c_int32, c.c_double, c.c_uint64, c.c_uint64, dp, dp, u8p]; L.orc4_bonds.restype = None
        L.orc4_labels.argtypes = [c.c_int32, u8p, i32p]; L.orc4_labels.restype = c.c_int
        L.orc4_selected.argtypes = [c.c_uint64, c.c_uint64, c.c_int64]; L.orc4_selected.restype = c.c_int
        L.orc4_reflect.argtypes = [c.c_int32, c.c_uint64, c.c_uint64, i32p, dp, dp]; L.orc4_reflect.restype = None
        L.orc4_observables.argtypes = [c.c_int32, dp, i32p, u8p, dp, i64p]; L.orc4_observables.restype = c.c_int
        L.orc4_sweep.argtypes = [c.c_int32, c.c_double, c.c_uint64, c.c_uint64, dp, dp, u8p, i32p, dp, i64p]
        L.orc4_sweep.restype = c.c_int
        L.orc4_run.argtypes = [c.c_int32, c.c_double, c.c_uint64, c.c_uint64, c.c_int64, dp, dp, i64p]
        L.orc4_run.restype = c.c_int
        _ready = True
    return L


def _d(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def init(L: int, seed: int) -> np.ndarray:
    phi = np.zeros((L ** 4, 4), dtype=np.float64)
    lib().orc4_init(L, seed, _d(phi))
    return phi


def direction(seed: int, t: int) -> Tuple[np.ndarray, int]:
    r = np.zeros(4, dtype=np.float64)
    n = lib().orc4_direction(seed, t, _d(r))
    return r, int(n)


def threshold(kappa: float, sx: float, sy: float) -> int:
    return int(lib().orc4_threshold(float(kappa), float(sx), float(sy)))


def bonds(L: int, kappa: float, seed: int, t: int, phi: np.ndarray, r: np.ndarray) -> np.ndarray:
    phi = np.ascontiguousarray(phi, dtype=np.float64); r = np.ascontiguousarray(r, dtype=np.float64)
    b = np.zeros(L ** 4, dtype=np.uint8)
    lib().orc4_bonds(L, float(kappa), seed, t, _d(phi), _d(r), b.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)))
    return b


def labels(L: int, bonds_: np.ndarray) -> np.ndarray:
    b = np.ascontiguousarray(bonds_, dtype=np.uint8)
    lab = np.zeros(L ** 4, dtype=np.int32)
    if lib().orc4_labels(L, b.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), lab.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))):
        raise MemoryError("orc4_labels")
    return lab


def selected(seed: int, t: int, label: int) -> int:
    return int(lib().orc4_selected(seed, t, int(label)))


def reflect(L: int, seed: int, t: int, label: np.ndarray, r: np.ndarray, phi: np.ndarray) -> np.ndarray:
    out = np.array(phi, dtype=np.float64, copy=True)
    lab = np.ascontiguousarray(label, dtype=np.int32); r = np.ascontiguousarray(r, dtype=np.float64)
    lib().orc4_reflect(L, seed, t, lab.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _d(r), _d(out))
    return out


def observables(L: int, phi: np.ndarray, label: Optional[np.ndarray] = None, bonds_: Optional[np.ndarray] = None):
    """((link, M0, M1, M2, M3), (clusters, largest cluster, bonds))."""
    phi = np.ascontiguousarray(phi, dtype=np.float64)
    d = np.zeros(5, dtype=np.float64); i3 = np.zeros(3, dtype=np.int64)
    lp = None if label is None else np.ascontiguousarray(label, dtype=np.int32).ctypes.data_as(ctypes.POINTER(ctypes.c_int32))
    bp = None if bonds_ is None else np.ascontiguousarray(bonds_, dtype=np.uint8).ctypes.data_as(ctypes.POINTER(ctypes.c_uint8))
    if lib().orc4_observables(L, _d(phi), lp, bp, _d(d), i3.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))):
        raise MemoryError("orc4_observables")
    return tuple(float(v) for v in d), tuple(int(v) for v in i3)


def sweep(L: int, kappa: float, seed: int, t: int, phi: np.ndarray):
    """One update with sweep index t: (new phi, r, bonds, labels, (link, M0..M3), (clusters, largest, bonds))."""
    out = np.array(phi, dtype=np.float64, copy=True)
    V = L ** 4
    r = np.zeros(4); b = np.zeros(V, dtype=np.uint8); lab = np.zeros(V, dtype=np.int32)
    d = np.zeros(5); i3 = np.zeros(3, dtype=np.int64)
    rc = lib().orc4_sweep(L, float(kappa), seed, t, _d(out), _d(r), b.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)),
                          lab.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)), _d(d), i3.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)))
    if rc:
        raise MemoryError("orc4_sweep")
    return out, r, b, lab, tuple(float(v) for v in d), tuple(int(v) for v in i3)


def run(L: int, kappa: float, seed: int, n: int, phi: Optional[np.ndarray] = None, t0: int = 0):
    """n updates t0 .. t0+n-1 from `phi` (default: the start of `seed`): (final phi, series (n, 5), iseries (n, 3))."""
    out = init(L, seed) if phi is None else np.array(phi, dtype=np.float64, copy=True)
    ser = np.zeros((n, 5)); iser = np.zeros((n, 3), dtype=np.int64)
    if lib().orc4_run(L, float(kappa), seed, t0, n, _d(out), _d(ser), iser.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))):
        raise MemoryError("orc4_run")
    return out, ser, iser
