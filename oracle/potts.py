"""ORACLE (test infrastructure, not product code): q-state Potts Swendsen-Wang, SURVEY.md 8(f) NEXT-3.

PAPER.md:33 ("can be generalized to other discrete spin systems") and PAPER.md:166 name the generalisation but give
no formulas; the readings (textbook Potts SW) are stated in the header of the Potts part of
``sw_oracle.c``, where the arithmetic lives.  This module only marshals numpy arrays.  Bond formation and labelling
are the Ising oracle's own functions (their rule is "equal values and word < thr").  Shares nothing with the CUDA
path.  Pins: tests/test_oracle_potts.py.
"""
from __future__ import annotations

import ctypes
from typing import Optional

import numpy as np

from . import _p, lib as _base_lib, bonds, labels  # noqa: F401  (bonds / labels re-exported)

_ready = False


def lib() -> ctypes.CDLL:
    global _ready
    L = _base_lib()
    if not _ready:
        c = ctypes
        i8p, u8p, i32p, i64p = (c.POINTER(c.c_int8), c.POINTER(c.c_uint8), c.POINTER(c.c_int32), c.POINTER(c.c_int64))
        L.orc_potts_threshold.argtypes = [c.c_double]
        L.orc_potts_threshold.restype = c.c_uint32
        L.orc_potts_colour.argtypes = [c.c_uint64, c.c_uint64, c.c_uint32, c.c_int64, c.c_int32]
        L.orc_potts_colour.restype = c.c_int
        L.orc_potts_init_random.argtypes = [c.c_int32, c.c_int32, c.c_uint64, i8p]
        L.orc_potts_init_random.restype = None
        L.orc_potts_assign.argtypes = [c.c_int32, c.c_int32, c.c_uint64, c.c_uint64, i32p, i8p]
        L.orc_potts_assign.restype = None
        L.orc_potts_observables.argtypes = [c.c_int32, c.c_int32, i8p, i32p, i64p, i64p]
        L.orc_potts_observables.restype = c.c_int
        L.orc_potts_sweep.argtypes = [c.c_int32, c.c_int32, c.c_uint32, c.c_uint64, c.c_uint64,
                                      i8p, u8p, u8p, i32p, i64p]
        L.orc_potts_sweep.restype = c.c_int
        L.orc_potts_run.argtypes = [c.c_int32, c.c_int32, c.c_double, c.c_uint64, c.c_uint64, c.c_int64, i8p, i64p]
        L.orc_potts_run.restype = c.c_int
        _ready = True
    return L


def threshold(T: float) -> int:
    return int(lib().orc_potts_threshold(float(T)))


def colour(seed: int, t: int, tag: int, idx: int, q: int) -> int:
    return int(lib().orc_potts_colour(seed, t, tag, idx, q))


def init_random(L: int, q: int, seed: int) -> np.ndarray:
    s = np.empty(L * L, dtype=np.int8)
    lib().orc_potts_init_random(L, q, seed, _p(s, ctypes.c_int8))
    return s


def observables(L: int, q: int, colours: np.ndarray, label: Optional[np.ndarray] = None):
    """((E, M, ncl, maxcl), counts[q])"""
    s = np.ascontiguousarray(colours, dtype=np.int8)
    out = np.zeros(4, dtype=np.int64)
    cnt = np.zeros(q, dtype=np.int64)
    lp = None
    if label is not None:
        label = np.ascontiguousarray(label, dtype=np.int32)
        lp = _p(label, ctypes.c_int32)
    rc = lib().orc_potts_observables(L, q, _p(s, ctypes.c_int8), lp, _p(out, ctypes.c_int64), _p(cnt, ctypes.c_int64))
    if rc != 0:
        raise RuntimeError("orc_potts_observables: %d" % rc)
    return tuple(int(v) for v in out), cnt


def sweep(L: int, q: int, T: float, seed: int, t: int, colours: np.ndarray):
    """One sweep with index t from `colours` (not modified): (new colours, bondE, bondS, label, (E, M, ncl, maxcl))."""
    s = np.array(colours, dtype=np.int8, copy=True).reshape(-1)
    N = L * L
    bE = np.empty(N, dtype=np.uint8)
    bS = np.empty(N, dtype=np.uint8)
    lab = np.empty(N, dtype=np.int32)
    obs = np.zeros(4, dtype=np.int64)
    rc = lib().orc_potts_sweep(L, q, threshold(T), seed, t, _p(s, ctypes.c_int8), _p(bE, ctypes.c_uint8),
                               _p(bS, ctypes.c_uint8), _p(lab, ctypes.c_int32), _p(obs, ctypes.c_int64))
    if rc != 0:
        raise MemoryError("orc_potts_sweep")
    return s, bE, bS, lab, tuple(int(v) for v in obs)


def run(L: int, q: int, T: float, seed: int, n: int, colours: Optional[np.ndarray] = None, t0: int = 0):
    """n sweeps; returns (final colours, series (n, 4) int64 of (E, M, ncl, maxcl))."""
    s = init_random(L, q, seed) if colours is None else np.array(colours, dtype=np.int8, copy=True).reshape(-1)
    ser = np.zeros((n, 4), dtype=np.int64)
    rc = lib().orc_potts_run(L, q, float(T), seed, t0, n, _p(s, ctypes.c_int8), _p(ser, ctypes.c_int64))
    if rc != 0:
        raise MemoryError("orc_potts_run")
    return s, ser
