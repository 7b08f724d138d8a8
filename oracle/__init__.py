"""Serial CPU Swendsen-Wang oracle -- TEST INFRASTRUCTURE, NOT PRODUCT.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2302_14720_b200`` (the CUDA path) and neither imports the other.

The arithmetic lives in ``sw_oracle.c`` (plain serial C99, one site at a time,
following PAPER.md:33-63 under the readings of SURVEY.md section 8(c)); this
module only compiles it with gcc, loads it with ctypes and marshals numpy
arrays.  Parity pins: see the header of ``sw_oracle.c`` and DESIGN.md.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sw_oracle.c")
_SO = os.path.join(_HERE, "liboracle_sw.so")

TAG_INIT, TAG_BOND, TAG_FLIP = 0, 1, 2


_SRC4 = os.path.join(os.path.dirname(os.path.abspath(__file__)), "phi4_oracle.c")


def build(force: bool = False) -> str:
    """Compile sw_oracle.c + phi4_oracle.c -> liboracle_sw.so with gcc -O2 (no tuning flags; -std=c99 keeps
    floating-point contraction off, stated explicitly: no fused multiply-add anywhere)."""
    stale = (not os.path.exists(_SO)) or os.path.getmtime(_SO) < max(os.path.getmtime(_SRC), os.path.getmtime(_SRC4))
    if force or stale:
        tmp = _SO + ".tmp%d" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-ffp-contract=off", "-fPIC", "-shared", "-o", tmp, _SRC, _SRC4, "-lm"])
        os.replace(tmp, _SO)
    return _SO


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        c = ctypes
        u32p, i8p = c.POINTER(c.c_uint32), c.POINTER(c.c_int8)
        u8p, i32p, i64p = c.POINTER(c.c_uint8), c.POINTER(c.c_int32), c.POINTER(c.c_int64)
        _lib.orc_philox4x32_10.argtypes = [u32p, u32p, u32p]
        _lib.orc_philox4x32_10.restype = None
        _lib.orc_bit.argtypes = [c.c_uint64, c.c_uint64, c.c_uint32, c.c_int64]
        _lib.orc_bit.restype = c.c_int
        _lib.orc_threshold.argtypes = [c.c_double]
        _lib.orc_threshold.restype = c.c_uint32
        _lib.orc_init_random.argtypes = [c.c_int32, c.c_uint64, i8p]
        _lib.orc_init_random.restype = None
        _lib.orc_init_cold.argtypes = [c.c_int32, i8p]
        _lib.orc_init_cold.restype = None
        _lib.orc_bonds.argtypes = [c.c_int32, c.c_uint32, c.c_uint64, c.c_uint64, i8p, u8p, u8p]
        _lib.orc_bonds.restype = None
        _lib.orc_labels.argtypes = [c.c_int32, u8p, u8p, i32p]
        _lib.orc_labels.restype = c.c_int
        _lib.orc_assign.argtypes = [c.c_int32, c.c_uint64, c.c_uint64, i32p, i8p]
        _lib.orc_assign.restype = None
        _lib.orc_observables.argtypes = [c.c_int32, i8p, i32p, i64p]
        _lib.orc_observables.restype = c.c_int
        _lib.orc_sweep.argtypes = [c.c_int32, c.c_uint32, c.c_uint64, c.c_uint64,
                                   i8p, u8p, u8p, i32p, i64p]
        _lib.orc_sweep.restype = c.c_int
        _lib.orc_run.argtypes = [c.c_int32, c.c_double, c.c_uint64, c.c_uint64, c.c_int64,
                                 i8p, i64p]
        _lib.orc_run.restype = c.c_int
    return _lib


def _p(a: np.ndarray, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().orc_philox4x32_10(_p(c, ctypes.c_uint32), _p(k, ctypes.c_uint32), _p(out, ctypes.c_uint32))
    return out


def bit(seed: int, t: int, tag: int, idx: int) -> int:
    return int(lib().orc_bit(seed, t, tag, idx))


def threshold(T: float) -> int:
    return int(lib().orc_threshold(float(T)))


def init_random(L: int, seed: int) -> np.ndarray:
    s = np.empty(L * L, dtype=np.int8)
    lib().orc_init_random(L, seed, _p(s, ctypes.c_int8))
    return s


def init_cold(L: int) -> np.ndarray:
    s = np.empty(L * L, dtype=np.int8)
    lib().orc_init_cold(L, _p(s, ctypes.c_int8))
    return s


def bonds(L: int, thr: int, seed: int, t: int, spins: np.ndarray) -> Tuple[np.ndarray, np.ndarray]:
    spins = np.ascontiguousarray(spins, dtype=np.int8)
    bE = np.empty(L * L, dtype=np.uint8)
    bS = np.empty(L * L, dtype=np.uint8)
    lib().orc_bonds(L, thr, seed, t, _p(spins, ctypes.c_int8), _p(bE, ctypes.c_uint8), _p(bS, ctypes.c_uint8))
    return bE, bS


def labels(L: int, bondE: np.ndarray, bondS: np.ndarray) -> np.ndarray:
    bE = np.ascontiguousarray(bondE, dtype=np.uint8)
    bS = np.ascontiguousarray(bondS, dtype=np.uint8)
    lab = np.empty(L * L, dtype=np.int32)
    rc = lib().orc_labels(L, _p(bE, ctypes.c_uint8), _p(bS, ctypes.c_uint8), _p(lab, ctypes.c_int32))
    if rc != 0:
        raise MemoryError("orc_labels")
    return lab


def assign(L: int, seed: int, t: int, label: np.ndarray) -> np.ndarray:
    label = np.ascontiguousarray(label, dtype=np.int32)
    s = np.empty(L * L, dtype=np.int8)
    lib().orc_assign(L, seed, t, _p(label, ctypes.c_int32), _p(s, ctypes.c_int8))
    return s


def observables(L: int, spins: np.ndarray, label: Optional[np.ndarray] = None) -> Tuple[int, int, int, int]:
    spins = np.ascontiguousarray(spins, dtype=np.int8)
    out = np.zeros(4, dtype=np.int64)
    lp = None
    if label is not None:
        label = np.ascontiguousarray(label, dtype=np.int32)
        lp = _p(label, ctypes.c_int32)
    rc = lib().orc_observables(L, _p(spins, ctypes.c_int8), lp, _p(out, ctypes.c_int64))
    if rc != 0:
        raise MemoryError("orc_observables")
    return tuple(int(v) for v in out)


def sweep(L: int, T: float, seed: int, t: int, spins: np.ndarray):
    """One sweep with index t from `spins` (not modified).

    Returns (new_spins, bondE, bondS, label, (E, M, ncl, maxcl)); bond arrays
    hold one byte (0/1) per site.
    """
    s = np.array(spins, dtype=np.int8, copy=True).reshape(-1)
    N = L * L
    bE = np.empty(N, dtype=np.uint8)
    bS = np.empty(N, dtype=np.uint8)
    lab = np.empty(N, dtype=np.int32)
    obs = np.zeros(4, dtype=np.int64)
    rc = lib().orc_sweep(L, threshold(T), seed, t, _p(s, ctypes.c_int8), _p(bE, ctypes.c_uint8),
                         _p(bS, ctypes.c_uint8), _p(lab, ctypes.c_int32), _p(obs, ctypes.c_int64))
    if rc != 0:
        raise MemoryError("orc_sweep")
    return s, bE, bS, lab, tuple(int(v) for v in obs)


def run(L: int, T: float, seed: int, n: int, spins: Optional[np.ndarray] = None, t0: int = 0,
        series: bool = True):
    """n sweeps t0..t0+n-1.  Start: `spins` if given, else the random start of `seed`.

    Returns (final_spins, series) with series an (n, 4) int64 array of
    (E, M, ncl, maxcl) after each sweep, or None.
    """
    s = init_random(L, seed) if spins is None else np.array(spins, dtype=np.int8, copy=True).reshape(-1)
    ser = np.zeros((n, 4), dtype=np.int64) if series else None
    rc = lib().orc_run(L, float(T), seed, t0, n, _p(s, ctypes.c_int8),
                       _p(ser, ctypes.c_int64) if series else None)
    if rc != 0:
        raise MemoryError("orc_run")
    return s, ser
