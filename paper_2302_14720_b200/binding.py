"""Thin ctypes binding of libsw_b200.so -- same names as include/sw.h, argument marshalling only.

PyTorch is used for device memory (the workspace every handle lives in, and zero-copy tensor views
of the library's device buffers), pinned host staging buffers and CUDA streams.  Every step of the
sweep runs in the library's kernels.  There is no CPU fallback: if the shared library is missing,
or no CUDA device is usable, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libsw_b200.so")

SW_OK, SW_EINVAL, SW_ENOMEM, SW_ECUDA, SW_ESTATE = 0, -1, -2, -3, -4


class sw_obs(C.Structure):
    _fields_ = [("energy", C.c_int64), ("magnetisation", C.c_int64), ("n_clusters", C.c_int64),
                ("largest_cluster", C.c_int64), ("sweep", C.c_uint64),
                ("e_per_site", C.c_double), ("abs_m_per_site", C.c_double)]

    def as_tuple(self):
        return (self.energy, self.magnetisation, self.n_clusters, self.largest_cluster)


class sw_mom(C.Structure):
    """Mirror of include/sw.h sw_mom (moments of the per-sweep observables)."""
    _fields_ = [("n", C.c_int64), ("e_mean", C.c_double), ("e2_mean", C.c_double), ("absm_mean", C.c_double),
                ("m2_mean", C.c_double), ("m4_mean", C.c_double), ("specific_heat", C.c_double),
                ("susceptibility", C.c_double), ("binder", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class sw_binstat(C.Structure):
    """Mirror of include/sw.h sw_binstat."""
    _fields_ = [("n_bins", C.c_int64), ("mean", C.c_double), ("err", C.c_double)]


class sw_taustat(C.Structure):
    """Mirror of include/sw.h sw_taustat."""
    _fields_ = [("tau_int", C.c_double), ("window", C.c_int64), ("tmax", C.c_int64), ("c0", C.c_double)]


class SwError(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"sw error {code}: {text}")
        self.code = code


_lib = None

# name -> (restype, argtypes); this table is also what tests/test_abi.py checks against include/sw.h
_VP, _I32, _I64, _U32, _U64, _DBL = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_uint64, C.c_double
PROTOTYPES = {
    "sw_create": (_VP, [_I32, _DBL, _U64]),
    "sw_create_batch": (_VP, [_I32, _I32, C.POINTER(_DBL), C.POINTER(_U64)]),
    "sw_workspace_bytes": (_U64, [_I32, _I32]),
    "sw_create_in": (_VP, [_VP, _U64, _I32, _I32, C.POINTER(_DBL), C.POINTER(_U64)]),
    "sw_destroy": (None, [_VP]),
    "sw_sweep": (C.c_int, [_VP, _I64]),
    "sw_labels": (_VP, [_VP]),
    "sw_observables": (C.c_int, [_VP, C.POINTER(sw_obs)]),
    "sw_spins": (_VP, [_VP]),
    "sw_bonds": (C.c_int, [_VP, C.POINTER(_VP), C.POINTER(_VP)]),
    "sw_set_spins": (C.c_int, [_VP, _VP, C.c_int]),
    "sw_set_cold": (C.c_int, [_VP]),
    "sw_get_spins": (C.c_int, [_VP, _VP]),
    "sw_set_spins_bits": (C.c_int, [_VP, _VP]),
    "sw_get_spins_bits": (C.c_int, [_VP, _VP]),
    "sw_get_labels": (C.c_int, [_VP, _VP]),
    "sw_set_sweep_index": (C.c_int, [_VP, _U64]),
    "sw_sweep_index": (_U64, [_VP]),
    "sw_set_stream": (C.c_int, [_VP, _VP]),
    "sw_series": (_I64, [_VP, C.POINTER(sw_obs), _I64]),
    "sw_set_series_capacity": (C.c_int, [_VP, _I64]),
    "sw_moments": (C.c_int, [_VP, C.POINTER(sw_mom)]),
    "sw_moments_reset": (C.c_int, [_VP]),
    "sw_bins": (C.c_int, [_VP, _I32, C.c_int64, C.POINTER(C.c_double), C.c_int64, C.POINTER(sw_binstat)]),
    "sw_autocorr": (C.c_int, [_VP, _I32, C.c_int64, C.c_double, C.POINTER(C.c_double), C.POINTER(sw_taustat)]),
    "sw_bins_noalloc": (C.c_int, [_VP, _I32, C.c_int64, _VP]),
    "sw_set_stage_timing": (C.c_int, [_VP, C.c_int]),
    "sw_stage_ms": (C.c_int, [_VP, C.POINTER(C.c_float)]),
    "sw_kernel_ms": (C.c_int, [_VP, C.POINTER(C.c_float), _I32]),
    "sw_kernel_name": (C.c_char_p, [_I32]),
    "sw_set_path": (C.c_int, [_VP, C.c_int]),
    "sw_set_tma": (C.c_int, [_VP, C.c_int]),
    "sw_set_cluster": (C.c_int, [_VP, C.c_int]),
    "sw_label_passes": (C.c_int, [_VP, C.POINTER(C.c_int32)]),
    "sw_sweep_ms": (C.c_int64, [_VP, C.POINTER(C.c_float), C.c_int64]),
    "sw_create_potts": (_VP, [C.c_int32, C.c_int32, C.c_double, C.c_uint64]),
    "sw_create_potts_in": (_VP, [_VP, C.c_uint64, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_double), C.POINTER(C.c_uint64)]),
    "sw_q": (C.c_int32, [_VP]),
    "sw_set_eager_labels": (C.c_int, [_VP, C.c_int]),
    "sw_set_graphs": (C.c_int, [_VP, C.c_int]),
    "sw_last_launch_count": (_I64, [_VP]),
    "sw_threshold": (_U32, [_VP, _I32]),
    "sw_L": (_I32, [_VP]),
    "sw_batch": (_I32, [_VP]),
    "sw_test_philox": (C.c_int, [_VP, _VP, _VP, _I64]),
    "sw_test_label": (C.c_int, [_VP, _VP, _VP, _VP]),
    "sw_test_philox_ceiling": (C.c_int, [C.c_int64, C.c_int32, C.POINTER(C.c_float)]),
    "sw_last_error": (C.c_char_p, []),
    "sw_version": (C.c_char_p, []),
}


def lib() -> C.CDLL:
    """Load libsw_b200.so (built by paper_2302_14720_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} is not built; run `python -m paper_2302_14720_b200.build` "
                              "(there is no CPU fallback)")
        l = C.CDLL(_SO)
        for name, (res, args) in PROTOTYPES.items():
            f = getattr(l, name)
            f.restype, f.argtypes = res, args
        _lib = l
    return _lib


def sw_last_error() -> str:
    return lib().sw_last_error().decode()


def _check(rc: int) -> int:
    if rc < 0:
        raise SwError(rc, sw_last_error())
    return rc


def _ptr(h) -> int:
    if not h:
        raise SwError(SW_EINVAL, "null handle")
    return h


# ---- plain functions with the C names ---------------------------------------------------------
def sw_version() -> str:
    return lib().sw_version().decode()

def sw_workspace_bytes(L: int, nb: int = 1) -> int:
    return int(lib().sw_workspace_bytes(L, nb))

def sw_create(L: int, T: float, seed: int):
    h = lib().sw_create(L, float(T), seed)
    if not h:
        raise SwError(SW_EINVAL, sw_last_error())
    return h

def sw_create_potts(L: int, q: int, T: float, seed: int):
    h = lib().sw_create_potts(L, q, float(T), seed)
    if not h:
        raise SwError(SW_EINVAL, sw_last_error())
    return h

def sw_create_potts_in(ws_ptr: int, ws_bytes: int, L: int, q: int, T: Sequence[float], seed: Sequence[int]):
    nb = len(T)
    Ta = (C.c_double * nb)(*[float(t) for t in T]); Sa = (C.c_uint64 * nb)(*[int(s) for s in seed])
    h = lib().sw_create_potts_in(ws_ptr, ws_bytes, L, q, nb, Ta, Sa)
    if not h:
        raise SwError(SW_EINVAL, sw_last_error())
    return h

def sw_q(h) -> int:
    return int(lib().sw_q(_ptr(h)))

def sw_create_batch(L: int, T: Sequence[float], seed: Sequence[int]):
    nb = len(T)
    Ta = (C.c_double * nb)(*[float(t) for t in T]); Sa = (C.c_uint64 * nb)(*[int(s) for s in seed])
    h = lib().sw_create_batch(L, nb, Ta, Sa)
    if not h:
        raise SwError(SW_EINVAL, sw_last_error())
    return h

def sw_create_in(workspace_ptr: int, workspace_bytes: int, L: int, T: Sequence[float], seed: Sequence[int]):
    nb = len(T)
    Ta = (C.c_double * nb)(*[float(t) for t in T]); Sa = (C.c_uint64 * nb)(*[int(s) for s in seed])
    h = lib().sw_create_in(workspace_ptr, workspace_bytes, L, nb, Ta, Sa)
    if not h:
        raise SwError(SW_EINVAL, sw_last_error())
    return h

def sw_destroy(h) -> None:
    lib().sw_destroy(h)

def sw_sweep(h, n: int) -> None:
    _check(lib().sw_sweep(_ptr(h), n))

def sw_labels(h) -> int:
    p = lib().sw_labels(_ptr(h))
    if not p:
        raise SwError(SW_ESTATE, sw_last_error())
    return p

def sw_spins(h) -> int:
    p = lib().sw_spins(_ptr(h))
    if not p:
        raise SwError(SW_EINVAL, sw_last_error())
    return p

def sw_bonds(h):
    e, s = C.c_void_p(), C.c_void_p()
    _check(lib().sw_bonds(_ptr(h), C.byref(e), C.byref(s)))
    return e.value, s.value

def sw_observables(h) -> List[sw_obs]:
    nb = lib().sw_batch(_ptr(h))
    out = (sw_obs * nb)()
    _check(lib().sw_observables(h, out))
    return list(out)

def sw_series(h, cap: Optional[int] = None) -> np.ndarray:
    """History of the last sw_sweep call as an int64 array [sweeps, nb, 4] = (E, M, ncl, maxcl)."""
    nb = lib().sw_batch(_ptr(h))
    kept = _check(lib().sw_series(h, (sw_obs * 1)(), 0))
    n = kept if cap is None else min(kept, cap)
    buf = (sw_obs * max(1, n * nb))()
    _check(lib().sw_series(h, buf, n))
    a = np.zeros((n, nb, 4), dtype=np.int64)
    for k in range(n * nb):
        a[k // nb, k % nb] = buf[k].as_tuple()
    return a

def sw_moments(h) -> List[dict]:
    """Moments of the per-sweep observables since creation / the last reset, one dict per lattice."""
    nb = lib().sw_batch(_ptr(h))
    out = (sw_mom * nb)()
    _check(lib().sw_moments(h, out))
    return [m.as_dict() for m in out]

def sw_moments_reset(h) -> None:
    _check(lib().sw_moments_reset(_ptr(h)))

def sw_bins(h, which: int, bin_len: int, want_means: bool = True):
    """Binning of the last call's series (which: 0 = E/N, 1 = |M|/N): per lattice (n_bins, mean, err[, bin means])."""
    nb = lib().sw_batch(_ptr(h))
    out = (sw_binstat * nb)()
    _check(lib().sw_bins(h, which, bin_len, None, 0, out))           # first the number of bins
    nbins = int(out[0].n_bins)
    means = np.zeros((nb, max(nbins, 1)), dtype=np.float64)
    if want_means and nbins > 0:
        _check(lib().sw_bins(h, which, bin_len, means.ctypes.data_as(C.POINTER(C.c_double)), means.shape[1], out))
    return [{"n_bins": int(o.n_bins), "mean": o.mean, "err": o.err, "bin_means": means[b, :nbins].copy()} for b, o in enumerate(out)]

SW_BINS_NOALLOC_MAX = 65536              # include/sw.h

def sw_bins_noalloc(h, which: int, bin_len: int, out_dev_ptr: int) -> None:
    """sw_bins without any allocation: nb records (int64 n_bins, double mean, double err) into DEVICE memory at
    out_dev_ptr, asynchronously on the handle's stream (argument marshalling only)."""
    _check(lib().sw_bins_noalloc(h, which, bin_len, C.c_void_p(out_dev_ptr)))

def sw_autocorr(h, which: int, tmax: int, c: float = 6.0):
    """Normalised autocorrelation rho(0 .. tmax) of the last call's series and the windowed tau_int, per lattice."""
    nb = lib().sw_batch(_ptr(h))
    out = (sw_taustat * nb)()
    rho = np.zeros((nb, tmax + 1), dtype=np.float64)
    _check(lib().sw_autocorr(h, which, tmax, c, rho.ctypes.data_as(C.POINTER(C.c_double)), out))
    return [{"tau_int": o.tau_int, "window": int(o.window), "tmax": int(o.tmax), "c0": o.c0, "rho": rho[b, :int(o.tmax) + 1].copy()}
            for b, o in enumerate(out)]

def sw_set_graphs(h, on: bool) -> None:
    _check(lib().sw_set_graphs(_ptr(h), 1 if on else 0))

def sw_set_series_capacity(h, sweeps: int) -> None:
    _check(lib().sw_set_series_capacity(_ptr(h), sweeps))

def sw_set_spins(h, ptr: int, is_host: bool) -> None:
    _check(lib().sw_set_spins(_ptr(h), ptr, 1 if is_host else 0))

def sw_set_cold(h) -> None:
    _check(lib().sw_set_cold(_ptr(h)))

def sw_get_spins(h, host_ptr: int) -> None:
    _check(lib().sw_get_spins(_ptr(h), host_ptr))

def sw_set_spins_bits(h, host_ptr: int) -> None:
    _check(lib().sw_set_spins_bits(_ptr(h), host_ptr))

def sw_get_spins_bits(h, host_ptr: int) -> None:
    _check(lib().sw_get_spins_bits(_ptr(h), host_ptr))

def sw_get_labels(h, host_ptr: int) -> None:
    _check(lib().sw_get_labels(_ptr(h), host_ptr))

def sw_set_sweep_index(h, t: int) -> None:
    _check(lib().sw_set_sweep_index(_ptr(h), t))

def sw_sweep_index(h) -> int:
    return int(lib().sw_sweep_index(_ptr(h)))

def sw_set_stream(h, cuda_stream: int) -> None:
    _check(lib().sw_set_stream(_ptr(h), cuda_stream))

def sw_set_stage_timing(h, on: bool) -> None:
    _check(lib().sw_set_stage_timing(_ptr(h), 1 if on else 0))

def sw_stage_ms(h):
    out = (C.c_float * 4)()
    _check(lib().sw_stage_ms(_ptr(h), out))
    return dict(zip(("bond", "label", "flip", "observe"), (float(v) for v in out)))

def sw_kernel_ms(h):
    out = (C.c_float * 32)()
    n = _check(lib().sw_kernel_ms(_ptr(h), out, 32))
    return {lib().sw_kernel_name(i).decode(): float(out[i]) for i in range(n)}

def sw_sweep_ms(h) -> np.ndarray:
    """ms of every timed sweep of the last sw_sweep call (stage timing on), in order."""
    n = _check(lib().sw_sweep_ms(_ptr(h), (C.c_float * 1)(), 0))
    out = (C.c_float * max(1, n))()
    _check(lib().sw_sweep_ms(_ptr(h), out, n))
    return np.array(out[:n], dtype=np.float64)

def sw_set_tma(h, on: bool) -> None:
    _check(lib().sw_set_tma(_ptr(h), 1 if on else 0))

def sw_set_cluster(h, on: bool) -> None:
    _check(lib().sw_set_cluster(_ptr(h), 1 if on else 0))

def sw_set_path(h, path: int) -> None:
    _check(lib().sw_set_path(_ptr(h), path))

def sw_label_passes(h) -> int:
    out = C.c_int32(0)
    _check(lib().sw_label_passes(_ptr(h), C.byref(out)))
    return int(out.value)

def sw_set_eager_labels(h, on: bool) -> None:
    _check(lib().sw_set_eager_labels(_ptr(h), 1 if on else 0))

def sw_last_launch_count(h) -> int:
    return int(lib().sw_last_launch_count(_ptr(h)))

def sw_threshold(h, b: int = 0) -> int:
    return int(lib().sw_threshold(_ptr(h), b))

def sw_test_philox(ctr: np.ndarray, key: np.ndarray) -> np.ndarray:
    ctr = np.ascontiguousarray(ctr, dtype=np.uint32).reshape(-1, 4)
    key = np.ascontiguousarray(key, dtype=np.uint32).reshape(-1, 2)
    out = np.zeros_like(ctr)
    _check(lib().sw_test_philox(ctr.ctypes.data, key.ctypes.data, out.ctypes.data, len(ctr)))
    return out

def sw_test_philox_ceiling(sites: int, reps: int = 20) -> float:
    """ms per launch of the Philox-only kernel for one sweep of `sites` sites (the bond stage's ALU ceiling)."""
    out = C.c_float(0.0)
    _check(lib().sw_test_philox_ceiling(sites, reps, C.byref(out)))
    return float(out.value)

def sw_test_label(h, bondE_words: np.ndarray, bondS_words: np.ndarray) -> np.ndarray:
    L = lib().sw_L(_ptr(h))
    e = np.ascontiguousarray(bondE_words, dtype=np.uint32); s = np.ascontiguousarray(bondS_words, dtype=np.uint32)
    out = np.empty(L * L, dtype=np.int32)
    _check(lib().sw_test_label(h, e.ctypes.data, s.ctypes.data, out.ctypes.data))
    return out


# ---- convenience wrapper: torch owns the memory and the stream ------------------------------------
class SwendsenWang:
    """One handle (nb >= 1 lattices) whose device buffers live in a torch uint8 workspace tensor."""

    def __init__(self, L: int, T, seed, device: str = "cuda:0", path: int = 0, q: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2302_14720_b200 needs a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.T = [float(T)] if np.isscalar(T) else [float(t) for t in T]
        self.seed = [int(seed)] if np.isscalar(seed) else [int(s) for s in seed]
        assert len(self.T) == len(self.seed)
        self.L, self.nb, self.N = int(L), len(self.T), int(L) * int(L)
        self.words = (self.N + 31) // 32
        self.device = torch.device(device)
        nbytes = sw_workspace_bytes(self.L, self.nb)
        if nbytes == 0:
            raise SwError(SW_EINVAL, f"invalid lattice side {L} / batch {self.nb}")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_off = (-base) % 256
            self.q = int(q)                            # 0: Ising; >= 2: q-state Potts (colours 0 .. q-1)
            if self.q:
                self.h = sw_create_potts_in(base + self._ws_off, nbytes, self.L, self.q, self.T, self.seed)
            else:
                self.h = sw_create_in(base + self._ws_off, nbytes, self.L, self.T, self.seed)
            sw_set_stream(self.h, torch.cuda.current_stream(self.device).cuda_stream)
        if path:
            sw_set_path(self.h, path)

    # -- lifetime
    def close(self):
        if getattr(self, "h", None):
            sw_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- zero-copy tensor views of the borrowed device pointers (they point into self.workspace)
    def _view(self, ptr: int, nbytes: int):
        off = ptr - self.workspace.data_ptr()
        assert 0 <= off and off + nbytes <= self.workspace.numel(), "pointer outside the workspace"
        return self.workspace[off:off + nbytes]

    def spins(self):
        return self._view(sw_spins(self.h), self.nb * self.N).view(self.torch.int8).view(self.nb, self.L, self.L)

    def labels(self):
        """Flat int32 labels of the last sweep: a zero-copy tensor over the library's own label array (allocated by the
        library on first use, outside the torch workspace; valid until the next sweep / sw_destroy)."""
        ptr = sw_labels(self.h)

        class _Raw:                                   # (__cuda_array_interface__: pointer + shape, no copy)
            __cuda_array_interface__ = {"shape": (self.nb, self.L, self.L), "typestr": "<i4", "data": (ptr, False),
                                        "version": 2, "strides": None}
        with self.torch.cuda.device(self.device):
            return self.torch.as_tensor(_Raw(), device=self.device)

    def bonds(self):
        e, s = sw_bonds(self.h)
        n = self.nb * self.words * 4
        return (self._view(e, n).view(self.torch.int32).view(self.nb, self.words),
                self._view(s, n).view(self.torch.int32).view(self.nb, self.words))

    # -- the hot path
    def use_current_stream(self):
        sw_set_stream(self.h, self.torch.cuda.current_stream(self.device).cuda_stream)

    def sweep(self, n: int = 1):
        sw_sweep(self.h, n)

    def observables(self):
        return sw_observables(self.h)

    def series(self, cap=None):
        return sw_series(self.h, cap)

    def set_graphs(self, on: bool):
        sw_set_graphs(self.h, on)

    def moments(self):
        return sw_moments(self.h)

    def moments_reset(self):
        sw_moments_reset(self.h)

    def bins(self, which: int, bin_len: int):
        return sw_bins(self.h, which, bin_len)

    def bins_noalloc(self, which: int, bin_len: int, out):
        """`out`: a device tensor of nb * 3 float64 (= nb records of 24 bytes: n_bins as int64 bits, mean, err)."""
        assert out.is_cuda and out.is_contiguous() and out.element_size() * out.numel() >= 24 * self.nb
        sw_bins_noalloc(self.h, which, bin_len, out.data_ptr())

    def autocorr(self, which: int, tmax: int, c: float = 6.0):
        return sw_autocorr(self.h, which, tmax, c)

    # -- state
    def set_spins(self, spins):
        """spins: torch tensor on the device or on the host, or a numpy array; nb*N int8 of +-1."""
        torch = self.torch
        if isinstance(spins, np.ndarray):
            spins = torch.from_numpy(np.ascontiguousarray(spins, dtype=np.int8))
        spins = spins.contiguous().view(-1)
        assert spins.dtype == torch.int8 and spins.numel() == self.nb * self.N
        sw_set_spins(self.h, spins.data_ptr(), not spins.is_cuda)

    def set_cold(self):
        sw_set_cold(self.h)

    def set_sweep_index(self, t: int):
        sw_set_sweep_index(self.h, t)

    @property
    def sweep_index(self) -> int:
        return sw_sweep_index(self.h)

    def set_stage_timing(self, on: bool):
        sw_set_stage_timing(self.h, on)

    def stage_ms(self):
        return sw_stage_ms(self.h)

    def kernel_ms(self):
        return sw_kernel_ms(self.h)

    def sweep_ms(self):
        return sw_sweep_ms(self.h)

    def threshold(self, b: int = 0) -> int:
        return sw_threshold(self.h, b)

    def label_passes(self) -> int:
        """Path 11: passes of the last label-equivalence iteration."""
        return sw_label_passes(self.h)

    def launch_count(self) -> int:
        return sw_last_launch_count(self.h)

    # -- host copies (numpy) for the parity tests
    def spins_host(self) -> np.ndarray:
        return self.spins().cpu().numpy().reshape(self.nb, self.N)

    def labels_host(self) -> np.ndarray:
        return self.labels().cpu().numpy().reshape(self.nb, self.N)

    def bonds_host(self):
        e, s = self.bonds()
        return (e.cpu().numpy().view(np.uint32).reshape(self.nb, self.words),
                s.cpu().numpy().view(np.uint32).reshape(self.nb, self.words))
