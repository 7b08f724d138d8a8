"""ctypes binding of include/phi4.h (the Wolff-type embedded cluster update for O(4) phi^4 in four dimensions): argument
marshalling only -- every step of the update runs in the kernels of csrc/phi4_api.cu.  Same library as the Ising path
(libsw_b200.so); no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
from typing import List

import numpy as np

from . import binding as _b

_VP, _I32, _I64, _U64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64

PHI4_OK, PHI4_EINVAL, PHI4_ENOMEM, PHI4_ECUDA, PHI4_ESTATE = 0, -1, -2, -3, -4
PHI4_MAX_L = 128


class phi4_obs(C.Structure):
    """Mirror of include/phi4.h phi4_obs."""
    _fields_ = [("link", C.c_double), ("m", C.c_double * 4), ("n_clusters", C.c_int64), ("largest_cluster", C.c_int64),
                ("n_bonds", C.c_int64), ("sweep", C.c_uint64), ("link_per_link", C.c_double), ("abs_m_per_site", C.c_double)]

    def ints(self):
        return (int(self.n_clusters), int(self.largest_cluster), int(self.n_bonds))

    def doubles(self):
        return (self.link, self.m[0], self.m[1], self.m[2], self.m[3])


PROTOTYPES = {
    "phi4_last_error": (C.c_char_p, []),
    "phi4_create": (_VP, [_I32, C.c_double, _U64]),
    "phi4_destroy": (None, [_VP]),
    "phi4_sweep": (C.c_int, [_VP, _I64]),
    "phi4_field": (_VP, [_VP]),
    "phi4_labels": (_VP, [_VP]),
    "phi4_bonds": (_VP, [_VP]),
    "phi4_direction": (C.c_int, [_VP, C.POINTER(C.c_double)]),
    "phi4_observables": (C.c_int, [_VP, C.POINTER(phi4_obs)]),
    "phi4_series": (_I64, [_VP, C.POINTER(phi4_obs), _I64]),
    "phi4_set_field": (C.c_int, [_VP, _VP, C.c_int]),
    "phi4_get_field": (C.c_int, [_VP, _VP]),
    "phi4_get_labels": (C.c_int, [_VP, _VP]),
    "phi4_get_bonds": (C.c_int, [_VP, _VP]),
    "phi4_set_sweep_index": (C.c_int, [_VP, _U64]),
    "phi4_sweep_index": (_U64, [_VP]),
    "phi4_set_stream": (C.c_int, [_VP, _VP]),
    "phi4_set_graphs": (C.c_int, [_VP, C.c_int]),
    "phi4_L": (_I32, [_VP]),
    "phi4_last_launch_count": (_I64, [_VP]),
}

_ready = False


class Phi4Error(RuntimeError):
    def __init__(self, code: int, text: str):
        super().__init__(f"phi4 error {code}: {text}")
        self.code = code


def lib() -> C.CDLL:
    global _ready
    l = _b.lib()
    if not _ready:
        for name, (res, args) in PROTOTYPES.items():
            f = getattr(l, name)
            f.restype, f.argtypes = res, args
        _ready = True
    return l


def _check(rc: int) -> int:
    if rc < 0:
        raise Phi4Error(rc, lib().phi4_last_error().decode())
    return rc


class Phi4:
    """One L^4 lattice of four-component fields on the current CUDA device."""

    def __init__(self, L: int, kappa: float, seed: int, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2302_14720_b200 needs a CUDA device; there is no CPU fallback")
        self.torch, self.device = torch, torch.device(device)
        self.L, self.V, self.kappa, self.seed = int(L), int(L) ** 4, float(kappa), int(seed)
        with torch.cuda.device(self.device):
            self.h = lib().phi4_create(self.L, self.kappa, self.seed)
            if not self.h:
                raise Phi4Error(PHI4_EINVAL, lib().phi4_last_error().decode())
            _check(lib().phi4_set_stream(self.h, torch.cuda.current_stream(self.device).cuda_stream))

    def close(self):
        if getattr(self, "h", None):
            lib().phi4_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def sweep(self, n: int = 1):
        _check(lib().phi4_sweep(self.h, n))

    def set_graphs(self, on: bool):
        _check(lib().phi4_set_graphs(self.h, 1 if on else 0))

    @property
    def sweep_index(self) -> int:
        return int(lib().phi4_sweep_index(self.h))

    def set_sweep_index(self, t: int):
        _check(lib().phi4_set_sweep_index(self.h, t))

    def field_host(self) -> np.ndarray:
        out = np.empty((self.V, 4), dtype=np.float64)
        _check(lib().phi4_get_field(self.h, out.ctypes.data))
        return out

    def set_field(self, phi: np.ndarray):
        a = np.ascontiguousarray(phi, dtype=np.float64).reshape(self.V, 4)
        _check(lib().phi4_set_field(self.h, a.ctypes.data, 1))

    def labels_host(self) -> np.ndarray:
        out = np.empty(self.V, dtype=np.int32)
        _check(lib().phi4_get_labels(self.h, out.ctypes.data))
        return out

    def bonds_host(self) -> np.ndarray:
        out = np.empty(self.V, dtype=np.uint8)
        _check(lib().phi4_get_bonds(self.h, out.ctypes.data))
        return out

    def direction(self) -> np.ndarray:
        r = (C.c_double * 4)()
        _check(lib().phi4_direction(self.h, r))
        return np.array(list(r), dtype=np.float64)

    def observables(self) -> phi4_obs:
        o = phi4_obs()
        _check(lib().phi4_observables(self.h, C.byref(o)))
        return o

    def series(self) -> List[phi4_obs]:
        cap = 4096
        buf = (phi4_obs * cap)()
        n = _check(lib().phi4_series(self.h, buf, cap))
        return [buf[k] for k in range(min(n, cap))]

    def launch_count(self) -> int:
        return int(lib().phi4_last_launch_count(self.h))
