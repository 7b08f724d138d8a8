"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NONE of the method's arithmetic: no Philox, no thresholds, no
bond rule, no labelling.  It only names the workloads (lattice side, temperature,
seed, start, sweep count) and builds injected start states / bond patterns with
numpy's own generator.  Random numbers the method itself draws are defined by the
counter-based generator that oracle/ and csrc/ each implement on their own.

The paper's workloads are RNG-generated Ising lattices (L = 128
... 4096, 10^4 iterations); there is no external dataset.  The five configurations
below are BASELINE.json's `configs`, made concrete as in SURVEY.md section 8(d).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import List, Tuple

import numpy as np

#: critical temperature of the 2D square-lattice Ising model, J = k_B = 1 (a workload parameter)
T_C = 2.0 / math.log(1.0 + math.sqrt(2.0))   # 2.269185314213022
#: the literal BASELINE.json prints for configs 1 and 2 (SURVEY.md 8(c) reading c-11)
T_C_PRINTED = 2.26919


@dataclass(frozen=True)
class Workload:
    name: str
    L: int
    T: Tuple[float, ...]          # one temperature per lattice of the batch
    seed: Tuple[int, ...]         # one seed per lattice
    start: str                    # "random" (Philox TAG_INIT stream of the seed) or "cold" (all +1)
    sweeps: int
    thermalise: int = 0
    note: str = ""

    @property
    def nb(self) -> int:
        return len(self.T)

    @property
    def sites(self) -> int:
        return self.L * self.L * self.nb


def scan_temperatures(nb: int = 32, lo: float = 1.5, hi: float = 3.5) -> Tuple[float, ...]:
    return tuple(lo + b * (hi - lo) / (nb - 1) for b in range(nb))


CONFIGS: List[Workload] = [
    Workload("c1_L64_Tc", 64, (T_C_PRINTED,), (2024,), "random", 1000,
             note="BASELINE configs[0], first half"),
    Workload("c1_4x4_T1.5", 4, (1.5,), (7,), "random", 100000, 100, "configs[0]: 4x4 vs exact enumeration"),
    Workload("c1_4x4_T2.269", 4, (2.269,), (8,), "random", 100000, 100, "configs[0]"),
    Workload("c1_4x4_T3.5", 4, (3.5,), (9,), "random", 100000, 100, "configs[0]"),
    Workload("c2_L1024_T2.0", 1024, (2.0,), (1,), "random", 2000, 200, "configs[1]"),
    Workload("c2_L1024_Tc", 1024, (T_C_PRINTED,), (2,), "random", 2000, 200, "configs[1]"),
    Workload("c2_L1024_T3.0", 1024, (3.0,), (3,), "random", 2000, 200, "configs[1]"),
    Workload("c3_L4096_cold", 4096, (T_C,), (4,), "cold", 1000, note="configs[2]"),
    Workload("c3_L4096_random", 4096, (T_C,), (5,), "random", 1000, note="configs[2]"),
    Workload("c4_L16384_Tc", 16384, (T_C,), (6,), "random", 200, note="configs[3]: headline roofline run"),
    Workload("c5_scan32_L2048", 2048, scan_temperatures(32), tuple(1000 + b for b in range(32)),
             "random", 1000, note="configs[4]: temperature scan, one launch per stage for the batch"),
]


def by_name(name: str) -> Workload:
    for w in CONFIGS:
        if w.name == name:
            return w
    raise KeyError(name)


# ---------------------------------------------------------------------------
# injected start states (int8 +-1, row-major i = y*L + x)
# ---------------------------------------------------------------------------
def spins_cold(L: int) -> np.ndarray:
    return np.ones(L * L, dtype=np.int8)

def spins_all_down(L: int) -> np.ndarray:
    return -np.ones(L * L, dtype=np.int8)

def spins_numpy_random(L: int, seed: int, p_up: float = 0.5) -> np.ndarray:
    """A start state from numpy's generator (NOT the method's stream)."""
    rng = np.random.default_rng(seed)
    return np.where(rng.random(L * L) < p_up, 1, -1).astype(np.int8)

def spins_checkerboard(L: int) -> np.ndarray:
    y, x = np.divmod(np.arange(L * L), L)
    return np.where((x + y) % 2 == 0, 1, -1).astype(np.int8)

def spins_stripes(L: int, width: int = 1, vertical: bool = False) -> np.ndarray:
    y, x = np.divmod(np.arange(L * L), L)
    c = x if vertical else y
    return np.where((c // width) % 2 == 0, 1, -1).astype(np.int8)

def spins_blocks(L: int, block: int) -> np.ndarray:
    """Square domains of side `block` (clusters that cross every tile edge when block > tile)."""
    y, x = np.divmod(np.arange(L * L), L)
    return np.where(((x // block) + (y // block)) % 2 == 0, 1, -1).astype(np.int8)


# ---------------------------------------------------------------------------
# injected bond patterns for labelling-only tests (one byte per site, 0/1)
# bondE[i]: edge i -- East(i);  bondS[i]: edge i -- South(i)
# ---------------------------------------------------------------------------
def bonds_random(L: int, seed: int, density: float) -> Tuple[np.ndarray, np.ndarray]:
    rng = np.random.default_rng(seed)
    bE = (rng.random(L * L) < density).astype(np.uint8)
    bS = (rng.random(L * L) < density).astype(np.uint8)
    return bE, bS

def bonds_none(L: int):
    return np.zeros(L * L, np.uint8), np.zeros(L * L, np.uint8)

def bonds_all(L: int):
    return np.ones(L * L, np.uint8), np.ones(L * L, np.uint8)

def bonds_row_wrap(L: int, row: int):
    """One full row of East bonds, closing around the torus."""
    bE, bS = bonds_none(L)
    bE[row * L:(row + 1) * L] = 1
    return bE, bS

def bonds_col_wrap(L: int, col: int):
    bE, bS = bonds_none(L)
    bS[col::L] = 1
    return bE, bS

def bonds_spiral(L: int):
    """A single path spiralling inwards from site 0 (long, thin cluster; worst case for pointer chains)."""
    bE, bS = bonds_none(L)
    x = y = 0
    dx, dy = 1, 0
    x0, y0, x1, y1 = 0, 0, L - 1, L - 1       # remaining box (inclusive), shrinks by 2 per turn for a gap
    visited = np.zeros((L, L), dtype=bool)
    visited[0, 0] = True
    while True:
        nx, ny = x + dx, y + dy
        def free(ax, ay):
            if not (0 <= ax < L and 0 <= ay < L) or visited[ay, ax]:
                return False
            # keep one empty lane between successive arms of the spiral
            for bx, by in ((ax + 1, ay), (ax - 1, ay), (ax, ay + 1), (ax, ay - 1)):
                if (bx, by) != (x, y) and 0 <= bx < L and 0 <= by < L and visited[by, bx]:
                    return False
            return True
        if not free(nx, ny):
            dx, dy = -dy, dx                   # turn right (screen coordinates: E -> S -> W -> N)
            nx, ny = x + dx, y + dy
            if not free(nx, ny):
                break
        if dx == 1:
            bE[y * L + x] = 1
        elif dx == -1:
            bE[ny * L + nx] = 1
        elif dy == 1:
            bS[y * L + x] = 1
        else:
            bS[ny * L + nx] = 1
        x, y = nx, ny
        visited[y, x] = True
    return bE, bS

def bonds_comb(L: int):
    """Top row fully bonded plus every second column hanging from it (many merges into one root)."""
    bE, bS = bonds_none(L)
    bE[0:L - 1] = 1
    for x in range(0, L, 2):
        bS[x:(L - 2) * L + x + 1:L] = 1
    return bE, bS


def bonds_ladder(L: int, every: int = 2, phase: int = 1):
    """Every column bonded top to bottom (not around the torus), rungs of East bonds on every `every`-th row: at each
    rung a whole row of distinct column labels meets at once -- far more label meetings and merges per 32 x 32 block than any
    equilibrium bond graph has (the kernels' lists of meetings / hooked nodes overflow into their fallback paths)."""
    bE, bS = bonds_none(L)
    bS[: (L - 1) * L] = 1
    for y in range(phase, L, every):
        bE[y * L: y * L + L - 1] = 1
    return bE, bS


def bonds_u_shapes(L: int):
    """Clusters of 2 x 3 sites: two columns of South bonds joined by one East bond at the bottom -- one merge of two labels
    per six sites (more hooked nodes per tile than the kernels' list holds)."""
    bE, bS = bonds_none(L)
    y = np.arange(L * L) // L
    x = np.arange(L * L) % L
    bS[(y % 3 != 2) & (y < L - 1)] = 1
    bE[(y % 3 == 2) & (x % 2 == 0) & (x < L - 1)] = 1
    return bE, bS


def bonds_dense_meetings(L: int, seed: int):
    """Columns broken at random places, rungs on random rows: many meetings, many separate clusters."""
    rng = np.random.default_rng(seed)
    bE, bS = bonds_none(L)
    bS[:] = (rng.random(L * L) < 0.9)
    rows = rng.random(L) < 0.5
    for y in np.nonzero(rows)[0]:
        bE[y * L:(y + 1) * L] = (rng.random(L) < 0.95)
    return bE, bS


def pack_bits(bytes01: np.ndarray) -> np.ndarray:
    """Canonical bit-plane layout of the C ABI: bit (i & 31) of uint32 word (i >> 5)."""
    b = np.asarray(bytes01, dtype=np.uint8).reshape(-1)
    pad = (-len(b)) % 32
    if pad:
        b = np.concatenate([b, np.zeros(pad, np.uint8)])
    return np.packbits(b, bitorder="little").view("<u4").copy()

def unpack_bits(words: np.ndarray, n: int) -> np.ndarray:
    w = np.ascontiguousarray(words, dtype="<u4")
    return np.unpackbits(w.view(np.uint8), bitorder="little")[:n].copy()
