"""ORACLE (test infrastructure, not product code): the paper's own cluster labelling, SURVEY.md 8(f) NEXT-2.

PAPER.md:49-53 (section 2.3, "Cluster Formation") describes a label-equivalence iteration (after Kalentev et
al., the paper's ref. [2]) in three steps per pass, restated here in the paper's order:

  init      "each site is labeled with a unique integer incrementing from zero":   label[i] = i, ref[i] = i
  scan      "each site ... comparing its label to those of its neighbors and forming a reference to the lowest
            valued neighbor":   m_i = min(label[j] : j bonded to i);  if m_i < label[i]:
                                ref[label[i]] = min(ref[label[i]], m_i)        (a minimum: order-free)
  collapse  "these forests are then collapsed into trees by a function which follows and links each site to
            the lowest label in its chain of references":   for every label l still in use (label[l] == l):
                                r = l;  while ref[r] != r: r = ref[r];  ref[l] = r
  relabel   "it then looks up the label it has been decided it is equivalent to, and assigns it to itself":
                                label[i] = ref[label[i]]
  "This process will repeat until every site is divided into its appropriate cluster": until a scan forms no
  reference.

Readings: a site's neighbours are the up to four sites it shares a bond with (periodic);
the relabel step is ONE lookup (after the collapse every label in use points at the end of its chain); `passes`
counts the scans, including the last one that finds nothing to do.  Every step is a minimum or a walk to a fixed
point, so labels AND the pass count are the same for every execution order -- exactly one result is correct, and
the final labels are the minimum site index of each cluster (the definition oracle.labels computes by BFS).

Two statements of the same algorithm: `label_equivalence_loops` (plain Python loops, one site at a time in index
order -- for tiny lattices) and `label_equivalence` (the same three steps with numpy array operations, for the
parity sizes).  Pinned (tests/test_oracle_label_equivalence.py): final labels against the definition
(oracle.labels, breadth-first search, independent code); pass counts against cases worked by hand (no bonds: 1;
a straight chain: 2; a U-shaped chain: 3; a chain whose labels after the first pass form the path 0 - (L+2) - 4: 4
-- derivations in the test file) and the two statements against each other.  Shares nothing with the CUDA path.
"""
from __future__ import annotations

from typing import Tuple

import numpy as np


def _neighbour_tables(L: int, bondE: np.ndarray, bondS: np.ndarray):
    """(nbr[4][N], has[4][N]): East, South, West, North neighbour of every site and whether a bond joins them."""
    N = L * L
    i = np.arange(N, dtype=np.int64)
    y, x = i // L, i % L
    east = y * L + (x + 1) % L
    south = ((y + 1) % L) * L + x
    west = y * L + (x - 1) % L
    north = ((y - 1) % L) * L + x
    bE = np.asarray(bondE).reshape(-1) != 0
    bS = np.asarray(bondS).reshape(-1) != 0
    return (east, south, west, north), (bE, bS, bE[west], bS[north])


def label_equivalence_loops(L: int, bondE, bondS, max_passes: int = 1 << 20) -> Tuple[np.ndarray, int]:
    """The three steps, one site at a time.  Returns (label[N] int32, passes)."""
    N = L * L
    nbr, has = _neighbour_tables(L, bondE, bondS)
    label = list(range(N))
    ref = list(range(N))
    passes = 0
    while passes < max_passes:
        passes += 1
        formed = False
        for i in range(N):                                   # scan
            m = label[i]
            for d in range(4):
                if has[d][i]:
                    m = min(m, label[int(nbr[d][i])])
            if m < label[i]:
                ref[label[i]] = min(ref[label[i]], m)
                formed = True
        if not formed:
            break
        for l in range(N):                                   # collapse
            if label[l] == l:
                r = l
                while ref[r] != r:
                    r = ref[r]
                ref[l] = r
        for i in range(N):                                   # relabel
            label[i] = ref[label[i]]
    return np.asarray(label, dtype=np.int32), passes


def label_equivalence(L: int, bondE, bondS, max_passes: int = 1 << 20) -> Tuple[np.ndarray, int]:
    """The same three steps on whole arrays.  Returns (label[N] int32, passes)."""
    N = L * L
    nbr, has = _neighbour_tables(L, bondE, bondS)
    big = np.int64(N)
    label = np.arange(N, dtype=np.int64)
    ref = np.arange(N, dtype=np.int64)
    passes = 0
    while passes < max_passes:
        passes += 1
        m = label.copy()                                     # scan
        for d in range(4):
            m = np.minimum(m, np.where(has[d], label[nbr[d]], big))
        lower = m < label
        if not lower.any():
            break
        np.minimum.at(ref, label[lower], m[lower])
        live = np.nonzero(label == np.arange(N))[0]          # collapse: walk every chain to its fixed point
        r = live.copy()
        while True:
            nxt = ref[r]
            if np.array_equal(nxt, r):
                break
            r = nxt
        ref[live] = r
        label = ref[label]                                   # relabel
    return label.astype(np.int32), passes
