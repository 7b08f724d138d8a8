"""Per-sweep invariants of a Swendsen-Wang sweep, checked with numpy/scipy only.

Used on the oracle's output (pins, SURVEY.md section 8(c) pin 6 and 9) and again on the CUDA
path's output at sizes where the oracle is too slow.  Nothing here imports oracle/ or the
CUDA binding; the labelling reference is scipy's connected_components (a library routine).
"""
from __future__ import annotations

import numpy as np
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components


def east(L: int) -> np.ndarray:
    i = np.arange(L * L, dtype=np.int64)
    y, x = np.divmod(i, L)
    return y * L + (x + 1) % L


def south(L: int) -> np.ndarray:
    i = np.arange(L * L, dtype=np.int64)
    y, x = np.divmod(i, L)
    return ((y + 1) % L) * L + x


def min_index_components(L: int, bondE: np.ndarray, bondS: np.ndarray) -> np.ndarray:
    """Connected components of the bond graph, each named by its minimum site index."""
    N = L * L
    i = np.arange(N, dtype=np.int64)
    e, s = east(L), south(L)
    mE, mS = bondE.astype(bool), bondS.astype(bool)
    rows = np.concatenate([i[mE], i[mS]])
    cols = np.concatenate([e[mE], s[mS]])
    g = coo_matrix((np.ones(len(rows), np.int8), (rows, cols)), shape=(N, N))
    _, comp = connected_components(g, directed=False)
    first = np.full(comp.max() + 1, N, dtype=np.int64)
    np.minimum.at(first, comp, i)
    return first[comp].astype(np.int32)


def flood_fill_labels(L: int, bondE, bondS):
    """Pure-Python flood fill for tiny lattices (a second, independent brute force)."""
    N = L * L
    adj = [[] for _ in range(N)]
    for i in range(N):
        y, x = divmod(i, L)
        e = y * L + (x + 1) % L
        s = ((y + 1) % L) * L + x
        if bondE[i]:
            adj[i].append(e); adj[e].append(i)
        if bondS[i]:
            adj[i].append(s); adj[s].append(i)
    lab = [-1] * N
    for r in range(N):
        if lab[r] >= 0:
            continue
        stack = [r]; lab[r] = r
        while stack:
            u = stack.pop()
            for v in adj[u]:
                if lab[v] < 0:
                    lab[v] = r; stack.append(v)
    return np.array(lab, dtype=np.int32)


def energy_magnetisation(L: int, spins: np.ndarray):
    s = spins.astype(np.int64)
    E = -int(np.sum(s * (s[east(L)] + s[south(L)])))
    return E, int(s.sum())


def check_sweep(L: int, spins_before, bondE, bondS, label, spins_after, obs=None, thr=None):
    """Assert every invariant of SURVEY.md 8(c) pin 6; bond arrays hold one byte per site."""
    N = L * L
    sb = np.asarray(spins_before).reshape(-1)
    sa = np.asarray(spins_after).reshape(-1)
    bE = np.asarray(bondE).reshape(-1).astype(bool)
    bS = np.asarray(bondS).reshape(-1).astype(bool)
    lab = np.asarray(label).reshape(-1).astype(np.int64)
    e, s = east(L), south(L)
    i = np.arange(N)
    assert set(np.unique(sb)) <= {-1, 1} and set(np.unique(sa)) <= {-1, 1}
    # bonds only between equal (pre-sweep) spins
    assert np.all(sb[i[bE]] == sb[e[bE]]), "East bond between unequal spins"
    assert np.all(sb[i[bS]] == sb[s[bS]]), "South bond between unequal spins"
    # canonical labels: root = minimum index, idempotent
    assert np.all(lab <= i) and np.all(lab >= 0)
    assert np.all(lab[lab] == lab)
    # closed under bonds (=> maximal)
    assert np.all(lab[i[bE]] == lab[e[bE]]) and np.all(lab[i[bS]] == lab[s[bS]])
    # connected through bonds and equal to the true components (library routine)
    ref = min_index_components(L, bE, bS)
    assert np.array_equal(ref, lab.astype(np.int32)), "labels differ from connected components"
    # single-spin clusters before the sweep, constant new spin on each cluster after it
    assert np.all(sb == sb[lab]), "cluster holds both spin values"
    assert np.all(sa == sa[lab]), "new spins not constant on a cluster"
    if obs is not None:
        E, M, ncl, maxcl = (int(v) for v in obs)
        E2, M2 = energy_magnetisation(L, sa)
        sizes = np.bincount(lab, minlength=N)
        assert (E, M) == (E2, M2)
        assert ncl == int(np.count_nonzero(lab == i))
        assert maxcl == int(sizes.max())
        assert int(sizes.sum()) == N
        assert abs(E) <= 2 * N and (M - N) % 2 == 0
        if L % 2 == 0:
            assert (E - 2 * N) % 4 == 0
