"""Pins of oracle/label_equivalence.py (section 2.3) -- CPU only.

What fixes the result other than the oracle itself:
  * the final labels are the minimum site index of every connected component: the definition, computed by
    breadth-first search in oracle/sw_oracle.c (orc_labels) -- independent code;
  * the number of passes on bond graphs small enough to work by hand (derivations below);
  * the two statements (site-at-a-time loops, whole-array numpy) against each other.
"""
import numpy as np
import pytest

import oracle
from oracle import label_equivalence as le
from paper_2302_14720_b200 import workloads as wl


def _empty(L):
    return np.zeros(L * L, dtype=np.uint8), np.zeros(L * L, dtype=np.uint8)


def _chain(L, n):
    """row 0: sites 0 .. n-1 joined by East bonds."""
    bE, bS = _empty(L)
    bE[0:n - 1] = 1
    return bE, bS


def _u_shape(L, k):
    """column 0 rows 0..k, row k columns 0..2, column 2 rows 0..k."""
    bE, bS = _empty(L)
    for y in range(k):
        bS[y * L + 0] = 1
        bS[y * L + 2] = 1
    bE[k * L + 0] = 1
    bE[k * L + 1] = 1
    return bE, bS


def _hook_shape(L, k):
    """column 0 rows 0..k, row k columns 0..2, column 2 rows 1..k, row 1 columns 2..4, column 4 rows 0..1."""
    bE, bS = _empty(L)
    for y in range(k):
        bS[y * L + 0] = 1
    bE[k * L + 0] = 1
    bE[k * L + 1] = 1
    for y in range(1, k):
        bS[y * L + 2] = 1
    bE[1 * L + 2] = 1
    bE[1 * L + 3] = 1
    bS[0 * L + 4] = 1
    return bE, bS


BOTH = [le.label_equivalence_loops, le.label_equivalence]


@pytest.mark.parametrize("f", BOTH)
def test_pass_counts_worked_by_hand(f):
    # no bonds: the first scan forms no reference                                              -> 1 pass
    lab, p = f(6, *_empty(6))
    assert p == 1 and lab.tolist() == list(range(36))
    # chain 0-1-...-4 on row 0: scan 1 gives ref[x] = x - 1, the collapse walks every chain to 0,
    # the relabel makes every label 0; scan 2 finds nothing                                   -> 2 passes
    lab, p = f(6, *_chain(6, 5))
    assert p == 2 and lab[:5].tolist() == [0] * 5 and lab[5:].tolist() == list(range(5, 36))
    # a full row with the periodic bond: site L-1 sees 0 and L-2, still one collapse            -> 2 passes
    lab, p = f(6, *wl.bonds_row_wrap(6, 0))
    assert p == 2 and lab[:6].tolist() == [0] * 6
    # U: scan 1 sends column 0 and (k,1) down to 0, but (k,2) prefers (k-1,2) = (k-1)L+2 < kL+1, so column 2
    # collapses onto its top, site 2.  Scan 2: (k,2) [label 2] sees (k,1) [label 0]: ref[2] = 0.  Scan 3: nothing.
    for L, k in ((4, 1), (6, 3), (8, 6)):
        lab, p = f(L, *_u_shape(L, k))
        assert p == 3, (L, k, p)
        members = [y * L for y in range(k + 1)] + [k * L + 1] + [y * L + 2 for y in range(k + 1)]
        assert all(lab[m] == 0 for m in members) and int((lab == 0).sum()) == len(members)
    # hook: local minima of the site index along the chain are 0, L+2 (at (1,2): neighbours (2,2), (1,3)) and 4
    # (at (0,4)).  After pass 1 the labels are 0 | L+2 | 4 along the chain.  Scan 2: L+2 sees 0 and 4 and refers to
    # 0; 4 sees only L+2 > 4 and stays.  After pass 2: 0 | 4.  Scan 3: ref[4] = 0.  Scan 4: nothing   -> 4 passes
    for L, k in ((6, 3), (8, 5)):
        lab, p = f(L, *_hook_shape(L, k))
        assert p == 4, (L, k, p)
        assert int((lab == 0).sum()) == (k + 1) + 1 + k + 2 + 1 and lab[4] == 0 and lab[L + 2] == 0


@pytest.mark.parametrize("L", [2, 3, 4, 5, 8, 13])
def test_loops_reach_the_definition_on_random_graphs(L):
    for k, d in enumerate((0.0, 0.2, 0.45, 0.5, 0.55, 0.8, 1.0)):
        bE, bS = wl.bonds_random(L, 11 * L + k, d)
        want = oracle.labels(L, bE, bS)
        lab, p = le.label_equivalence_loops(L, bE, bS)
        assert np.array_equal(lab, want), (L, d)
        lab2, p2 = le.label_equivalence(L, bE, bS)
        assert np.array_equal(lab2, want) and p2 == p, (L, d, p, p2)


@pytest.mark.parametrize("L", [16, 33, 64, 100, 256])
def test_numpy_statement_reaches_the_definition(L):
    graphs = [wl.bonds_none(L), wl.bonds_all(L), wl.bonds_row_wrap(L, L - 1), wl.bonds_col_wrap(L, L - 1),
              wl.bonds_comb(L), wl.bonds_spiral(L)]
    graphs += [wl.bonds_random(L, 7 * L + k, d) for k, d in enumerate((0.2, 0.45, 0.5, 0.55, 0.8))]
    for g, (bE, bS) in enumerate(graphs):
        lab, p = le.label_equivalence(L, bE, bS)
        assert np.array_equal(lab, oracle.labels(L, bE, bS)), (L, g)
        assert p >= 1
        assert np.array_equal(lab[lab], lab) and np.all(lab <= np.arange(L * L))


def test_statements_agree_on_structured_graphs():
    for L in (8, 12):
        for bE, bS in (wl.bonds_comb(L), wl.bonds_spiral(L), wl.bonds_all(L), wl.bonds_col_wrap(L, 3)):
            a, pa = le.label_equivalence_loops(L, bE, bS)
            b, pb = le.label_equivalence(L, bE, bS)
            assert np.array_equal(a, b) and pa == pb


def test_statements_agree_at_parity_size():
    """The numpy statement is what the GPU pass counts are compared with at L >= 64: labels AND pass count against the
    plain loops on random bond graphs of that size (sub-, near- and super-critical bond densities) and on the bond graph
    of a Swendsen-Wang sweep."""
    L = 64
    graphs = [wl.bonds_random(L, 900 + k, d) for k, d in enumerate((0.3, 0.5, 0.7))]
    s = oracle.init_random(L, 5)
    for t in range(3):
        s, bE, bS, _, _ = oracle.sweep(L, wl.T_C, 5, t, s)
    graphs.append((bE, bS))
    for g, (bE, bS) in enumerate(graphs):
        a, pa = le.label_equivalence_loops(L, bE, bS)
        b, pb = le.label_equivalence(L, bE, bS)
        assert np.array_equal(a, b) and pa == pb, (g, pa, pb)
        assert np.array_equal(a, oracle.labels(L, bE, bS))


def test_pass_count_on_sw_bond_graphs_is_small():
    # context, not a pin: PAPER.md:53 reports "5 or 6 parallel iterations" for 512 x 512 (variant and counting
    # convention unstated); this statement needs 5-8 scans (the last one idle) at L = 512 and T_c on the way to equilibrium
    L, T, seed = 128, wl.T_C, 6
    s = oracle.init_random(L, seed)
    for t in range(12):
        s, bE, bS, lab, _ = oracle.sweep(L, T, seed, t, s)
        got, p = le.label_equivalence(L, bE, bS)
        assert np.array_equal(got, lab)
        assert 3 <= p <= 10
