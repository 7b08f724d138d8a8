"""Pins for the serial oracle that do not depend on the oracle itself (SURVEY.md 8(c) pins 1, 2, 6-9).

Run with -m "not gpu".  Each test is chosen so that a plausible mistake in the oracle (a dropped
round, a wrong word index, a transposed neighbour, a wrong sign) fails it.
"""
import hashlib
import json
import math
import os

import mpmath as mp
import numpy as np
import pytest

import oracle
from paper_2302_14720_b200 import workloads as wl
import invariants as inv

GOLD = os.path.join(os.path.dirname(__file__), "golden")
T_C = wl.T_C


# ---------------------------------------------------------------- pin 1: Philox known answers
def _kat_rows():
    rows = []
    for line in open(os.path.join(GOLD, "philox4x32_10_kat.txt")):
        if line.startswith("#") or not line.strip():
            continue
        v = [int(t, 16) for t in line.split()]
        rows.append((v[0:4], v[4:6], v[6:10]))
    return rows


def test_philox_known_answers():
    rows = _kat_rows()
    assert len(rows) == 3
    for ctr, key, out in rows:
        assert oracle.philox4x32_10(ctr, key).tolist() == out


def test_philox_is_a_bijection_of_the_counter_and_keyed():
    # distinct counters -> distinct outputs (Philox is a permutation for a fixed key); key matters
    outs = {tuple(oracle.philox4x32_10([c, 0, 0, 0], [1, 2]).tolist()) for c in range(2000)}
    assert len(outs) == 2000
    assert oracle.philox4x32_10([5, 0, 0, 0], [1, 2]).tolist() != oracle.philox4x32_10([5, 0, 0, 0], [1, 3]).tolist()


def test_bit_layout_128_site_bits_per_call():
    # bit(idx) = word (idx>>5)&3, bit idx&31 of Philox(ctr=(idx>>7, t_lo, t_hi, TAG), key=(seed_lo, seed_hi))
    seed, t = 0x1234567890ABCDEF, (7 << 32) | 11
    for idx in (0, 1, 31, 32, 95, 127, 128, 1000, 2 ** 28 - 1, 2 ** 30 - 1):
        w = oracle.philox4x32_10([idx >> 7, t & 0xFFFFFFFF, t >> 32, oracle.TAG_FLIP],
                                 [seed & 0xFFFFFFFF, seed >> 32])
        assert oracle.bit(seed, t, oracle.TAG_FLIP, idx) == (int(w[(idx >> 5) & 3]) >> (idx & 31)) & 1
    # the three streams are disjoint
    a = [oracle.bit(seed, 0, oracle.TAG_INIT, i) for i in range(256)]
    b = [oracle.bit(seed, 0, oracle.TAG_FLIP, i) for i in range(256)]
    assert a != b


def test_random_bits_are_fair():
    n = 200000
    s = oracle.init_random(448, 99)[:n].astype(np.int64)       # TAG_INIT stream
    assert abs(s.mean()) < 4 / math.sqrt(n)
    # neighbouring bits uncorrelated
    assert abs(np.mean(s[:-1] * s[1:])) < 4 / math.sqrt(n)


# ---------------------------------------------------------------- pin 2: thresholds
def _thr_exact(T):
    p = 1 - mp.e ** (mp.mpf(-2) / mp.mpf(T))
    return int(min(mp.floor(p * mp.mpf(2) ** 32), 2 ** 32 - 1))


def test_thresholds_against_50_digit_arithmetic():
    for line in open(os.path.join(GOLD, "thresholds.txt")):
        if line.startswith("#") or not line.strip():
            continue
        T, thr = line.split()
        T = float(T)
        assert oracle.threshold(T) == int(thr) == _thr_exact(T)


def test_threshold_closed_form_at_Tc_and_limits():
    # at T_c, p = 2 - sqrt(2) exactly (exp(-2/T_c) = sqrt(2) - 1)
    exact = int(mp.floor((2 - mp.sqrt(2)) * mp.mpf(2) ** 32))
    assert abs(oracle.threshold(T_C) - exact) <= 2          # T_c is a rounded double
    assert oracle.threshold(1e-3) == 0xFFFFFFFF              # p -> 1: clamp, never 2^32
    assert oracle.threshold(0.05) == 0xFFFFFFFF
    assert oracle.threshold(1e12) == 0                       # p ~ 2e-12 < 2^-32
    assert oracle.threshold(1e6) == _thr_exact(1e6)          # expm1 keeps small p accurate
    # the paper's printed form 1 - exp(-1/T) is a different number (reading c-1)
    assert oracle.threshold(2.269) != int(math.floor((1 - math.exp(-1 / 2.269)) * 2 ** 32))
    # monotone decreasing in T
    ts = np.linspace(0.5, 6.0, 56)
    th = [oracle.threshold(t) for t in ts]
    assert all(a > b for a, b in zip(th, th[1:]))


# ---------------------------------------------------------------- pin 8: survey golden vectors
def _pm(s):
    return "".join("+" if v > 0 else "-" for v in s)


def test_survey_vector_L4():
    g = json.load(open(os.path.join(GOLD, "survey_vectors.json")))["L4"]
    L, T, seed = g["L"], g["T"], g["seed"]
    s = oracle.init_random(L, seed)
    assert _pm(s) == g["start"]
    s1, bE, bS, lab, obs = oracle.sweep(L, T, seed, 0, s)
    assert "".join(map(str, bE)) == g["sweep0"]["bondE"]
    assert "".join(map(str, bS)) == g["sweep0"]["bondS"]
    assert lab.tolist() == g["sweep0"]["labels"]
    assert _pm(s1) == g["sweep0"]["spins"]
    assert list(obs) == g["sweep0"]["obs"]
    s2, *_, obs1 = oracle.sweep(L, T, seed, 1, s1)
    s3, *_, obs2 = oracle.sweep(L, T, seed, 2, s2)
    assert list(obs1) == g["sweep1_obs"] and list(obs2) == g["sweep2_obs"]


def test_survey_vector_L64():
    g = json.load(open(os.path.join(GOLD, "survey_vectors.json")))["L64"]
    L, seed = g["L"], g["seed"]
    s = oracle.init_random(L, seed)
    assert int(s.sum()) == g["sum_start"]
    for t in range(10):
        s, bE, bS, lab, obs = oracle.sweep(L, T_C, seed, t, s)
        if str(t) in g["obs"]:
            assert list(obs) == g["obs"][str(t)]
        if t == 0:
            assert [int(bE.sum()), int(bS.sum())] == g["bond_counts_sweep0"]
    assert hashlib.sha256(s.tobytes()).hexdigest()[:16] == g["sha256_spins_after_sweep9_first16"]


def test_survey_vector_L1024():
    g = json.load(open(os.path.join(GOLD, "survey_vectors.json")))["L1024"]
    _, ser = oracle.run(g["L"], T_C, g["seed"], 20)
    for k, v in g["obs"].items():
        assert ser[int(k)].tolist() == v


# ---------------------------------------------------------------- pin 9: labelling alone, brute force
def _patterns(L):
    yield "none", wl.bonds_none(L)
    yield "all", wl.bonds_all(L)
    yield "row_wrap", wl.bonds_row_wrap(L, L - 1)
    yield "col_wrap", wl.bonds_col_wrap(L, L - 1)
    yield "comb", wl.bonds_comb(L)
    if L >= 3:
        yield "spiral", wl.bonds_spiral(L)
    for k, d in enumerate((0.1, 0.3, 0.5, 0.7, 0.9)):
        yield f"random{d}", wl.bonds_random(L, 100 * L + k, d)


@pytest.mark.parametrize("L", [2, 3, 4, 5, 8, 13])
def test_labels_equal_brute_force_on_tiny_lattices(L):
    for name, (bE, bS) in _patterns(L):
        lab = oracle.labels(L, bE, bS)
        assert np.array_equal(lab, inv.flood_fill_labels(L, bE, bS)), name
        assert np.array_equal(lab, inv.min_index_components(L, bE, bS)), name
    # special results that are fixed by hand
    assert oracle.labels(L, *wl.bonds_none(L)).tolist() == list(range(L * L))
    assert oracle.labels(L, *wl.bonds_all(L)).tolist() == [0] * (L * L)
    rw = oracle.labels(L, *wl.bonds_row_wrap(L, L - 1))
    assert rw[(L - 1) * L:].tolist() == [(L - 1) * L] * L and rw[:(L - 1) * L].tolist() == list(range((L - 1) * L))


def test_L2_double_edges_are_independent():
    # L = 2: East(i) and West(i) are the same site, yet the two edges have separate draws and both
    # enter the energy (reading c-3).  All-up start at very low T: every one of the 8 edges bonds.
    L, T, seed = 2, 0.05, 3
    s, bE, bS, lab, obs = oracle.sweep(L, T, seed, 0, wl.spins_cold(L))
    assert bE.tolist() == [1, 1, 1, 1] and bS.tolist() == [1, 1, 1, 1]
    assert lab.tolist() == [0, 0, 0, 0]
    assert obs[0] == -8 and abs(obs[1]) == 4 and obs[2:] == (1, 4)


@pytest.mark.parametrize("L", [33, 64, 96])
def test_labels_equal_scipy_components(L):
    for name, (bE, bS) in _patterns(L):
        assert np.array_equal(oracle.labels(L, bE, bS), inv.min_index_components(L, bE, bS)), name


# ---------------------------------------------------------------- pin 6: per-sweep invariants
@pytest.mark.parametrize("L,T,seed", [(2, 2.0, 1), (3, 2.269, 2), (4, 1.5, 3), (5, 3.5, 4), (8, T_C, 5),
                                       (16, 2.0, 6), (33, T_C, 7), (64, T_C, 8), (100, 3.0, 9)])
def test_sweep_invariants(L, T, seed):
    s = oracle.init_random(L, seed)
    for t in range(6):
        s1, bE, bS, lab, obs = oracle.sweep(L, T, seed, t, s)
        inv.check_sweep(L, s, bE, bS, lab, s1, obs)
        s = s1


def test_sweep_is_a_pure_function_of_state_seed_and_t():
    L, T, seed = 24, T_C, 77
    s0 = wl.spins_numpy_random(L, 5)
    a = oracle.sweep(L, T, seed, 41, s0)
    b = oracle.sweep(L, T, seed, 41, s0)
    assert all(np.array_equal(x, y) for x, y in zip(a[:4], b[:4])) and a[4] == b[4]
    c = oracle.sweep(L, T, seed, 42, s0)
    assert not np.array_equal(a[1], c[1])
    d = oracle.sweep(L, T, seed + 1, 41, s0)
    assert not np.array_equal(a[1], d[1])
    # run() == repeated sweep(); t0 offsets the stream (one-step parity relies on this)
    s_run, ser = oracle.run(L, T, seed, 5, spins=s0, t0=40)
    s = s0
    for k in range(5):
        s, *_, obs = oracle.sweep(L, T, seed, 40 + k, s)
        assert ser[k].tolist() == list(obs)
    assert np.array_equal(s, s_run)
    # the 64-bit sweep index reaches the counter's third word
    hi = oracle.sweep(L, T, seed, (1 << 32) + 41, s0)
    assert not np.array_equal(a[1], hi[1])


def test_cold_and_special_starts():
    L = 16
    # T -> 0: every edge between equal spins bonds; cold start is one cluster
    s, bE, bS, lab, obs = oracle.sweep(L, 0.01, 1, 0, wl.spins_cold(L))
    assert bE.all() and bS.all() and not lab.any() and obs[2:] == (1, L * L) and obs[0] == -2 * L * L
    # checkerboard: no equal neighbours, no bonds at any T, N singleton clusters
    s, bE, bS, lab, obs = oracle.sweep(L, 0.01, 1, 0, wl.spins_checkerboard(L))
    assert not bE.any() and not bS.any() and lab.tolist() == list(range(L * L)) and obs[2:] == (L * L, 1)
    # T -> infinity: no bonds
    s, bE, bS, lab, obs = oracle.sweep(L, 1e12, 1, 0, wl.spins_cold(L))
    assert not bE.any() and not bS.any()
    # horizontal stripes of width 1 at T -> 0: East bonds only, L clusters of L sites, each wrapping
    s, bE, bS, lab, obs = oracle.sweep(L, 0.01, 1, 0, wl.spins_stripes(L, 1))
    assert bE.all() and not bS.any() and obs[2:] == (L, L)
    assert np.array_equal(lab, (np.arange(L * L) // L) * L)
    # vertical stripes: South bonds only
    s, bE, bS, lab, obs = oracle.sweep(L, 0.01, 1, 0, wl.spins_stripes(L, 1, vertical=True))
    assert bS.all() and not bE.any() and np.array_equal(lab, np.arange(L * L) % L)


# ---------------------------------------------------------------- pin 7: statistical identities
def test_acceptance_fraction_and_root_fairness():
    L, T, seed = 256, 2.5, 11
    thr = oracle.threshold(T)
    p = thr / 2.0 ** 32
    s = wl.spins_cold(L)                       # every pair equal: acceptance is exactly the draw
    bE, bS = oracle.bonds(L, thr, seed, 3, s)
    n = 2 * L * L
    acc = (int(bE.sum()) + int(bS.sum())) / n
    assert abs(acc - p) < 4 * math.sqrt(p * (1 - p) / n)
    # East and South use different words of the call
    assert abs(int(bE.sum()) / (n / 2) - p) < 4 * math.sqrt(p * (1 - p) / (n / 2))
    assert abs(int(bS.sum()) / (n / 2) - p) < 4 * math.sqrt(p * (1 - p) / (n / 2))
    assert not np.array_equal(bE, bS)
    # roots are assigned +1 with probability 1/2: no bonds -> N independent clusters
    lab = np.arange(L * L, dtype=np.int32)
    new = oracle.assign(L, seed, 3, lab).astype(np.int64)
    assert abs(new.mean()) < 4 / math.sqrt(L * L)
    # all sites in one cluster with root r get bit(r)
    for r in (0, 5, 127, 128, 4099):
        lab[:] = r
        new = oracle.assign(L, seed, 3, lab)
        assert np.all(new == (1 if oracle.bit(seed, 3, oracle.TAG_FLIP, r) else -1))
