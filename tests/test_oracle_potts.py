"""Pins of the q-state Potts oracle (oracle/potts.py + the Potts part of oracle/sw_oracle.c; SURVEY.md 8(f) NEXT-3;
PAPER.md:33, :166) -- CPU only.

What fixes the result other than the oracle itself:
  * threshold: closed forms p(T_c(q)) = sqrt(q) / (1 + sqrt(q)) at T_c(q) = 1 / ln(1 + sqrt(q)), and the identity with
    the Ising threshold (pinned to 50 digits elsewhere) at T_Ising = 2 T;
  * colour draw: floor(word q / 2^32) recomputed from the Philox words (known-answer pinned) in Python integers;
  * the whole sweep: exact enumeration of all 3^9 states of the 3 x 3 three-state lattice (written out below), and of the
    4 x 4 two-state lattice through the Ising table (E_Potts = (E_Ising - 2N) / 2 at T_Potts = T_Ising / 2), Kaufman's exact
    finite-lattice energy at L = 32 for q = 2, all within 4 sigma of binned Monte-Carlo error;
  * invariants per sweep: bonds only between equal colours, clusters single-coloured and maximal, labels = minimum index.
"""
import math

import numpy as np
import pytest

import exact_ising as ex
import invariants as inv
import oracle
from oracle import potts

TAG_INIT, TAG_FLIP = 0, 2


def t_c(q):
    return 1.0 / math.log(1.0 + math.sqrt(q))


def test_threshold_closed_forms():
    assert potts.threshold(t_c(4)) in (2863311530, 2863311531)          # p = 2/3 (the rounding of T_c decides the last unit)
    assert abs(potts.threshold(t_c(9)) - 0.75 * 2 ** 32) <= 2              # p = 3/4
    assert abs(potts.threshold(1.0 / math.log(2.0)) - 2 ** 31) <= 2        # p = 1/2
    for T in (0.3, 0.7, t_c(2), t_c(3), 1.5, 10.0):
        assert potts.threshold(T) == oracle.threshold(2.0 * T)            # 1 - exp(-1/T) = 1 - exp(-2/(2T)), same double
        assert potts.threshold(T) == min(int(math.floor(-math.expm1(-1.0 / T) * 2 ** 32)), 2 ** 32 - 1)
    assert potts.threshold(1e-3) == 0xFFFFFFFF and potts.threshold(1e12) == 0


def test_colour_is_floor_word_q_over_2_32():
    seed, t = 0x123456789ABCDEF, 77
    key = [seed & 0xFFFFFFFF, seed >> 32]
    for q in (2, 3, 5, 8, 127):
        for idx in (0, 1, 2, 3, 4, 5, 1023, 10 ** 6 + 3):
            w = oracle.philox4x32_10([idx >> 2, t, 0, TAG_FLIP], key)
            assert potts.colour(seed, t, TAG_FLIP, idx, q) == (int(w[idx & 3]) * q) >> 32
    # q = 2: the top bit of the word
    w = oracle.philox4x32_10([0, 0, 0, TAG_INIT], [5, 0])
    assert [potts.colour(5, 0, TAG_INIT, i, 2) for i in range(4)] == [int(x) >> 31 for x in w]
    # uniform: 30000 draws, every colour within 4.5 sigma
    for q in (3, 7):
        c = np.bincount(potts.init_random(174, q, 99).astype(np.int64), minlength=q)
        n = 174 * 174
        assert c.sum() == n and np.all(np.abs(c - n / q) < 4.5 * math.sqrt(n / q))


def _potts_enumeration(L, q):
    """E = -#(equal East / South pairs) and M = q max_c n_c - N of all q^N states, straight from the definition."""
    N = L * L
    idx = np.arange(q ** N, dtype=np.int64)
    s = np.empty((N, q ** N), dtype=np.int8)
    for i in range(N):
        s[i] = (idx // q ** i) % q
    E = np.zeros(q ** N, dtype=np.int64)
    for i in range(N):
        y, x = divmod(i, L)
        E -= (s[i] == s[y * L + (x + 1) % L]).astype(np.int64) + (s[i] == s[((y + 1) % L) * L + x]).astype(np.int64)
    nmax = np.max(np.stack([(s == c).sum(axis=0) for c in range(q)]), axis=0)
    return E, q * nmax - N


@pytest.mark.parametrize("T,seed", [(0.7, 7), (0.995, 8), (1.5, 9)])
def test_three_state_3x3_against_exact_enumeration(T, seed):
    L, q, n, therm = 3, 3, 120000, 100
    E, M = _potts_enumeration(L, q)
    w = np.exp(-(E - E.min()) / T)
    exact_E, exact_M = float((E * w).sum() / w.sum()), float((M * w).sum() / w.sum())
    _, ser = potts.run(L, q, T, seed, therm + n)
    e, de = ex.binned_mean_err(ser[therm:, 0])
    m, dm = ex.binned_mean_err(ser[therm:, 1])
    assert abs(e - exact_E) <= 4 * de and de < 0.05, (e, de, exact_E)
    assert abs(m - exact_M) <= 4 * dm and dm < 0.05, (m, dm, exact_M)
    # the two candidate misreadings are far outside: p = 1 - exp(-2/T) (the Ising rule) samples temperature T / 2
    w2 = np.exp(-(E - E.min()) / (T / 2))
    assert abs(float((E * w2).sum() / w2.sum()) - exact_E) > 20 * de


@pytest.mark.parametrize("T_ising,seed", [(1.5, 17), (2.269, 18), (3.5, 19)])
def test_two_state_4x4_is_the_ising_table(T_ising, seed):
    L, n, therm = 4, 100000, 100
    N = L * L
    r = ex.exact_small(L, T_ising)
    _, ser = potts.run(L, 2, T_ising / 2.0, seed, therm + n)
    e, de = ex.binned_mean_err(2.0 * ser[therm:, 0] / N + 2.0)          # E_Ising / N = 2 E_Potts / N + 2
    m, dm = ex.binned_mean_err(ser[therm:, 1] / N)                      # q = 2: M = |n_0 - n_1| = |M_Ising|
    assert abs(e - float(r["u"])) <= 4 * de, (e, de, float(r["u"]))
    assert abs(m - float(r["abs_m"])) <= 4 * dm, (m, dm, float(r["abs_m"]))


@pytest.mark.slow
def test_two_state_L32_matches_kaufman_at_the_critical_point():
    L, n, therm, seed = 32, 20000, 300, 41
    T = t_c(2)                                                         # = T_c(Ising) / 2
    _, ser = potts.run(L, 2, T, seed, therm + n)
    u, du = ex.binned_mean_err(2.0 * ser[therm:, 0] / (L * L) + 2.0)
    exact = float(ex.kaufman_u(L, 2.0 * T))
    assert abs(u - exact) <= 4 * du and du < 3e-3, (u, du, exact)


@pytest.mark.parametrize("L,q,T", [(5, 3, 0.9), (16, 3, 0.995), (16, 4, 0.91), (13, 7, 0.6), (24, 2, 1.1346)])
def test_invariants_every_sweep(L, q, T):
    seed = 100 + L + q
    s = potts.init_random(L, q, seed)
    assert s.min() >= 0 and s.max() <= q - 1
    thr = potts.threshold(T)
    for t in range(12):
        s1, bE, bS, lab, obs = potts.sweep(L, q, T, seed, t, s)
        e, so = inv.east(L), inv.south(L)
        assert np.all(s[bE != 0] == s[e][bE != 0]) and np.all(s[bS != 0] == s[so][bS != 0])     # bond => equal colours
        assert np.array_equal(lab, inv.min_index_components(L, bE, bS))
        assert np.array_equal(s1, s1[lab])                                                     # one colour per cluster
        assert np.array_equal(s1[lab == np.arange(L * L)],
                              [potts.colour(seed, t, TAG_FLIP, int(r), q) for r in np.nonzero(lab == np.arange(L * L))[0]])
        assert s1.min() >= 0 and s1.max() <= q - 1
        (E, M, ncl, maxcl), cnt = potts.observables(L, q, s1, lab)
        assert (E, M, ncl, maxcl) == obs
        assert E == -int((s1 == s1[e]).sum() + (s1 == s1[so]).sum())
        assert cnt.sum() == L * L and M == q * cnt.max() - L * L
        assert ncl == int((lab == np.arange(L * L)).sum()) and maxcl == int(np.bincount(lab).max())
        # the bond draws are the Ising oracle's own function (equal values AND word < thr)
        bE2, bS2 = oracle.bonds(L, thr, seed, t, s)
        assert np.array_equal(bE, bE2) and np.array_equal(bS, bS2)
        s = s1


def test_limits():
    L, q = 12, 5
    s0 = potts.init_random(L, q, 3)
    # T -> 0 from a single colour: one cluster; T -> infinity: every site its own cluster
    s1, bE, bS, lab, obs = potts.sweep(L, q, 1e-3, 3, 0, np.zeros(L * L, dtype=np.int8))
    assert obs[2] == 1 and obs[3] == L * L and obs[0] == -2 * L * L and obs[1] == (q - 1) * L * L
    s1, bE, bS, lab, obs = potts.sweep(L, q, 1e12, 3, 0, s0)
    assert obs[2] == L * L and obs[3] == 1 and not bE.any() and not bS.any()
