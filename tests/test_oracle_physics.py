"""Physics pins for the serial oracle: exact results it must reproduce within 4 sigma
(SURVEY.md 8(c) pins 3, 4, 5, 7; north_star's own list).  Run with -m "not gpu".

The exact numbers come from tests/exact_ising.py (enumeration / Kaufman / Onsager / Yang in
50-digit arithmetic); tests/golden/*.txt hold the survey's copies as a cross-check of THOSE.
"""
import math
import os

import mpmath as mp
import numpy as np
import pytest

import oracle
import exact_ising as ex
from paper_2302_14720_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")
T_C = wl.T_C


def _table(name):
    rows = []
    for line in open(os.path.join(GOLD, name)):
        if line.startswith("#") or not line.strip():
            continue
        rows.append([float(t) for t in line.split()])
    return rows


# ---------------------------------------------------------------- the exact side checks itself
def test_enumeration_matches_survey_table_and_level_counts():
    r = ex.exact_small(4, T_C)
    assert r["levels"] == {-32: 2, -24: 32, -20: 64, -16: 424, -12: 1728, -8: 6688, -4: 13568, 0: 20524,
                           4: 13568, 8: 6688, 12: 1728, 16: 424, 20: 64, 24: 32, 32: 2}
    assert sum(r["levels"].values()) == 2 ** 16
    assert abs(r["Z"] - 5509120) < 1e-6           # Z(T_c) is an integer for this lattice (p = 2 - sqrt 2)
    for T, u, am, m2, c in _table("ising4x4_exact.txt"):
        r = ex.exact_small(4, T)
        assert abs(r["u"] - u) < 2e-12 and abs(r["abs_m"] - am) < 2e-12
        assert abs(r["m2"] - m2) < 2e-12 and abs(r["c"] - c) < 2e-12


def test_kaufman_formula_trust_chain():
    # the formula, as typed in exact_ising.py, reproduces brute force on 4x4 (Z, u, c) ...
    for T in (1.5, 2.269, T_C, 3.5):
        r = ex.exact_small(4, T)
        assert abs(mp.e ** ex.kaufman_lnZ(4, 1 / mp.mpf(T)) / r["Z"] - 1) < mp.mpf(10) ** -25
        assert abs(ex.kaufman_u(4, T) - r["u"]) < 1e-16
        assert abs(ex.kaufman_c(4, T) - r["c"]) < 1e-14
    # ... on 3x3 (odd side) and 2x2 as well
    for L in (2, 3):
        r = ex.exact_small(L, 2.5)
        assert abs(ex.kaufman_u(L, 2.5) - r["u"]) < 1e-16
    # ... agrees with the survey's table at L = 64, and tends to Onsager away from T_c
    row = [r for r in _table("kaufman_u.txt") if r[0] == 64][0]
    for T, u in zip((2.0, 2.26919, T_C, 2.5, 3.0), row[1:]):
        assert abs(ex.kaufman_u(64, T) - u) < 2e-10
    assert abs(ex.kaufman_u(64, 2.0) - ex.onsager_u(2.0)) < 1e-10
    assert abs(ex.onsager_u(T_C * (1 + 1e-9)) + mp.sqrt(2)) < 1e-6      # u(T_c) = -sqrt 2
    assert abs(ex.onsager_u(2.0) - mp.mpf("-1.745564575313")) < 1e-11
    assert abs(ex.yang_m(2.0) - mp.mpf("0.911319377877")) < 1e-11


# ---------------------------------------------------------------- pin 3: 4x4 vs exact enumeration
@pytest.mark.slow
@pytest.mark.parametrize("T,seed", [(1.5, 7), (2.269, 8), (3.5, 9)])
def test_oracle_4x4_matches_exact_enumeration(T, seed):
    L, N, therm, n = 4, 16, 100, 100000
    _, ser = oracle.run(L, T, seed, therm + n)
    ser = ser[therm:]
    r = ex.exact_small(L, T)
    u, du = ex.binned_mean_err(ser[:, 0] / N)
    am, dam = ex.binned_mean_err(np.abs(ser[:, 1]) / N)
    m2, dm2 = ex.binned_mean_err((ser[:, 1] / N) ** 2)
    assert abs(u - float(r["u"])) <= 4 * du, (u, du, float(r["u"]))
    assert abs(am - float(r["abs_m"])) <= 4 * dam, (am, dam, float(r["abs_m"]))
    assert abs(m2 - float(r["m2"])) <= 4 * dm2
    assert du < 6e-3 and dam < 3e-3            # the test has resolving power
    # the paper's printed p = 1 - exp(-1/T) (with J = 1) would be off by hundreds of sigma (c-1)
    if T == 2.269:
        assert abs(u - (-0.524)) > 100 * du
    # signed magnetisation averages to zero (cluster spins are assigned, not kept)
    ms, dms = ex.binned_mean_err(ser[:, 1] / N)
    assert abs(ms) <= 4 * dms
    # every energy level is visited with its Boltzmann weight (chi^2-free check on the two extremes)
    pE = {int(e): float(g * mp.e ** (-mp.mpf(int(e)) / mp.mpf(T)) / r["Z"]) for e, g in r["levels"].items()}
    f_ground = float(np.mean(ser[:, 0] == -32))
    assert abs(f_ground - pE[-32]) < 5 * math.sqrt(max(pE[-32], 1e-5) * 20 / n) + 1e-4


# ---------------------------------------------------------------- pin 4: Kaufman finite-L energy
@pytest.mark.slow
@pytest.mark.parametrize("L,T,seed,n", [(32, T_C, 21, 30000), (64, 2.26919, 2024, 12000), (48, 2.5, 23, 12000)])
def test_oracle_energy_matches_kaufman(L, T, seed, n):
    therm = 300
    _, ser = oracle.run(L, T, seed, therm + n)
    u, du = ex.binned_mean_err(ser[therm:, 0] / (L * L))
    exact = float(ex.kaufman_u(L, T))
    assert abs(u - exact) <= 4 * du, (u, du, exact)
    assert du < 2.5e-3
    # Onsager's L -> infinity value at T_c is NOT within the error bar: the finite-L pin matters
    if abs(T - T_C) < 1e-4:
        assert abs(exact + math.sqrt(2)) > 4 * du


# ---------------------------------------------------------------- pin 5: Onsager / Yang away from T_c
@pytest.mark.slow
def test_oracle_matches_onsager_and_yang_below_Tc():
    L, T, seed, therm, n = 96, 2.0, 31, 300, 4000
    _, ser = oracle.run(L, T, seed, therm + n)
    N = L * L
    u, du = ex.binned_mean_err(ser[therm:, 0] / N)
    am, dam = ex.binned_mean_err(np.abs(ser[therm:, 1]) / N)
    assert abs(u - float(ex.onsager_u(T))) <= 4 * du, (u, du)
    assert abs(am - float(ex.yang_m(T))) <= 4 * dam + 2e-4, (am, dam)   # finite-L shift of |m| < 2e-4 at L = 96
    assert du < 1.5e-3 and dam < 1.5e-3
    # the largest cluster is the magnetised one: <maxcl>/N tracks <|m|> closely below T_c
    big, dbig = ex.binned_mean_err(ser[therm:, 3] / N)
    assert abs(big - am) < 0.02


@pytest.mark.slow
def test_oracle_matches_onsager_above_Tc_and_bond_identity():
    L, T, seed, therm, n = 96, 3.0, 32, 200, 3000
    N = L * L
    thr = oracle.threshold(T)
    p = thr / 2.0 ** 32
    s = oracle.init_random(L, seed)
    us, nb = [], []
    for t in range(therm + n):
        # <bonds>/N = p (1 - u/2) where u is the energy of the configuration the bonds are drawn on
        if t >= therm and t % 10 == 0:
            E, _, _, _ = oracle.observables(L, s)
            bE, bS = oracle.bonds(L, thr, seed, t, s)
            nb.append((int(bE.sum()) + int(bS.sum())) / N - p * (1 - (E / N) / 2))
        s, ser = oracle.run(L, T, seed, 1, spins=s, t0=t)
        if t >= therm:
            us.append(ser[0, 0] / N)
    u, du = ex.binned_mean_err(us)
    assert abs(u - float(ex.onsager_u(T))) <= 4 * du, (u, du)
    d, dd = ex.binned_mean_err(nb, nbins=30)
    assert abs(d) <= 4 * dd + 1e-9, (d, dd)
    # |m| -> 0 above T_c (Fig. 7)
    assert np.mean(np.abs(np.array(us))) > 0 and abs(np.mean(us)) < 1.0
