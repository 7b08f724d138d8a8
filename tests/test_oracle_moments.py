"""Pins for oracle/moments.py: the definitions of <e>, <e^2>, <|m|>, <m^2>, <m^4>,
C/N, chi', U_4 against closed forms, numpy's own statistics, and the exact 4x4 enumeration.  -m "not gpu"."""
import math

import numpy as np
import pytest

import oracle
from oracle import moments as om
import exact_ising as ex


def test_constant_series_has_no_fluctuations():
    r = om.moments([-24] * 10, [8] * 10, 16, 2.0)
    assert r["n"] == 10 and r["e_mean"] == -1.5 and r["e2_mean"] == 2.25
    assert r["absm_mean"] == 0.5 and r["m2_mean"] == 0.25 and r["m4_mean"] == 0.0625
    assert r["specific_heat"] == 0.0 and r["susceptibility"] == 0.0
    assert r["binder"] == pytest.approx(1.0 - 1.0 / 3.0)          # a delta distribution of |m|: U_4 = 2/3


def test_two_valued_series_closed_form():
    # e alternates between -2 and -1, m between +1 and -1/2 (sign must not matter for |m|, m^2, m^4)
    N, T, n = 64, 2.5, 1000
    E = [-128, -64] * (n // 2)
    M = [64, -32] * (n // 2)
    r = om.moments(E, M, N, T)
    assert r["e_mean"] == pytest.approx(-1.5, abs=1e-13) and r["e2_mean"] == pytest.approx(2.5, abs=1e-13)
    assert r["specific_heat"] == pytest.approx(N * 0.25 / T ** 2, rel=1e-12)       # var(e) = 1/4
    assert r["absm_mean"] == pytest.approx(0.75, abs=1e-13) and r["m2_mean"] == pytest.approx(0.625, abs=1e-13)
    assert r["susceptibility"] == pytest.approx(N * (0.625 - 0.5625) / T, rel=1e-12)
    assert r["m4_mean"] == pytest.approx((1 + 1 / 16) / 2, abs=1e-13)
    assert r["binder"] == pytest.approx(1 - 0.53125 / (3 * 0.625 ** 2), rel=1e-12)


def test_against_numpy_statistics_on_a_real_run():
    L, T = 16, 2.3
    _, ser = oracle.run(L, T, 5, 400)
    N = L * L
    r = om.moments(ser[:, 0], ser[:, 1], N, T)
    e = ser[:, 0].astype(np.float64) / N
    a = np.abs(ser[:, 1].astype(np.float64)) / N
    assert r["e_mean"] == pytest.approx(e.mean(), rel=1e-13)
    assert r["absm_mean"] == pytest.approx(a.mean(), rel=1e-13)
    assert r["specific_heat"] == pytest.approx(N * e.var() / T ** 2, rel=1e-9)
    assert r["susceptibility"] == pytest.approx(N * a.var() / T, rel=1e-9)
    assert r["binder"] == pytest.approx(1 - (a ** 4).mean() / (3 * (a ** 2).mean() ** 2), rel=1e-12)
    with pytest.raises(ValueError):
        om.moments([], [], N, T)


@pytest.mark.slow
@pytest.mark.parametrize("T,seed", [(1.5, 17), (2.269, 18), (3.5, 19)])
def test_4x4_specific_heat_and_m2_match_exact_enumeration(T, seed):
    """C/N and <m^2> of a long oracle run against all 2^16 states (golden/ising4x4_exact.txt, SURVEY pin 3).
    Error of C/N from 50 bins, each bin its own moments() call."""
    L, N, therm, n, nb = 4, 16, 100, 100000, 50
    _, ser = oracle.run(L, T, seed, therm + n)
    ser = ser[therm:]
    r = ex.exact_small(L, T)
    full = om.moments(ser[:, 0], ser[:, 1], N, T)
    per = [om.moments(b[:, 0], b[:, 1], N, T) for b in np.array_split(ser, nb)]
    for key, exact in (("specific_heat", float(r["c"])), ("m2_mean", float(r["m2"])),
                       ("e_mean", float(r["u"])), ("absm_mean", float(r["abs_m"]))):
        vals = np.array([p[key] for p in per])
        err = vals.std(ddof=1) / math.sqrt(nb)
        bias = abs(exact) / (n / nb) * 20 if key == "specific_heat" else 0.0     # 1/n_bin bias of a variance
        assert abs(full[key] - exact) <= 4 * err + bias, (key, full[key], exact, err)
        assert err < 0.05 * max(abs(exact), 0.05)                                # the test resolves something
