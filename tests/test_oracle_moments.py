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


# ------------------------------------------------------------------------------------------------------------
# binning and the integrated autocorrelation time (oracle/moments.py, second half): pinned by closed forms and by
# series whose autocorrelation is known -- none of these repeats the oracle's own formula
def test_bin_means_closed_form_and_dropped_remainder():
    N = 8
    E = list(range(11))                                   # 0 .. 10: bins of 4 -> (0..3), (4..7); 8, 9, 10 dropped
    b = om.bin_means(E, [0] * 11, N, 0, 4)
    assert b == [1.5 / N, 5.5 / N]
    assert om.bin_means(E, [0] * 11, N, 0, 12) == []
    m = om.bin_means([0] * 6, [3, -5, 4, -4, 0, 7], N, 1, 2)         # |M|: sign must not matter
    assert m == [4.0 / N, 4.0 / N, 3.5 / N]


def test_binned_error_of_a_constant_series_is_zero_and_of_one_bin_too():
    mean, err, nb = om.binned_error([-24] * 40, [8] * 40, 16, 0, 5)
    assert (mean, err, nb) == (-1.5, 0.0, 8)
    assert om.binned_error([-24, -20, -28], [0] * 3, 16, 0, 3) == (-1.5, 0.0, 1)
    tau, W, rho = om.tau_int([-24] * 40, [8] * 40, 16, 0, 10)
    assert tau == 0.5 and W == 0 and rho == [0.0] * 11


def test_binned_error_with_unit_bins_is_the_textbook_standard_error():
    rng = np.random.default_rng(3)
    E = rng.integers(-2000, 2000, size=500)
    N = 1000
    mean, err, nb = om.binned_error(E, np.zeros(500, dtype=int), N, 0, 1)
    x = E.astype(np.float64) / N
    assert nb == 500 and mean == pytest.approx(x.mean(), rel=1e-13)
    assert err == pytest.approx(x.std(ddof=1) / math.sqrt(500), rel=1e-12)
    # bins of 10 of an iid series give the same error within its own scatter (1 / sqrt(2 (nb - 1)) = 10 %)
    _, err10, nb10 = om.binned_error(E, np.zeros(500, dtype=int), N, 0, 10)
    assert nb10 == 50 and abs(err10 / err - 1.0) < 0.4


def test_white_noise_has_tau_one_half():
    rng = np.random.default_rng(11)
    n, N = 20000, 1 << 20
    E = rng.integers(-N, N, size=n)
    tau, W, rho = om.tau_int(E, np.zeros(n, dtype=int), N, 0, 40)
    sigma = 0.5 * math.sqrt(2.0 * (2 * W + 1) / n)                     # Madras-Sokal variance of the windowed estimator
    assert 1 <= W <= 6 and abs(tau - 0.5) <= 4.0 * sigma, (tau, W, sigma)
    assert rho[0] == 1.0 and max(abs(v) for v in rho[1:]) < 4.0 / math.sqrt(n) * 1.5


@pytest.mark.parametrize("r", [0.5, 0.8])
def test_ar1_series_has_the_known_autocorrelation(r):
    """x_{k+1} = r x_k + noise: rho(t) = r^t, tau_int = (1/2) (1 + r) / (1 - r)."""
    rng = np.random.default_rng(int(100 * r))
    n, N = 60000, 1
    x = np.empty(n)
    x[0] = 0.0
    noise = rng.standard_normal(n)
    for k in range(1, n):
        x[k] = r * x[k - 1] + noise[k]
    M = np.rint(1e6 * (x + 20.0)).astype(np.int64)          # which = 1 takes |M|: shifted to stay positive
    exact = 0.5 * (1.0 + r) / (1.0 - r)
    tau, W, rho = om.tau_int(np.zeros(n, dtype=int), M, N, 1, 80)
    sigma = exact * math.sqrt(2.0 * (2 * W + 1) / n)
    bias = r ** (W + 1) / (1.0 - r)                          # the tail the window cuts off
    assert abs(tau - exact) <= 4.0 * sigma + bias, (tau, exact, W, sigma)
    for t in (1, 2, 3):
        assert abs(rho[t] - r ** t) < 0.02, (t, rho[t])
    assert W >= 6 * tau - 1e-9 and (W == 1 or (W - 1) < 6 * (tau - rho[W]) + 1e-9)       # the smallest such window


def test_autocovariance_at_lag_zero_is_the_exact_4x4_variance_and_binning_agrees_with_tau():
    """C(0) of e on the 4 x 4 lattice against the exact enumeration (var e = (C/N) T^2 / N); and the two error
    estimates of the mean -- binned with long bins, and sqrt(2 tau C(0) / n) -- agree."""
    T, n, N = 2.269, 40000, 16
    _, ser = oracle.run(4, T, 7, n + 100)
    E, M = ser[100:, 0], ser[100:, 1]
    C = om.autocovariance(E, M, N, 0, 0)
    exact = ex.exact_small(4, T)
    var_e = float(exact["c"]) * T * T / N
    tau, W, _ = om.tau_int(E, M, N, 0, 60)
    rel = math.sqrt(2.0 * 2.0 * tau / n) * 1.5               # relative error of a variance estimate, generous kurtosis factor
    assert abs(C[0] / var_e - 1.0) <= 4.0 * rel, (C[0], var_e)
    _, err, nb = om.binned_error(E, M, N, 0, 100)
    assert nb == 400
    assert abs(err / math.sqrt(2.0 * tau * C[0] / n) - 1.0) < 0.25, (err, tau, C[0])
    assert 0.5 < tau < 3.0                                   # cluster updates: no critical slowing down to speak of
