"""ORACLE (test infrastructure, not product code): moments of the per-sweep observables, SURVEY.md 8(f) NEXT-1.

The paper validates its code on the energy, the specific heat and the magnetisation as functions of the
temperature (section 4, Figs. 5-7; M and H per configuration: PAPER.md:63).  This module
writes the plain definitions out, one sweep at a time in double precision, in the order stated:

    e_k = E_k / N,  a_k = |M_k| / N            (per configuration)
    <e> = (1/n) sum e_k,  <e^2>,  <|m|> = (1/n) sum a_k,  <m^2> = (1/n) sum a_k^2,  <m^4>
    C / N  = N (<e^2> - <e>^2) / T^2           (specific heat per site, Fig. 6)
    chi'   = N (<m^2> - <|m|>^2) / T           (susceptibility of |m|)
    U_4    = 1 - <m^4> / (3 <m^2>^2)           (Binder cumulant)

Pinned (tests/test_oracle_moments.py) by exact enumeration of the 4x4 lattice (<m^2>, C/N within 4 sigma of a
long oracle run), by closed-form inputs (constant series, two-valued series) and by numpy's own mean/var.
Shares nothing with the CUDA path.  Python floats are IEEE doubles; no reordering, no fused operations.
"""
from __future__ import annotations

from typing import Dict, Sequence


def accumulate(E: Sequence[int], M: Sequence[int], N: int) -> Dict[str, float]:
    """Running sums over the sweeps, in order: s_e, s_e2, s_am, s_m2, s_m4 (doubles) and n."""
    s_e = s_e2 = s_am = s_m2 = s_m4 = 0.0
    n = 0
    fN = float(N)
    for Ek, Mk in zip(E, M):
        e = float(int(Ek)) / fN
        a = abs(float(int(Mk)) / fN)
        a2 = a * a
        s_e = s_e + e
        s_e2 = s_e2 + e * e
        s_am = s_am + a
        s_m2 = s_m2 + a2
        s_m4 = s_m4 + a2 * a2
        n += 1
    return {"n": n, "s_e": s_e, "s_e2": s_e2, "s_am": s_am, "s_m2": s_m2, "s_m4": s_m4}


def moments(E: Sequence[int], M: Sequence[int], N: int, T: float) -> Dict[str, float]:
    """Means and the derived quantities of the header, from the per-sweep integer E and M."""
    s = accumulate(E, M, N)
    n = s["n"]
    if n == 0:
        raise ValueError("no sweeps")
    fn = float(n)
    e = s["s_e"] / fn
    e2 = s["s_e2"] / fn
    am = s["s_am"] / fn
    m2 = s["s_m2"] / fn
    m4 = s["s_m4"] / fn
    fN = float(N)
    out = {"n": n, "e_mean": e, "e2_mean": e2, "absm_mean": am, "m2_mean": m2, "m4_mean": m4}
    out["specific_heat"] = fN * (e2 - e * e) / (T * T)
    out["susceptibility"] = fN * (m2 - am * am) / T
    out["binder"] = 1.0 - m4 / (3.0 * (m2 * m2)) if m2 > 0.0 else 0.0
    return out


# ------------------------------------------------------------------------------------------------------------
# Error analysis of the per-sweep series ("binning, integrated autocorrelation time").
# The paper's motivation is the autocorrelation time tau ~ |g - g*|^(-z) of local updates near a critical point and
# its reduction by cluster updates (section 1; section 4 validates on time series of E
# and M).  It gives no formulas; the textbook definitions are taken (DESIGN.md 7b lists them as readings):
#
#   series        x_k = E_k / N  (which = 0)  or  |M_k| / N  (which = 1),  k = 0 .. n-1, in sweep order
#   bins          nb = floor(n / B) bins of B consecutive sweeps (a remainder at the END is dropped);
#                 bin mean b_j = (sum of the INTEGER E_k or |M_k| of the bin) / (B N): one division of an exact sum
#   binned error  bbar = (1/nb) sum b_j ;  err = sqrt( sum (b_j - bbar)^2 / (nb (nb - 1)) )
#   autocovariance, with xbar = (1/n) sum x_k:
#                 C(t) = (1/(n - t)) sum_{k=0}^{n-t-1} (x_k - xbar)(x_{k+t} - xbar),   rho(t) = C(t) / C(0)
#   integrated autocorrelation time with the self-consistent window of Madras and Sokal:
#                 tau(W) = 1/2 + sum_{t=1}^{W} rho(t);  W = the smallest W >= 1 with W >= c tau(W) (c = 6 by default),
#                 or tmax if there is none
# Every sum runs in index order in double precision with separate (unfused) operations; a constant series
# (C(0) = 0) has rho = 0 and tau = 1/2 by convention.
# ------------------------------------------------------------------------------------------------------------
from math import sqrt
from typing import List, Tuple


def _ints(E: Sequence[int], M: Sequence[int], which: int) -> List[int]:
    if which == 0:
        return [int(v) for v in E]
    if which == 1:
        return [abs(int(v)) for v in M]
    raise ValueError("which is 0 (energy per site) or 1 (|magnetisation| per site)")


def bin_means(E: Sequence[int], M: Sequence[int], N: int, which: int, B: int) -> List[float]:
    xs = _ints(E, M, which)
    if B < 1:
        raise ValueError("bin length")
    nb = len(xs) // B
    out = []
    for j in range(nb):
        tot = 0
        for k in range(j * B, (j + 1) * B):
            tot += xs[k]                     # exact (Python integers)
        out.append(float(tot) / float(B * N))
    return out


def binned_error(E: Sequence[int], M: Sequence[int], N: int, which: int, B: int) -> Tuple[float, float, int]:
    """(mean of the bin means, its standard error, number of bins); the error is 0 with fewer than two bins."""
    b = bin_means(E, M, N, which, B)
    nb = len(b)
    if nb == 0:
        return 0.0, 0.0, 0
    tot = 0.0
    for v in b:
        tot = tot + v
    bbar = tot / float(nb)
    if nb < 2:
        return bbar, 0.0, nb
    ss = 0.0
    for v in b:
        d = v - bbar
        ss = ss + d * d
    return bbar, sqrt(ss / float(nb * (nb - 1))), nb


def autocovariance(E: Sequence[int], M: Sequence[int], N: int, which: int, tmax: int) -> List[float]:
    """C(0) .. C(tmax) of the series (tmax is clipped to n - 1)."""
    xs = _ints(E, M, which)
    n = len(xs)
    if n == 0:
        raise ValueError("no sweeps")
    fN = float(N)
    x = [float(v) / fN for v in xs]
    tot = 0.0
    for v in x:
        tot = tot + v
    xbar = tot / float(n)
    tmax = min(int(tmax), n - 1)
    out = []
    for t in range(tmax + 1):
        acc = 0.0
        for k in range(n - t):
            acc = acc + (x[k] - xbar) * (x[k + t] - xbar)
        out.append(acc / float(n - t))
    return out


def tau_int(E: Sequence[int], M: Sequence[int], N: int, which: int, tmax: int, c: float = 6.0) -> Tuple[float, int, List[float]]:
    """(tau_int, window W, [rho(0) .. rho(tmax)])."""
    C = autocovariance(E, M, N, which, tmax)
    tmax = len(C) - 1
    if not (C[0] > 0.0):
        return 0.5, 0, [0.0] * (tmax + 1)
    rho = [v / C[0] for v in C]
    tau = 0.5
    for W in range(1, tmax + 1):
        tau = tau + rho[W]
        if float(W) >= c * tau:
            return tau, W, rho
    return tau, tmax, rho
