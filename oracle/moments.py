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
