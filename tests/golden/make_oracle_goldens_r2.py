"""Writes tests/golden/oracle_r2_vectors.json: small worked examples of the round-2 oracles (phi^4 cluster update, binning /
integrated autocorrelation time), computed by calling ONLY oracle/ -- no value here comes from the CUDA path.  They guard the
oracles against accidental change (tests/test_oracle_goldens_r2.py compares the oracles as they stand with this file); what
the oracles must compute is fixed by the pins of tests/test_oracle_phi4.py and tests/test_oracle_moments.py, not by this file.

    python tests/golden/make_oracle_goldens_r2.py
"""
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import oracle                                   # noqa: E402
from oracle import moments as om, phi4          # noqa: E402


def main():
    out = {"_note": "written by tests/golden/make_oracle_goldens_r2.py from oracle/ alone; doubles as hex strings (bit patterns)"}
    # phi^4: L = 3, kappa = 0.304, seed 11 (readings: DESIGN.md 7e)
    L, kappa, seed = 3, 0.304, 11
    phi = phi4.init(L, seed)
    out["phi4"] = {"L": L, "kappa": kappa, "seed": seed, "start_first_site": [float(v).hex() for v in phi[0]], "updates": []}
    for t in range(3):
        phi, r, b, lab, d, i3 = phi4.sweep(L, kappa, seed, t, phi)
        out["phi4"]["updates"].append({"t": t, "direction": [float(v).hex() for v in r], "bonds": b.tolist(), "labels": lab.tolist(),
                                       "link": float(d[0]).hex(), "ints": list(i3), "field_site_40": [float(v).hex() for v in phi[40]]})
    # error analysis of the L = 16 Ising series at T = 2.269, seed 5, 300 sweeps (readings: DESIGN.md 7b)
    Li, T, sd, n = 16, 2.269, 5, 300
    _, ser = oracle.run(Li, T, sd, n)
    E, M, N = ser[:, 0], ser[:, 1], Li * Li
    mean, err, nb = om.binned_error(E, M, N, 0, 20)
    tau, W, rho = om.tau_int(E, M, N, 1, 40)
    out["series"] = {"L": Li, "T": T, "seed": sd, "sweeps": n, "E_last": int(E[-1]), "M_last": int(M[-1]),
                     "bins20_e": {"n_bins": nb, "mean": float(mean).hex(), "err": float(err).hex()},
                     "tau_absm": {"tau": float(tau).hex(), "window": int(W), "rho5": float(rho[5]).hex()}}
    p = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_r2_vectors.json")
    with open(p, "w") as f:
        json.dump(out, f, indent=1)
    print("wrote", p)


if __name__ == "__main__":
    main()
