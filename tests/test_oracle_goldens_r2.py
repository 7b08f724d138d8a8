"""The round-2 oracles as they stand against the worked examples stored by tests/golden/make_oracle_goldens_r2.py (a committed
script that calls only oracle/): guards against accidental change of oracle/phi4_oracle.c and oracle/moments.py.  -m "not gpu"."""
import json
import os

import numpy as np

import oracle
from oracle import moments as om, phi4

G = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "oracle_r2_vectors.json")))


def test_phi4_worked_example():
    g = G["phi4"]
    L, kappa, seed = g["L"], g["kappa"], g["seed"]
    phi = phi4.init(L, seed)
    assert [float(v).hex() for v in phi[0]] == g["start_first_site"]
    for u in g["updates"]:
        phi, r, b, lab, d, i3 = phi4.sweep(L, kappa, seed, u["t"], phi)
        assert [float(v).hex() for v in r] == u["direction"]
        assert b.tolist() == u["bonds"] and lab.tolist() == u["labels"] and list(i3) == u["ints"]
        assert float(d[0]).hex() == u["link"] and [float(v).hex() for v in phi[40]] == u["field_site_40"]


def test_series_analysis_worked_example():
    g = G["series"]
    _, ser = oracle.run(g["L"], g["T"], g["seed"], g["sweeps"])
    E, M, N = ser[:, 0], ser[:, 1], g["L"] ** 2
    assert (int(E[-1]), int(M[-1])) == (g["E_last"], g["M_last"])
    mean, err, nb = om.binned_error(E, M, N, 0, 20)
    assert nb == g["bins20_e"]["n_bins"] and float(mean).hex() == g["bins20_e"]["mean"] and float(err).hex() == g["bins20_e"]["err"]
    tau, W, rho = om.tau_int(E, M, N, 1, 40)
    assert W == g["tau_absm"]["window"] and float(tau).hex() == g["tau_absm"]["tau"] and float(rho[5]).hex() == g["tau_absm"]["rho5"]
