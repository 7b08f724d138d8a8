"""GPU <-> oracle parity for the second workload (-m gpu): the Wolff-type embedded cluster update for O(4) phi^4 in four
dimensions (Eq. 2-3) through the C ABI of include/phi4.h against
oracle/phi4_oracle.c on the same seeds.  Bar: direction, bond bytes, labels and the FIELD bit for bit after every update
(every floating-point operation on the path is a separately rounded IEEE operation in the oracle's order; the one library
function, expm1, only feeds an integer threshold); integer observables equal; the double sums (link, magnetisation) within
1e-12 of the sum of the magnitudes of their terms (the device adds in a tree, the oracle in index order).
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from oracle import phi4 as o4


@pytest.fixture(scope="module")
def P():
    from paper_2302_14720_b200 import phi4
    phi4.lib()
    return phi4


def _check_sums(L, phi, obs, d):
    V = L ** 4
    scale_link = 4.0 * float((np.linalg.norm(phi, axis=1) ** 2).sum())       # >= sum of |terms| (Cauchy-Schwarz)
    assert abs(obs.link - d[0]) <= 1e-12 * scale_link
    for a in range(4):
        assert abs(obs.m[a] - d[1 + a]) <= 1e-12 * float(np.abs(phi[:, a]).sum())
    assert obs.link_per_link == obs.link / (4.0 * V)
    assert abs(obs.abs_m_per_site - math.sqrt(sum(obs.m[a] ** 2 for a in range(4))) / V) <= 1e-15


def _compare(P, L, kappa, seed, n, start=None, t0=0):
    g = P.Phi4(L, kappa, seed)
    if start is None:
        phi = o4.init(L, seed)
        assert np.array_equal(g.field_host(), phi), "start differs"
    else:
        phi = np.array(start, dtype=np.float64)
        g.set_field(phi)
    if t0:
        g.set_sweep_index(t0)
    o = g.observables()
    d0, _ = o4.observables(L, phi)
    _check_sums(L, phi, o, d0)
    assert o.ints() == (0, 0, 0) and o.sweep == t0
    for k in range(n):
        t = t0 + k
        new, r, b, lab, d, i3 = o4.sweep(L, kappa, seed, t, phi)
        g.sweep(1)
        assert np.array_equal(g.direction(), r), f"direction differs at update {t}"
        assert np.array_equal(g.bonds_host(), b), f"bonds differ at update {t}"
        assert np.array_equal(g.labels_host(), lab), f"labels differ at update {t}"
        assert np.array_equal(g.field_host(), new), f"field differs at update {t}"
        o = g.observables()
        assert o.ints() == i3 and o.sweep == t + 1, (o.ints(), i3)
        _check_sums(L, new, o, d)
        phi = new
    g.close()


@pytest.mark.parametrize("L", [2, 3, 4, 5, 6, 8])
def test_every_update_matches_the_oracle(P, L):
    for kappa, seed in ((0.1, 1), (0.304, 2), (0.6, 3)):
        _compare(P, L, kappa, seed + L, 6)


def test_paper_size_one_update_at_a_time(P):
    """L = 16 at kappa = 0.304 (Fig. 9): the paper's smallest timed lattice."""
    _compare(P, 16, 0.304, 7, 4)


def test_special_fields_and_limits(P):
    L = 4
    V = L ** 4
    rng = np.random.default_rng(5)
    ordered = np.tile(np.array([0.8, 0.1, -0.3, 0.5]), (V, 1))
    staggered = ordered * (1.0 - 2.0 * (np.indices((L,) * 4).sum(axis=0).reshape(-1) % 2))[:, None]
    big = 30.0 * rng.standard_normal((V, 4))
    zero = np.zeros((V, 4))
    for f in (ordered, staggered, big, zero):
        for kappa in (0.0, 0.304, 50.0):
            _compare(P, L, kappa, 11, 2, start=f)
    _compare(P, 4, 0.304, 12, 2, t0=(1 << 32) + 5)           # 64-bit sweep index


@pytest.mark.parametrize("L,n", [(4, 40), (6, 25), (8, 13)])
def test_many_updates_per_call_with_and_without_graphs(P, L, n):
    kappa, seed = 0.304, 50 + L
    ref, ser, iser = o4.run(L, kappa, seed, n)
    for graphs in (True, False):
        g = P.Phi4(L, kappa, seed)
        g.set_graphs(graphs)
        g.sweep(n)
        assert np.array_equal(g.field_host(), ref), f"field differs (graphs={graphs})"
        got = g.series()
        assert len(got) == n
        for k in range(n):
            assert got[k].ints() == tuple(int(v) for v in iser[k]) and got[k].sweep == k + 1
            assert abs(got[k].link - ser[k, 0]) <= 1e-12 * 4.0 * float((ref ** 2).sum())
        # a second call continues the same chain
        g.sweep(5)
        ref2, _, iser2 = o4.run(L, kappa, seed, 5, phi=ref, t0=n)
        assert np.array_equal(g.field_host(), ref2) and g.observables().ints() == tuple(int(v) for v in iser2[-1])
        assert g.sweep_index == n + 5 and g.launch_count() > 0
        g.close()


def test_update_is_reproducible_whatever_the_race_order(P):
    L, kappa, seed = 8, 0.304, 3
    g = P.Phi4(L, kappa, seed)
    g.sweep(5)
    f5 = g.field_host()
    ref = None
    for rep in range(4):
        g.set_field(f5); g.set_sweep_index(5); g.sweep(1)
        cur = (g.field_host(), g.labels_host(), g.observables().doubles(), g.observables().ints())
        if ref is None:
            ref = cur
        assert np.array_equal(cur[0], ref[0]) and np.array_equal(cur[1], ref[1]) and cur[2] == ref[2] and cur[3] == ref[3]
    g.close()


def test_moduli_are_kept_and_the_o4_weight_is_sampled_on_the_gpu(P):
    """The CUDA path against the physics without the oracle in between: unit moduli on a 2^4 lattice at kappa = 0.25, the
    mean link energy against a numpy Metropolis simulation of exp(2 kappa sum phi_x . phi_y) (tests/test_oracle_phi4.py)."""
    import test_oracle_phi4 as T
    L, kappa = 2, 0.25
    V = L ** 4
    want, dw = T._metropolis_link(L, kappa, np.ones(V), sweeps=100, therm=400, replicas=1200, seed=9)
    rng = np.random.default_rng(4)
    v = rng.standard_normal((V, 4))
    g = P.Phi4(L, kappa, 77)
    g.set_field(v / np.linalg.norm(v, axis=1, keepdims=True))
    g.sweep(500)
    tot = []
    for _ in range(15):
        g.sweep(4000)
        tot.append(np.mean([o.link for o in g.series()]))
    assert np.allclose(np.linalg.norm(g.field_host(), axis=1), 1.0, rtol=1e-10)
    got, dg = float(np.mean(tot)), float(np.std(tot, ddof=1) / math.sqrt(len(tot)))
    assert abs(got - want) <= 4.0 * math.hypot(dg, dw), (got, dg, want, dw)
    g.close()


def test_argument_errors(P):
    for L, kappa in ((1, 0.3), (129, 0.3), (4, -0.1), (4, float("nan"))):
        assert not P.lib().phi4_create(L, kappa, 1)
    g = P.Phi4(4, 0.3, 1)
    with pytest.raises(P.Phi4Error):
        g.labels_host()
    with pytest.raises(P.Phi4Error):
        g.direction()
    with pytest.raises(P.Phi4Error):
        g.sweep(-1)
    g.sweep(0)
    g.close()
    P.lib().phi4_destroy(None)
