"""Pins for oracle/phi4_oracle.c (the Wolff-type embedded cluster update for the O(4) phi^4 theory in
four dimensions, Eq. 2-3).  -m "not gpu".  Nothing here repeats the oracle's own arithmetic: the direction
is checked against the moments of the uniform distribution on the sphere, Eq. 2 against 1 - exp(-4 kappa s^2) in mpmath on a
constant field, the clusters against scipy on a graph built apart, Eq. 3 against the invariants of a reflection, and the
whole update against a Metropolis simulation of the same Boltzmann weight written with numpy."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy.sparse import coo_matrix
from scipy.sparse.csgraph import connected_components

from oracle import phi4


def _coords(L):
    x = np.arange(L ** 4)
    return np.stack([(x // L ** k) % L for k in range(4)], axis=1)


def _fwd(L, mu):
    c = _coords(L)
    c[:, mu] = (c[:, mu] + 1) % L
    return (c * (L ** np.arange(4))).sum(axis=1)


def test_start_is_deterministic_and_inside_the_cube():
    a, b = phi4.init(3, 5), phi4.init(3, 5)
    assert np.array_equal(a, b) and not np.array_equal(a, phi4.init(3, 6))
    assert a.shape == (81, 4) and np.all(np.abs(a) < 1.0)
    big = phi4.init(8, 1)
    assert abs(big.mean()) < 4.0 / math.sqrt(3.0 * big.size) and abs((big ** 2).mean() - 1.0 / 3.0) < 4.0 * 0.3 / math.sqrt(big.size)


def test_direction_is_a_unit_vector_uniform_on_the_sphere():
    n = 40000
    R = np.array([phi4.direction(77, t)[0] for t in range(n)])
    tries = np.array([phi4.direction(77, t)[1] for t in range(2000)])
    assert np.all(np.abs((R ** 2).sum(axis=1) - 1.0) < 1e-15)
    # uniform on S^3: <r_a> = 0, <r_a r_b> = delta_ab / 4, <r_a^4> = 3 / (4 * 6) = 1/8, <r_a^2 r_b^2> = 1/24
    assert np.all(np.abs(R.mean(axis=0)) < 4.0 * 0.5 / math.sqrt(n))
    C = R.T @ R / n
    assert np.all(np.abs(C - np.eye(4) / 4.0) < 4.0 * 0.25 / math.sqrt(n))
    assert np.all(np.abs((R ** 4).mean(axis=0) - 0.125) < 4.0 * 0.15 / math.sqrt(n))       # a cube-corner bias would show here
    assert abs((R[:, 0] ** 2 * R[:, 1] ** 2).mean() - 1.0 / 24.0) < 4.0 * 0.06 / math.sqrt(n)
    # rejection from the cube to the ball: acceptance pi^2 / 32
    assert abs(1.0 / tries.mean() - math.pi ** 2 / 32.0) < 0.03
    assert not np.array_equal(phi4.direction(77, 0)[0], phi4.direction(78, 0)[0])


@pytest.mark.parametrize("kappa,vec", [(0.304, (0.9, -0.3, 0.5, 0.2)), (0.1, (1.5, 0.0, 0.0, 0.0)), (1.0, (0.2, 0.2, 0.2, 0.2))])
def test_bond_probability_on_a_constant_field_is_equation_2(kappa, vec):
    """phi_x = v everywhere: every link has the same projections, so the bond fraction is 1 - exp(-4 kappa (v.r)^2)."""
    L, seed = 6, 3
    phi = np.tile(np.array(vec, dtype=np.float64), (L ** 4, 1))
    tot, want, nl = 0, 0.0, 0
    for t in range(6):
        r, _ = phi4.direction(seed, t)
        b = phi4.bonds(L, kappa, seed, t, phi, r)
        s = mp.fsum(mp.mpf(float(a)) * mp.mpf(float(c)) for a, c in zip(vec, r))
        p = float(1 - mp.e ** (-4 * mp.mpf(kappa) * s * s))
        k = int(sum(((b >> mu) & 1).sum() for mu in range(4)))
        n = 4 * L ** 4
        assert abs(k - n * p) <= 4.0 * math.sqrt(n * p * (1 - p)) + 1, (t, k, n * p)
        tot += k; want += n * p; nl += n
    assert abs(tot - want) <= 4.0 * math.sqrt(want) + 1


def test_thresholds_closed_forms():
    assert phi4.threshold(0.3, 0.5, -0.5) == 0 and phi4.threshold(0.3, 0.0, 1.0) == 0 and phi4.threshold(0.0, 1.0, 1.0) == 0
    assert phi4.threshold(1e6, 1.0, 1.0) == 2 ** 32 - 1
    for kappa, sx, sy in ((0.304, 0.7, 0.9), (0.25, 1.0, math.log(2.0)), (0.05, 0.01, 0.02)):
        exact = mp.floor((1 - mp.e ** (-4 * mp.mpf(kappa) * mp.mpf(sx) * mp.mpf(sy))) * 2 ** 32)
        assert abs(phi4.threshold(kappa, sx, sy) - int(exact)) <= 1
    assert phi4.threshold(0.25, 1.0, math.log(2.0)) in (2 ** 31 - 1, 2 ** 31)            # p = 1/2
    assert phi4.threshold(0.3, -0.5, -0.8) == phi4.threshold(0.3, 0.5, 0.8)               # the product decides


def test_bonds_only_between_projections_of_one_sign():
    L, kappa, seed = 4, 0.5, 9
    phi = phi4.init(L, seed)
    for t in range(5):
        r, _ = phi4.direction(seed, t)
        b = phi4.bonds(L, kappa, seed, t, phi, r)
        s = phi @ r
        for mu in range(4):
            on = ((b >> mu) & 1).astype(bool)
            assert np.all(s[on] * s[_fwd(L, mu)][on] > 0.0)
        assert np.all(phi4.bonds(L, 0.0, seed, t, phi, r) == 0)
        # kappa -> infinity: every link between projections of one sign
        full = phi4.bonds(L, 1e9, seed, t, phi, r)
        for mu in range(4):
            assert np.array_equal(((full >> mu) & 1).astype(bool), s * s[_fwd(L, mu)] > 1e-12)
    assert b.max() < 16


@pytest.mark.parametrize("L", [2, 3, 4, 5])
def test_clusters_are_the_connected_components(L):
    rng = np.random.default_rng(L)
    V = L ** 4
    for dens in (0.0, 0.1, 0.2, 0.35, 1.0):
        b = np.zeros(V, dtype=np.uint8)
        for mu in range(4):
            b |= ((rng.random(V) < dens).astype(np.uint8) << mu)
        lab = phi4.labels(L, b)
        rows, cols = [], []
        for mu in range(4):
            on = ((b >> mu) & 1).astype(bool)
            rows.append(np.arange(V)[on]); cols.append(_fwd(L, mu)[on])
        rows, cols = np.concatenate(rows), np.concatenate(cols)
        ncomp, comp = connected_components(coo_matrix((np.ones(len(rows)), (rows, cols)), shape=(V, V)), directed=False)
        mins = np.full(ncomp, V); np.minimum.at(mins, comp, np.arange(V))
        assert np.array_equal(lab, mins[comp]), (L, dens)
    # one line of bonds that wraps around the lattice in direction 3
    b = np.zeros(V, dtype=np.uint8); line = np.arange(L) * L ** 3; b[line] = 8
    lab = phi4.labels(L, b)
    assert np.all(lab[line] == 0) and np.count_nonzero(lab == 0) == L


def test_reflection_is_equation_3():
    L, kappa, seed = 4, 0.4, 21
    phi = phi4.init(L, seed)
    nsel = ncl = 0
    for t in range(8):
        new, r, b, lab, d, i3 = phi4.sweep(L, kappa, seed, t, phi)
        sel = np.array([phi4.selected(seed, t, l) for l in lab], dtype=bool)
        s = phi @ r
        # selected sites: reflected in the hyperplane normal to r; the others untouched
        assert np.array_equal(new[~sel], phi[~sel])
        assert np.allclose(new[sel], phi[sel] - 2.0 * s[sel, None] * r[None, :], rtol=0, atol=1e-15)
        assert np.allclose(new[sel] @ r, -s[sel], rtol=0, atol=1e-15)
        assert np.allclose((new ** 2).sum(axis=1), (phi ** 2).sum(axis=1), rtol=1e-14, atol=0)     # |phi_x| is kept
        for mu in range(4):                                  # a reflection is orthogonal: phi_x . phi_y is kept inside a cluster
            on = ((b >> mu) & 1).astype(bool)
            y = _fwd(L, mu)
            assert np.allclose((new[on] * new[y][on]).sum(axis=1), (phi[on] * phi[y][on]).sum(axis=1), rtol=0, atol=1e-14)
            assert np.array_equal(lab[on], lab[y][on])
        roots = np.unique(lab)
        assert np.array_equal(roots, np.nonzero(lab == np.arange(L ** 4))[0]) and i3[0] == len(roots)
        assert i3[1] == np.bincount(lab).max() and i3[2] == sum(int(((b >> mu) & 1).sum()) for mu in range(4))
        nsel += int(sel[roots].sum()); ncl += len(roots)
        link = sum(float((new * new[_fwd(L, mu)]).sum()) for mu in range(4))
        assert abs(d[0] - link) <= 1e-12 * abs(link) and np.allclose(d[1:], new.sum(axis=0), rtol=0, atol=1e-12)
        phi = new
    assert abs(nsel - 0.5 * ncl) <= 4.0 * 0.5 * math.sqrt(ncl)                                     # selected with probability 1/2


def _metropolis_link(L, kappa, rho, sweeps, therm, replicas, seed):
    """Mean link energy <sum_{x,mu} phi_x . phi_{x+mu}> of the weight exp(2 kappa sum phi_x . phi_y) over the DIRECTIONS at fixed
    moduli rho_x: single-site Metropolis with a fresh uniform direction as the proposal, many independent replicas at once."""
    rng = np.random.default_rng(seed)
    V = L ** 4
    nbr = [np.stack([_fwd(L, mu), np.argsort(_fwd(L, mu))], axis=0) for mu in range(4)]     # forward and backward neighbours

    def unit(shape):
        v = rng.standard_normal(shape + (4,))
        return v / np.linalg.norm(v, axis=-1, keepdims=True)

    n = unit((replicas, V))
    phi = n * rho[None, :, None]
    acc = []
    for it in range(therm + sweeps):
        for x in range(V):
            h = np.zeros((replicas, 4))
            for mu in range(4):
                h += phi[:, nbr[mu][0][x]] + phi[:, nbr[mu][1][x]]
            new = unit((replicas,)) * rho[x]
            dS = 2.0 * kappa * ((new - phi[:, x]) * h).sum(axis=1)
            take = np.log(rng.random(replicas)) < dS
            phi[take, x] = new[take]
        if it >= therm:
            acc.append(sum((phi * phi[:, _fwd(L, mu)]).sum(axis=(1, 2)) for mu in range(4)))
    e = np.mean(acc, axis=0)                                 # one number per replica: independent samples
    return e.mean(), e.std(ddof=1) / math.sqrt(replicas)


@pytest.mark.parametrize("L,kappa,moduli", [(2, 0.25, "unit"), (2, 0.5, "unequal"), (3, 0.2, "unit")])
def test_cluster_update_samples_the_o4_weight_at_fixed_moduli(L, kappa, moduli):
    """The update leaves |phi_x| alone and must sample exp(2 kappa sum_links phi_x . phi_y) over the directions (the hopping
    term of the lattice action): the mean link energy against an independent Metropolis simulation, within 4 sigma."""
    V = L ** 4
    rng = np.random.default_rng(100 + L)
    rho = np.ones(V) if moduli == "unit" else 0.5 + 1.5 * rng.random(V)
    # (uniform proposals are accepted rarely where the couplings 2 kappa rho_x rho_y are strong: 400 sweeps to thermalise)
    want, dw = _metropolis_link(L, kappa, rho, sweeps=100 if L == 2 else 60, therm=400, replicas=1200 if L == 2 else 500, seed=L)
    v = rng.standard_normal((V, 4))
    phi = v / np.linalg.norm(v, axis=1, keepdims=True) * rho[:, None]
    n, therm = 60000 if L == 2 else 20000, 500
    out, ser, _ = phi4.run(L, kappa, 42, n + therm, phi=phi)
    assert np.allclose(np.linalg.norm(out, axis=1), rho, rtol=1e-10)
    x = ser[therm:, 0]
    nb = 50
    bins = x[: len(x) // nb * nb].reshape(nb, -1).mean(axis=1)
    got, dg = bins.mean(), bins.std(ddof=1) / math.sqrt(nb)
    assert abs(got - want) <= 4.0 * math.hypot(dg, dw), (got, dg, want, dw)
    assert dg < 0.02 * abs(want) + 0.05 and dw < 0.02 * abs(want) + 0.05       # the comparison is sharp enough to mean something
