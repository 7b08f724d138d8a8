"""GPU <-> oracle parity (-m gpu): the CUDA path through the C ABI against the serial oracle, element by
element on the same seeded inputs.  Bar (north_star): bit-exact spins, bond planes, labels and integer
observables after every sweep; double observables within 1e-12 relative.
"""
import math

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
import invariants as inv
from paper_2302_14720_b200 import workloads as wl

T_C = wl.T_C


@pytest.fixture(scope="module")
def B():
    from paper_2302_14720_b200 import binding
    binding.lib()
    return binding


def _obs_tuple(o):
    return (o.energy, o.magnetisation, o.n_clusters, o.largest_cluster)


def _check_double_obs(o, N):
    e = o.energy / N
    m = abs(o.magnetisation) / N
    assert abs(o.e_per_site - e) <= 1e-12 * max(1.0, abs(e))
    assert abs(o.abs_m_per_site - m) <= 1e-12 * max(1.0, abs(m))


def _compare_sweeps(B, L, T, seed, n, path=0, start=None, t0=0, every=1):
    """n sweeps on the GPU, one at a time, each compared in full with the oracle."""
    sw = B.SwendsenWang(L, T, seed, path=path)
    N = L * L
    if start is None:
        s = oracle.init_random(L, seed)
        assert np.array_equal(sw.spins_host()[0], s), "random start differs"
    else:
        s = np.asarray(start, dtype=np.int8)
        sw.set_spins(s)
    if t0:
        sw.set_sweep_index(t0)
    assert sw.threshold() == oracle.threshold(T)
    for k in range(n):
        t = t0 + k
        s1, bE, bS, lab, obs = oracle.sweep(L, T, seed, t, s)
        sw.sweep(1)
        if k % every == 0 or k == n - 1:
            gE, gS = sw.bonds_host()
            assert np.array_equal(gE[0], wl.pack_bits(bE)), f"bondE differs at sweep {t}"
            assert np.array_equal(gS[0], wl.pack_bits(bS)), f"bondS differs at sweep {t}"
            assert np.array_equal(sw.labels_host()[0], lab), f"labels differ at sweep {t}"
            assert np.array_equal(sw.spins_host()[0], s1), f"spins differ at sweep {t}"
            o = sw.observables()[0]
            assert _obs_tuple(o) == obs, f"observables differ at sweep {t}: {_obs_tuple(o)} vs {obs}"
            assert o.sweep == t + 1
            _check_double_obs(o, N)
        s = s1
    sw.close()


# ------------------------------------------------------------------------------------------------
def test_philox_on_device_matches_oracle_and_known_answers(B):
    rng = np.random.default_rng(1)
    ctr = rng.integers(0, 2 ** 32, size=(4096, 4), dtype=np.uint64).astype(np.uint32)
    key = rng.integers(0, 2 ** 32, size=(4096, 2), dtype=np.uint64).astype(np.uint32)
    ctr[0] = 0; key[0] = 0
    ctr[1] = 0xFFFFFFFF; key[1] = 0xFFFFFFFF
    ctr[2] = [0x243f6a88, 0x85a308d3, 0x13198a2e, 0x03707344]; key[2] = [0xa4093822, 0x299f31d0]
    out = B.sw_test_philox(ctr, key)
    assert out[0].tolist() == [0x6627e8d5, 0xe169c58d, 0xbc57ac4c, 0x9b00dbd8]
    assert out[1].tolist() == [0x408f276d, 0x41c83b0e, 0xa20bc7c6, 0x6d5451fd]
    assert out[2].tolist() == [0xd16cfe09, 0x94fdcceb, 0x5001e420, 0x24126ea1]
    for i in range(0, 4096, 37):
        assert out[i].tolist() == oracle.philox4x32_10(ctr[i], key[i]).tolist()


def test_thresholds_match_oracle(B):
    for T in (0.05, 1.5, 2.0, 2.269, 2.26919, T_C, 2.5, 3.0, 3.5, 10.0, 1e6, 1e12):
        sw = B.SwendsenWang(8, T, 1)
        assert sw.threshold() == oracle.threshold(T)
        sw.close()


@pytest.mark.parametrize("L", [2, 3, 4, 5, 8, 13, 31, 33, 64, 100])
def test_generic_path_every_sweep(B, L):
    for T, seed in ((1.5, 7), (T_C, 8), (3.5, 9)):
        _compare_sweeps(B, L, T, seed + L, 8, path=1)


@pytest.mark.parametrize("L,path", [(64, 0), (128, 0), (192, 0), (256, 0), (320, 0), (512, 0), (384, 0), (512, 6), (768, 0),
                                    (128, 6), (192, 6), (1024, 0), (640, 0)])
def test_tiled_path_every_sweep(B, L, path):
    for T, seed in ((2.0, 1), (T_C, 2), (3.0, 3)):
        _compare_sweeps(B, L, T, seed + L, 6, path=path)


# the bond threshold at its ends: T = 1e11 -> threshold 0 (no bond at all), T = 1e9 -> 8, T = 0.01 -> 2^32 - 1 (the draw bits
# come out of the carry of word + (2^32 - threshold), k_bond_label); both tile shapes, the cluster kernel and the generic path
@pytest.mark.parametrize("L,path", [(64, 0), (128, 0), (256, 0), (2048, 0), (20, 1)])
def test_bond_threshold_at_its_ends(B, L, path):
    for T in (1e11, 1e9, 0.01):
        assert oracle.threshold(T) == {1e11: 0, 1e9: 8, 0.01: 2 ** 32 - 1}[T]
        _compare_sweeps(B, L, T, 40 + L, 2, path=path)
        _compare_sweeps(B, L, T, 41 + L, 2, path=path, start=np.ones(L * L, dtype=np.int8))


def test_config1_L64_many_sweeps(B):
    # BASELINE configs[0]: L = 64, T = 2.26919, seed 2024 -- every one of the 1000 sweeps, in full
    _compare_sweeps(B, 64, wl.T_C_PRINTED, 2024, 1000)


def test_survey_golden_vector_on_gpu(B):
    sw = B.SwendsenWang(4, 2.269, 12345)
    assert "".join("+" if v > 0 else "-" for v in sw.spins_host()[0]) == "+------+-+++++--"
    sw.sweep(1)
    assert sw.labels_host()[0].tolist() == [0, 1, 2, 2, 4, 4, 4, 7, 4, 0, 7, 7, 0, 0, 2, 2]
    assert _obs_tuple(sw.observables()[0]) == (-16, -10, 5, 4)
    sw.sweep(2)
    assert _obs_tuple(sw.observables()[0]) == (-16, -10, 4, 11)
    assert sw.series()[:, 0, :].tolist() == [[-20, -12, 5, 10], [-16, -10, 4, 11]]
    sw.close()


@pytest.mark.parametrize("L,path", [(64, 0), (256, 0), (100, 1), (128, 0), (256, 6), (192, 0)])
def test_special_starts(B, L, path):
    for name, s0 in (("cold", wl.spins_cold(L)), ("down", wl.spins_all_down(L)),
                     ("checker", wl.spins_checkerboard(L)), ("hstripes", wl.spins_stripes(L, 1)),
                     ("vstripes", wl.spins_stripes(L, 1, vertical=True)), ("blocks", wl.spins_blocks(L, 24)),
                     ("wide", wl.spins_stripes(L, 5))):
        for T in (0.05, T_C, 1e12):      # all bonds / critical / no bonds
            _compare_sweeps(B, L, T, 5, 2, path=path, start=s0)


def _label_patterns(L):
    yield "none", wl.bonds_none(L)
    yield "all", wl.bonds_all(L)
    yield "row_wrap", wl.bonds_row_wrap(L, L - 1)
    yield "col_wrap", wl.bonds_col_wrap(L, L - 1)
    yield "row0", wl.bonds_row_wrap(L, 0)
    yield "comb", wl.bonds_comb(L)
    yield "spiral", wl.bonds_spiral(L)
    yield "ladder", wl.bonds_ladder(L)
    yield "u_shapes", wl.bonds_u_shapes(L)
    yield "ladder3", wl.bonds_ladder(L, 3, 0)
    yield "dense_meetings", wl.bonds_dense_meetings(L, L)
    for k, d in enumerate((0.2, 0.45, 0.5, 0.55, 0.8)):
        yield f"random{d}", wl.bonds_random(L, 7 * L + k, d)


@pytest.mark.parametrize("L,path", [(64, 0), (128, 0), (256, 0), (320, 0), (100, 1), (512, 0), (192, 6), (1152, 0), (2048, 0)])
def test_labelling_of_injected_bond_graphs(B, L, path):
    """Labelling alone on adversarial bond graphs (long thin spiral, comb, wrap-around rows)."""
    sw = B.SwendsenWang(L, 2.0, 1, path=path)
    for name, (bE, bS) in _label_patterns(L):
        got = B.sw_test_label(sw.h, wl.pack_bits(bE), wl.pack_bits(bS))
        ref = oracle.labels(L, bE, bS)
        assert np.array_equal(got, ref), f"{name}: {np.count_nonzero(got != ref)} labels differ"
    sw.close()


@pytest.mark.parametrize("L,nb", [(2048, 1), (2048, 2)])
def test_assignment_kernel_with_and_without_tma_staging(B, L, nb):
    """k_flip16_tma (16-bit root plane staged by cp.async.bulk.tensor boxes, persistent CTAs) against the oracle, and the
    direct-load kernel on the same handle: identical spins and observables, every sweep."""
    Ts, seeds = [T_C, 2.0, 3.0][:nb], [71, 72, 73][:nb]
    sw = B.SwendsenWang(L, Ts, seeds)
    refs = [oracle.init_random(L, s) for s in seeds]
    for t in range(6):
        B.sw_set_tma(sw.h, t % 2 == 0)
        sw.sweep(1)
        gs, obs = sw.spins_host(), sw.observables()
        for b in range(nb):
            s1, _, _, _, o = oracle.sweep(L, Ts[b], seeds[b], t, refs[b])
            assert np.array_equal(gs[b], s1), (t, b)
            assert _obs_tuple(obs[b]) == o, (t, b)
            refs[b] = s1
    # many sweeps in one call (graph replay) on either kernel
    for on in (True, False):
        B.sw_set_tma(sw.h, on)
        t0 = sw.sweep_index
        sw.sweep(9)
        gs = sw.spins_host()
        for b in range(nb):
            refs[b], _ = oracle.run(L, Ts[b], seeds[b], 9, spins=refs[b], t0=t0, series=False)
            assert np.array_equal(gs[b], refs[b]), (on, b)
    sw.close()


def test_labels_of_a_sweep_survive_a_path_switch(B):
    """sw_labels flattens the 16-bit roots of the LAST sweep with the tile shape that wrote them, whatever path is selected
    afterwards (sw_set_path between the sweep and the first sw_labels call)."""
    L, T, seed = 256, T_C, 19
    for new_path in (1, 6, 11):
        sw = B.SwendsenWang(L, T, seed)
        s = oracle.init_random(L, seed)
        for t in range(3):
            s, _, _, lab, _ = oracle.sweep(L, T, seed, t, s)
        sw.sweep(3)
        B.sw_set_path(sw.h, new_path)
        assert np.array_equal(sw.labels_host()[0], lab), new_path
        sw.sweep(1)                                   # and the chain goes on, on the new path
        s, _, _, lab, o = oracle.sweep(L, T, seed, 3, s)
        assert np.array_equal(sw.labels_host()[0], lab) and np.array_equal(sw.spins_host()[0], s)
        assert _obs_tuple(sw.observables()[0]) == o
        sw.close()


def test_series_through_the_raw_c_call_with_a_batch(B):
    """include/sw.h: `cap` of sw_series counts SWEEPS; the caller's buffer holds cap * nb records."""
    import ctypes
    L, Ts, seeds, n = 64, [2.0, T_C, 3.0], [5, 6, 7], 9
    sw = B.SwendsenWang(L, Ts, seeds)
    sw.sweep(n)
    cap = 4                                           # fewer sweeps than retained: only cap * nb records may be written
    buf = (B.sw_obs * (cap * 3 + 1))()
    buf[cap * 3].energy = 123456789
    kept = B.lib().sw_series(sw.h, buf, cap)
    assert kept == n and buf[cap * 3].energy == 123456789
    for b in range(3):
        _, ser = oracle.run(L, Ts[b], seeds[b], n)
        for k in range(cap):
            r = buf[k * 3 + b]
            assert (r.energy, r.magnetisation, r.n_clusters, r.largest_cluster) == tuple(int(v) for v in ser[k]) and r.sweep == k + 1
    sw.close()


def test_handle_on_a_device_that_is_not_current(B):
    """A handle lives on the device it was created on; every call switches to it (needs two GPUs)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("one GPU")
    L, T, seed = 256, T_C, 3
    sw = B.SwendsenWang(L, T, seed, device="cuda:1")
    torch.cuda.set_device(0)
    s = oracle.init_random(L, seed)
    for t in range(3):
        s, _, _, lab, o = oracle.sweep(L, T, seed, t, s)
        sw.sweep(1)
    assert np.array_equal(sw.spins_host()[0], s) and np.array_equal(sw.labels_host()[0], lab) and _obs_tuple(sw.observables()[0]) == o
    sw.close()


def test_random_sizes_temperatures_and_seeds(B):
    """A sweep of (L, T, seed) drawn from a fixed generator over both tile shapes and the generic path: every sweep in full."""
    rng = np.random.default_rng(20260511)
    sides = [64, 128, 192, 256, 320, 384, 448, 576, 704, 1088, 1152, 1280, 96, 160, 40]
    for k in range(18):
        L = int(sides[k % len(sides)])
        T = float(rng.choice([0.9, 1.6, 2.1, T_C, 2.4, 2.9, 4.5, 9.0]))
        seed = int(rng.integers(1, 2 ** 62))
        _compare_sweeps(B, L, T, seed, 4 if L < 1000 else 3)


def test_race_order_independence(B):
    """Same state, same sweep index, repeated: identical bits every time (min-index labels)."""
    L, T, seed = 512, T_C, 3
    sw = B.SwendsenWang(L, T, seed)
    sw.sweep(5)
    s5 = sw.spins_host().copy()
    ref = None
    for rep in range(5):
        sw.set_spins(s5)
        sw.set_sweep_index(5)
        sw.sweep(1)
        cur = (sw.labels_host().copy(), sw.spins_host().copy(), _obs_tuple(sw.observables()[0]))
        if ref is None:
            ref = cur
        assert np.array_equal(cur[0], ref[0]) and np.array_equal(cur[1], ref[1]) and cur[2] == ref[2]
    sw.close()


def test_multi_sweep_call_equals_single_sweeps_and_series(B):
    L, T, seed, n = 128, T_C, 11, 40
    _, ser = oracle.run(L, T, seed, n)
    sw = B.SwendsenWang(L, T, seed)
    sw.sweep(n)
    got = sw.series()
    assert got.shape == (n, 1, 4) and np.array_equal(got[:, 0, :], ser)
    assert _obs_tuple(sw.observables()[0]) == tuple(ser[-1])
    sfin, _ = oracle.run(L, T, seed, n, series=False)
    assert np.array_equal(sw.spins_host()[0], sfin)
    sw.close()


def test_series_ring_keeps_the_last_sweeps(B):
    L, T, seed, n, cap = 64, 2.5, 4, 50, 16
    _, ser = oracle.run(L, T, seed, n)
    sw = B.SwendsenWang(L, T, seed)
    B.sw_set_series_capacity(sw.h, cap)
    sw.sweep(n)
    got = sw.series()
    assert got.shape == (cap, 1, 4) and np.array_equal(got[:, 0, :], ser[-cap:])
    sw.close()


def test_batch_of_independent_lattices(B):
    """BASELINE configs[4] in small: several temperatures and seeds in one launch per stage."""
    L, Ts, seeds, n = 256, [1.5, T_C, 3.5, 2.0], [1000, 1012, 1031, 5], 12
    sw = B.SwendsenWang(L, Ts, seeds)
    refs = [oracle.init_random(L, s) for s in seeds]
    got0 = sw.spins_host()
    for b in range(len(Ts)):
        assert np.array_equal(got0[b], refs[b])
        assert sw.threshold(b) == oracle.threshold(Ts[b])
    for t in range(n):
        sw.sweep(1)
        gs, gl = sw.spins_host(), sw.labels_host()
        gE, gS = sw.bonds_host()
        obs = sw.observables()
        for b in range(len(Ts)):
            s1, bE, bS, lab, o = oracle.sweep(L, Ts[b], seeds[b], t, refs[b])
            assert np.array_equal(gE[b], wl.pack_bits(bE)) and np.array_equal(gS[b], wl.pack_bits(bS))
            assert np.array_equal(gl[b], lab) and np.array_equal(gs[b], s1)
            assert _obs_tuple(obs[b]) == o
            refs[b] = s1
    sw.close()


def test_batch_generic_path_odd_side(B):
    L, Ts, seeds = 27, [2.0, T_C, 3.0], [1, 2, 3]
    sw = B.SwendsenWang(L, Ts, seeds)
    refs = [oracle.init_random(L, s) for s in seeds]
    for t in range(6):
        sw.sweep(1)
        gs, gl = sw.spins_host(), sw.labels_host()
        obs = sw.observables()
        for b in range(3):
            s1, bE, bS, lab, o = oracle.sweep(L, Ts[b], seeds[b], t, refs[b])
            assert np.array_equal(gl[b], lab) and np.array_equal(gs[b], s1) and _obs_tuple(obs[b]) == o
            refs[b] = s1
    sw.close()


def test_resume_from_checkpoint(B):
    L, T, seed = 192, T_C, 21
    a = B.SwendsenWang(L, T, seed)
    a.sweep(7)
    s7 = a.spins_host().copy()
    a.sweep(5)
    b = B.SwendsenWang(L, T, seed)
    b.set_spins(s7)
    b.set_sweep_index(7)
    b.sweep(5)
    assert np.array_equal(a.spins_host(), b.spins_host()) and a.sweep_index == b.sweep_index == 12
    assert _obs_tuple(a.observables()[0]) == _obs_tuple(b.observables()[0])
    # 64-bit sweep index reaches the counter's third word
    t_big = (1 << 32) + 3
    b.set_spins(s7); b.set_sweep_index(t_big); b.sweep(1)
    s1, *_ , o = oracle.sweep(L, T, seed, t_big, s7[0])
    assert np.array_equal(b.spins_host()[0], s1) and _obs_tuple(b.observables()[0]) == o
    a.close(); b.close()


def test_observables_before_any_sweep_and_after_set_spins(B):
    L = 96
    sw = B.SwendsenWang(L, 2.0, 5, path=1)
    s = oracle.init_random(L, 5)
    o = sw.observables()[0]
    E, M, _, _ = oracle.observables(L, s)
    assert (o.energy, o.magnetisation, o.n_clusters, o.largest_cluster, o.sweep) == (E, M, 0, 0, 0)
    sw.set_cold()
    o = sw.observables()[0]
    assert (o.energy, o.magnetisation) == (-2 * L * L, L * L) and o.e_per_site == -2.0 and o.abs_m_per_site == 1.0
    with pytest.raises(B.SwError):
        sw.labels()
    with pytest.raises(B.SwError):
        sw.bonds()
    sw.close()


def test_argument_errors(B):
    for bad in ((1, 2.0), (0, 2.0), (32769, 2.0), (8, 0.0), (8, -1.0), (8, float("nan")), (8, float("inf"))):
        with pytest.raises(B.SwError):
            B.sw_create(bad[0], bad[1], 1)
    assert B.sw_workspace_bytes(1, 1) == 0 and B.sw_workspace_bytes(8, 0) == 0
    h = B.sw_create(8, 2.0, 1)
    with pytest.raises(B.SwError):
        B.sw_sweep(h, -1)
    B.sw_sweep(h, 0)
    B.sw_destroy(h)
    B.sw_destroy(None)


# ---- one-step parity at the sizes the bench times ----------------------------------
def _one_step(B, sw, L, T, seed):
    t = sw.sweep_index
    s = sw.spins_host()[0].copy()
    sw.sweep(1)
    s1, bE, bS, lab, obs = oracle.sweep(L, T, seed, t, s)
    gE, gS = sw.bonds_host()
    assert np.array_equal(gE[0], wl.pack_bits(bE)) and np.array_equal(gS[0], wl.pack_bits(bS))
    assert np.array_equal(sw.labels_host()[0], lab)
    assert np.array_equal(sw.spins_host()[0], s1)
    o = sw.observables()[0]
    assert _obs_tuple(o) == obs
    _check_double_obs(o, L * L)


@pytest.mark.parametrize("L,T,seed,start", [(1024, 2.0, 1, "random"), (1024, wl.T_C_PRINTED, 2, "random"),
                                            (1024, 3.0, 3, "random"), (2048, T_C, 1012, "random"),
                                            (4096, T_C, 4, "cold"), (4096, T_C, 5, "random")])
def test_one_step_parity_configs_2_3_5(B, L, T, seed, start):
    sw = B.SwendsenWang(L, T, seed)
    if start == "cold":
        sw.set_cold()
    _one_step(B, sw, L, T, seed)          # t = 0
    _one_step(B, sw, L, T, seed)          # t = 1
    sw.sweep(30)
    _one_step(B, sw, L, T, seed)          # t = 32, after the clusters have grown
    sw.close()


def test_one_step_parity_headline_L16384(B):
    """BASELINE configs[3]: L = 16384, T_c, seed 6 -- in the launch configuration bench.py times."""
    L, T, seed = 16384, T_C, 6
    sw = B.SwendsenWang(L, T, seed)
    for t in (0, 1, 2, 100, 199):         # the random start, then the state the bench times
        sw.sweep(t - sw.sweep_index)
        _one_step(B, sw, L, T, seed)
    sw.close()


def test_one_step_parity_headline_cold_start(B):
    """L = 16384 from the cold start: the first sweep's bonds percolate (p = 0.586 per edge): one cluster holds most
    sites, every tile has ~100 open roots hanging under one node."""
    L, T, seed = 16384, T_C, 6
    sw = B.SwendsenWang(L, T, seed)
    sw.set_cold()
    _one_step(B, sw, L, T, seed)          # t = 0
    _one_step(B, sw, L, T, seed)          # t = 1
    sw.close()


def test_one_step_parity_at_the_largest_side(B):
    """SW_MAX_L = 32768: N = 2^30, the int32 edge the ABI advertises (labels up to 2^30 - 1, 32-bit word and site
    indices in every kernel)."""
    L, T, seed = 32768, T_C, 9
    sw = B.SwendsenWang(L, T, seed)
    _one_step(B, sw, L, T, seed)          # t = 0
    sw.close()


def test_config2_every_sweep(B):
    """BASELINE configs[1]: L = 1024, T in {2.0, 2.26919, 3.0}, seeds 1, 2, 3 -- the first 200 sweeps, each in full."""
    for T, seed in ((2.0, 1), (wl.T_C_PRINTED, 2), (3.0, 3)):
        _compare_sweeps(B, 1024, T, seed, 200)


@pytest.mark.parametrize("seed,start", [(4, "cold"), (5, "random")])
def test_config3_sweeps_0_to_9_then_every_100th(B, seed, start):
    """BASELINE configs[2]: L = 4096, T_c, 1000 sweeps -- sweeps 0 .. 9 in full, then one-step parity at every 100th."""
    L, T = 4096, T_C
    sw = B.SwendsenWang(L, T, seed)
    if start == "cold":
        sw.set_cold()
    for t in list(range(10)) + list(range(100, 1001, 100)):
        sw.sweep(t - sw.sweep_index)
        _one_step(B, sw, L, T, seed)
    sw.close()


def test_config5_at_size(B):
    """BASELINE configs[4]: 32 lattices of L = 2048, T_b = 1.5 + 2 b / 31, seeds 1000 + b, one launch per stage for the
    batch.  Lattices b = 0, 12, 31 against three oracle runs, every sweep for 20 sweeps, then one step after 200."""
    L, nb = 2048, 32
    Ts, seeds = wl.scan_temperatures(nb), [1000 + b for b in range(nb)]
    sw = B.SwendsenWang(L, Ts, seeds)
    pick = (0, 12, 31)
    ref = {b: oracle.init_random(L, seeds[b]) for b in pick}
    g0 = sw.spins()
    for b in pick:
        assert np.array_equal(g0[b].cpu().numpy().reshape(-1), ref[b])

    def check(t):
        before = {b: ref[b] for b in pick}
        sw.sweep(1)
        gs, gl = sw.spins(), sw.labels()
        gE, gS = sw.bonds()
        obs = sw.observables()
        for b in pick:
            s1, bE, bS, lab, o = oracle.sweep(L, Ts[b], seeds[b], t, before[b])
            assert np.array_equal(gE[b].cpu().numpy().view(np.uint32), wl.pack_bits(bE)), (b, t)
            assert np.array_equal(gS[b].cpu().numpy().view(np.uint32), wl.pack_bits(bS)), (b, t)
            assert np.array_equal(gl[b].cpu().numpy().reshape(-1), lab), (b, t)
            assert np.array_equal(gs[b].cpu().numpy().reshape(-1), s1), (b, t)
            assert _obs_tuple(obs[b]) == o, (b, t)
            ref[b] = s1

    for t in range(20):
        check(t)
    sw.sweep(180)
    g = sw.spins()
    for b in pick:
        ref[b] = g[b].cpu().numpy().reshape(-1).copy()
    check(200)
    sw.close()


def test_invariants_hold_at_size_without_the_oracle(B):
    """Properties that hold at any size, checked with numpy/scipy only (L = 2048 after 50 sweeps)."""
    L, T, seed = 2048, T_C, 77
    sw = B.SwendsenWang(L, T, seed)
    sw.sweep(50)
    before = sw.spins_host()[0].copy()
    sw.sweep(1)
    gE, gS = sw.bonds_host()
    bE, bS = wl.unpack_bits(gE[0], L * L), wl.unpack_bits(gS[0], L * L)
    o = sw.observables()[0]
    inv.check_sweep(L, before, bE, bS, sw.labels_host()[0], sw.spins_host()[0], _obs_tuple(o))
    sw.close()


# ------------------------------------------------------------------------------------------------
# moments accumulated on the device against oracle/moments.py on the oracle's series
@pytest.mark.parametrize("L,path,T", [(64, 0, T_C), (256, 0, 2.0), (128, 0, 3.0), (20, 1, T_C), (192, 0, T_C), (256, 6, 2.5)])
def test_moments_match_oracle(B, L, path, T):
    from oracle import moments as om
    seed, therm, n = 31 + L, 7, 40
    N = L * L
    sw = B.SwendsenWang(L, T, seed, path=path)
    assert sw.moments()[0]["n"] == 0
    sw.sweep(therm)
    sw.moments_reset()                               # discard thermalisation
    sw.sweep(25)                                     # several calls: the scan path closes each with its own pass
    sw.sweep(1)
    sw.sweep(n - 26)
    got = sw.moments()[0]
    _, ser = oracle.run(L, T, seed, therm + n)
    ref = om.moments(ser[therm:, 0], ser[therm:, 1], N, T)
    assert got["n"] == n
    # the device adds the same doubles in the same order with unfused operations: the means are the oracle's to the
    # last bit, and so are the derived quantities (same formula on the same doubles); the bar is north_star's 1e-12
    for k in ("e_mean", "e2_mean", "absm_mean", "m2_mean", "m4_mean"):
        assert got[k] == ref[k], (k, got[k], ref[k])
    for k in ("specific_heat", "susceptibility", "binder"):
        assert abs(got[k] - ref[k]) <= 1e-12 * abs(ref[k]), (k, got[k], ref[k])
    sw.close()


def test_moments_of_a_batch(B):
    from oracle import moments as om
    L, nb, n = 128, 3, 12
    Ts = [2.0, T_C, 3.0]
    seeds = [1000, 1001, 1002]
    sw = B.SwendsenWang(L, Ts, seeds)
    sw.sweep(n)
    got = sw.moments()
    for b in range(nb):
        _, ser = oracle.run(L, Ts[b], seeds[b], n)
        ref = om.moments(ser[:, 0], ser[:, 1], L * L, Ts[b])
        assert got[b]["n"] == n
        for k in ("e_mean", "absm_mean", "m2_mean"):
            assert abs(got[b][k] - ref[k]) <= 1e-12 * max(1.0, abs(ref[k]))
    sw.close()


# SURVEY.md 8(f) NEXT-1, second half: binning and the integrated autocorrelation time over the device series ring
@pytest.mark.parametrize("L,path,T,n,cap", [(64, 0, T_C, 400, None), (128, 0, 2.0, 300, None), (20, 1, T_C, 257, None),
                                            (64, 0, 3.0, 300, 128)])
def test_binning_and_autocorrelation_match_oracle(B, L, path, T, n, cap):
    from oracle import moments as om
    seed, N = 900 + L, L * L
    sw = B.SwendsenWang(L, T, seed, path=path)
    if cap:
        B.sw_set_series_capacity(sw.h, cap)          # the ring keeps the last `cap` sweeps of the call
    sw.sweep(n)
    _, ser = oracle.run(L, T, seed, n)
    ser = ser[-cap:] if cap else ser
    E, M = ser[:, 0], ser[:, 1]
    for which in (0, 1):
        for bl in (1, 7, 50, len(E), len(E) + 1):
            got = sw.bins(which, bl)[0]
            means = om.bin_means(E, M, N, which, bl)
            mean, err, nb = om.binned_error(E, M, N, which, bl)
            assert got["n_bins"] == nb == len(means)
            assert got["bin_means"].tolist() == means                      # exact integer sums, one division
            assert abs(got["mean"] - mean) <= 1e-12 * abs(mean) and abs(got["err"] - err) <= 1e-12 * err
        for tmax, c in ((60, 6.0), (5, 6.0), (len(E) + 10, 4.0)):
            got = sw.autocorr(which, tmax, c)[0]
            tau, W, rho = om.tau_int(E, M, N, which, tmax, c)
            assert got["window"] == W and got["tmax"] == len(rho) - 1
            assert abs(got["tau_int"] - tau) <= 1e-12 * abs(tau)
            assert np.all(np.abs(got["rho"] - np.array(rho)) <= 1e-12 * np.maximum(1.0, np.abs(rho)))
            assert abs(got["c0"] - om.autocovariance(E, M, N, which, 0)[0]) <= 1e-12 * got["c0"]
    sw.close()


def test_binning_of_a_batch_and_without_a_series(B):
    from oracle import moments as om
    L, Ts, seeds, n = 64, [2.0, T_C, 3.0], [31, 32, 33], 200
    sw = B.SwendsenWang(L, Ts, seeds)
    with pytest.raises(B.SwError):
        sw.bins(0, 10)                               # no sweep yet
    sw.sweep(n)
    gb, gt = sw.bins(1, 20), sw.autocorr(0, 30)
    for b in range(3):
        _, ser = oracle.run(L, Ts[b], seeds[b], n)
        mean, err, nb = om.binned_error(ser[:, 0], ser[:, 1], L * L, 1, 20)
        assert gb[b]["n_bins"] == nb and abs(gb[b]["mean"] - mean) <= 1e-12 * mean and abs(gb[b]["err"] - err) <= 1e-12 * err
        tau, W, _ = om.tau_int(ser[:, 0], ser[:, 1], L * L, 0, 30)
        assert gt[b]["window"] == W and abs(gt[b]["tau_int"] - tau) <= 1e-12 * tau
    with pytest.raises(B.SwError):
        sw.bins(2, 10)
    with pytest.raises(B.SwError):
        sw.autocorr(0, 10, c=0.0)
    sw.close()


def test_critical_slowing_down_is_absent(B):
    """The paper's motivation made visible: tau_int of the energy stays of order one for cluster updates,
    at T_c as away from it (config 2's temperatures, L = 256)."""
    L, n = 256, 2000
    sw = B.SwendsenWang(L, [2.0, T_C, 3.0], [1, 2, 3])
    sw.sweep(200)
    sw.sweep(n)
    taus = [r["tau_int"] for r in sw.autocorr(0, 100)]
    assert all(0.4 < t < 12.0 for t in taus), taus
    assert taus[1] > taus[0] and taus[1] > taus[2]   # largest at the critical point, but small (z ~ 0.2)
    sw.close()


# ------------------------------------------------------------------------------------------------
# many sweeps in ONE call: the steady sweep is replayed from CUDA graphs (sw_set_graphs, default on)
@pytest.mark.parametrize("L,path,n", [(128, 0, 37), (256, 0, 12), (192, 0, 21), (64, 0, 50), (512, 6, 9)])
def test_many_sweeps_per_call_with_and_without_graphs(B, L, path, n):
    T, seed = T_C, 77 + L
    s_ref, ser_ref = oracle.run(L, T, seed, n)
    for graphs in (True, False):
        sw = B.SwendsenWang(L, T, seed, path=path)
        sw.set_graphs(graphs)
        B.sw_set_cluster(sw.h, False)                # (L = 64, 128 would otherwise run the whole call inside k_sweeps_cluster)
        sw.sweep(n)
        assert np.array_equal(sw.series()[:, 0, :], ser_ref), f"series differ (graphs={graphs})"
        assert np.array_equal(sw.spins_host()[0], s_ref)
        assert _obs_tuple(sw.observables()[0]) == tuple(int(v) for v in ser_ref[-1])
        # a second call continues the same Markov chain (graphs are reused)
        sw.sweep(5)
        s2, ser2 = oracle.run(L, T, seed, 5, spins=s_ref, t0=n)
        assert np.array_equal(sw.series()[:, 0, :], ser2)
        assert np.array_equal(sw.labels_host()[0], oracle.sweep(L, T, seed, n + 4, oracle.run(L, T, seed, 4, spins=s_ref, t0=n)[0])[3])
        sw.close()


# lattices of at most 8 tiles: the whole call inside one kernel, a thread-block cluster per lattice (sw_cluster.cuh, default)
# against the kernels of the fast path one by one (sw_set_cluster(h, 0)); the oracle decides which is right
@pytest.mark.parametrize("L,nb,cap", [(64, 1, None), (128, 1, None), (128, 3, 16), (64, 5, 7), (128, 8, None)])
def test_cluster_kernel_and_separate_kernels_agree(B, L, nb, cap):
    Ts = [1.8 + 0.25 * b for b in range(nb)]
    seeds = [500 + L + b for b in range(nb)]
    a, k = B.SwendsenWang(L, Ts, seeds), B.SwendsenWang(L, Ts, seeds)
    B.sw_set_cluster(k.h, False)
    if cap:
        B.sw_set_series_capacity(a.h, cap); B.sw_set_series_capacity(k.h, cap)      # the ring wraps inside the kernel
    s = [oracle.init_random(L, sd) for sd in seeds]
    t = 0
    for n in (1, 2, 37, 5, 1):
        a.sweep(n); k.sweep(n)
        for b in range(nb):
            for _ in range(n):
                s[b], bE, bS, lab, obs = oracle.sweep(L, Ts[b], seeds[b], t + _, s[b])
            assert np.array_equal(a.spins_host()[b], s[b]) and np.array_equal(a.labels_host()[b], lab), (n, b)
            assert _obs_tuple(a.observables()[b]) == obs
        t += n
        assert np.array_equal(a.spins_host(), k.spins_host()) and np.array_equal(a.labels_host(), k.labels_host())
        ga, gk = a.bonds_host(), k.bonds_host()
        assert np.array_equal(ga[0], gk[0]) and np.array_equal(ga[1], gk[1])
        assert np.array_equal(a.series(), k.series())
        ma, mk = a.moments(), k.moments()
        for b in range(nb):
            assert _obs_tuple(a.observables()[b]) == _obs_tuple(k.observables()[b])
            assert ma[b] == mk[b] and ma[b]["n"] == t                 # (dicts of the nine fields: the same sums in the same order)
    assert a.sweep_index == k.sweep_index == t
    a.close(); k.close()


def test_cluster_kernels_of_two_handles_on_two_streams(B):
    """Two lattices, each swept by its own cluster kernel on its own stream, launched back to back with no synchronisation in
    between: nothing is shared between handles, so both must land where the oracle does."""
    import torch
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    with torch.cuda.stream(s1):
        a = B.SwendsenWang(128, T_C, 71)
    with torch.cuda.stream(s2):
        b = B.SwendsenWang(64, 2.0, 72)
    for n in (30, 1, 12):
        with torch.cuda.stream(s1):
            a.use_current_stream(); a.sweep(n)
        with torch.cuda.stream(s2):
            b.use_current_stream(); b.sweep(n)
    torch.cuda.synchronize()
    sa, sera = oracle.run(128, T_C, 71, 43)
    sb, serb = oracle.run(64, 2.0, 72, 43)
    assert np.array_equal(a.spins_host()[0], sa) and np.array_equal(b.spins_host()[0], sb)
    assert _obs_tuple(a.observables()[0]) == tuple(int(v) for v in sera[-1])
    assert _obs_tuple(b.observables()[0]) == tuple(int(v) for v in serb[-1])
    assert np.array_equal(a.series()[:, 0, :], sera[-12:]) and np.array_equal(b.series()[:, 0, :], serb[-12:])
    a.close(); b.close()


# ------------------------------------------------------------------------------------------------
# the paper's own labelling as path 11.  Labels are the same canonical
# minimum-index labels (bit-exact with the definition), and the number of passes is a deterministic function of
# the bond graph: it must equal the oracle's step-by-step statement of the iteration.
from oracle import label_equivalence as le


@pytest.mark.parametrize("L", [2, 3, 4, 13, 33, 64, 100, 128, 256])
def test_label_equivalence_path_every_sweep(B, L):
    for T, seed in ((2.0, 1), (T_C, 2), (3.0, 3)):
        sw = B.SwendsenWang(L, T, seed + L, path=11)
        s = oracle.init_random(L, seed + L)
        for t in range(5):
            s1, bE, bS, lab, obs = oracle.sweep(L, T, seed + L, t, s)
            sw.sweep(1)
            gE, gS = sw.bonds_host()
            assert np.array_equal(gE[0], wl.pack_bits(bE)) and np.array_equal(gS[0], wl.pack_bits(bS))
            assert np.array_equal(sw.labels_host()[0], lab), f"labels differ at sweep {t}"
            assert np.array_equal(sw.spins_host()[0], s1), f"spins differ at sweep {t}"
            assert _obs_tuple(sw.observables()[0]) == obs
            assert sw.label_passes() == le.label_equivalence(L, bE, bS)[1], f"pass count differs at sweep {t}"
            s = s1
        sw.close()


@pytest.mark.parametrize("L", [64, 100, 256, 512])
def test_label_equivalence_on_injected_bond_graphs(B, L):
    sw = B.SwendsenWang(L, 2.0, 1, path=11)
    for name, (bE, bS) in _label_patterns(L):
        got = B.sw_test_label(sw.h, wl.pack_bits(bE), wl.pack_bits(bS))
        ref = oracle.labels(L, bE, bS)
        assert np.array_equal(got, ref), f"{name}: {np.count_nonzero(got != ref)} labels differ"
        assert sw.label_passes() == le.label_equivalence(L, bE, bS)[1], name
    sw.close()


def test_label_equivalence_pass_counts_worked_by_hand(B):
    # the cases derived in tests/test_oracle_label_equivalence.py: no bonds 1, chain 2, U 3, hook 4
    L = 8
    sw = B.SwendsenWang(L, 2.0, 1, path=11)

    def passes(bE, bS):
        got = B.sw_test_label(sw.h, wl.pack_bits(bE), wl.pack_bits(bS))
        assert np.array_equal(got, oracle.labels(L, bE, bS))
        return sw.label_passes()

    z = lambda: (np.zeros(L * L, dtype=np.uint8), np.zeros(L * L, dtype=np.uint8))
    bE, bS = z()
    assert passes(bE, bS) == 1
    bE[0:4] = 1
    assert passes(bE, bS) == 2
    bE, bS = z()                                     # U: column 0 rows 0..5, row 5 columns 0..2, column 2 rows 0..5
    for y in range(5):
        bS[y * L] = 1; bS[y * L + 2] = 1
    bE[5 * L] = 1; bE[5 * L + 1] = 1
    assert passes(bE, bS) == 3
    bE, bS = z()                                     # hook: ... column 2 rows 1..5, row 1 columns 2..4, column 4 rows 0..1
    for y in range(5):
        bS[y * L] = 1
    bE[5 * L] = 1; bE[5 * L + 1] = 1
    for y in range(1, 5):
        bS[y * L + 2] = 1
    bE[L + 2] = 1; bE[L + 3] = 1; bS[4] = 1
    assert passes(bE, bS) == 4
    sw.close()


def test_label_equivalence_batch_and_errors(B):
    L, Ts, seeds = 96, [1.5, T_C, 3.5], [11, 12, 13]
    sw = B.SwendsenWang(L, Ts, seeds, path=11)
    with pytest.raises(Exception):
        sw.label_passes()                            # SW_ESTATE before any labelling
    refs = [oracle.init_random(L, s) for s in seeds]
    for t in range(4):
        sw.sweep(1)
        gs, gl, obs = sw.spins_host(), sw.labels_host(), sw.observables()
        want = 0
        for b in range(3):
            s1, bE, bS, lab, o = oracle.sweep(L, Ts[b], seeds[b], t, refs[b])
            assert np.array_equal(gl[b], lab) and np.array_equal(gs[b], s1) and _obs_tuple(obs[b]) == o
            want = max(want, le.label_equivalence(L, bE, bS)[1])
            refs[b] = s1
        assert sw.label_passes() == want             # the lattices of a batch iterate together
    sw.close()
    sw = B.SwendsenWang(64, 2.0, 1)
    sw.sweep(1)
    with pytest.raises(Exception):
        sw.label_passes()                            # not path 11
    sw.close()


# ------------------------------------------------------------------------------------------------
# q-state Potts model on the same sweep.  Bit-exact with oracle/potts.py:
# colours, both bond planes, labels and the integer observables after every sweep.
from oracle import potts as opotts


def _compare_potts(B, L, q, T, seed, n, path=0, start=None, t0=0):
    sw = B.SwendsenWang(L, T, seed, path=path, q=q)
    assert B.sw_q(sw.h) == q
    N = L * L
    if start is None:
        s = opotts.init_random(L, q, seed)
        assert np.array_equal(sw.spins_host()[0], s), "random start differs"
    else:
        s = np.asarray(start, dtype=np.int8)
        sw.set_spins(s)
    if t0:
        sw.set_sweep_index(t0)
    assert sw.threshold() == opotts.threshold(T)
    o0 = sw.observables()[0]                         # before any sweep: E, M of the start, no clusters
    want0, _ = opotts.observables(L, q, s)
    assert (o0.energy, o0.magnetisation, o0.n_clusters, o0.largest_cluster) == (want0[0], want0[1], 0, 0)
    for k in range(n):
        t = t0 + k
        s1, bE, bS, lab, obs = opotts.sweep(L, q, T, seed, t, s)
        sw.sweep(1)
        gE, gS = sw.bonds_host()
        assert np.array_equal(gE[0], wl.pack_bits(bE)), f"bondE differs at sweep {t}"
        assert np.array_equal(gS[0], wl.pack_bits(bS)), f"bondS differs at sweep {t}"
        assert np.array_equal(sw.labels_host()[0], lab), f"labels differ at sweep {t}"
        assert np.array_equal(sw.spins_host()[0], s1), f"colours differ at sweep {t}"
        o = sw.observables()[0]
        assert _obs_tuple(o) == obs, f"observables differ at sweep {t}: {_obs_tuple(o)} vs {obs}"
        assert o.sweep == t + 1
        assert abs(o.e_per_site - obs[0] / N) <= 1e-12 and abs(o.abs_m_per_site - obs[1] / N) <= 1e-12
        s = s1
    sw.close()


@pytest.mark.parametrize("L,q", [(2, 2), (3, 3), (5, 4), (13, 3), (32, 5), (33, 7), (64, 3), (100, 127), (128, 2), (256, 3),
                                 (384, 5), (512, 127)])      # L % 128 == 0: scan-line tiles + k_assign16_potts
def test_potts_every_sweep(B, L, q):
    tc = 1.0 / math.log(1.0 + math.sqrt(q))
    for T, seed in ((0.7 * tc, 1), (tc, 2), (1.6 * tc, 3)):
        _compare_potts(B, L, q, T, seed + L, 6)


@pytest.mark.parametrize("L,q,path", [(64, 3, 11), (100, 4, 11), (96, 3, 1), (128, 4, 1), (128, 3, 11)])
def test_potts_on_other_paths(B, L, q, path):
    _compare_potts(B, L, q, 1.0 / math.log(1.0 + math.sqrt(q)), 77, 5, path=path)


@pytest.mark.parametrize("L", [48, 128])
def test_potts_special_starts_limits_and_sweep_index(B, L):
    q = 3
    one = np.zeros(L * L, dtype=np.int8)
    stripes = (np.arange(L * L, dtype=np.int64) // L % q).astype(np.int8)
    for s0 in (one, stripes):
        for T in (1e-3, 0.995, 1e12):                # all bonds between equal colours / critical / none
            _compare_potts(B, L, q, T, 9, 2, start=s0)
    _compare_potts(B, L, q, 0.995, 5, 3, t0=(1 << 40) + 3)


def test_potts_many_sweeps_per_call_series_and_batch(B):
    for L in (64, 128):                              # generic kernels / scan-line tiles
        q, Ts, seeds, n = 3, [0.8, 0.995, 1.4], [21, 22, 23], 15
        sw = B.SwendsenWang(L, Ts, seeds, q=q)
        sw.sweep(n)
        ser = sw.series()                            # (n, nb, 4)
        got, lab = sw.spins_host(), sw.labels_host()
        for b in range(3):
            s, want = opotts.run(L, q, Ts[b], seeds[b], n - 1)
            s1, bE, bS, lab_b, o = opotts.sweep(L, q, Ts[b], seeds[b], n - 1, s)
            assert np.array_equal(got[b], s1) and np.array_equal(lab[b], lab_b)
            assert np.array_equal(ser[:n - 1, b, :], want) and tuple(ser[n - 1, b, :]) == o
        sw.close()


def test_potts_argument_errors(B):
    for q in (1, -3, 128):
        with pytest.raises(Exception):
            B.sw_create_potts(16, q, 1.0, 1)
    h = B.sw_create_potts(16, 3, 1.0, 1)
    with pytest.raises(Exception):
        B.sw_set_path(h, 6)                          # the stand-alone Ising bond kernel reads sign bits
    B.sw_destroy(h)


# ------------------------------------------------------------------------------------------------
# bit-packed host interface (sw_set_spins_bits / sw_get_spins_bits): the same spins, 1 bit per site
@pytest.mark.parametrize("L,nb", [(64, 1), (13, 1), (27, 3), (128, 2), (5, 1)])
def test_bit_packed_host_interface(B, L, nb):
    N, words = L * L, (L * L + 31) // 32
    Ts, seeds = [T_C] * nb, [40 + b for b in range(nb)]
    sw = B.SwendsenWang(L, Ts, seeds)
    bits = np.zeros(nb * words, dtype=np.uint32)
    B.sw_get_spins_bits(sw.h, bits.ctypes.data)
    s0 = sw.spins_host()
    for b in range(nb):
        assert np.array_equal(bits[b * words:(b + 1) * words], wl.pack_bits((s0[b] > 0).astype(np.uint8)))
        assert np.array_equal(s0[b], oracle.init_random(L, seeds[b]))
    # inject a different state through the packed interface, sweep, read back both ways
    rng = np.random.default_rng(L)
    s = [np.where(rng.random(N) < 0.4, 1, -1).astype(np.int8) for _ in range(nb)]
    inj = np.concatenate([wl.pack_bits((x > 0).astype(np.uint8)) for x in s]).astype(np.uint32)
    B.sw_set_spins_bits(sw.h, inj.ctypes.data)
    got = sw.spins_host()
    for b in range(nb):
        assert np.array_equal(got[b], s[b])
    sw.sweep(1)
    B.sw_get_spins_bits(sw.h, bits.ctypes.data)
    got = sw.spins_host()
    for b in range(nb):
        s1 = oracle.sweep(L, Ts[b], seeds[b], 0, s[b])[0]
        assert np.array_equal(got[b], s1)
        assert np.array_equal(bits[b * words:(b + 1) * words], wl.pack_bits((s1 > 0).astype(np.uint8)))
    sw.close()
    swp = B.SwendsenWang(16, 1.0, 1, q=3)
    with pytest.raises(Exception):
        B.sw_get_spins_bits(swp.h, bits.ctypes.data)
    swp.close()


def test_switching_paths_keeps_one_state(B):
    """The fused path sweeps on the bit-packed plane, the others on the int8 plane: one handle walked through the
    paths must follow the oracle without a break (the planes are converted on demand)."""
    L, T, seed = 256, T_C, 77
    sw = B.SwendsenWang(L, T, seed)
    s = oracle.init_random(L, seed)
    t = 0
    for path, n in ((0, 2), (1, 2), (0, 1), (6, 2), (11, 1), (0, 2), (6, 1), (0, 2)):
        B.sw_set_path(sw.h, path)
        for _ in range(n):
            s, bE, bS, lab, obs = oracle.sweep(L, T, seed, t, s)
            sw.sweep(1)
            t += 1
            assert np.array_equal(sw.labels_host()[0], lab), (path, t)
            assert _obs_tuple(sw.observables()[0]) == obs, (path, t)
        assert np.array_equal(sw.spins_host()[0], s), (path, t)
    # several sweeps per call across a switch, spins read only at the end
    B.sw_set_path(sw.h, 0); sw.sweep(5)
    B.sw_set_path(sw.h, 1); sw.sweep(2)
    B.sw_set_path(sw.h, 0); sw.sweep(4)
    s, _ = oracle.run(L, T, seed, 11, spins=s, t0=t)
    assert np.array_equal(sw.spins_host()[0], s)
    sw.close()


def test_observables_of_an_injected_packed_state(B):
    L = 128
    sw = B.SwendsenWang(L, T_C, 3)
    s = wl.spins_numpy_random(L, 5, 0.3)
    bits = wl.pack_bits((s > 0).astype(np.uint8)).astype(np.uint32)
    B.sw_set_spins_bits(sw.h, bits.ctypes.data)
    o = sw.observables()[0]                          # no sweep yet: E, M of the injected state, no clusters
    assert _obs_tuple(o) == oracle.observables(L, s)[:2] + (0, 0)
    s1, bE, bS, lab, obs = oracle.sweep(L, T_C, 3, 0, s)
    sw.sweep(1)
    assert _obs_tuple(sw.observables()[0]) == obs and np.array_equal(sw.spins_host()[0], s1)
    sw.close()


# ------------------------------------------------------------------------------------------------
# The GPU path against what the physics fixes, without the oracle in between
import exact_ising as ex


def _golden_kaufman(L):
    import os
    with open(os.path.join(os.path.dirname(__file__), "golden", "kaufman_u.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            v = line.split()
            if int(v[0]) == L:
                return dict(zip((2.0, 2.26919, "Tc", 2.5, 3.0), (float(x) for x in v[1:])))
    raise KeyError(L)


@pytest.mark.parametrize("T,seed", [(2.0, 1), (2.26919, 2), (3.0, 3)])
def test_config2_L1024_energy_against_kaufman_on_the_gpu(B, T, seed):
    L, therm, n = 1024, 200, 2000
    sw = B.SwendsenWang(L, T, seed)
    sw.sweep(therm)
    sw.sweep(n)
    ser = sw.series()[:, 0, :]
    assert ser.shape[0] == n
    u, du = ex.binned_mean_err(ser[:, 0] / (L * L), nbins=40)
    exact = _golden_kaufman(L)[T]
    assert abs(u - exact) <= 4 * du and du < 2e-3, (u, du, exact)
    if T == 2.0:                                     # Yang's spontaneous magnetisation (finite-size shift << error bar)
        m, dm = ex.binned_mean_err(np.abs(ser[:, 1]) / (L * L), nbins=40)
        assert abs(m - 0.911319) <= 4 * dm + 1e-5, (m, dm)
    sw.close()


@pytest.mark.parametrize("T,seed", [(1.5, 7), (2.269, 8), (3.5, 9)])
def test_config1_4x4_against_exact_enumeration_on_the_gpu(B, T, seed):
    L, calls, per = 4, 25, 4000
    r = ex.exact_small(L, T)
    sw = B.SwendsenWang(L, T, seed)
    sw.sweep(100)
    E, M = [], []
    for _ in range(calls):
        sw.sweep(per)
        ser = sw.series()[:, 0, :]
        E.append(ser[:, 0]); M.append(np.abs(ser[:, 1]))
    u, du = ex.binned_mean_err(np.concatenate(E) / 16.0)
    m, dm = ex.binned_mean_err(np.concatenate(M) / 16.0)
    assert abs(u - float(r["u"])) <= 4 * du, (u, du, float(r["u"]))
    assert abs(m - float(r["abs_m"])) <= 4 * dm, (m, dm, float(r["abs_m"]))
    sw.close()


def test_specific_heat_against_kaufman_on_the_gpu(B):
    """The paper's own validation (Fig. 6: the specific-heat peak), with the on-device moments
    (NEXT-1): 16 independent L = 64 lattices at T_c, C/N of each from sw_moments, mean +- standard error against
    Kaufman's exact finite-lattice value."""
    L, nb, therm, n = 64, 16, 500, 20000
    T = T_C
    sw = B.SwendsenWang(L, [T] * nb, [900 + b for b in range(nb)])
    sw.sweep(therm)
    sw.moments_reset()
    sw.sweep(n)
    mom = sw.moments()
    c = np.array([m["specific_heat"] for m in mom])
    u = np.array([m["e_mean"] for m in mom])
    assert all(m["n"] == n for m in mom)
    c_exact, u_exact = float(ex.kaufman_c(L, T)), float(ex.kaufman_u(L, T))
    assert abs(c.mean() - c_exact) <= 4 * c.std(ddof=1) / np.sqrt(nb), (c.mean(), c.std(ddof=1) / np.sqrt(nb), c_exact)
    assert abs(u.mean() - u_exact) <= 4 * u.std(ddof=1) / np.sqrt(nb), (u.mean(), u_exact)
    assert c.std(ddof=1) / np.sqrt(nb) < 0.03 * c_exact
    sw.close()


@pytest.mark.parametrize("T,seed", [(0.7, 7), (0.995, 8)])
def test_potts_3x3_against_exact_enumeration_on_the_gpu(B, T, seed):
    from test_oracle_potts import _potts_enumeration
    L, q, calls, per = 3, 3, 20, 4000
    E, M = _potts_enumeration(L, q)
    w = np.exp(-(E - E.min()) / T)
    exact_E, exact_M = float((E * w).sum() / w.sum()), float((M * w).sum() / w.sum())
    sw = B.SwendsenWang(L, T, seed, q=q)
    sw.sweep(100)
    es, ms = [], []
    for _ in range(calls):
        sw.sweep(per)
        ser = sw.series()[:, 0, :]
        es.append(ser[:, 0]); ms.append(ser[:, 1])
    e, de = ex.binned_mean_err(np.concatenate(es))
    m, dm = ex.binned_mean_err(np.concatenate(ms))
    assert abs(e - exact_E) <= 4 * de and de < 0.06, (e, de, exact_E)
    assert abs(m - exact_M) <= 4 * dm and dm < 0.06, (m, dm, exact_M)
    sw.close()


def test_per_sweep_time_series(B):
    sw = B.SwendsenWang(256, T_C, 1)
    with pytest.raises(Exception):
        sw.sweep(2); sw.sweep_ms()                   # no stage timing: SW_ESTATE
    sw.set_stage_timing(True)
    sw.sweep(7)
    per = sw.sweep_ms()
    assert per.shape == (7,) and np.all(per > 0)
    km = sw.kernel_ms()                              # (on this path the "energy" slot is the pass after the last sweep)
    assert abs(per.sum() - (sum(km.values()) - km["energy"])) < 1e-3 * per.sum() + 1e-3
    sw.close()


def test_philox_ceiling_hook(B):
    ms = B.sw_test_philox_ceiling(1 << 22, 5)
    assert 0.0 < ms < 50.0
    with pytest.raises(Exception):
        B.sw_test_philox_ceiling(8, 1)


def test_temperature_scan_batch_against_kaufman_on_the_gpu(B):
    """BASELINE configs[4] in small (the paper's Fig. 5): a batch of lattices at temperatures across the
    transition, one launch per stage; the mean energy of every lattice against Kaufman's exact finite-lattice value."""
    L, nb, therm, n = 128, 16, 300, 3000
    Ts = [1.5 + b * 2.0 / (nb - 1) for b in range(nb)]
    sw = B.SwendsenWang(L, Ts, [1000 + b for b in range(nb)])
    sw.sweep(therm)
    sw.sweep(n)
    ser = sw.series()
    assert ser.shape == (n, nb, 4)
    worst = 0.0
    for b, T in enumerate(Ts):
        u, du = ex.binned_mean_err(ser[:, b, 0] / (L * L), nbins=30)
        exact = float(ex.kaufman_u(L, T))
        worst = max(worst, abs(u - exact) / du)
        assert abs(u - exact) <= 4.0 * du and du < 3e-3, (T, u, du, exact)
    assert worst > 0.0
    sw.close()
