"""sw_bins_noalloc (include/sw.h): the binning of sw_bins for callers that cannot call cudaMalloc -- its scratch (the bin
means) is a static device array of SW_BINS_NOALLOC_MAX doubles, its result goes to DEVICE memory the caller passes.
Checked against the existing path (sw_bins) on two calls in a row that leave different contents in the shared scratch,
then once more with the first arguments (a stale array must not show), and beyond the limit.  The file sorts last on
purpose: the suite runs with pytest -x, and a failure here must not hide the parity tests.  -m gpu."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    from paper_2302_14720_b200 import binding
    binding.lib()
    return binding


def _records(out, nb):
    """(n_bins, mean, err) per lattice from the device buffer of nb records of (int64, double, double)."""
    host = out.cpu().numpy()
    return [(int(host[3 * b:3 * b + 1].view(np.int64)[0]), float(host[3 * b + 1]), float(host[3 * b + 2])) for b in range(nb)]


def _check(sw, out, which, bin_len, nb):
    import torch
    want = sw.bins(which, bin_len)                       # the existing path: cudaMalloc'ed scratch, host results
    out.fill_(float("nan"))
    sw.bins_noalloc(which, bin_len, out)                 # asynchronous on the handle's stream (here: the current one)
    torch.cuda.synchronize()
    got = _records(out, nb)
    for b in range(nb):
        assert got[b][0] == want[b]["n_bins"]
        # the same kernels on the same series: the tolerance of the binning parity tests (1e-12) is met with equality
        assert abs(got[b][1] - want[b]["mean"]) <= 1e-12 * abs(want[b]["mean"]) and got[b][1] == want[b]["mean"]
        assert abs(got[b][2] - want[b]["err"]) <= 1e-12 * abs(want[b]["err"]) and got[b][2] == want[b]["err"]
    return got


def test_no_alloc_binning_matches_the_existing_path_on_two_calls_in_a_row(B):
    import torch
    from paper_2302_14720_b200 import workloads as wl
    L, Ts, seeds, n = 64, [2.0, wl.T_C, 3.0], [41, 42, 43], 300
    sw = B.SwendsenWang(L, Ts, seeds)
    out = torch.empty(3 * 3, dtype=torch.float64, device=sw.device)
    with pytest.raises(B.SwError):
        sw.bins_noalloc(0, 10, out)                      # no series yet: SW_ESTATE, as sw_bins
    sw.sweep(n)
    first = _check(sw, out, 0, 7, 3)                     # 42 bins of the energy per lattice
    second = _check(sw, out, 1, 1, 3)                    # straight after it: 300 bins of |m| (overwrites the scratch, and more of it)
    again = _check(sw, out, 0, 7, 3)                     # the first call again: nothing of the second one's contents shows
    assert again == first and second != first
    _check(sw, out, 0, n + 1, 3)                         # no bin at all: n_bins = 0, mean = err = 0
    _check(sw, out, 1, n, 3)                             # one bin: err = 0
    sw.close()


def test_no_alloc_binning_rejects_sizes_beyond_the_static_scratch(B):
    import torch
    nb, n = 32, 2100                                     # 32 x 2100 bins of one sweep = 67200 > SW_BINS_NOALLOC_MAX
    assert nb * n > B.SW_BINS_NOALLOC_MAX >= nb * (n // 2)
    sw = B.SwendsenWang(64, [2.0 + 0.03 * b for b in range(nb)], list(range(100, 100 + nb)))
    out = torch.zeros(3 * nb, dtype=torch.float64, device=sw.device)
    sw.sweep(n)
    with pytest.raises(B.SwError) as e:
        sw.bins_noalloc(0, 1, out)
    assert "SW_BINS_NOALLOC_MAX" in str(e.value) and e.value.code == -1      # SW_EINVAL, with the limit in the text
    assert torch.count_nonzero(out).item() == 0          # nothing was launched
    _check(sw, out, 0, 2, nb)                            # 32 x 1050 fits
    with pytest.raises(B.SwError):
        sw.bins_noalloc(2, 10, out)                      # bad `which`
    sw.close()
