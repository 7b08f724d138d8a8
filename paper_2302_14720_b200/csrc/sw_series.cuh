// sw_series.cuh -- error analysis of the per-sweep series on the device (binning and the
// integrated autocorrelation time; PAPER.md:15 -- the autocorrelation time is the paper's motivation -- and
// PAPER.md:113, section 4).  Reductions over the series ring the sweeps leave on the device (sw_series): nothing
// is copied to the host but the results.  Every sum runs in index order with separate (unfused) double operations,
// so the results do not depend on the launch shape.
//   x_k = E_k / N (which = 0) or |M_k| / N (which = 1) of retained sweep k, oldest first
#pragma once
#include "sw_common.cuh"

namespace sw {

struct SeriesView {            // the retained sweeps of the last sw_sweep call inside the ring
    const Rec* rec; long long first, ring, n; int nb, which;
    __device__ __forceinline__ long long val(long long k, int b) const {
        const Rec& r = rec[(size_t)((first + k) % ring) * nb + b];
        return which == 0 ? r.E : (r.M < 0 ? -r.M : r.M);
    }
};
struct BinStat { long long n_bins; double mean, err; };
struct TauStat { double tau_int; long long window, tmax; double c0; };

// bin j of lattice b: the exact integer sum of its B sweeps, divided once
__global__ void __launch_bounds__(256)
k_series_bins(SeriesView s, double* __restrict__ bins, long long B, long long nbins, int N) {
    const long long j = (long long)blockIdx.x * 256 + threadIdx.x;
    const int b = blockIdx.y;
    if (j >= nbins) return;
    long long tot = 0;
    for (long long k = j * B; k < (j + 1) * B; ++k) tot += s.val(k, b);
    bins[(size_t)b * nbins + j] = __ddiv_rn((double)tot, (double)(B * (long long)N));
}
// mean of the bin means and its standard error: one thread per lattice, bins in order
__global__ void k_series_binerr(const double* __restrict__ bins, BinStat* __restrict__ out, long long nbins, int nb) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    BinStat r; r.n_bins = nbins; r.mean = 0.0; r.err = 0.0;
    if (nbins > 0) {
        const double* v = bins + (size_t)b * nbins;
        double tot = 0.0;
        for (long long j = 0; j < nbins; ++j) tot = __dadd_rn(tot, v[j]);
        r.mean = __ddiv_rn(tot, (double)nbins);
        if (nbins > 1) {
            double ss = 0.0;
            for (long long j = 0; j < nbins; ++j) { const double d = __dsub_rn(v[j], r.mean); ss = __dadd_rn(ss, __dmul_rn(d, d)); }
            r.err = __dsqrt_rn(__ddiv_rn(ss, (double)(nbins * (nbins - 1))));
        }
    }
    out[b] = r;
}
// x_k as doubles, and their mean (one thread per lattice adds them in order)
__global__ void __launch_bounds__(256)
k_series_x(SeriesView s, double* __restrict__ x, int N) {
    const long long k = (long long)blockIdx.x * 256 + threadIdx.x;
    const int b = blockIdx.y;
    if (k < s.n) x[(size_t)b * s.n + k] = __ddiv_rn((double)s.val(k, b), (double)N);
}
__global__ void k_series_mean(const double* __restrict__ x, double* __restrict__ xbar, long long n, int nb) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    double tot = 0.0;
    for (long long k = 0; k < n; ++k) tot = __dadd_rn(tot, x[(size_t)b * n + k]);
    xbar[b] = __ddiv_rn(tot, (double)n);
}
// C(t) = (1 / (n - t)) sum_k (x_k - xbar)(x_{k+t} - xbar): one thread per lag and lattice
__global__ void __launch_bounds__(128)
k_series_autocov(const double* __restrict__ x, const double* __restrict__ xbar, double* __restrict__ C,
                 long long n, long long tmax) {
    const long long t = (long long)blockIdx.x * 128 + threadIdx.x;
    const int b = blockIdx.y;
    if (t > tmax) return;
    const double* v = x + (size_t)b * n;
    const double m = xbar[b];
    double acc = 0.0;
    for (long long k = 0; k < n - t; ++k) acc = __dadd_rn(acc, __dmul_rn(__dsub_rn(v[k], m), __dsub_rn(v[k + t], m)));
    C[(size_t)b * (tmax + 1) + t] = __ddiv_rn(acc, (double)(n - t));
}
// rho(t) = C(t) / C(0) and the integrated autocorrelation time with the self-consistent window: tau(W) = 1/2 +
// sum_{t <= W} rho(t), W the smallest W >= 1 with W >= c tau(W), else tmax; C(0) = 0: rho = 0, tau = 1/2, W = 0
__global__ void k_series_tau(const double* __restrict__ C, double* __restrict__ rho, TauStat* __restrict__ out,
                             long long tmax, double c, int nb) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const double* cv = C + (size_t)b * (tmax + 1);
    double* rv = rho + (size_t)b * (tmax + 1);
    TauStat r; r.tau_int = 0.5; r.window = 0; r.tmax = tmax; r.c0 = cv[0];
    if (!(cv[0] > 0.0)) {
        for (long long t = 0; t <= tmax; ++t) rv[t] = 0.0;
        out[b] = r;
        return;
    }
    for (long long t = 0; t <= tmax; ++t) rv[t] = __ddiv_rn(cv[t], cv[0]);
    double tau = 0.5;
    long long W = tmax;
    for (long long w = 1; w <= tmax; ++w) {
        tau = __dadd_rn(tau, rv[w]);
        if ((double)w >= __dmul_rn(c, tau)) { W = w; break; }
    }
    r.tau_int = tau; r.window = W;
    out[b] = r;
}

} // namespace sw
