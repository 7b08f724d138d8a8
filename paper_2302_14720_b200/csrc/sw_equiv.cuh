// sw_equiv.cuh -- the paper's own cluster labelling as a second labelling kernel (path 11).
// Product code (CUDA path); shares nothing with oracle/.
//
// PAPER.md:49-53 (section 2.3): a label-equivalence iteration.  Every site starts with its own index as label; a
// pass is (scan) every site refers its label to the lowest label among the sites it is bonded to, (collapse) every
// label in use follows its chain of references to the end and links itself there, (relabel) every site looks up
// the label its own was found equivalent to; passes repeat until a scan forms no reference.  Every step is a
// minimum or a walk to a fixed point, so the labels (minimum site index of each cluster) and the number of passes
// do not depend on the execution order.
//
// The paper drives the three kernels of a pass from a "maintenance kernel" launched with dynamic parallelism, so
// that no flag crosses to the host.  Here the whole iteration is ONE persistent cooperative kernel:
// as many CTAs as the B200 holds at once (148 SMs x resident CTAs), grid-wide barriers between the steps, the
// "anything formed" flag of pass p in flags[p], the pass count left in flags[EQ_MAX_PASSES].
#pragma once
#include <cooperative_groups.h>
#include "sw_common.cuh"
#include "sw_scan.cuh"          // DivL / div_l

namespace sw {

constexpr int EQ_THREADS = 256;
constexpr int EQ_MAX_PASSES = 1024;       // flags[0 .. EQ_MAX_PASSES - 1]: pass p formed a reference; [EQ_MAX_PASSES]: passes

__global__ void __launch_bounds__(EQ_THREADS)
k_label_equiv(int* label, int* ref, const uint32_t* __restrict__ bondE, const uint32_t* __restrict__ bondS,
              int* flags, DivL dv, int L, int N, int words, int nb) {
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const int stride = gridDim.x * EQ_THREADS;
    const int i0 = blockIdx.x * EQ_THREADS + threadIdx.x, lane = threadIdx.x & 31;

    // "each site is labeled with a unique integer incrementing from zero"
    for (int b = 0; b < nb; ++b)
        for (int i = i0; i < N; i += stride) { label[(size_t)b * N + i] = i; ref[(size_t)b * N + i] = i; }
    grid.sync();

    int pass = 0;
    for (;;) {
        // ---- scan: refer my label to the lowest label among my bonded neighbours ----
        int formed = 0;
        for (int b = 0; b < nb; ++b) {
            const int* lab = label + (size_t)b * N;
            int* rf = ref + (size_t)b * N;
            const uint32_t* E = bondE + (size_t)b * words;
            const uint32_t* S = bondS + (size_t)b * words;
            for (int base = i0 - lane; base < N; base += stride) {   // whole warps stay together (aggregated atomics)
                const int i = base + lane;
                int l = 0, m = 0;
                if (i < N) {
                    const int y = div_l(i, dv), x = i - y * L;
                    const int ie = x + 1 == L ? i - L + 1 : i + 1, is = y + 1 == L ? i - N + L : i + L;
                    const int iw = x ? i - 1 : i + L - 1,          in = y ? i - L : i + N - L;
                    l = lab[i];
                    m = l;
                    if ((E[i >> 5] >> (i & 31)) & 1u)   m = min(m, lab[ie]);
                    if ((S[i >> 5] >> (i & 31)) & 1u)   m = min(m, lab[is]);
                    if ((E[iw >> 5] >> (iw & 31)) & 1u) m = min(m, lab[iw]);
                    if ((S[in >> 5] >> (in & 31)) & 1u) m = min(m, lab[in]);
                }
                const unsigned need = __ballot_sync(0xffffffffu, m < l);
                if (m < l) {
                    // lanes with the same label send one minimum (at T_c a third of all sites share one label)
                    const unsigned grp = __match_any_sync(need, l);
                    const int mn = __reduce_min_sync(grp, m);
                    if (lane == __ffs(grp) - 1 && mn < ld_cg(rf + l)) atomicMin(rf + l, mn);
                    formed = 1;
                }
            }
        }
        formed = __syncthreads_or(formed);
        if (formed && threadIdx.x == 0) flags[pass] = 1;            // (every writer stores the same value)
        grid.sync();
        const int any = ld_cg(flags + pass);
        ++pass;
        if (!any || pass >= EQ_MAX_PASSES) break;
        // ---- collapse: every label in use walks its chain of references to the end ----
        for (int b = 0; b < nb; ++b) {
            const int* lab = label + (size_t)b * N;
            int* rf = ref + (size_t)b * N;
            for (int i = i0; i < N; i += stride) {
                if (lab[i] != i) continue;
                int r = ld_cg(rf + i);
                if (r == i) continue;
                int q;
                while ((q = ld_cg(rf + r)) != r) r = q;             // (others shorten their own entries meanwhile: any
                rf[i] = r;                                          //  value seen is further along the same chain)
            }
        }
        grid.sync();
        // ---- relabel: look up the label mine was found equivalent to ----
        for (int b = 0; b < nb; ++b) {
            int* lab = label + (size_t)b * N;
            const int* rf = ref + (size_t)b * N;
            for (int i = i0; i < N; i += stride) {
                const int l = lab[i];
                const int r = rf[l];
                if (r != l) lab[i] = r;
            }
        }
        grid.sync();
    }
    if (blockIdx.x == 0 && threadIdx.x == 0) flags[EQ_MAX_PASSES] = pass;
}

// cluster count and sizes from FLAT labels (a7): no find, so no walk through the giant cluster's root.  A CTA
// covers EQ_COUNT_SPAN sites; lanes of one cluster add their count once, into a small shared-memory table that
// is flushed at the end (one global atomic per cluster and CTA: at T_c one cluster owns a third of all sites,
// and its counter would otherwise take every warp's atomic).  k_maxsize_generic then takes the maximum and
// clears gsize.
constexpr int EQ_COUNT_SPAN = 16 * EQ_THREADS, EQ_SLOTS = 256;
__global__ void __launch_bounds__(EQ_THREADS)
k_count_flat(const int* __restrict__ label, int* __restrict__ gsize, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
             int N, int nb) {
    __shared__ int s_key[EQ_SLOTS], s_cnt[EQ_SLOTS];
    for (int k = threadIdx.x; k < EQ_SLOTS; k += EQ_THREADS) { s_key[k] = -1; s_cnt[k] = 0; }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    int* gs = gsize + (size_t)blockIdx.y * N;
    int nroot = 0;
    const int first = blockIdx.x * EQ_COUNT_SPAN + threadIdx.x;
#pragma unroll 4
    for (int k = 0; k < EQ_COUNT_SPAN / EQ_THREADS; ++k) {
        const int i = first + k * EQ_THREADS;
        const unsigned act = __ballot_sync(0xffffffffu, i < N);
        if (i < N) {
            const int r = label[(size_t)blockIdx.y * N + i];
            nroot += (r == i);
            const unsigned grp = __match_any_sync(act, r);
            if (lane == __ffs(grp) - 1) {
                const int c = __popc(grp);
                const int slot = (int)(((uint32_t)r * 2654435761u) >> 24) & (EQ_SLOTS - 1);
                const int old = atomicCAS(&s_key[slot], -1, r);
                if (old == -1 || old == r) atomicAdd(&s_cnt[slot], c);
                else atomicAdd(gs + r, c);                          // slot taken by another cluster
            }
        }
    }
    __syncthreads();
    for (int k = threadIdx.x; k < EQ_SLOTS; k += EQ_THREADS)
        if (s_cnt[k]) atomicAdd(gs + s_key[k], s_cnt[k]);
    nroot = warp_sum_i(nroot);
    if (lane == 0 && nroot) atomic_add_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].ncl, nroot);
}

} // namespace sw
