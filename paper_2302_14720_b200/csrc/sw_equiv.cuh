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
    const int i0 = blockIdx.x * EQ_THREADS + threadIdx.x;

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
            for (int i = i0; i < N; i += stride) {
                const int y = div_l(i, dv), x = i - y * L;
                const int ie = x + 1 == L ? i - L + 1 : i + 1, is = y + 1 == L ? i - N + L : i + L;
                const int iw = x ? i - 1 : i + L - 1,          in = y ? i - L : i + N - L;
                const int l = lab[i];
                int m = l;
                if ((E[i >> 5] >> (i & 31)) & 1u)   m = min(m, lab[ie]);
                if ((S[i >> 5] >> (i & 31)) & 1u)   m = min(m, lab[is]);
                if ((E[iw >> 5] >> (iw & 31)) & 1u) m = min(m, lab[iw]);
                if ((S[in >> 5] >> (in & 31)) & 1u) m = min(m, lab[in]);
                if (m < l) { atomicMin(rf + l, m); formed = 1; }
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

} // namespace sw
