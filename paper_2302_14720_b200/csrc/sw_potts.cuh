// sw_potts.cuh -- q-state Potts model on the same sweep.  Product code (CUDA path).
//
// "The approach can be generalized to other discrete spin systems" (also PAPER.md:166).  The paper
// gives no formulas; the readings are the textbook ones: colours 0 .. q-1 in the int8 spin plane,
// H = -sum_<ij> delta(c_i, c_j), bond between EQUAL colours with p = 1 - exp(-1/T) (k_bond_generic tests equality, so
// it serves unchanged with the Potts threshold), labelling as for the Ising model, every cluster assigned the colour
// floor(word q / 2^32) with word = 32-bit field `root` of the TAG_FLIP stream (call root >> 2, word root & 3).
// Observables: E = -#(equal East / South pairs), M = q max_c n_c - N.
#pragma once
#include "sw_common.cuh"
#include "sw_generic.cuh"

namespace sw {

constexpr int POTTS_MAX_Q = 127;          // colours live in int8

// 32-bit field idx of the (t, tag) stream: word idx & 3 of call idx >> 2
__device__ __forceinline__ uint32_t potts_word(uint32_t idx, uint32_t tlo, uint32_t thi, uint32_t tag,
                                               const PhiloxKey& key) {
    const uint4 r = philox4x32_10(idx >> 2, tlo, thi, tag, key);
    const uint32_t s = idx & 3u;
    return s == 0 ? r.x : s == 1 ? r.y : s == 2 ? r.z : r.w;
}

// start configuration: colour[i] = floor(word_INIT(i) q / 2^32); one thread per call = 4 sites
__global__ void __launch_bounds__(GEN_THREADS)
k_init_potts(int8_t* __restrict__ colours, const Lat* __restrict__ lat, int q, int N) {
    const int g = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (4 * g >= N) return;
    const Lat la = lat[blockIdx.y];
    const PhiloxKey key(la.key0, la.key1);
    const uint4 r = philox4x32_10((uint32_t)g, 0u, 0u, TAG_INIT, key);
    const uint32_t w[4] = { r.x, r.y, r.z, r.w };
    int8_t* s = colours + (size_t)blockIdx.y * N;
#pragma unroll
    for (int k = 0; k < 4; ++k)
        if (4 * g + k < N) s[4 * g + k] = (int8_t)__umulhi(w[k], (uint32_t)q);
}

// assignment (generalised): every site takes the colour drawn for its cluster's label (labels flat)
__global__ void __launch_bounds__(GEN_THREADS)
k_assign_potts(int8_t* __restrict__ colours, const int* __restrict__ label, const Lat* __restrict__ lat,
               const Ctl* __restrict__ ctl, int q, int N) {
    const int i = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (i >= N) return;
    const Lat la = lat[blockIdx.y];
    const PhiloxKey key(la.key0, la.key1);
    const unsigned long long t = ctl->t;
    const int r = label[(size_t)blockIdx.y * N + i];
    const uint32_t w = potts_word((uint32_t)r, (uint32_t)t, (uint32_t)(t >> 32), TAG_FLIP, key);
    colours[(size_t)blockIdx.y * N + i] = (int8_t)__umulhi(w, (uint32_t)q);
}

// observables (generalised): E = -#(equal East / South pairs); sites per colour into cnt[b][c]
__global__ void __launch_bounds__(GEN_THREADS)
k_observe_potts(const int8_t* __restrict__ colours, Rec* __restrict__ rec, int* __restrict__ cnt,
                const Ctl* __restrict__ ctl, int use_slot, int q, int L, int N, int nb) {
    __shared__ int s_cnt[POTTS_MAX_Q + 1];
    __shared__ int s_e;
    for (int c = threadIdx.x; c <= POTTS_MAX_Q; c += GEN_THREADS) s_cnt[c] = 0;
    if (threadIdx.x == 0) s_e = 0;
    __syncthreads();
    const int i = blockIdx.x * GEN_THREADS + threadIdx.x;
    int e = 0;
    const unsigned act = __ballot_sync(0xffffffffu, i < N);
    if (i < N) {
        const int8_t* s = colours + (size_t)blockIdx.y * N;
        const int y = i / L, x = i - y * L;
        const int v = s[i];
        e = -(int)(v == s[y * L + (x + 1 == L ? 0 : x + 1)]) - (int)(v == s[(y + 1 == L ? 0 : y + 1) * L + x]);
        const unsigned grp = __match_any_sync(act, v);
        if ((threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(&s_cnt[v & POTTS_MAX_Q], __popc(grp));
    }
    e = warp_sum_i(e);
    if ((threadIdx.x & 31) == 0 && e) atomicAdd(&s_e, e);
    __syncthreads();
    for (int c = threadIdx.x; c < q; c += GEN_THREADS)
        if (s_cnt[c]) atomicAdd(cnt + (size_t)blockIdx.y * q + c, s_cnt[c]);
    if (threadIdx.x == 0 && s_e) {
        Rec* r = rec + (use_slot ? (size_t)ctl->slot * nb : 0) + blockIdx.y;
        atomic_add_ll(&r->E, s_e);
    }
}

// M = q max_c n_c - N from the colour counts, which are cleared for the next sweep; one thread per lattice
__global__ void k_potts_finish(Rec* __restrict__ rec, int* __restrict__ cnt, const Ctl* __restrict__ ctl,
                               int use_slot, int q, int N, int nb) {
    for (int b = threadIdx.x; b < nb; b += blockDim.x) {
        int m = 0;
        for (int c = 0; c < q; ++c) { m = max(m, cnt[(size_t)b * q + c]); cnt[(size_t)b * q + c] = 0; }
        rec[(use_slot ? (size_t)ctl->slot * nb : 0) + b].M = (long long)q * m - N;
    }
}

} // namespace sw
