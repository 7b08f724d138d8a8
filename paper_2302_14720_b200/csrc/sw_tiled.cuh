// sw_tiled.cuh -- row kernels on the int8 spin plane and flat int32 labels (lattice side a multiple of 64):
// the stand-alone stages of the unfused path 6 (per-stage timing, BASELINE config 3) and of path 11 (the paper's
// labelling, sw_equiv.cuh).
//
//   a1 k_bond_rows      Philox bond draws, one thread per bit-plane word (32 sites, 16 Philox calls)
//   a6 k_flip_rows      spins = gather(D, label); labels are flat
//   a7 k_energy_rows    energy of the new configuration from sign masks + popc
#pragma once
#include "sw_common.cuh"

namespace sw {

constexpr int ROW_THREADS = 256;

// ---------------------------------------------------------------------------------------------
// a1 bond formation, PAPER.md:37-39 (section 2.1).  Thread w owns sites 32w .. 32w+31 of one row.
// Equal-spin masks come from the sign bits of the int8 spins; the draw masks from 16 Philox calls
// (call c covers sites 2c, 2c+1: words x,y = East,South of the even site, z,w of the odd one).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ROW_THREADS)
k_bond_rows(const int8_t* __restrict__ spins, uint32_t* __restrict__ bondE, uint32_t* __restrict__ bondS,
            const Lat* __restrict__ lat, const Ctl* __restrict__ ctl, int L, int N, int words,
            Rec* __restrict__ rec, int nb, int obs_prev) {
    const int w = blockIdx.x * ROW_THREADS + threadIdx.x;
    if (w >= words) return;                          // (words is a multiple of 32 here: whole warps leave)
    const int wpr = L >> 5;
    const int y = w / wpr, xw = w - y * wpr;
    const int8_t* s = spins + (size_t)blockIdx.y * N;
    const int8_t* row  = s + (size_t)y * L + xw * 32;
    const int8_t* rowS = s + (size_t)(y + 1 == L ? 0 : y + 1) * L + xw * 32;
    const uint4 a0 = *reinterpret_cast<const uint4*>(row),  a1 = *reinterpret_cast<const uint4*>(row + 16);
    const uint4 b0 = *reinterpret_cast<const uint4*>(rowS), b1 = *reinterpret_cast<const uint4*>(rowS + 16);
    const int8_t nx = s[(size_t)y * L + (xw + 1 == wpr ? 0 : (xw + 1) * 32)];
    const uint32_t own = neg_mask32(a0, a1), south = neg_mask32(b0, b1);
    const uint32_t eastm = (own >> 1) | (nx < 0 ? 0x80000000u : 0u);
    const uint32_t eqE = ~(own ^ eastm), eqS = ~(own ^ south);
    if (obs_prev) {     // scan path: E, M of the configuration the previous sweep left (see k_bond_label)
        const int eo = warp_sum_i(64 - 2 * (__popc(eqE) + __popc(eqS)));
        const int mo = warp_sum_i(32 - 2 * __popc(own));
        if ((threadIdx.x & 31) == 0) {
            Rec* rp = rec + (size_t)(ctl->slot == 0 ? ctl->cap - 1 : ctl->slot - 1) * nb + blockIdx.y;
            if (eo) atomic_add_ll(&rp->E, eo);
            if (mo) atomic_add_ll(&rp->M, mo);
        }
    }

    const Lat la = lat[blockIdx.y];
    const PhiloxKey key(la.key0, la.key1);
    const unsigned long long t = ctl->t;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);
    uint32_t dE = 0, dS = 0;
#pragma unroll
    for (int c = 0; c < 16; ++c) {
        const uint4 r = philox4x32_10((uint32_t)w * 16u + c, tlo, thi, TAG_BOND, key);
        dE |= (r.x < la.thr ? 1u : 0u) << (2 * c) | (r.z < la.thr ? 1u : 0u) << (2 * c + 1);
        dS |= (r.y < la.thr ? 1u : 0u) << (2 * c) | (r.w < la.thr ? 1u : 0u) << (2 * c + 1);
    }
    bondE[(size_t)blockIdx.y * words + w] = eqE & dE;
    bondS[(size_t)blockIdx.y * words + w] = eqS & dS;
}

// ---------------------------------------------------------------------------------------------
// a6 assignment, PAPER.md:57 (section 2.4): 16 sites per thread; labels are flat.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ROW_THREADS)
k_flip_rows(int8_t* __restrict__ spins, const int* __restrict__ label, const uint32_t* __restrict__ D,
            Rec* __restrict__ rec, const Ctl* __restrict__ ctl, int N, int words, int nb) {
    const int g = blockIdx.x * ROW_THREADS + threadIdx.x;       // group of 16 sites
    int m = 0;
    if (g * 16 < N) {
        const int* lab = label + (size_t)blockIdx.y * N + (size_t)g * 16;
        const uint32_t* d = D + (size_t)blockIdx.y * words;
        uint32_t out[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint4 v = ld_stream_u4(lab + q * 4);
            const uint32_t r[4] = { v.x, v.y, v.z, v.w };
            uint32_t o = 0;
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t up = (__ldg(d + (r[k] >> 5)) >> (r[k] & 31)) & 1u;
                o |= (up ? 0x01u : 0xFFu) << (8 * k);
                m += up ? 1 : -1;
            }
            out[q] = o;
        }
        st_stream_u4(spins + (size_t)blockIdx.y * N + (size_t)g * 16, make_uint4(out[0], out[1], out[2], out[3]));
    }
    m = warp_sum_i(m);
    if ((threadIdx.x & 31) == 0 && m) atomic_add_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].M, m);
}

// ---------------------------------------------------------------------------------------------
// a7 energy, PAPER.md:63 (section 2.5): E = -sum over East and South edges of s_i s_j
//    = (#edges) - 2 (#equal pairs); 32 sites per thread from sign masks.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ROW_THREADS)
k_energy_rows(const int8_t* __restrict__ spins, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
              int L, int N, int words, int nb) {
    const int w = blockIdx.x * ROW_THREADS + threadIdx.x;
    int e = 0;
    if (w < words) {
        const int wpr = L >> 5;
        const int y = w / wpr, xw = w - y * wpr;
        const int8_t* s = spins + (size_t)blockIdx.y * N;
        const int8_t* row  = s + (size_t)y * L + xw * 32;
        const int8_t* rowS = s + (size_t)(y + 1 == L ? 0 : y + 1) * L + xw * 32;
        const uint4 a0 = *reinterpret_cast<const uint4*>(row),  a1 = *reinterpret_cast<const uint4*>(row + 16);
        const uint4 b0 = *reinterpret_cast<const uint4*>(rowS), b1 = *reinterpret_cast<const uint4*>(rowS + 16);
        const int8_t nx = s[(size_t)y * L + (xw + 1 == wpr ? 0 : (xw + 1) * 32)];
        const uint32_t own = neg_mask32(a0, a1), south = neg_mask32(b0, b1);
        const uint32_t eastm = (own >> 1) | (nx < 0 ? 0x80000000u : 0u);
        e = 64 - 2 * (__popc(~(own ^ eastm)) + __popc(~(own ^ south)));
    }
    e = warp_sum_i(e);
    if ((threadIdx.x & 31) == 0 && e) atomic_add_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].E, e);
}

} // namespace sw
