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
#include "sw_scan.cuh"

namespace sw {

constexpr int POTTS_MAX_Q = 127;          // colours live in int8

// Philox4x32-10 with the round keys advanced on the fly (2 registers instead of the 20 of PhiloxKey): for the
// kernels here, which draw once per cluster or per site next to other register-hungry work
__device__ __forceinline__ uint4 philox4x32_10_rk(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                  uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;
        const unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
        k0 += PHILOX_W0; k1 += PHILOX_W1;
    }
    return make_uint4(c0, c1, c2, c3);
}

// 32-bit field idx of the (t, tag) stream: word idx & 3 of call idx >> 2
__device__ __forceinline__ uint32_t potts_word(uint32_t idx, uint32_t tlo, uint32_t thi, uint32_t tag,
                                               uint32_t key0, uint32_t key1) {
    const uint4 r = philox4x32_10_rk(idx >> 2, tlo, thi, tag, key0, key1);
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
    const unsigned long long t = ctl->t;
    const int r = label[(size_t)blockIdx.y * N + i];
    const uint32_t w = potts_word((uint32_t)r, (uint32_t)t, (uint32_t)(t >> 32), TAG_FLIP, la.key0, la.key1);
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

// ---------------------------------------------------------------------------------------------------
// Fast path (L a multiple of 128): the fused bond + scan-line labelling kernel of sw_scan.cuh in its POTTS variant
// (k_bond_label<4, 64, FUSE, POTTS>: equal-colour masks by byte-wise compares of the int8 plane, same draws), then
// k_merge_nodes and k_roots_nodes, leaving the 16-bit tile-local root of every site and the node array of the open
// tile roots.  k_assign16_potts is the Potts counterpart of k_flip16: one
// colour per TILE ROOT in shared memory (a Philox call per root: closed roots draw for their own site index, open
// ones for the minimum site index under their root node), then every site looks its colour up by its 16-bit root.
// Also counts the clusters that span tiles and maximises their sizes, as k_flip16 does.
// ---------------------------------------------------------------------------------------------------
template <int NW, int TH>
__global__ void __launch_bounds__(NW * TH, 1536 / (NW * TH))
k_assign16_potts(int8_t* __restrict__ colours, const uint16_t* __restrict__ lab16, const int4* __restrict__ nodes,
                 const int* __restrict__ ocount, Rec* __restrict__ rec, const Lat* __restrict__ lat,
                 const Ctl* __restrict__ ctl, DivL dv, int q, int L, int N, int nb, int* __restrict__ cnt) {
    constexpr int TW = 32 * NW, SITES = TW * TH, THREADS = NW * TH;
    constexpr int CAP = 2 * (TW + TH);
    constexpr int OSTEPS = SITES / 8 / THREADS;      // = 4
    constexpr int LOG_TW = ilog2_c(TW);
    __shared__ uint8_t col[SITES];                   // colour of the tile root with local index l
    __shared__ uint4 sv[SITES / 8];                  // my sites' 16-bit roots, parked while the colours are drawn

    const int tid = threadIdx.x;
    const int tilesX = L / TW;
    const int ty = blockIdx.x / tilesX, tx = blockIdx.x - ty * tilesX;
    const int y0 = ty * TH, x0 = tx * TW;
    const int tilebase = y0 * L + x0;
    const size_t tile = (size_t)blockIdx.y * gridDim.x + blockIdx.x;

    uint4 v[OSTEPS];
#pragma unroll
    for (int k = 0; k < OSTEPS; ++k) {
        const int l = 8 * (k * THREADS + tid);
        v[k] = ld_stream_u4(lab16 + (size_t)blockIdx.y * N + (size_t)(y0 + (l >> LOG_TW)) * L + x0 + (l & (TW - 1)));
    }
    const int n = ocount[tile];
    const Lat la = lat[blockIdx.y];
    const unsigned long long t = ctl->t;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);
    uint32_t ncol[2] = { 0u, 0u };                   // my sites per colour, a byte each (at most 32): colours 0-3, 4-7

    // which of my 32 sites are tile roots (their 16-bit root is their own local index)
    uint32_t rootmask = 0;
#pragma unroll
    for (int k = 0; k < OSTEPS; ++k) {
        const int l = 8 * (k * THREADS + tid);
        const uint32_t w4[4] = { v[k].x, v[k].y, v[k].z, v[k].w };
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t r = (u & 1) ? (w4[u >> 1] >> 16) : (w4[u >> 1] & 0xFFFFu);
            rootmask |= (r == (uint32_t)(l + u) ? 1u : 0u) << (8 * k + u);
        }
        sv[k * THREADS + tid] = v[k];
    }
    while (rootmask) {                               // one Philox call per tile root
        const int b = __ffs(rootmask) - 1;
        rootmask &= rootmask - 1;
        const int l = 8 * ((b >> 3) * THREADS + tid) + (b & 7);
        const int g = tilebase + (l >> LOG_TW) * L + (l & (TW - 1));
        col[l] = (uint8_t)__umulhi(potts_word((uint32_t)g, tlo, thi, TAG_FLIP, la.key0, la.key1), (uint32_t)q);
    }
    __syncthreads();
    {   // open tile roots take the colour of their cluster root = the minimum site index under their root node
        const size_t lb = (size_t)blockIdx.y * gridDim.x * CAP;
        const int nodebase = blockIdx.x * CAP;
        int nroot = 0, big = 0;
        for (int e = tid; e < n; e += THREADS) {
            const int4 me = nodes[lb + nodebase + e];                  // (root node, size, min site, site of the tile root)
            const int R = me.x == nodebase + e ? me.z : nodes[lb + me.x].z;
            if (me.x == nodebase + e) { ++nroot; big = max(big, me.y); }
            const int delta = me.w - tilebase;
            const int ry = div_l(delta, dv);
            col[ry * TW + (delta - ry * L)] = (uint8_t)__umulhi(potts_word((uint32_t)R, tlo, thi, TAG_FLIP, la.key0, la.key1), (uint32_t)q);
        }
        if (tid < ((n + 31) & ~31)) {                                  // (whole warps)
            nroot = warp_sum_i(nroot); big = warp_max_i(big);
            if ((tid & 31) == 0) {
                Rec* r = rec + (size_t)ctl->slot * nb + blockIdx.y;
                if (nroot) atomic_add_ll(&r->ncl, nroot);
                if (big) atomic_max_ll(&r->maxcl, big);
            }
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < OSTEPS; ++k) {
        const int l = 8 * (k * THREADS + tid);
        const uint4 vk = sv[k * THREADS + tid];
        const uint32_t w4[4] = { vk.x, vk.y, vk.z, vk.w };
        uint32_t out[2] = { 0u, 0u };
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t r = (u & 1) ? (w4[u >> 1] >> 16) : (w4[u >> 1] & 0xFFFFu);
            out[u >> 2] |= (uint32_t)col[r] << (8 * (u & 3));
        }
        *reinterpret_cast<uint2*>(colours + (size_t)blockIdx.y * N + (size_t)(y0 + (l >> LOG_TW)) * L + x0 + (l & (TW - 1))) =
            make_uint2(out[0], out[1]);
        if (cnt) {                                   // (q <= 8) sites per colour, for M: equal bytes against the splat of the colour
#pragma unroll
            for (int c = 0; c < 8; ++c)
                if (c < q) {
                    const uint32_t pat = (uint32_t)c * 0x01010101u;
                    ncol[c >> 2] += (uint32_t)((__popc(__vcmpeq4(out[0], pat)) + __popc(__vcmpeq4(out[1], pat))) >> 3) << (8 * (c & 3));
                }
        }
    }
    if (cnt) {
        // the colour counts of the new configuration, a7 (the order parameter needs max_c n_c): one add per warp and colour
        // into shared memory, one per CTA into the lattice's counters (k_potts_finish turns them into M)
        __shared__ int s_ncol[8];
        if (tid < 8) s_ncol[tid] = 0;
        __syncthreads();
#pragma unroll
        for (int c = 0; c < 8; ++c)
            if (c < q) {
                const int n_c = warp_sum_i((int)((ncol[c >> 2] >> (8 * (c & 3))) & 0xFFu));
                if ((tid & 31) == 0 && n_c) atomicAdd(&s_ncol[c], n_c);
            }
        __syncthreads();
        if (tid < q && s_ncol[tid]) atomicAdd(cnt + (size_t)blockIdx.y * q + tid, s_ncol[tid]);
    }
}

// observables on rows (L a multiple of 16): 16 sites per thread, byte-wise compares (__vcmpeq4) with the East-
// shifted and the South words; colour counts through a shared-memory histogram (lanes of one colour add once)
__global__ void __launch_bounds__(GEN_THREADS)
k_observe_potts_rows(const int8_t* __restrict__ colours, Rec* __restrict__ rec, int* __restrict__ cnt,
                     const Ctl* __restrict__ ctl, int use_slot, int q, int L, int N, int nb) {
    // use_slot: 0 record 0 (sw_observables of a state no sweep produced), 1 the running sweep's slot, 2 the slot BEFORE it and
    // the energy only (end of a sw_sweep call on the fast path: E of a sweep otherwise comes out of the next sweep's bond test)
    __shared__ int s_cnt[POTTS_MAX_Q + 1];
    __shared__ int s_e;
    for (int c = threadIdx.x; c <= POTTS_MAX_Q; c += GEN_THREADS) s_cnt[c] = 0;
    if (threadIdx.x == 0) s_e = 0;
    __syncthreads();
    const int g = blockIdx.x * GEN_THREADS + threadIdx.x;              // group of 16 sites (N / 16 is a multiple of 32)
    int e = 0;
    const bool on = g * 16 < N;                                        // (warp-uniform: N / 16 is a multiple of 32)
    uint32_t w[4] = { 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu, 0xFFFFFFFFu };   // 0xFF: no colour
    if (on) {
        const int8_t* s = colours + (size_t)blockIdx.y * N;
        const int i = g * 16;
        const int y = i / L, x = i - y * L;
        const uint4 a = *reinterpret_cast<const uint4*>(s + i);
        const uint4 b = *reinterpret_cast<const uint4*>(s + (size_t)(y + 1 == L ? 0 : y + 1) * L + x);
        const uint32_t nx = (uint8_t)s[(size_t)y * L + (x + 16 == L ? 0 : x + 16)];
        const uint32_t so[4] = { b.x, b.y, b.z, b.w };
        w[0] = a.x; w[1] = a.y; w[2] = a.z; w[3] = a.w;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t east = __funnelshift_r(w[k], k < 3 ? w[k < 3 ? k + 1 : 3] : nx, 8);
            e -= (__popc(__vcmpeq4(w[k], east)) + __popc(__vcmpeq4(w[k], so[k]))) >> 3;
        }
    }
    if (use_slot == 2) {
        // (energy only)
    } else if (q <= 8) {
        // few colours: sites of colour c among my 16 = equal bytes against the splat of c; one add per warp and colour
        for (int c = 0; c < q; ++c) {
            const uint32_t pat = (uint32_t)c * 0x01010101u;
            int n = (__popc(__vcmpeq4(w[0], pat)) + __popc(__vcmpeq4(w[1], pat)) +
                     __popc(__vcmpeq4(w[2], pat)) + __popc(__vcmpeq4(w[3], pat))) >> 3;
            n = warp_sum_i(n);
            if ((threadIdx.x & 31) == 0 && n) atomicAdd(&s_cnt[c], n);
        }
    } else if (on) {
#pragma unroll
        for (int k = 0; k < 4; ++k)
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int c = (w[k] >> (8 * u)) & POTTS_MAX_Q;
                const unsigned grp = __match_any_sync(0xffffffffu, c);
                if ((threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(&s_cnt[c], __popc(grp));
            }
    }
    e = warp_sum_i(e);
    if ((threadIdx.x & 31) == 0 && e) atomicAdd(&s_e, e);
    __syncthreads();
    for (int c = threadIdx.x; c < q; c += GEN_THREADS)
        if (use_slot != 2 && s_cnt[c]) atomicAdd(cnt + (size_t)blockIdx.y * q + c, s_cnt[c]);
    if (threadIdx.x == 0 && s_e) {
        const uint32_t slot = use_slot == 2 ? (ctl->slot == 0 ? ctl->cap - 1 : ctl->slot - 1) : ctl->slot;
        Rec* r = rec + (use_slot ? (size_t)slot * nb : 0) + blockIdx.y;
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
