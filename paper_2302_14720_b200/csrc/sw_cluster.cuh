// sw_cluster.cuh -- small lattices (the paper's own sizes): a whole sw_sweep(h, n) call inside ONE kernel.
//
// A lattice of at most 8 tiles is swept by one thread-block CLUSTER, one CTA per tile, all n sweeps inside the kernel: the
// four dependent steps of a sweep (a1+a2 bond_label_persist -- the text of k_bond_label --, a3 merge, a3 roots, a4-a6
// assignment) are separated by the cluster's hardware barrier (barrier.cluster, ~1 us for 8 CTAs) instead of by kernel
// boundaries (4 launches of ~4 us each even when replayed from a graph with programmatic dependent launches: what a sweep of
// L <= 256 cost).  A batch runs one cluster per lattice, each at its own pace: nothing is shared between lattices, so the
// sweep index and the series slot are computed from the call's first ones instead of being read from Ctl.
// Everything a CTA reads that another CTA of the cluster wrote goes to L2 (ld.global.cg / atomics), never through L1 or
// the read-only path; the barrier orders it (release / acquire at cluster scope).  Same RNG convention, same results: the
// parity tests run unchanged.
#pragma once
#include "sw_scan.cuh"

namespace sw {

__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t ld_cg_u16(const uint16_t* p) {
    uint16_t v; asm volatile("ld.global.cg.u16 %0, [%1];" : "=h"(v) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ uint4 ld_cg_u4(const void* p) {
    uint4 v; asm volatile("ld.global.cg.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory"); return v;
}
__device__ __forceinline__ int ld_cg_i32(const int* p) {
    int v; asm volatile("ld.global.cg.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}

// a1 + a2 for the CTA's own tile: the body of k_bond_label with the sweep's control values as arguments and the spins
// loaded through L2 (the plane is rewritten by the assignment step of the same kernel).  Returns the tile's number of
// open roots (= ocount[tile]).
__device__ __forceinline__ uint32_t ld_cg_u32(const uint32_t* p) {
    uint32_t v; asm volatile("ld.global.cg.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
template <int NW, int TH, int BAND_T>
__device__ __forceinline__ int
bond_label_persist(const uint32_t* sbits, uint32_t* bondE, uint32_t* bondS, uint16_t* __restrict__ lab16, int4* __restrict__ nodes,
                   int* __restrict__ ocount, uint16_t* __restrict__ bslot, Rec* __restrict__ rec, const Lat* __restrict__ lat,
                   const unsigned long long t_now, const uint32_t slot_now, const uint32_t cap_now,
                   int L, int N, int words, int nb, int obs_prev) {
    constexpr bool FUSE = true, POTTS = false;
#define BL_LDSPIN(p, i) ld_cg_u32((p) + (i))
#define BL_T t_now
#define BL_SLOT slot_now
#define BL_CAP cap_now
#include "sw_bond_label_body.inc"
#undef BL_LDSPIN
#undef BL_T
#undef BL_SLOT
#undef BL_CAP
    return s_nopen;                                     // (final since the barrier in front of phase 6)
}

// a3 for the CTA's own tile: its South row against the North row of the tile below, its East column against the West
// column of the tile to the East (k_merge_nodes, one tile)
template <int TW, int TH, int THREADS>
__device__ __forceinline__ void merge_tile(int4* nd, const uint16_t* bs, const int ta, const int tilesX, const int tilesY, const int tid) {
    constexpr int CAP = 2 * (TW + TH), PER = TW + TH;
    const int r = ta / tilesX, c = ta - r * tilesX;
    for (int j = tid; j < PER; j += THREADS) {
        int ka, tb, kb;
        if (j < TW) { ka = TW + j;                 tb = (r + 1 == tilesY ? 0 : r + 1) * tilesX + c; kb = j; }
        else        { ka = 2 * TW + TH + (j - TW); tb = r * tilesX + (c + 1 == tilesX ? 0 : c + 1); kb = 2 * TW + (j - TW); }
        const int sa = (int)ld_cg_u16(bs + (size_t)ta * CAP + ka), sb = (int)ld_cg_u16(bs + (size_t)tb * CAP + kb);
        if (sa != 0xFFFF) nd_union<true>(nd, ta * CAP + sa, tb * CAP + sb);
    }
}

// a4-a6 for the CTA's own tile (k_flip16<NW, TH, BITS, FUSED> with any number of threads): one decision bit per tile
// root in shared memory -- drawn here: word w of the decision plane is word w & 3 of Philox call (w >> 2, t, TAG_FLIP) --,
// the open roots take their cluster root's, every site looks its bit up by its 16-bit root; the new spins go out bit-packed
template <int NW, int TH, int THREADS>
__device__ __forceinline__ void flip_tile(uint32_t* sbits, const uint16_t* lab16, const int4* nd, const int n, Rec* rc,
                                          const Lat la, const unsigned long long t, const DivL dv, const int L, const int N) {
    constexpr int TW = 32 * NW, SITES = TW * TH, CAP = 2 * (TW + TH), LOG_TW = ilog2_c(TW);
    __shared__ uint32_t dec[TH * NW];
    const int tid = threadIdx.x;
    const int tilesX = L / TW;
    const int ty = blockIdx.x / tilesX, tx = blockIdx.x - ty * tilesX;
    const int y0 = ty * TH, x0 = tx * TW;
    const int tilebase = y0 * L + x0;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);
    const PhiloxKey key(la.key0, la.key1);
    // my sites' 16-bit roots and my open root's node: the loads are issued first, the Philox calls run under them
    constexpr int OSTEPS = (SITES / 8 + THREADS - 1) / THREADS;
    uint4 v[OSTEPS];
#pragma unroll
    for (int k = 0; k < OSTEPS; ++k) {
        const int l = 8 * (k * THREADS + tid);
        if (l < SITES) v[k] = ld_cg_u4(lab16 + (size_t)blockIdx.y * N + (size_t)(y0 + (l >> LOG_TW)) * L + x0 + (l & (TW - 1)));
    }
    int4 me0 = make_int4(0, 0, 0, 0);
    if (tid < n) me0 = ld_cg_int4(nd + blockIdx.x * CAP + tid);
    for (int i = tid; i < TH * NW; i += THREADS) {
        const int row = i / NW, wx = i - row * NW;
        const int w = (y0 + row) * (L >> 5) + (x0 >> 5) + wx;            // my word of the decision plane
        const uint4 r = philox4x32_10((uint32_t)w >> 2, tlo, thi, TAG_FLIP, key);
        dec[i] = (w & 2) ? ((w & 1) ? r.w : r.z) : ((w & 1) ? r.y : r.x);
    }
    __syncthreads();
    {
        const int nodebase = blockIdx.x * CAP;
        int nroot = 0, big = 0;
        for (int e0 = 0; e0 < n; e0 += THREADS) {                          // (whole warps: the reductions below)
            const int e = e0 + tid;
            if (e < n) {
                const int4 me = e0 == 0 ? me0 : ld_cg_int4(nd + nodebase + e);   // (root node, size, min site, site of the tile root)
                const int R = me.x == nodebase + e ? me.z : ld_cg_i32(&nd[me.x].z);
                if (me.x == nodebase + e) { ++nroot; big = max(big, me.y); }
                const uint4 r = philox4x32_10((uint32_t)R >> 7, tlo, thi, TAG_FLIP, key);
                const uint32_t wsel = (R & 64) ? ((R & 32) ? r.w : r.z) : ((R & 32) ? r.y : r.x);
                const int delta = me.w - tilebase;
                const int ry = div_l(delta, dv);
                const int l = ry * TW + (delta - ry * L);
                if ((wsel >> (R & 31)) & 1u) atomicOr(&dec[l >> 5], 1u << (l & 31));
                else                         atomicAnd(&dec[l >> 5], ~(1u << (l & 31)));
            }
        }
        nroot = warp_sum_i(nroot); big = warp_max_i(big);
        if ((tid & 31) == 0) {
            if (nroot) atomic_add_ll(&rc->ncl, nroot);
            if (big) atomic_max_ll(&rc->maxcl, big);
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < OSTEPS; ++k) {
        const int l = 8 * (k * THREADS + tid);
        if (l >= SITES) break;
        const size_t gsite = (size_t)blockIdx.y * N + (size_t)(y0 + (l >> LOG_TW)) * L + x0 + (l & (TW - 1));
        const uint32_t w4[4] = { v[k].x, v[k].y, v[k].z, v[k].w };
        uint32_t b8 = 0;                                                   // bit u: site l + u goes up
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t r = (u & 1) ? (w4[u >> 1] >> 16) : (w4[u >> 1] & 0xFFFFu);
            b8 |= (__funnelshift_r(dec[r >> 5], 0u, r) & 1u) << u;
        }
        reinterpret_cast<uint8_t*>(sbits)[gsite >> 3] = (uint8_t)b8;
    }
}

// grid = (tiles per lattice, nb), cluster = (tiles per lattice, 1, 1); sweeps t0 .. t0 + nsweeps - 1 into the series slots
// 0, 1, .. (mod cap) -- sw_sweep zeroes slot 0 before the launch and sets Ctl after it.  obs_first: the first sweep's bond
// test also delivers E, M of the configuration before it (never within one sw_sweep call: 0).
template <int NW, int TH, int BAND_T>
__global__ void __launch_bounds__(NW * TH * (32 / BAND_T))
k_sweeps_cluster(uint32_t* sbits, uint32_t* bondE, uint32_t* bondS, uint16_t* lab16, int4* nodes, int* ocount, uint16_t* bslot,
                 Rec* rec, const Lat* __restrict__ lat, Mom* mom, const unsigned long long t0, const uint32_t cap,
                 const long long nsweeps, const int obs_first, const DivL dv, const int L, const int N, const int words, const int nb) {
    constexpr int TW = 32 * NW, THREADS = NW * TH * (32 / BAND_T), CAP = 2 * (TW + TH);
    constexpr int WPT = THREADS / 32 < 4 ? THREADS / 32 : 4;              // warps that walk the tile's open pieces
    const int tid = threadIdx.x, tile = blockIdx.x, tiles = gridDim.x, b = blockIdx.y;
    int4* nd = nodes + (size_t)b * tiles * CAP;
    const uint16_t* bs = bslot + (size_t)b * tiles * CAP;
    const Lat la = lat[b];
    for (long long k = 0; k < nsweeps; ++k) {
        const unsigned long long t = t0 + (unsigned long long)k;
        const uint32_t slot = (uint32_t)(k % cap), next = slot + 1 == cap ? 0u : slot + 1, prev = slot == 0 ? cap - 1 : slot - 1;
        // a1 + a2 (its first barrier comes after its shared-memory set-up; the sweep before ended with a cluster barrier)
        const int nopen = bond_label_persist<NW, TH, BAND_T>(sbits, bondE, bondS, lab16, nodes, ocount, bslot, rec, lat,
                                                             t, slot, cap, L, N, words, nb, (k > 0 || obs_first) ? 1 : 0);
        cluster_sync_all();
        // the record of sweep k - 1 is complete now (its E, M came with this sweep's bond test): running moments, in sweep
        // order, one thread per lattice; then the slot of sweep k + 1 is cleared (nobody touches it before three more barriers;
        // with a ring of two slots it is the slot just consumed)
        if (tile == 0 && tid == 0) {
            if (k > 0) {
                const unsigned long long* rp = reinterpret_cast<const unsigned long long*>(rec + (size_t)prev * nb + b);
                Mom m = mom[b];
                mom_add(m, (long long)ld_cg64(rp), (long long)ld_cg64(rp + 1), N);
                mom[b] = m;
            }
            rec[(size_t)next * nb + b] = Rec{0, 0, 0, 0};
        }
        merge_tile<TW, TH, THREADS>(nd, bs, tile, L / TW, L / TH, tid);    // a3
        cluster_sync_all();
        if (tid < 32 * WPT)                                                // a3: sizes and minimum sites of the spanning clusters
            roots_warp<CAP, true>(nd, nopen, tile, tid >> 5, WPT, tid & 31);
        cluster_sync_all();
        flip_tile<NW, TH, THREADS>(sbits, lab16, nd, nopen, rec + (size_t)slot * nb + b, la, t, dv, L, N);
        cluster_sync_all();
    }
}

} // namespace sw
