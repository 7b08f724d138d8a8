// sw_scan.cuh -- the fast path (lattice side a multiple of 64): 128 x 64 tiles above L = 1024, 64 x 32 tiles up to it.
//
// Stage map; one CTA per tile of TW x TH sites, TW = 32 * NW; the tile is NW x TH / BAND blocks of
// 32 x BAND sites, one warp each (BAND = 32: one thread per 32-site word; BAND = 8: four threads per word -- small lattices).
//   a1+a2 k_bond_label<NW, TH, FUSE, POTTS, BAND>
//       phase 1  per 32-site word: the word's spins from the BIT-PACKED plane (FUSE; bit 1 = +1; the int8 plane is derived
//                on demand, sw_spins), 16 Philox4x32-10 calls, bond words to shared memory and to the canonical global
//                bit-planes; E, M of the previous sweep's configuration from the same equal-pair masks; the bonds that enter
//                the tile from its North and West neighbours are recomputed (TW/2 + TH extra calls)
//       phase 2  scan-line labelling, lane = column, the block's rows in sequence, uniform control flow: runs of East bonds
//                from bit tricks on the row's bond word; a run takes the label of the first of its sites that has a South
//                bond from the row above (one shuffle), or opens a new label (its head's index); where another site of the
//                run is bonded to a different label above, the lane notes the row in a bit mask; after the block every lane
//                unites the pairs of its column (atomicMin hooking; hooked nodes go into a tile-wide list)
//       phase 3  seams between blocks (East bonds across strips, South bonds across band seams); every site counted at its label
//       phase 3b the label nodes (heads of runs with no bond from above) are counted; the hooked ones point at their roots and
//                hand them their counts
//       phase 4  per site: root = parent(parent(site)) -> 16-bit tile-local root to global memory (2 B / site); largest count
//       phase 5  border sites with a bond across the tile edge claim their root: node (parent, size, min site, site), slot
//       phase 6  per border site with a bond across the tile edge: the slot of its root
//   a3    k_merge_nodes (union-find over the nodes of neighbouring tiles), k_roots_nodes (sizes and minimum
//         site index of the clusters that span tiles)
//   a4-a6 k_flip16<NW, TH, BITS, FUSED>: one decision bit per tile root in shared memory, spins = lookup by 16-bit root,
//         written bit-packed (BITS: a byte per 8 sites) or as int8 (unfused path 6); on 128 x 64 tiles of large lattices the
//         TMA-staged, warp-specialised k_flip16_tma (sw_flip_tma.cuh) does the same;
//         k_labels16<NW, TH>: flat int32 labels from the 16-bit roots, on demand (sw_labels)
//   a7    E, M: by-product of the next sweep's bond test, k_observe_bits / k_observe_rows at the end of a call; cluster count
//         and largest cluster: k_bond_label (closed roots, largest tile-local count) + the assignment kernel (root nodes)
#pragma once
#include "sw_common.cuh"

namespace sw {

#ifndef SCAN_UNROLL_N
#define SCAN_UNROLL_N 32
#endif
constexpr int SCAN_UNROLL = SCAN_UNROLL_N;      // rows of the scan loop unrolled together
constexpr int BAND = 32;                        // rows a warp walks by default; a tile is TH / BAND bands of NW strips
constexpr uint32_t OPEN_BIT = 0x40000000u;      // bit 30 of a root's word: the cluster has a bond across the tile edge
// A root's word: bits 0 .. LS-1 tile-local index (LS = log2 of the sites per tile <= 14), bits LS .. 2 LS the
// cluster size (<= 2^LS), bit 30 open.
__host__ __device__ constexpr int ilog2_c(int v) { return v <= 1 ? 0 : 1 + ilog2_c(v >> 1); }

// ---- the shared parent array of k_bond_label -------------------------------------------------------------
// One 32-bit word per site of the tile:
//   bits 16 .. 29  parent (tile-local index); a root points at itself
//   bits  0 .. 13  sites counted at this node: every run adds its length to the label it takes (phase 2); the
//                  flatten (phase 3b) moves the counts of the nodes that were hooked to their roots, so that a
//                  root ends up with the size of its tile-local cluster
//   bit  14        CLAIMED (roots with a bond across the tile edge, phase 5): the low 14 bits now hold the root's
//                  slot in the tile's node list instead of the count
// The parent sits in the HIGH half so that hooking "larger under smaller" stays one atomicMin on the whole
// word: (b << 16) is below every word whose parent is above b.  The count the atomicMin wipes out comes back
// in its return value and is added again by the thread that hooked.
// All accesses go through the shared window (32-bit addresses, ld / st / atom / red .shared): word x sits at
// par_s + 4 x, its parent at par_s + 4 x + 2.
constexpr uint32_t CLAIMED16 = 0x4000u, CNT16 = 0x3FFFu;

__device__ __forceinline__ uint32_t lds_u16(uint32_t a) {
    uint16_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=h"(v) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ uint32_t lds_u32(uint32_t a) {
    uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ uint4 lds_u128(uint32_t a) {
    uint4 v; asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ void sts_u16(uint32_t a, uint32_t v) {
    asm volatile("st.shared.u16 [%0], %1;" :: "r"(a), "h"((uint16_t)v) : "memory");
}
__device__ __forceinline__ void sts_u128(uint32_t a, uint4 v) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" :: "r"(a), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
__device__ __forceinline__ void red_add_s(uint32_t a, uint32_t v) {
    asm volatile("red.shared.add.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ uint32_t atom_min_s(uint32_t a, uint32_t v) {
    uint32_t o; asm volatile("atom.shared.min.u32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory"); return o;
}
__device__ __forceinline__ uint32_t atom_or_s(uint32_t a, uint32_t v) {
    uint32_t o; asm volatile("atom.shared.or.b32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory"); return o;
}

__device__ __forceinline__ int sc_find(uint32_t par_s, int x) {
    int p = (int)lds_u16(par_s + 4u * x + 2u);
    while (p != x) { x = p; p = (int)lds_u16(par_s + 4u * x + 2u); }
    return x;
}
// unite the trees of a and b (any nodes); hooking "larger under smaller" with atomicMin so the root of a
// component is its minimum index whatever the interleaving.  A node stops being a root exactly once, and the
// call whose atomicMin did it (the return value still shows the node as its own parent) returns that node --
// at most one per call, NO_NODE otherwise.  Phase 3b flattens exactly these hooked nodes: ~0.03 per site at T_c,
// against ~0.2 label nodes per site.
constexpr int NO_NODE = 0xFFFF;
__device__ __forceinline__ uint32_t atom_add_s(uint32_t a, uint32_t v) {
    uint32_t o; asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(o) : "r"(a), "r"(v) : "memory"); return o;
}
// the tile's list of hooked nodes (phase 3b flattens from it with all threads); the counter runs on past the capacity
// (it also gives the number of roots), and phase 3b then visits every label node instead
struct HookList { uint32_t items_s, count_s; int cap; uint32_t one; };     // (shared-window addresses; one = 1)
__device__ __forceinline__ void hooked(const HookList& hk, int node) {
    if (node == NO_NODE) return;
    // (the increment is a 1 that ptxas cannot prove to be one -- `one` comes from a kernel argument: it would otherwise
    // turn the add into a warp-aggregated one -- vote, popc, shuffle: 20 instructions -- for the few lanes that get here
    // together)
    const int pos = (int)atom_add_s(hk.count_s, hk.one);
    if (pos < hk.cap) sts_u16(hk.items_s + 2u * pos, (uint32_t)node);
}
__device__ __forceinline__ int sc_union(uint32_t par_s, int a, int b) {
    while (a != b) {
        if (a < b) { const int s = a; a = b; b = s; }      // a is the larger
        const uint32_t nv = (uint32_t)b << 16;
        const uint32_t old = atom_min_s(par_s + 4u * a, nv);
        if (old > nv && (old & 0xFFFFu)) red_add_s(par_s + 4u * a, old & 0xFFFFu);   // the count the minimum replaced
        const int p = (int)(old >> 16);
        if (p == a) return a;                               // a was a root: hooked under b
        a = p;                                              // a had parent p: unite that with b
    }
    return NO_NODE;
}
// point a hooked node at its root and hand it the node's count
__device__ __forceinline__ void sc_flatten(uint32_t par_s, int n) {
    const uint32_t wn = lds_u32(par_s + 4u * n);
    const int p0 = (int)(wn >> 16);
    int r = p0, q = (int)lds_u16(par_s + 4u * r + 2u);
    while (q != r) { r = q; q = (int)lds_u16(par_s + 4u * r + 2u); }
    if (r != p0) sts_u16(par_s + 4u * n + 2u, (uint32_t)r);
    if (wn & 0xFFFFu) red_add_s(par_s + 4u * r, wn & 0xFFFFu);    // (a hooked node receives nothing any more)
}

// exact v / d for 0 <= v < 2^30 with a host-made magic (m, p): q = (v * m) >> p
struct DivL { uint32_t m; int p; int d; };
__device__ __forceinline__ int div_l(int v, const DivL& D) {
    return (int)(((unsigned long long)(uint32_t)v * D.m) >> D.p);
}

// FUSE = true: phase 1 draws the bonds (a1 fused into a2).  FUSE = false: phase 1 reads the bond planes
// that k_bond_rows (or a test) wrote -- per-stage timing (BASELINE config 3) and labelling-only tests.
// POTTS (with FUSE; sw_potts.cuh): `sbits` is the int8 COLOUR plane; a bond needs equal colours (byte compares).
// BAND_T: rows of the block a warp scans (32: one thread per 32-site word; 8: four threads per word, each with a quarter
// of the word's Philox calls -- the variant for small lattices, whose sweep time is the latency of ONE tile through this
// kernel: 4 x less serial work per warp).
template <int NW, int TH, bool FUSE, bool POTTS = false, int BAND_T = 32>
__global__ void __launch_bounds__(NW * TH * (32 / BAND_T))
k_bond_label(const uint32_t* __restrict__ sbits, uint32_t* bondE, uint32_t* bondS,
             uint16_t* __restrict__ lab16, int4* __restrict__ nodes, int* __restrict__ ocount,
             uint16_t* __restrict__ bslot,
             Rec* __restrict__ rec, const Lat* __restrict__ lat, const Ctl* __restrict__ ctl,
             int L, int N, int words, int nb, int obs_prev) {
    pdl_wait();
    constexpr int BAND = BAND_T;                // (shadows the default: rows per warp block in this instantiation)
    constexpr int TPW = 32 / BAND;              // threads per 32-site word (one warp per 32 x BAND block)
    constexpr int TW = 32 * NW, SITES = TW * TH, WORDS = NW * TH, THREADS = WORDS * TPW;
    constexpr int CAP = 2 * (TW + TH);
    static_assert(TPW == 1 || TPW == 2 || TPW == 4, "threads per word");
    constexpr int HKCAP = 1024;                 // hooked nodes the tile can list (~250 at T_c)
    static_assert(TH % BAND == 0 && TH <= 64 && SITES <= 8192 && CAP < 0x3FFF, "tile shape");
    extern __shared__ __align__(16) uint32_t par[];  // [SITES] (see above); dynamic: 32 KB at 128 x 64
    __shared__ uint2 es[TH * NW];              // [row][strip] = (East word, South word)
    __shared__ uint16_t hkitems[HKCAP];        // nodes hooked in phases 2 and 3
    __shared__ uint32_t nIn[NW];               // South bonds entering from the tile above, per strip
    __shared__ uint32_t wIn[2];                // East bonds entering from the tile to the West, bit = row
    __shared__ int s_nopen, s_max, s_nlab, s_nhook, s_obs[2];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lanebit = 1u << lane, lt = lanebit - 1u;
    const int tilesX = L / TW;
    const int ty = blockIdx.x / tilesX, tx = blockIdx.x - ty * tilesX;
    const int y0 = ty * TH, x0 = tx * TW;
    const int wprL = L >> 5;
    // FUSE: the spins come bit-packed (bit 1 = +1; word w = sites 32w .. 32w+31), 1/8 of the int8 plane's bytes
    const uint32_t* sb = sbits + (size_t)blockIdx.y * words;
    const int8_t* col = reinterpret_cast<const int8_t*>(sbits) + (size_t)blockIdx.y * N;   // (POTTS)
    const Lat la = lat[blockIdx.y];
    const unsigned long long t = ctl->t;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);

    if (tid < NW) nIn[tid] = 0;
    if (tid == 0) { wIn[0] = 0; wIn[1] = 0; s_nopen = 0; s_max = 0; s_nlab = 0; s_nhook = 0; s_obs[0] = 0; s_obs[1] = 0; }
    uint32_t par_s = (uint32_t)__cvta_generic_to_shared(par);        // shared-window address of word 0
    asm volatile("mov.u32 %0, %0;" : "+r"(par_s));                   // (opaque: kept in a register, not recomputed at every use)
    const HookList hk = { (uint32_t)__cvta_generic_to_shared(hkitems), (uint32_t)__cvta_generic_to_shared(&s_nhook), HKCAP, (uint32_t)(L > -tid) };   // (1, but neither constant nor warp-uniform for ptxas)
#pragma unroll
    for (int k = 0; k < SITES / 4 / THREADS; ++k)                    // counts start at 0 (the scan stores parents only)
        sts_u128(par_s + 16u * (k * THREADS + tid), make_uint4(0u, 0u, 0u, 0u));
    __syncthreads();

    // ---- phase 1: bonds of the tile, PAPER.md:37-39 (section 2.1) --------------------------------------
    if (!FUSE) {
        const uint32_t* bE = bondE + (size_t)blockIdx.y * words;
        const uint32_t* bS = bondS + (size_t)blockIdx.y * words;
        if (tid < WORDS) {
            const int row = tid / NW, wx = tid - row * NW;
            const size_t gw = (size_t)(y0 + row) * wprL + (x0 >> 5) + wx;
            es[tid] = make_uint2(bE[gw], bS[gw]);
        }
        if (tid < NW) nIn[tid] = bS[(size_t)(y0 == 0 ? L - 1 : y0 - 1) * wprL + (x0 >> 5) + tid];
        if (tid < TH) {
            const int wl = (x0 >> 5) == 0 ? wprL - 1 : (x0 >> 5) - 1;
            if (bE[(size_t)(y0 + tid) * wprL + wl] >> 31) atomicOr(&wIn[tid >> 5], 1u << (tid & 31));
        }
    } else {
        const PhiloxKey key(la.key0, la.key1);
        {
            const int wid = tid / TPW, part = tid - wid * TPW;      // this thread's 32-site word (and which part of its draws)
            const int row = wid / NW, wx = wid - row * NW;
            const int y = y0 + row;
            const int xw = (x0 >> 5) + wx;
            const int w = y * wprL + xw;                              // word index within the lattice
            uint32_t own = 0, eqE = 0, eqS = 0;
            if (POTTS) {
                const int8_t* r0 = col + (size_t)y * L + xw * 32;
                const int8_t* r1 = col + (size_t)(y + 1 == L ? 0 : y + 1) * L + xw * 32;
                const uint4 a0 = *reinterpret_cast<const uint4*>(r0), a1 = *reinterpret_cast<const uint4*>(r0 + 16);
                const uint4 b0 = *reinterpret_cast<const uint4*>(r1), b1 = *reinterpret_cast<const uint4*>(r1 + 16);
                const uint32_t nx = (uint8_t)col[(size_t)y * L + (xw + 1 == wprL ? 0 : (xw + 1) * 32)];
                const uint32_t a[9] = { a0.x, a0.y, a0.z, a0.w, a1.x, a1.y, a1.z, a1.w, nx };
                const uint32_t b[8] = { b0.x, b0.y, b0.z, b0.w, b1.x, b1.y, b1.z, b1.w };
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    eqE |= neg_nibble(__vcmpeq4(a[k], __funnelshift_r(a[k], a[k + 1], 8))) << (4 * k);
                    eqS |= neg_nibble(__vcmpeq4(a[k], b[k])) << (4 * k);
                }
            } else {
                own = ~sb[w];                                            // bit = 1: spin -1
                const uint32_t south = ~sb[(y + 1 == L ? 0 : y + 1) * wprL + xw];
                const uint32_t nxw = sb[y * wprL + (xw + 1 == wprL ? 0 : xw + 1)];
                const uint32_t eastm = (own >> 1) | ((~nxw & 1u) << 31);
                eqE = ~(own ^ eastm); eqS = ~(own ^ south);
            }
            if (POTTS && obs_prev) {
                // Potts: E = -#(equal East / South pairs) of the configuration the previous sweep left (M comes from the colour
                // counts of the assignment kernel)
                const int eo = warp_sum_i(-(__popc(eqE) + __popc(eqS)));
                if (lane == 0) atomicAdd(&s_obs[0], eo);
            }
            if (!POTTS && obs_prev) {
                // a7 for free: the equal-pair masks of the bond test are the energy of the
                // configuration the previous sweep left: E = (#edges) - 2 (#equal pairs), M = N - 2 (#down)
                const int eo = warp_sum_i(part == 0 ? 64 - 2 * (__popc(eqE) + __popc(eqS)) : 0);
                const int mo = warp_sum_i(part == 0 ? 32 - 2 * __popc(own) : 0);
                if (lane == 0) { atomicAdd(&s_obs[0], eo); atomicAdd(&s_obs[1], mo); }
            }
            uint32_t dE = 0, dS = 0;
#pragma unroll
            for (int cc = 0; cc < 16 / TPW; ++cc) {
                const int c = part * (16 / TPW) + cc;
                const uint4 r = philox4x32_10((uint32_t)w * 16u + c, tlo, thi, TAG_BOND, key);
                if (r.x < la.thr) dE |= 1u << (2 * c);               // (a compare and a predicated OR per word)
                if (r.z < la.thr) dE |= 2u << (2 * c);
                if (r.y < la.thr) dS |= 1u << (2 * c);
                if (r.w < la.thr) dS |= 2u << (2 * c);
            }
#pragma unroll
            for (int o = 1; o < TPW; o <<= 1) {                      // the word's TPW threads are neighbouring lanes
                dE |= __shfl_xor_sync(0xffffffffu, dE, o);
                dS |= __shfl_xor_sync(0xffffffffu, dS, o);
            }
            const uint32_t e = eqE & dE, so = eqS & dS;
            if (part == 0) {
                es[wid] = make_uint2(e, so);
                bondE[(size_t)blockIdx.y * words + w] = e;
                bondS[(size_t)blockIdx.y * words + w] = so;
            }
        }
        // bonds entering the tile: South bonds of the row above (TW / 2 calls), East bonds of the column to
        // the West (32 calls).  They are owned by the neighbouring tiles; recomputed here from the same draws.
        for (int j = tid; j < TW / 2 + TH; j += THREADS) {
            if (j < TW / 2) {
                const int yn = y0 == 0 ? L - 1 : y0 - 1;
                const int x = x0 + 2 * j;
                const int i = yn * L + x;                                  // even site; call covers i, i + 1
                const uint4 r = philox4x32_10((uint32_t)(i >> 1), tlo, thi, TAG_BOND, key);
                const int id = y0 * L + x;                                 // (x is even: both sites in one word)
                const uint32_t eq = POTTS ? ((col[i] == col[id] ? 1u : 0u) | (col[i + 1] == col[id + 1] ? 2u : 0u))
                                          : ~((sb[i >> 5] >> (i & 31)) ^ (sb[id >> 5] >> (id & 31)));
                const uint32_t bits = (eq & ((r.y < la.thr ? 1u : 0u) | (r.w < la.thr ? 2u : 0u))) & 3u;
                if (bits) atomicOr(&nIn[(2 * j) >> 5], bits << ((2 * j) & 31));
            } else {
                const int row = j - TW / 2;
                const int xwst = x0 == 0 ? L - 1 : x0 - 1;                 // odd column
                const int i = (y0 + row) * L + xwst;
                const uint4 r = philox4x32_10((uint32_t)(i >> 1), tlo, thi, TAG_BOND, key);
                const int ie = (y0 + row) * L + x0;
                const bool same = POTTS ? col[i] == col[ie] : !(((sb[i >> 5] >> (i & 31)) ^ (sb[ie >> 5] >> (ie & 31))) & 1u);
                if (same && r.z < la.thr)
                    atomicOr(&wIn[row >> 5], 1u << (row & 31));
            }
        }
    }
    __syncthreads();

    // ---- phase 2: scan-line labelling of this warp's block (32 columns x 32 rows), PAPER.md:49-51 -------
    // Lane = column, the block's rows in sequence, uniform control flow.  A run of East bonds takes the label of the
    // first of its sites that has a South bond from the row above (one shuffle), or opens a new label = its head's
    // own index (a root).  Where another site of the run is bonded to a different label above, the two labels are
    // equivalent: the lane notes the row in a bit mask (no divergent work in the loop, no list) and unites the pairs of
    // its column once the block is scanned.  Labels are never refreshed on the way down, so the only loop-carried
    // dependency of a row is the shuffle.
    {
        const int strip = warp % NW, yb = (warp / NW) * BAND;
        int rowbase = yb * TW + strip * 32;                          // first site of the row in this strip
        uint32_t rowaddr = par_s + 4u * (rowbase + lane) + 2u;       // my site's parent field in this row
        uint32_t prev = 0;                                           // label of the site above
        uint32_t s_up = 0;                                           // (a band's first row adopts nothing: seams come later)
        uint32_t mymeet = 0;                                         // rows of the block where two labels met at my column
#pragma unroll SCAN_UNROLL
        for (int y = yb; y < yb + BAND; ++y, rowbase += TW, rowaddr += 4u * TW) {
            const uint2 w = es[y * NW + strip];
            const uint32_t nz = ~w.x | 0x80000000u;                  // bit k: no bond between columns k, k + 1 of the strip
            const uint32_t below = nz & lt, above = nz & ~lt;        // run boundaries left of me / at or right of me
            const int h = bfind_u32(below) + 1;                      // head column of my run
            // my run: bits h .. tail, tail = lowest set bit of `above` (bit 31 is always set)
            const uint32_t runmask = (above ^ (above - 1u)) & ~((1u << h) - 1u);
            const uint32_t upm = s_up & runmask;                     // sites of my run bonded to the row above
            const uint32_t got = __shfl_sync(0xffffffffu, prev, __ffs(upm) - 1);   // (source lane is taken mod 32)
            const uint32_t c = upm ? got : (uint32_t)(rowbase + h);  // a new label: the head's own index (its own root)
            sts_u16(rowaddr, c);
            const bool meet = (s_up & lanebit) && prev != c;         // two labels meet at my site: the one above, my run's
            mymeet = (mymeet >> 1) | (meet ? 0x80000000u : 0u);
            prev = c;
            s_up = w.y;
        }
        __syncwarp();                                                // the block's parents are written
        // The meetings (~2.5 per lane at T_c, up to ~7) are united by all lanes, 32 at a time: every lane writes the sites of
        // its column into the warp's list at the positions a prefix sum gives it.  The list lives in the (still unused)
        // count fields of the warp's own block: entry k in the low half of the block's word (k >> 5, k & 31) -- no memory of
        // its own (6 CTAs per SM), no capacity to overflow (a block has fewer meetings than sites).
        mymeet >>= 32 - BAND;                                        // bit r: row yb + r
        const uint32_t pl_s = par_s + 4u * (uint32_t)(yb * TW + strip * 32);
        const int cnt = __popc(mymeet);
        int pos = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, pos, o);
            if (lane >= o) pos += v;
        }
        const int npend = __shfl_sync(0xffffffffu, pos, 31);
        pos -= cnt;
        const int colbase = yb * TW + strip * 32 + lane;
        while (mymeet) {
            const int i = colbase + (__ffs(mymeet) - 1) * TW;
            mymeet &= mymeet - 1u;
            sts_u16(pl_s + 4u * (uint32_t)((pos >> 5) * TW + (pos & 31)), (uint32_t)i);
            ++pos;
        }
        // An entry is read and its field cleared (the counts start at 0 in phase 3) while no union of this warp is in
        // flight: a hook wipes the low half of the word it replaces and adds it back, and only this warp's unions touch
        // this block's words before the barrier below.
        for (int j0 = 0; j0 < npend; j0 += 32) {
            __syncwarp();
            const int j = j0 + lane;
            const uint32_t slot = pl_s + 4u * (uint32_t)((j >> 5) * TW + (j & 31));
            uint32_t i = 0;
            if (j < npend) { i = lds_u16(slot); sts_u16(slot, 0u); }
            __syncwarp();
            if (j < npend) {
                const int a = (int)lds_u16(par_s + 4u * (i - TW) + 2u), c = (int)lds_u16(par_s + 4u * i + 2u);
                hooked(hk, sc_union(par_s, a, c));                   // (labels are mostly still roots: sc_union takes any nodes)
            }
        }
    }
    __syncthreads();

    // ---- phase 3: seams between the warps' blocks: East bonds across strip edges, South bonds across bands
    for (int j = tid; j < (NW - 1) * TH + (TH / BAND - 1) * TW; j += THREADS) {
        if (j < (NW - 1) * TH) {
            const int row = j / (NW - 1), st = j - row * (NW - 1);
            if (es[row * NW + st].x >> 31) {
                const int i = row * TW + st * 32 + 31;
                hooked(hk, sc_union(par_s, (int)lds_u16(par_s + 4u * i + 2u), (int)lds_u16(par_s + 4u * i + 6u)));   // the two sites' labels
            }
        } else {
            const int k = j - (NW - 1) * TH;
            const int row = (k / TW + 1) * BAND - 1, c = k % TW;
            if ((es[row * NW + (c >> 5)].y >> (c & 31)) & 1u) {
                const int i = row * TW + c;
                hooked(hk, sc_union(par_s, (int)lds_u16(par_s + 4u * i + 2u), (int)lds_u16(par_s + 4u * (i + TW) + 2u)));
            }
        }
    }
    // ... and, in the same phase, every site is counted at its label (any node of its tree will do: the flatten
    // moves the counts to the roots); four consecutive sites per thread, one add where they share the label
#pragma unroll 2
    for (int k = 0; k < SITES / 4 / THREADS; ++k) {
        const uint4 v = lds_u128(par_s + 16u * (k * THREADS + tid));
        const uint32_t n0 = v.x >> 16, n1 = v.y >> 16, n2 = v.z >> 16, n3 = v.w >> 16;
        if (n0 == n1 && n2 == n3 && n0 == n2) red_add_s(par_s + 4u * n0, 4u);
        else {
            red_add_s(par_s + 4u * n0, 1u); red_add_s(par_s + 4u * n1, 1u);
            red_add_s(par_s + 4u * n2, 1u); red_add_s(par_s + 4u * n3, 1u);
        }
    }
    // (the label nodes are counted here, in front of the barrier: bit tricks on the bond words only)
    uint32_t o;                                                      // heads of runs without an uplink in this thread's word
    int mybase;
    {
        const int wd = tid < WORDS ? tid : 0;                        // (with several threads per word the first WORDS threads count)
        mybase = (wd / NW) * TW + (wd % NW) * 32;
        const uint32_t ew = es[wd].x & 0x7FFFFFFFu;
        uint32_t up = (wd / NW) % BAND ? es[wd - NW].y : 0u;         // South bonds of the row above, within the band
        uint32_t m = ew;                                             // OR of the run's uplinks, gathered at its head
        up |= (up >> 1) & m;  m &= m >> 1;
        up |= (up >> 2) & m;  m &= m >> 2;
        up |= (up >> 4) & m;  m &= m >> 4;
        up |= (up >> 8) & m;  m &= m >> 8;
        up |= (up >> 16) & m;
        o = ~(ew << 1) & ~up;
        if (tid >= WORDS) o = 0;
        const int nl = warp_sum_i(__popc(o));
        if (lane == 0) atomicAdd(&s_nlab, nl);
    }
    __syncthreads();

    // ---- phase 3b: flatten ---------------------------------------------------------------------------
    // The scan gave every site of a run the run's label = a root at that time; the only nodes that ever were
    // roots are the heads of runs with no bond from the row above ("label nodes", ~0.2 per site at T_c), and
    // the only ones that no longer are were hooked (~0.03 per site): each of those is pointed at its root and hands
    // it its count, so that afterwards root(site) = parent(parent(site)) for every site, without a loop, and a
    // root's count is the size of its tile-local cluster.  The label nodes themselves are only COUNTED (bit tricks
    // on the bond words): roots = label nodes - hooked nodes.
    {
        const int nh = s_nhook;                                      // (complete: the barrier above)
        if (nh <= HKCAP) {
            for (int j = tid; j < nh; j += THREADS) sc_flatten(par_s, hkitems[j]);
        } else {                                                     // more hooks than the list holds: visit every label node
            while (o) {
                const int n = mybase + __ffs(o) - 1;
                o &= o - 1;
                if ((int)lds_u16(par_s + 4u * n + 2u) != n) sc_flatten(par_s, n);
            }
        }
    }
    __syncthreads();

    // ---- phase 4: the root of every site -> 16-bit tile-local label; the largest count of the tile ---------
    constexpr int QSTEPS = SITES / 4 / THREADS;                      // = 8
    constexpr int LOG_TW = ilog2_c(TW);
    static_assert((1 << LOG_TW) == TW, "tile width is a power of two");
    const int tilebase = y0 * L + x0;
    {
        // the tile-local 16-bit root of every site is all the sweep stores per site (2 B); the int32 labels
        // of the C ABI are derived from it on demand (k_labels16)
        uint16_t* out = lab16 + (size_t)blockIdx.y * N + (size_t)(y0 + ((4 * tid) >> LOG_TW)) * L + x0 + ((4 * tid) & (TW - 1));
        const size_t step = (size_t)(4 * THREADS / TW) * L;          // rows a step of the CTA covers
        uint32_t mx = 0;
#pragma unroll
        for (int k = 0; k < QSTEPS; ++k) {
            const uint4 v = lds_u128(par_s + 16u * (k * THREADS + tid));
            // site -> its label node -> root (label nodes are flat)
            const uint32_t r0 = lds_u16(par_s + 4u * (v.x >> 16) + 2u), r1 = lds_u16(par_s + 4u * (v.y >> 16) + 2u),
                           r2 = lds_u16(par_s + 4u * (v.z >> 16) + 2u), r3 = lds_u16(par_s + 4u * (v.w >> 16) + 2u);
            *reinterpret_cast<uint2*>(out + k * step) = make_uint2(r0 | (r1 << 16), r2 | (r3 << 16));
            // counts sit at label nodes only (0 elsewhere); a root holds its cluster's size, a hooked node a part of
            // one: the maximum over all words is the largest tile-local cluster (a piece of a cluster that spans
            // tiles may enter: its total, which k_flip16 maximises, is no smaller)
            mx = max(max(mx, v.x & CNT16), max(v.y & CNT16, max(v.z & CNT16, v.w & CNT16)));
        }
        mx = (uint32_t)warp_max_i((int)mx);
        if (lane == 0) atomicMax(&s_max, (int)mx);
    }
    __syncthreads();

    // ---- phase 5: a root with a bond across the tile edge becomes a node of the global union-find --------
    // (order of the border sites: North row, South row, West column, East column).  The first border site to
    // reach a root claims it: slot in the tile's list, node, and the slot in place of the count in the root's word.
    // Dense node arrays of CAP entries per tile (L2-resident at L = 16384) instead of the N-entry label array.
    {
        const int nodebase = blockIdx.x * CAP;                       // node ids are local to the lattice
        const size_t lb = (size_t)blockIdx.y * gridDim.x * CAP;
        int4* mynodes = nodes + lb + nodebase;
        for (int j = tid; j < 2 * (TW + TH); j += THREADS) {
            int site; bool open;
            if (j < TW)               { site = j;                              open = (nIn[j >> 5] >> (j & 31)) & 1u; }
            else if (j < 2 * TW)      { const int c = j - TW; site = (TH - 1) * TW + c;
                                        open = (es[(TH - 1) * NW + (c >> 5)].y >> (c & 31)) & 1u; }
            else if (j < 2 * TW + TH) { const int r = j - 2 * TW; site = r * TW; open = (wIn[r >> 5] >> (r & 31)) & 1u; }
            else                      { const int r = j - 2 * TW - TH; site = r * TW + TW - 1;
                                        open = es[r * NW + NW - 1].x >> 31; }
            if (open) {
                const uint32_t l = lds_u16(par_s + 4u * lds_u16(par_s + 4u * site + 2u) + 2u);   // site -> label node -> root
                const uint32_t old = atom_or_s(par_s + 4u * l, CLAIMED16);
                if (!(old & CLAIMED16)) {
                    const int pos = atomicAdd(&s_nopen, 1);
                    const int cnt = (int)(old & CNT16);
                    const int g = tilebase + (int)(l >> LOG_TW) * L + (int)(l & (TW - 1));
                    // node = (parent: its own root, size of the cluster rooted here: so far this piece,
                    //         minimum site index of the cluster rooted here, site index of this tile root)
                    mynodes[pos] = make_int4(nodebase + pos, cnt, g, g);
                    red_add_s(par_s + 4u * l, (uint32_t)(pos - cnt));     // the root's word now carries its slot
                }
            }
        }
    }
    __syncthreads();
    if (tid == 0) {
        ocount[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = s_nopen;
        Rec* rc = rec + (size_t)ctl->slot * nb + blockIdx.y;
        const int nclosed = s_nlab - s_nhook - s_nopen;              // roots = label nodes - hooked nodes; closed = not claimed
        if (s_max) atomic_max_ll(&rc->maxcl, s_max);
        if (nclosed) atomic_add_ll(&rc->ncl, nclosed);               // a closed tile root is a cluster root
        if (FUSE && obs_prev) {                                      // E, M of the previous sweep's configuration
            Rec* rp = rec + (size_t)(ctl->slot == 0 ? ctl->cap - 1 : ctl->slot - 1) * nb + blockIdx.y;
            if (s_obs[0]) atomic_add_ll(&rp->E, s_obs[0]);
            if (s_obs[1]) atomic_add_ll(&rp->M, s_obs[1]);
        }
    }

    // ---- phase 6: slot of the root of every border site with a bond across the tile edge ----------------
    // (what k_merge_nodes reads instead of label[])
    {
        uint16_t* myb = bslot + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * CAP;
        for (int j = tid; j < 2 * (TW + TH); j += THREADS) {
            int site; bool open;
            if (j < TW)               { site = j;                              open = (nIn[j >> 5] >> (j & 31)) & 1u; }
            else if (j < 2 * TW)      { const int c = j - TW; site = (TH - 1) * TW + c;
                                        open = (es[(TH - 1) * NW + (c >> 5)].y >> (c & 31)) & 1u; }
            else if (j < 2 * TW + TH) { const int r = j - 2 * TW; site = r * TW; open = (wIn[r >> 5] >> (r & 31)) & 1u; }
            else                      { const int r = j - 2 * TW - TH; site = r * TW + TW - 1;
                                        open = es[r * NW + NW - 1].x >> 31; }
            uint32_t slot = 0xFFFFu;
            if (open) {
                const uint32_t l = lds_u16(par_s + 4u * lds_u16(par_s + 4u * site + 2u) + 2u);
                slot = lds_u32(par_s + 4u * l) & CNT16;
            }
            myb[j] = (uint16_t)slot;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// a3 global boundary merge on the NODE arrays (north_star stage 2): one thread per site on a
// tile's East column or South row; if its bond crosses the edge (its border entry holds a slot), the two tile
// roots (slots from the border arrays of the two tiles) are united: find through L1, hook "larger id under smaller" with atomicMin.
// Node id = tile * CAP + slot.  Any total order gives a valid forest; the canonical label (minimum SITE index,
// PAPER.md:51) is accumulated per root in nmin[] by k_roots_nodes.
// ---------------------------------------------------------------------------------------------------
// union-find on the node array: the parent is field x of the node.  Walks go through L1 (a stale line shows an
// older parent = still an ancestor); the atomicMin in L2 decides whether a node still is a root.
__device__ __forceinline__ int nd_find(const int4* nodes, int x) {
    int p = ld_ca(&nodes[x].x);
    while (p != x) { x = p; p = ld_ca(&nodes[x].x); }
    return x;
}
__device__ __forceinline__ void nd_union(int4* nodes, int a, int b) {
    a = nd_find(nodes, a); b = nd_find(nodes, b);
    while (a != b) {
        if (a < b) { const int s = a; a = b; b = s; }      // a is the larger
        const int old = atomicMin(&nodes[a].x, b);
        if (old == a) break;
        a = old;
    }
}

template <int TW, int TH>
__global__ void __launch_bounds__(256)
k_merge_nodes(int4* nodes, const uint16_t* __restrict__ bslot, int tilesX, int tilesY) {
    pdl_wait();
    constexpr int CAP = 2 * (TW + TH), PER = TW + TH;       // per tile: TW South-row sites, TH East-column sites
    const int idx = blockIdx.x * 256 + threadIdx.x;
    const int tiles = tilesX * tilesY;
    if (idx >= tiles * PER) return;
    const size_t lb = (size_t)blockIdx.y * tiles * CAP;
    const uint16_t* bs = bslot + lb;
    const int ta = idx / PER, j = idx - ta * PER;
    const int r = ta / tilesX, c = ta - r * tilesX;
    int ka, tb, kb;
    if (j < TW) { ka = TW + j;                tb = (r + 1 == tilesY ? 0 : r + 1) * tilesX + c; kb = j; }            // South row -> North row below
    else        { ka = 2 * TW + TH + (j - TW); tb = r * tilesX + (c + 1 == tilesX ? 0 : c + 1); kb = 2 * TW + (j - TW); }  // East column -> West column
    const int sa = bs[(size_t)ta * CAP + ka], sb = bs[(size_t)tb * CAP + kb];   // (both loads in flight before the test)
    if (sa == 0xFFFF) return;                               // no bond across the edge here
    nd_union(nodes + lb, ta * CAP + sa, tb * CAP + sb);
}

// After the merge: every open piece adds its size and its site index to the node it hangs under (sum -> cluster
// size, min -> canonical label) and points straight at it.  The root of the largest piece of a warp's first round is
// carried in registers across rounds (at T_c one cluster owns many pieces in every tile); a piece whose root no other
// lane of the round shares goes there with one pair of reductions (no return value to wait for); only roots that
// several lanes share are combined inside the warp first.  (Combining ALL pieces per root -- __match_any_sync and
// reductions over the groups' masks, which run group after group, 18 groups of 1.7 lanes per round -- took half of
// this kernel's time; combining none is fastest on the young lattice of the bench, 1.270 ms per sweep, but loses on
// the equilibrated one: 1.367 ms at sweeps 200-249 against 1.314 for this version and 1.320 for combining all.)  wpt warps per tile (1 for large lattices; 4 for small ones, where the kernel is
// the latency of one warp walking its tile's ~100 pieces 32 at a time): warp `sub` takes rounds sub, sub + wpt, ...
template <int CAP>
__global__ void __launch_bounds__(256)
k_roots_nodes(int4* nodes, const int* __restrict__ ocount, int tiles, int wpt) {
    pdl_wait();
    const int gw = blockIdx.x * 8 + (threadIdx.x >> 5);
    const int tile = gw / wpt, sub = gw - tile * wpt;
    const int lane = threadIdx.x & 31;
    if (tile >= tiles) return;                              // (warp-uniform)
    int4* nd = nodes + (size_t)blockIdx.y * tiles * CAP;
    const int n = ocount[(size_t)blockIdx.y * tiles + tile];
    int hot = -1, hotacc = 0, hotmin = 0x7fffffff;
    for (int e0 = 32 * sub; e0 < n; e0 += 32 * wpt) {
        const int e = e0 + lane;
        const bool on = e < n;
        int root = -1 - lane, add = 0, g = 0x7fffffff;      // idle lanes: distinct keys, nothing to add
        if (on) {
            const int id = tile * CAP + e;
            const int4 me = nd[id];
            root = me.x;
            if (root != id) {                               // hooked: (no root changes during this kernel)
                root = nd_find(nd, root);
                if (root != me.x) nd[id].x = root;          // only ever an ancestor: safe while others walk
                add = me.y;                                 // a root's own piece is already in its size / min
            }
            g = me.w;
        }
        if (e0 == 32 * sub) {                               // (my first round) the hot root: the one of the round's largest piece
            const int best = __reduce_max_sync(0xffffffffu, add);
            const unsigned who = __ballot_sync(0xffffffffu, add == best && on);
            if (who) hot = __shfl_sync(0xffffffffu, root, __ffs(who) - 1);
        }
        const bool cold = on && root != hot;
        if (on && !cold) { hotacc += add; hotmin = min(hotmin, g); }
        // the other roots: most appear once in a round and get their pair of reductions straight away (fire and forget); the
        // few that appear several times (another large cluster with many pieces in this tile: the equilibrated lattice has
        // them) are combined first, group after group
        const unsigned grp = __match_any_sync(0xffffffffu, cold ? root : -1 - lane);
        if (cold) {
            if (grp == (1u << lane)) { if (add) { atomicAdd(&nd[root].y, add); atomicMin(&nd[root].z, g); } }
            else {
                const int tot = __reduce_add_sync(grp, add);
                const int gm = __reduce_min_sync(grp, g);
                if (tot && lane == __ffs(grp) - 1) { atomicAdd(&nd[root].y, tot); atomicMin(&nd[root].z, gm); }
            }
        }
    }
    hotacc = warp_sum_i(hotacc);
    hotmin = __reduce_min_sync(0xffffffffu, hotmin);
    if (lane == 0 && hotacc) { atomicAdd(&nd[hot].y, hotacc); atomicMin(&nd[hot].z, hotmin); }
}

// a4 on demand (sw_labels; every sweep with sw_set_eager_labels): flat int32 labels from the 16-bit tile-local
// roots.  One CTA per tile: a table in shared memory holds, for every open tile root, its cluster's canonical
// label (minimum site index under its root node); a closed tile root IS its cluster's label.  PAPER.md:51.
template <int NW, int TH>
__global__ void __launch_bounds__(NW * TH)
k_labels16(int* __restrict__ label, const uint16_t* __restrict__ lab16, const int4* __restrict__ nodes,
           const int* __restrict__ ocount, DivL dv, int L, int N) {
    pdl_wait();
    constexpr int TW = 32 * NW, SITES = TW * TH, THREADS = NW * TH, CAP = 2 * (TW + TH);
    constexpr int LOG_TW = ilog2_c(TW);
    extern __shared__ int tab[];                     // [SITES] canonical label of the open tile root with this local index, else -1
    const int tid = threadIdx.x;
    const int tilesX = L / TW;
    const int ty = blockIdx.x / tilesX, tx = blockIdx.x - ty * tilesX;
    const int y0 = ty * TH, x0 = tx * TW;
    const int tilebase = y0 * L + x0;
    for (int i = tid; i < SITES; i += THREADS) tab[i] = -1;
    __syncthreads();
    {
        const size_t lb = (size_t)blockIdx.y * gridDim.x * CAP;
        const int nodebase = blockIdx.x * CAP;
        const int n = ocount[(size_t)blockIdx.y * gridDim.x + blockIdx.x];
        for (int e = tid; e < n; e += THREADS) {
            const int4 me = nodes[lb + nodebase + e];
            const int R = me.x == nodebase + e ? me.z : nodes[lb + me.x].z;
            const int delta = me.w - tilebase;
            const int ry = div_l(delta, dv);
            tab[ry * TW + (delta - ry * L)] = R;
        }
    }
    __syncthreads();
    for (int q = tid; q < SITES / 4; q += THREADS) {
        const int l = 4 * q;
        const size_t gsite = (size_t)(y0 + (l >> LOG_TW)) * L + x0 + (l & (TW - 1));
        const uint2 w = *reinterpret_cast<const uint2*>(lab16 + (size_t)blockIdx.y * N + gsite);
        const int r[4] = { (int)(w.x & 0xFFFFu), (int)(w.x >> 16), (int)(w.y & 0xFFFFu), (int)(w.y >> 16) };
        int g[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int t = tab[r[u]];
            g[u] = t >= 0 ? t : tilebase + (r[u] >> LOG_TW) * L + (r[u] & (TW - 1));
        }
        *reinterpret_cast<int4*>(label + (size_t)blockIdx.y * N + gsite) = make_int4(g[0], g[1], g[2], g[3]);
    }
}

// ---------------------------------------------------------------------------------------------------
// a4-a6 fused: assignment PAPER.md:57 (section 2.4).  One CTA per tile (the tiles of k_bond_label), 32 sites
// per thread.  (a7: E and M of the new configuration fall out of the NEXT sweep's bond test, or of
// k_observe_rows after the last sweep of a call.)
//
// The decision of a site is the decision bit of its cluster root.  The kernel first builds, in shared
// memory, one decision bit per TILE ROOT, indexed by the root's tile-local index:
//   closed tile root g (cluster inside the tile): the cluster root is g itself -> bit D[g]: the tile's own
//                      words of the decision plane, copied in bulk;
//   open tile root g:  its cluster root R was found by k_roots_nodes and sits next to g in the tile's list ->
//                      bit D[R] overwrites the copied bit (a few hundred per tile).
// Then every site reads its 16-bit tile-local root index (2 B / site, written by k_bond_label) and looks the
// bit up in shared memory: no global gather, no index arithmetic per site.
// ---------------------------------------------------------------------------------------------------
// BITS: the new spins go out bit-packed (one byte = 8 sites per thread and step, 32 MiB instead of 256 MiB at
// L = 16384) into the plane k_bond_label<FUSE> reads; else as the int8 plane (unfused path 6).
// FUSED (small lattices, where a sweep is the sum of its kernels' latencies): no decision plane and no separate end-of-sweep
// kernel -- the decision words of the tile's own sites and of the cluster roots of its open tile roots are drawn here (word w
// of the plane is word w & 3 of Philox call (w >> 2, t, TAG_FLIP): the same bits k_flipbits would have stored), and the CTA
// that finishes last advances the sweep (advance_sweep).  4 launches per sweep instead of 6.  (At L = 16384 the extra draws
// cost more than the two launches: not used there.)
template <int NW, int TH, bool BITS, bool FUSED = false>
__global__ void __launch_bounds__(NW * TH, 1536 / (NW * TH))
k_flip16(int8_t* __restrict__ spins, uint32_t* __restrict__ sbits, const uint16_t* __restrict__ lab16, const uint32_t* __restrict__ D,
         const int4* __restrict__ nodes, const int* __restrict__ ocount, Rec* __restrict__ rec, Ctl* __restrict__ ctl,
         const Lat* __restrict__ lat, Mom* __restrict__ mom, int adv_acc,
         DivL dv, int L, int N, int words, int nb) {
    pdl_wait();
    constexpr int TW = 32 * NW, SITES = TW * TH, THREADS = NW * TH;
    constexpr int CAP = 2 * (TW + TH);
    constexpr int OSTEPS = SITES / 8 / THREADS;      // = 4
    constexpr int LOG_TW = ilog2_c(TW);
    __shared__ uint32_t dec[TH * NW];                // decision bit of the tile root with local index l: bit l & 31 of word l >> 5

    const int tid = threadIdx.x;
    const int tilesX = L / TW;
    const int ty = blockIdx.x / tilesX, tx = blockIdx.x - ty * tilesX;
    const int y0 = ty * TH, x0 = tx * TW;
    const int tilebase = y0 * L + x0;
    const uint32_t* d = D + (size_t)blockIdx.y * words;
    const size_t tile = (size_t)blockIdx.y * gridDim.x + blockIdx.x;

    // my sites' tile-root indices: issue the loads first
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
    {
        const int row = tid / NW, wx = tid - row * NW;
        const int w = (y0 + row) * (L >> 5) + (x0 >> 5) + wx;            // my word of the decision plane
        if (FUSED) {
            const PhiloxKey key(la.key0, la.key1);
            const uint4 r = philox4x32_10((uint32_t)w >> 2, tlo, thi, TAG_FLIP, key);
            dec[tid] = (w & 2) ? ((w & 1) ? r.w : r.z) : ((w & 1) ? r.y : r.x);
        } else {
            dec[tid] = d[w];
        }
    }
    __syncthreads();
    // open tile roots take the decision of their cluster root = the minimum site index under their root node;
    // the nodes that are roots are the clusters that span tiles: counted, and their sizes maximised, here
    {
        const size_t lb = (size_t)blockIdx.y * gridDim.x * CAP;
        const int nodebase = blockIdx.x * CAP;
        int nroot = 0, big = 0;
        for (int e = tid; e < n; e += THREADS) {
            const int4 me = nodes[lb + nodebase + e];                  // (root node, size, min site, site of the tile root)
            const int R = me.x == nodebase + e ? me.z : nodes[lb + me.x].z;
            if (me.x == nodebase + e) { ++nroot; big = max(big, me.y); }
            uint32_t up;
            if (FUSED) {
                const PhiloxKey key(la.key0, la.key1);
                const uint4 r = philox4x32_10((uint32_t)R >> 7, tlo, thi, TAG_FLIP, key);
                const uint32_t wsel = (R & 64) ? ((R & 32) ? r.w : r.z) : ((R & 32) ? r.y : r.x);
                up = (wsel >> (R & 31)) & 1u;
            } else {
                up = (__ldg(d + (R >> 5)) >> (R & 31)) & 1u;
            }
            const int delta = me.w - tilebase;
            const int ry = div_l(delta, dv);
            const int l = ry * TW + (delta - ry * L);
            if (up) atomicOr(&dec[l >> 5], 1u << (l & 31));
            else    atomicAnd(&dec[l >> 5], ~(1u << (l & 31)));
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
        const uint32_t w4[4] = { v[k].x, v[k].y, v[k].z, v[k].w };
        uint32_t b8 = 0;                                               // bit u: site l + u goes up
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const uint32_t r = (u & 1) ? (w4[u >> 1] >> 16) : (w4[u >> 1] & 0xFFFFu);
            b8 |= (__funnelshift_r(dec[r >> 5], 0u, r) & 1u) << u;
        }
        const size_t gsite = (size_t)blockIdx.y * N + (size_t)(y0 + (l >> LOG_TW)) * L + x0 + (l & (TW - 1));
        if (BITS) reinterpret_cast<uint8_t*>(sbits)[gsite >> 3] = (uint8_t)b8;
        else *reinterpret_cast<uint2*>(spins + gsite) = make_uint2(spin_bytes4(b8 & 15u), spin_bytes4(b8 >> 4));
    }
    if (FUSED) {
        // the CTA that finishes last closes the sweep (its own and every other CTA's record updates are done)
        __shared__ int s_last;
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            s_last = atomicAdd(&ctl->done, 1u) == gridDim.x * gridDim.y - 1;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            if (tid == 0) ctl->done = 0;
            advance_sweep(ctl, rec, nb, mom, N, adv_acc);
        }
    }
}

// a7 of the configuration a sw_sweep call ends with (the sweeps before it get theirs from the next sweep's
// bond test): E and M from sign masks, 32 sites per thread, into the slot of the sweep that just finished.
__global__ void __launch_bounds__(256)
k_observe_rows(const int8_t* __restrict__ spins, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
               int L, int N, int words, int nb) {
    pdl_wait();
    const int w = blockIdx.x * 256 + threadIdx.x;
    int e = 0, m = 0;
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
        m = 32 - 2 * __popc(own);
    }
    e = warp_sum_i(e); m = warp_sum_i(m);
    __shared__ int se[8], sm[8];
    if ((threadIdx.x & 31) == 0) { se[threadIdx.x >> 5] = e; sm[threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int te = 0, tm = 0;
        for (int k = 0; k < 8; ++k) { te += se[k]; tm += sm[k]; }
        Rec* r = rec + (size_t)(ctl->slot == 0 ? ctl->cap - 1 : ctl->slot - 1) * nb + blockIdx.y;
        if (te) atomic_add_ll(&r->E, te);
        if (tm) atomic_add_ll(&r->M, tm);
    }
}

// the same from the bit-packed plane (fused path): one word per thread
__global__ void __launch_bounds__(256)
k_observe_bits(const uint32_t* __restrict__ sbits, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
               int L, int N, int words, int nb) {
    pdl_wait();
    const int w = blockIdx.x * 256 + threadIdx.x;
    int e = 0, m = 0;
    if (w < words) {
        const int wpr = L >> 5;
        const int y = w / wpr, xw = w - y * wpr;
        const uint32_t* sb = sbits + (size_t)blockIdx.y * words;
        const uint32_t own = ~sb[w], south = ~sb[(y + 1 == L ? 0 : y + 1) * wpr + xw];
        const uint32_t eastm = (own >> 1) | ((~sb[y * wpr + (xw + 1 == wpr ? 0 : xw + 1)] & 1u) << 31);
        e = 64 - 2 * (__popc(~(own ^ eastm)) + __popc(~(own ^ south)));
        m = 32 - 2 * __popc(own);
    }
    e = warp_sum_i(e); m = warp_sum_i(m);
    __shared__ int se[8], sm[8];
    if ((threadIdx.x & 31) == 0) { se[threadIdx.x >> 5] = e; sm[threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int te = 0, tm = 0;
        for (int k = 0; k < 8; ++k) { te += se[k]; tm += sm[k]; }
        Rec* r = rec + (size_t)(ctl->slot == 0 ? ctl->cap - 1 : ctl->slot - 1) * nb + blockIdx.y;
        if (te) atomic_add_ll(&r->E, te);
        if (tm) atomic_add_ll(&r->M, tm);
    }
}

} // namespace sw
