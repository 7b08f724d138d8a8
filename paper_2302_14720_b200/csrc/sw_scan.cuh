// sw_scan.cuh -- the fast path (lattice side a multiple of 64): 128 x 64 tiles above L = 1024, 64 x 32 tiles up to it.
//
// Stage map; one CTA per tile of TW x TH sites, TW = 32 * NW; the tile is NW x TH / BAND blocks of
// 32 x BAND sites, one warp each (BAND = 32: one thread per 32-site word; BAND = 8: four threads per word -- small lattices).
//   a1+a2 k_bond_label<NW, TH, FUSE, POTTS, BAND>   (body: sw_bond_label_body.inc, shared with k_sweeps_cluster, sw_cluster.cuh)
//       phase 1  per 32-site word: the word's spins from the BIT-PACKED plane (FUSE; bit 1 = +1; the int8 plane is derived
//                on demand, sw_spins), 16 Philox4x32-10 calls, bond words to shared memory and to the canonical global
//                bit-planes; E, M of the previous sweep's configuration from the same equal-pair masks; the bonds that enter
//                the tile from its North and West neighbours are recomputed (TW/2 + TH extra calls)
//       phase 2  scan-line labelling, lane = column, the block's rows in sequence, uniform control flow: runs of East bonds
//                from bit tricks on the row's bond word; a run takes the label of the last of its sites that has a South
//                bond from the row above (one shuffle), or opens a new label (its head's index); where another site of the
//                run is bonded to a different label above, the lane notes the row in a bit mask; after the block the masks
//                become one list (prefix sum; it lives in the unused count fields of the block's own words) and the warp
//                unites the pairs 32 at a time (atomicMin hooking; hooked nodes go into a tile-wide list)
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
//   bits  0 .. 13  sites counted at this node: 0 from the scan's store, then every site is counted at its label (phase 3);
//                  the flatten (phase 3b) moves the counts of the nodes that were hooked to their roots, so that a
//                  root ends up with the size of its tile-local cluster.  (Between the scan of a block and its unions the
//                  fields of the block's first words hold the warp's list of meetings.)
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
__device__ __forceinline__ void sts_u32(uint32_t a, uint32_t v) {
    asm volatile("st.shared.u32 [%0], %1;" :: "r"(a), "r"(v) : "memory");
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

// m * 2 + (a >= thr) for 1 <= thr < 2^32, given nthr = 2^32 - thr: the carry of a + nthr goes straight into the mask
// (add.cc + addc: two instructions per bit instead of a compare, a select and half an OR)
__device__ __forceinline__ uint32_t shift_in_ge(uint32_t m, uint32_t a, uint32_t nthr) {
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %0, %0;\n\t}" : "+r"(m) : "r"(a), "r"(nthr));
    return m;
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
// The list and its counter sit behind the parent array in the kernel's DYNAMIC shared memory, so that their addresses are
// the parent array's (kept in a register) plus a constant.  Bytes of dynamic shared memory k_bond_label needs:
constexpr int BL_HKCAP = 1024;                  // hooked nodes a tile can list (~250 at T_c)
__host__ __device__ constexpr size_t bond_label_smem(int sites) { return (size_t)sites * 4 + (size_t)BL_HKCAP * 2 + 16; }
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
#define BL_LDSPIN(p, i) (p)[i]
#define BL_T ctl->t
#define BL_SLOT ctl->slot
#define BL_CAP ctl->cap
#include "sw_bond_label_body.inc"
#undef BL_LDSPIN
#undef BL_T
#undef BL_SLOT
#undef BL_CAP
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
// (CG -- k_sweeps_cluster, where the node array is rewritten sweep after sweep inside one kernel: every walk goes to L2)
template <bool CG = false>
__device__ __forceinline__ int nd_find(const int4* nodes, int x) {
    int p = CG ? ld_cg(&nodes[x].x) : ld_ca(&nodes[x].x);
    while (p != x) { x = p; p = CG ? ld_cg(&nodes[x].x) : ld_ca(&nodes[x].x); }
    return x;
}
template <bool CG = false>
__device__ __forceinline__ void nd_union(int4* nodes, int a, int b) {
    a = nd_find<CG>(nodes, a); b = nd_find<CG>(nodes, b);
    while (a != b) {
        if (a < b) { const int s = a; a = b; b = s; }      // a is the larger
        const int old = atomicMin(&nodes[a].x, b);
        if (old == a) break;
        a = old;
    }
}

template <int TW, int TH>
__global__ void __launch_bounds__(256)
k_merge_nodes(int4* nodes, const uint16_t* __restrict__ bslot, int tilesX, int tilesY, DivL dx) {   // dx: division by tilesX
    pdl_wait();
    constexpr int CAP = 2 * (TW + TH), PER = TW + TH;       // per tile: TW South-row sites, TH East-column sites
    const int idx = blockIdx.x * 256 + threadIdx.x;
    const int tiles = tilesX * tilesY;
    if (idx >= tiles * PER) return;
    const size_t lb = (size_t)blockIdx.y * tiles * CAP;
    const uint16_t* bs = bslot + lb;
    const int ta = idx / PER, j = idx - ta * PER;
    const int r = div_l(ta, dx), c = ta - r * tilesX;
    int ka, tb, kb;
    if (j < TW) { ka = TW + j;                tb = (r + 1 == tilesY ? 0 : r + 1) * tilesX + c; kb = j; }            // South row -> North row below
    else        { ka = 2 * TW + TH + (j - TW); tb = r * tilesX + (c + 1 == tilesX ? 0 : c + 1); kb = 2 * TW + (j - TW); }  // East column -> West column
    const int sa = bs[(size_t)ta * CAP + ka], sb = bs[(size_t)tb * CAP + kb];   // (both loads in flight before the test)
    if (sa == 0xFFFF) return;                               // no bond across the edge here
    int4* nd = nodes + lb;
    int a = ta * CAP + sa, b = tb * CAP + sb;
    int pa = ld_ca(&nd[a].x), pb = ld_ca(&nd[b].x);         // the first hops of both walks in flight together
    while (pa != a) { a = pa; pa = ld_ca(&nd[a].x); }
    while (pb != b) { b = pb; pb = ld_ca(&nd[b].x); }
    while (a != b) {
        if (a < b) { const int s = a; a = b; b = s; }      // a is the larger
        const int old = atomicMin(&nd[a].x, b);
        if (old == a) break;
        a = old;
    }
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
__device__ __forceinline__ int4 ld_cg_int4(const int4* p) {
    int4 v; asm volatile("ld.global.cg.v4.s32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p) : "memory"); return v;
}
// one warp: the pieces sub * 32 .., (sub + wpt) * 32 .. of `tile` (n of them) on the lattice's node array nd
template <int CAP, bool CG>
__device__ __forceinline__ void roots_warp(int4* nd, const int n, const int tile, const int sub, const int wpt, const int lane) {
    int hot = -1, hotacc = 0, hotmin = 0x7fffffff;
    for (int e0 = 32 * sub; e0 < n; e0 += 32 * wpt) {
        const int e = e0 + lane;
        const bool on = e < n;
        int root = -1 - lane, add = 0, g = 0x7fffffff;      // idle lanes: distinct keys, nothing to add
        if (on) {
            const int id = tile * CAP + e;
            const int4 me = CG ? ld_cg_int4(nd + id) : nd[id];
            root = me.x;
            if (root != id) {                               // hooked: (no root changes during this kernel)
                root = nd_find<CG>(nd, root);
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
template <int CAP>
__global__ void __launch_bounds__(256)
k_roots_nodes(int4* nodes, const int* __restrict__ ocount, int tiles, int wpt) {
    pdl_wait();
    const int gw = blockIdx.x * 8 + (threadIdx.x >> 5);
    const int tile = gw / wpt, sub = gw - tile * wpt;
    if (tile >= tiles) return;                              // (warp-uniform)
    roots_warp<CAP, false>(nodes + (size_t)blockIdx.y * tiles * CAP, ocount[(size_t)blockIdx.y * tiles + tile], tile, sub, wpt, threadIdx.x & 31);
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
