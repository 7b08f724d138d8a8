// sw_tiled.cuh -- the fast path for lattice sides that are a multiple of the tile width.
//
// Stage map:
//   a1 k_bond_rows      Philox bond draws, one thread per bit-plane word (32 sites, 16 Philox calls)
//   a2 k_tile_label     shared-memory union-find of one TW x TH tile: rows are pre-united by run
//                       length from the East-bond word (bit tricks, no atomics), vertical unions only
//                       where a South bond starts a new overlap of two runs; writes label[i] = global
//                       index of the tile-local root; tile-local cluster sizes; the list of "open"
//                       clusters (those with a bond across the tile edge)
//   a3 k_merge_tiled    one thread per tile-edge bond: atomicMin hooking on the global parent array
//      k_roots_open     points every hooked tile root at its global root; sizes of clusters that span
//                       tiles (closed clusters were maximised in a2)
//   a4 k_compress_tiled label[i] = label[label[i]] (two hops), 128-bit loads/stores; counts roots
//   a5 k_flipbits       (sw_generic.cuh) decision bit-plane
//   a6 k_flip_rows      spins = gather(D, label); magnetisation
//   a7 k_energy_rows    energy of the new configuration from sign masks + popc
#pragma once
#include "sw_common.cuh"

namespace sw {

constexpr int ROW_THREADS = 256;
constexpr uint32_t OPEN_FLAG = 0x40000000u;

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
// a2 tile-local labelling, PAPER.md:49-51 (section 2.3) with the algorithm north_star names:
// shared-memory union-find, min-index roots.
// ---------------------------------------------------------------------------------------------
template <int TW, int TH>
struct TileCfg {
    static constexpr int SITES = TW * TH;
    static constexpr int WPR = TW / 32;              // bond words per tile row
    static constexpr int RW = TH * WPR;              // row-words per tile
    static constexpr int THREADS = 1024;
    static constexpr int RW_PER_WARP = RW / 32;      // each warp owns RW/32 row-words, lane = x in the word
    static constexpr int CAP = 2 * (TW + TH);        // upper bound on open clusters per tile
    static_assert(TW % 32 == 0 && RW % 32 == 0, "tile shape");
};

// Shared-memory union-find.  Roots are hooked "larger under smaller" with a CAS that only succeeds
// on a node that is still a root, so a parent is always a smaller index, trees never split, and
// non-root parents change only through path halving (to an ancestor) -- safe under any interleaving.
__device__ __forceinline__ int s_find(int* lab_, int x) {
    volatile int* lab = lab_;
    int p = lab[x];
    while (p != x) {
        const int g = lab[p];
        if (g == p) return p;
        lab[x] = g;                      // path halving
        x = g; p = lab[x];
    }
    return x;
}
__device__ __forceinline__ void s_union(int* lab, int a, int b) {
    a = s_find(lab, a); b = s_find(lab, b);
    while (a != b) {
        if (a < b) { int s = a; a = b; b = s; }           // a is the larger root
        const int old = atomicCAS(lab + a, a, b);
        if (old == a) break;                               // hooked
        a = s_find(lab, old);                              // a had been hooked meanwhile: climb on
    }
}

template <int TW, int TH>
__global__ void __launch_bounds__(TileCfg<TW, TH>::THREADS)
k_tile_label(int* __restrict__ label, const uint32_t* __restrict__ bondE, const uint32_t* __restrict__ bondS,
             int2* __restrict__ olist, int* __restrict__ ocount, Rec* __restrict__ rec,
             const Ctl* __restrict__ ctl, int L, int N, int words, int nb) {
    using C = TileCfg<TW, TH>;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    int* lab = reinterpret_cast<int*>(smem_raw);                  // [SITES] parent, tile-local index
    int* cnt = lab + C::SITES;                                    // [SITES] size at roots (+ OPEN_FLAG)
    uint32_t* eW = reinterpret_cast<uint32_t*>(cnt + C::SITES);   // [RW] East-bond words of the tile
    uint32_t* sW = eW + C::RW;                                    // [RW] South-bond words
    uint32_t* nIn = sW + C::RW;                                   // [WPR] South bonds entering from the North tile
    int* s_misc = reinterpret_cast<int*>(nIn + C::WPR);           // [2] open-list cursor, closed maximum
    uint8_t* wIn = reinterpret_cast<uint8_t*>(s_misc + 2);        // [TH] East bonds entering from the West tile
    int& s_nopen = s_misc[0];
    int& s_max = s_misc[1];

    const int tilesX = L / TW;
    const int ty = blockIdx.x / tilesX, tx = blockIdx.x - ty * tilesX;
    const int y0 = ty * TH, x0 = tx * TW;
    const int wprL = L >> 5;
    const uint32_t* bE = bondE + (size_t)blockIdx.y * words;
    const uint32_t* bS = bondS + (size_t)blockIdx.y * words;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // phase 0: the tile's bond words, plus the bonds that enter it from the West and North tiles
    for (int idx = tid; idx < C::RW; idx += C::THREADS) {
        const int row = idx / C::WPR, wx = idx - row * C::WPR;
        const size_t gw = (size_t)(y0 + row) * wprL + (x0 >> 5) + wx;
        eW[idx] = bE[gw]; sW[idx] = bS[gw];
    }
    if (tid < TH) {
        const int wl = (x0 >> 5) == 0 ? wprL - 1 : (x0 >> 5) - 1;
        wIn[tid] = (uint8_t)(bE[(size_t)(y0 + tid) * wprL + wl] >> 31);
    }
    if (tid < C::WPR) {
        const int yn = y0 == 0 ? L - 1 : y0 - 1;
        nIn[tid] = bS[(size_t)yn * wprL + (x0 >> 5) + tid];
    }
    if (tid == 0) { s_nopen = 0; s_max = 0; }
    __syncthreads();

    // phase 1: every site starts at the head of its horizontal run inside its 32-site word
#pragma unroll
    for (int k = 0; k < C::RW_PER_WARP; ++k) {
        const int rw = warp + 32 * k;
        const uint32_t e = eW[rw];
        const int ones = lane ? __clz(~(e << (32 - lane))) : 0;      // bonded sites directly to my left
        const int row = rw / C::WPR, wx = rw - row * C::WPR;
        const int l = row * TW + wx * 32 + lane;
        lab[l] = l - ones;
        cnt[l] = 0;
    }
    __syncthreads();

    // phase 2: unions -- runs that continue across a word boundary, and South bonds.  A South bond
    // is skipped when its left neighbour already joins the same two runs.
#pragma unroll
    for (int k = 0; k < C::RW_PER_WARP; ++k) {
        const int rw = warp + 32 * k;
        const int row = rw / C::WPR, wx = rw - row * C::WPR;
        const int l = row * TW + wx * 32 + lane;
        if (lane == 0 && wx > 0 && (eW[rw - 1] >> 31)) s_union(lab, l - 1, l);
        if (row < TH - 1) {
            const uint32_t sb = sW[rw];
            const uint32_t need = sb & ~((sb & eW[rw] & eW[rw + C::WPR]) << 1);
            if ((need >> lane) & 1u) s_union(lab, l, l + TW);
        }
    }
    __syncthreads();

    // phase 3: flatten (lab[l] = root), sizes (one shared atomic per run head), global labels
    int* glab = label + (size_t)blockIdx.y * N;
#pragma unroll
    for (int k = 0; k < C::RW_PER_WARP; ++k) {
        const int rw = warp + 32 * k;
        const int row = rw / C::WPR, wx = rw - row * C::WPR;
        const int l = row * TW + wx * 32 + lane;
        const int r = s_find(lab, l);
        lab[l] = r;
        const uint32_t e = eW[rw];
        const bool head = lane == 0 || !((e >> (lane - 1)) & 1u);
        if (head) {
            const uint32_t tbits = ~(e >> lane);                      // first 0 above me ends the run
            const int len = min(tbits ? __ffs(tbits) : 33, 32 - lane);
            atomicAdd(&cnt[r], len);
        }
        const int rr = r / TW, rx = r - rr * TW;
        glab[(size_t)(y0 + row) * L + x0 + wx * 32 + lane] = (y0 + rr) * L + x0 + rx;
    }
    __syncthreads();

    // phase 4: a cluster is "open" when one of its sites has a bond across the tile edge
#pragma unroll
    for (int k = 0; k < C::RW_PER_WARP; ++k) {
        const int rw = warp + 32 * k;
        const int row = rw / C::WPR, wx = rw - row * C::WPR;
        bool open = false;
        if (wx == C::WPR - 1 && lane == 31 && (eW[rw] >> 31)) open = true;
        if (wx == 0 && lane == 0 && wIn[row]) open = true;
        if (row == TH - 1 && ((sW[rw] >> lane) & 1u)) open = true;
        if (row == 0 && ((nIn[wx] >> lane) & 1u)) open = true;
        if (open) atomicOr(reinterpret_cast<unsigned int*>(&cnt[lab[row * TW + wx * 32 + lane]]), OPEN_FLAG);
    }
    __syncthreads();

    // phase 5: closed clusters are complete -> maximise their size; open ones go to the tile's list
    int mymax = 0;
    int2* mylist = olist + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * C::CAP;
#pragma unroll
    for (int k = 0; k < C::RW_PER_WARP; ++k) {
        const int rw = warp + 32 * k;
        const int row = rw / C::WPR, wx = rw - row * C::WPR;
        const int l = row * TW + wx * 32 + lane;
        if (lab[l] == l) {
            const uint32_t c = (uint32_t)cnt[l];
            if (c & OPEN_FLAG) {
                const int pos = atomicAdd(&s_nopen, 1);
                mylist[pos] = make_int2((y0 + row) * L + x0 + wx * 32 + lane, (int)(c & ~OPEN_FLAG));
            } else {
                mymax = max(mymax, (int)c);
            }
        }
    }
    mymax = warp_max_i(mymax);
    if (lane == 0 && mymax) atomicMax(&s_max, mymax);
    __syncthreads();
    if (tid == 0) {
        ocount[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = s_nopen;
        if (s_max) atomic_max_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].maxcl, s_max);
    }
}

// ---------------------------------------------------------------------------------------------
// a3 global boundary merge: one thread per site on a tile's East column or South row.  The union starts
// from the two sites' tile roots (label[site] after a2), so label[] of a non-root site is never written
// here and stays "my tile root": the later passes rely on site -> tile root -> global root (two hops).
// ---------------------------------------------------------------------------------------------
template <int TW, int TH>
__global__ void __launch_bounds__(ROW_THREADS)
k_merge_tiled(int* label, const uint32_t* __restrict__ bondE, const uint32_t* __restrict__ bondS,
              int L, int N, int words) {
    const int tilesX = L / TW, tilesY = L / TH;
    const int nV = L * tilesX;                       // East-edge sites
    const int idx = blockIdx.x * ROW_THREADS + threadIdx.x;
    if (idx >= nV + tilesY * L) return;
    int* lab = label + (size_t)blockIdx.y * N;
    const int wprL = L >> 5;
    if (idx < nV) {
        const int y = idx / tilesX, c = idx - y * tilesX;
        const int x = c * TW + TW - 1;
        if (bondE[(size_t)blockIdx.y * words + (size_t)y * wprL + (x >> 5)] >> 31)
            uf_union_l1(lab, ld_cg(lab + y * L + x), ld_cg(lab + y * L + (x + 1 == L ? 0 : x + 1)));
    } else {
        const int j = idx - nV;
        const int r = j / L, x = j - r * L;
        const int y = r * TH + TH - 1;
        if ((bondS[(size_t)blockIdx.y * words + (size_t)y * wprL + (x >> 5)] >> (x & 31)) & 1u)
            uf_union_l1(lab, ld_cg(lab + y * L + x), ld_cg(lab + (y + 1 == L ? 0 : y + 1) * L + x));
    }
}

// ---------------------------------------------------------------------------------------------
// a4 compress: label[i] = root(i); four sites per thread, 128-bit accesses; counts roots.
// k_roots_open has already pointed every hooked tile root at its global root, so every site is at
// most two hops from it: site -> tile root -> global root.  No loops, no divergence.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(ROW_THREADS)
k_compress_tiled(int* label, Rec* __restrict__ rec, const Ctl* __restrict__ ctl, int N, int nb, int count) {
    const int q = blockIdx.x * ROW_THREADS + threadIdx.x;       // quad index
    int nroot = 0;
    if (q * 4 < N) {
        int* lab = label + (size_t)blockIdx.y * N;
        int4 v = *reinterpret_cast<const int4*>(lab + q * 4);
        const int t0 = lab[v.x], t1 = lab[v.y], t2 = lab[v.z], t3 = lab[v.w];   // tile root's parent
        nroot = (v.x == q * 4) + (v.y == q * 4 + 1) + (v.z == q * 4 + 2) + (v.w == q * 4 + 3);
        if (t0 != v.x || t1 != v.y || t2 != v.z || t3 != v.w)
            *reinterpret_cast<int4*>(lab + q * 4) = make_int4(t0, t1, t2, t3);
    }
    if (!count) return;
    nroot = warp_sum_i(nroot);
    if ((threadIdx.x & 31) == 0 && nroot)
        atomic_add_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].ncl, nroot);
}

// After the merge: every open tile-local root is pointed straight at its global root (find + write
// back), and the sizes of the clusters that span tiles are accumulated: each open piece adds its size
// to its root's accumulator; the running total returned by the atomic peaks at the full size.
// The list entry (tile root, size) becomes (tile root, cluster root) for the assignment kernel.
// count_roots != 0 (scan path): open tile roots that are cluster roots are counted here (closed ones
// were counted by k_bond_label).  One warp per tile.
template <int CAP>
__global__ void __launch_bounds__(ROW_THREADS)
k_roots_open(int* label, int2* __restrict__ olist, const int* __restrict__ ocount,
             int* __restrict__ gsize, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
             int tiles, int N, int nb, int count_roots) {
    const int tile = blockIdx.x * (ROW_THREADS / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    int m = 0, nroot = 0;
    if (tile < tiles) {                                     // (warp-uniform)
        const size_t t = (size_t)blockIdx.y * tiles + tile;
        int* lab = label + (size_t)blockIdx.y * N;
        int* gs = gsize + (size_t)blockIdx.y * N;
        const int n = ocount[t];
        // At T_c one cluster owns many pieces in every tile; a per-piece atomic on its accumulator would
        // serialise in L2.  Pieces are summed per root inside the warp first (match + reduce), and the
        // root with the largest sum of the first round ("hot") is carried in a register across rounds.
        int hot = -1, hotacc = 0;
        for (int e0 = 0; e0 < n; e0 += 32) {
            const int e = e0 + lane;
            const bool on = e < n;
            int R = -1 - lane, sz = 0;                      // idle lanes: distinct keys, nothing to add
            if (on) {
                const int2 it = olist[t * CAP + e];
                const int p = ld_cg(lab + it.x);
                R = p; sz = it.y;
                if (p != it.x) {                            // hooked: walk to the root, point at it
                    R = uf_find_l1(lab, p);                 // (no root changes during this kernel)
                    if (R != p) lab[it.x] = R;              // only ever an ancestor: safe while others walk
                } else {
                    ++nroot;
                }
                olist[t * CAP + e].y = R;
            }
            const unsigned grp = __match_any_sync(0xffffffffu, R);
            const int tot = __reduce_add_sync(grp, sz);
            if (e0 == 0) {                                  // choose the hot root
                const int best = __reduce_max_sync(0xffffffffu, tot);
                const unsigned who = __ballot_sync(0xffffffffu, tot == best && on);
                if (who) hot = __shfl_sync(0xffffffffu, R, __ffs(who) - 1);
            }
            const bool leader = on && lane == __ffs(grp) - 1;
            if (leader) {
                if (R == hot) hotacc += tot;                // (at most one leader per round has R == hot)
                else m = max(m, atomicAdd(gs + R, tot) + tot);
            }
        }
        hotacc = warp_sum_i(hotacc);
        if (lane == 0 && hotacc) m = max(m, atomicAdd(gs + hot, hotacc) + hotacc);
    }
    m = warp_max_i(m);
    if (lane == 0 && m) atomic_max_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].maxcl, m);
    if (count_roots) {
        nroot = warp_sum_i(nroot);
        if (lane == 0 && nroot) atomic_add_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].ncl, nroot);
    }
}

template <int CAP>
__global__ void __launch_bounds__(ROW_THREADS)
k_sizes_reset(const int2* __restrict__ olist, const int* __restrict__ ocount, int* __restrict__ gsize,
              int tiles, int N) {
    const int tile = blockIdx.x * (ROW_THREADS / 32) + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (tile >= tiles) return;
    const size_t t = (size_t)blockIdx.y * tiles + tile;
    const int n = ocount[t];
    for (int e = lane; e < n; e += 32) gsize[(size_t)blockIdx.y * N + olist[t * CAP + e].y] = 0;
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
