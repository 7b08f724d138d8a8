// sw_word.cuh -- the fast path, second generation: one THREAD per 32-site bit-plane word.
//
// Why: the scan-line kernels (sw_scan.cuh) spend one lane per site, so every per-site step costs a warp
// instruction per 32 sites; ncu showed them issue-bound at ~200 thread instructions per site
// (profiles/r1a_ncu_full.md).  Here a thread owns a whole word: runs of East bonds come from bit tricks on
// the word, only run HEADS are union-find nodes, only the South bonds that join a new pair of runs are
// united, and everything per-site that remains (flat parents, global labels) is a vectorised copy.
//
// Stage map; one CTA per tile of TW x TH sites, TW = 32 * WPR, WPR * TH threads:
//   a1+a2 k_word_label<WPR, TH, FUSE>
//       phase 0  thread (row, wx): sign masks of the int8 spins, 16 Philox4x32-10 calls, bond words to shared
//                memory and to the canonical global bit-planes; bonds entering the tile from its North / West
//                neighbours recomputed from the same draws (TW/2 + TH extra calls); par[l] = l
//       phase 1  unions between run heads: the run that continues into the next word, and every South bond
//                whose left neighbour does not already join the same two runs.  find = path halving on the
//                shared parent array, hook = atomicMin "larger under smaller" (root = minimum index whatever
//                the interleaving; "lowest value label")
//       phase 2  per run: root of its head; flat parent for each of its sites; run lengths summed into the
//                spare bits of the root's word; open flag if the run has a bond across the tile edge
//       phase 3  closed clusters -> running maximum; open clusters -> the tile's list (root, size);
//                global label of every site = global index of its tile root (128-bit stores)
//   The global merge (a3) and the fused assignment kernel (a4-a7) are those of sw_tiled.cuh / sw_scan.cuh.
#pragma once
#include "sw_common.cuh"
#include "sw_scan.cuh"

namespace sw {

__host__ __device__ constexpr int ilog2_c(int v) { return v <= 1 ? 0 : 1 + ilog2_c(v >> 1); }

// root of x while unions are running (no size / flag bits yet): path halving, plain stores.
// A halving store only ever replaces a non-root's parent by one of its ancestors, so it is safe against
// concurrent hooks (which change roots) and other halvings.
__device__ __forceinline__ int wd_find(int* par_, int x) {
    volatile int* par = par_;
    int p = par[x];
    while (p != x) {
        const int g = par[p];
        if (g == p) return p;
        par[x] = g;
        x = g; p = par[x];
    }
    return x;
}
__device__ __forceinline__ void wd_union(int* par, int a, int b) {
    a = wd_find(par, a); b = wd_find(par, b);
    while (a != b) {
        if (a < b) { const int s = a; a = b; b = s; }      // a is the larger root
        const int old = atomicMin(par + a, b);
        if (old == a) break;                                // a was still a root: hooked under b
        a = wd_find(par, old);                              // a had been hooked meanwhile: climb on
    }
}
// column of the head of the run that holds column c; hm = ~(e << 1) has bit k set iff column k starts a run
__device__ __forceinline__ int run_head(uint32_t hm, int c) {
    return 31 - __clz(hm & ((2u << c) - 1u));
}

template <int WPR, int TH, bool FUSE>
__global__ void __launch_bounds__(WPR * TH)
k_word_label(const int8_t* __restrict__ spins, uint32_t* bondE, uint32_t* bondS,
             int* __restrict__ label, int2* __restrict__ olist, int* __restrict__ ocount,
             Rec* __restrict__ rec, const Lat* __restrict__ lat, const Ctl* __restrict__ ctl,
             int L, int N, int words, int nb) {
    constexpr int TW = 32 * WPR, SITES = TW * TH, THREADS = WPR * TH;
    constexpr int CAP = 2 * (TW + TH);
    constexpr int LOG_TW = ilog2_c(TW);
    constexpr int QSTEPS = SITES / 4 / THREADS;          // = 8
    static_assert(SITES <= 8192 && TH <= 64 && (TW & (TW - 1)) == 0, "tile shape");
    __shared__ __align__(16) int par[SITES];   // parent, tile-local index (+ size / open bits at roots)
    __shared__ uint2 es[THREADS];              // [row][wx] = (East word, South word)
    __shared__ uint32_t nIn[WPR];              // South bonds entering from the tile above
    __shared__ uint32_t wIn[2];                // East bonds entering from the tile to the West, bit = row
    __shared__ int s_nopen, s_max;

    const int tid = threadIdx.x, lane = tid & 31;
    const int tilesX = L / TW;
    const int ty = blockIdx.x / tilesX, tx = blockIdx.x - ty * tilesX;
    const int y0 = ty * TH, x0 = tx * TW;
    const int wprL = L >> 5;
    const int row = tid / WPR, wx = tid - row * WPR;
    const int8_t* s = spins + (size_t)blockIdx.y * N;
    const Lat la = lat[blockIdx.y];
    const unsigned long long t = ctl->t;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);

    if (tid < WPR) nIn[tid] = 0;
    if (tid < 2) wIn[tid] = 0;
    if (tid == 0) { s_nopen = 0; s_max = 0; }
#pragma unroll
    for (int k = 0; k < QSTEPS; ++k) {
        const int q = k * THREADS + tid;
        *reinterpret_cast<int4*>(par + 4 * q) = make_int4(4 * q, 4 * q + 1, 4 * q + 2, 4 * q + 3);
    }
    __syncthreads();

    // ---- phase 0: bonds of the tile, PAPER.md:37-39 (section 2.1) --------------------------------------
    uint32_t e, so;
    if (!FUSE) {
        const uint32_t* bE = bondE + (size_t)blockIdx.y * words;
        const uint32_t* bS = bondS + (size_t)blockIdx.y * words;
        const size_t gw = (size_t)(y0 + row) * wprL + (x0 >> 5) + wx;
        e = bE[gw]; so = bS[gw];
        if (tid < WPR) nIn[tid] = bS[(size_t)(y0 == 0 ? L - 1 : y0 - 1) * wprL + (x0 >> 5) + tid];
        if (tid >= THREADS - TH) {                                   // (not the threads that wrote nIn)
            const int r = tid - (THREADS - TH);
            const int wl = (x0 >> 5) == 0 ? wprL - 1 : (x0 >> 5) - 1;
            if (bE[(size_t)(y0 + r) * wprL + wl] >> 31) atomicOr(&wIn[r >> 5], 1u << (r & 31));
        }
    } else {
        const PhiloxKey key(la.key0, la.key1);
        {
            const int y = y0 + row;
            const int xw = (x0 >> 5) + wx;
            const int w = y * wprL + xw;                              // word index within the lattice
            const int8_t* r0 = s + (size_t)y * L + xw * 32;
            const int8_t* r1 = s + (size_t)(y + 1 == L ? 0 : y + 1) * L + xw * 32;
            const uint4 a0 = *reinterpret_cast<const uint4*>(r0), a1 = *reinterpret_cast<const uint4*>(r0 + 16);
            const uint4 b0 = *reinterpret_cast<const uint4*>(r1), b1 = *reinterpret_cast<const uint4*>(r1 + 16);
            const int8_t nx = s[(size_t)y * L + (xw + 1 == wprL ? 0 : (xw + 1) * 32)];
            const uint32_t own = neg_mask32(a0, a1), south = neg_mask32(b0, b1);
            const uint32_t eastm = (own >> 1) | (nx < 0 ? 0x80000000u : 0u);
            const uint32_t eqE = ~(own ^ eastm), eqS = ~(own ^ south);
            uint32_t dE = 0, dS = 0;
#pragma unroll
            for (int c = 0; c < 16; ++c) {
                const uint4 r = philox4x32_10((uint32_t)w * 16u + c, tlo, thi, TAG_BOND, key);
                dE |= (r.x < la.thr ? 1u : 0u) << (2 * c) | (r.z < la.thr ? 1u : 0u) << (2 * c + 1);
                dS |= (r.y < la.thr ? 1u : 0u) << (2 * c) | (r.w < la.thr ? 1u : 0u) << (2 * c + 1);
            }
            e = eqE & dE; so = eqS & dS;
            bondE[(size_t)blockIdx.y * words + w] = e;
            bondS[(size_t)blockIdx.y * words + w] = so;
        }
        // bonds entering the tile: South bonds of the row above (TW / 2 calls), East bonds of the column to
        // the West (TH calls).  They are owned by the neighbouring tiles; recomputed here from the same draws.
        for (int j = tid; j < TW / 2 + TH; j += THREADS) {
            if (j < TW / 2) {
                const int yn = y0 == 0 ? L - 1 : y0 - 1;
                const int x = x0 + 2 * j;
                const int i = yn * L + x;                                  // even site; call covers i, i + 1
                const uint4 r = philox4x32_10((uint32_t)(i >> 1), tlo, thi, TAG_BOND, key);
                const int8_t u0 = s[i], u1 = s[i + 1];
                const int8_t d0 = s[(size_t)y0 * L + x], d1 = s[(size_t)y0 * L + x + 1];
                const uint32_t bits = ((u0 == d0 && r.y < la.thr) ? 1u : 0u) | ((u1 == d1 && r.w < la.thr) ? 2u : 0u);
                if (bits) atomicOr(&nIn[(2 * j) >> 5], bits << ((2 * j) & 31));
            } else {
                const int r_ = j - TW / 2;
                const int xwst = x0 == 0 ? L - 1 : x0 - 1;                 // odd column
                const int i = (y0 + r_) * L + xwst;
                const uint4 r = philox4x32_10((uint32_t)(i >> 1), tlo, thi, TAG_BOND, key);
                if (s[i] == s[(size_t)(y0 + r_) * L + x0] && r.z < la.thr) atomicOr(&wIn[r_ >> 5], 1u << (r_ & 31));
            }
        }
    }
    es[tid] = make_uint2(e, so);
    __syncthreads();

    // ---- phase 1: unions between run heads, PAPER.md:49-51 (section 2.3) -------------------------------
    const int base = row * TW + wx * 32;
    const uint32_t hm = ~(e << 1);                                   // bit c: column c starts a run
    if (wx + 1 < WPR && (e >> 31)) wd_union(par, base + run_head(hm, 31), base + 32);
    if (row + 1 < TH) {
        const uint32_t eb = es[tid + WPR].x;
        const uint32_t hb = ~(eb << 1);
        uint32_t need = so & ~((so & e & eb) << 1);                  // skip a bond whose left neighbour joins the same runs
        while (need) {
            const int c = __ffs(need) - 1;
            need &= need - 1;
            wd_union(par, base + run_head(hm, c), base + TW + run_head(hb, c));
        }
    }
    __syncthreads();

    // ---- phase 2: per run -- root, flat parents, size, open flag ----------------------------------------
    uint32_t rootbits = 0;                                           // bit c: my column c is a tile-local root
    {
        uint32_t X = 0;                                              // my sites with a bond across the tile edge
        if (row == 0) X |= nIn[wx];
        if (row == TH - 1) X |= so;
        if (wx == 0) X |= (wIn[row >> 5] >> (row & 31)) & 1u;
        if (wx == WPR - 1) X |= e & 0x80000000u;
        uint32_t h = hm;
        int lastr = -1; uint32_t acc = 0;
        while (h) {
            const int c = __ffs(h) - 1;
            h &= h - 1;
            const int nxt = h ? __ffs(h) - 1 : 32;
            const int x = base + c;
            int r = x, p = par[x] & (int)IDX_MASK;
            while (p != r) { r = p; p = par[r] & (int)IDX_MASK; }
            if (r == x) rootbits |= 1u << c;
            else par[x] = r;
            for (int k = c + 1; k < nxt; ++k) par[base + k] = r;
            const uint32_t runmask = (nxt == 32 ? 0u : (1u << nxt)) - (1u << c);
            if (X & runmask) atomicOr(reinterpret_cast<unsigned int*>(par + r), OPEN_BIT);
            if (r != lastr) {
                if (acc) atomicAdd(reinterpret_cast<unsigned int*>(par + lastr), acc << CNT_SHIFT);
                lastr = r; acc = 0;
            }
            acc += (uint32_t)(nxt - c);
        }
        if (acc) atomicAdd(reinterpret_cast<unsigned int*>(par + lastr), acc << CNT_SHIFT);
    }
    __syncthreads();

    // ---- phase 3: lists of open clusters, maximum of the closed ones, global labels ---------------------
    {
        int mymax = 0;
        int2* mylist = olist + ((size_t)blockIdx.y * gridDim.x + blockIdx.x) * CAP;
        while (rootbits) {
            const int c = __ffs(rootbits) - 1;
            rootbits &= rootbits - 1;
            const uint32_t v = (uint32_t)par[base + c];
            const int cnt = (int)((v >> CNT_SHIFT) & CNT_MASK);
            if (v & OPEN_BIT) {
                const int pos = atomicAdd(&s_nopen, 1);
                mylist[pos] = make_int2((y0 + row) * L + x0 + wx * 32 + c, cnt);
            } else {
                mymax = max(mymax, cnt);
            }
        }
        mymax = warp_max_i(mymax);
        if (lane == 0 && mymax) atomicMax(&s_max, mymax);
    }
    {
        int* glab = label + (size_t)blockIdx.y * N;
        const int tilebase = y0 * L + x0;
#pragma unroll
        for (int k = 0; k < QSTEPS; ++k) {
            const int q = k * THREADS + tid;
            const int r_ = (4 * q) >> LOG_TW, col = (4 * q) & (TW - 1);
            const int4 v = *reinterpret_cast<const int4*>(par + 4 * q);
            int4 g;
            { const int r = v.x & (int)IDX_MASK; g.x = tilebase + (r >> LOG_TW) * L + (r & (TW - 1)); }
            { const int r = v.y & (int)IDX_MASK; g.y = tilebase + (r >> LOG_TW) * L + (r & (TW - 1)); }
            { const int r = v.z & (int)IDX_MASK; g.z = tilebase + (r >> LOG_TW) * L + (r & (TW - 1)); }
            { const int r = v.w & (int)IDX_MASK; g.w = tilebase + (r >> LOG_TW) * L + (r & (TW - 1)); }
            *reinterpret_cast<int4*>(glab + (size_t)(y0 + r_) * L + x0 + col) = g;
        }
    }
    __syncthreads();
    if (tid == 0) {
        ocount[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = s_nopen;
        if (s_max) atomic_max_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].maxcl, s_max);
    }
}

} // namespace sw
