// sw_flip_tma.cuh -- a4-a6 of the fast path with the 16-bit root plane staged by the TMA engine (north_star: "TMA or
// cp.async staging ... into shared memory").  PAPER.md:57 (section 2.4); same result as k_flip16<4, 64, BITS> (sw_scan.cuh).
//
// k_flip16 keeps 16 KB of roots in flight per CTA (four 16-byte loads per thread) and then waits on a chain of
// dependent loads (open-root count -> node -> root node -> decision word) before it can use them: ~3.0 TB/s on the
// 537 MB plane at L = 16384.  Here a CTA is persistent over the tiles blockIdx.x, blockIdx.x + gridDim.x, ...; one
// thread issues cp.async.bulk.tensor.2d loads of the NEXT tiles' 128 x 64 x 2 B boxes into a ring of shared-memory
// stages (mbarrier complete_tx), so the plane streams while the chain of the current tile resolves.
#pragma once
#include <cuda.h>
#include "sw_scan.cuh"

namespace sw {

constexpr int FT_TILE_BYTES = 128 * 64 * 2;

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "W_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra D_%=;\n"
        "bra W_%=;\n"
        "D_%=:\n"
        "}\n" :: "r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* tm, int c0, int c1, uint32_t bar) {
    asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                 :: "r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar) : "memory");
}

__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" :: "r"(bar) : "memory");
}
__device__ __forceinline__ void bar_consumers() { asm volatile("bar.sync 1, 256;" ::: "memory"); }
__device__ __forceinline__ uint32_t lds_u8(uint32_t a) {
    uint32_t v; asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a) : "memory"); return v;
}
__device__ __forceinline__ void sts_u8(uint32_t a, uint32_t v) {
    asm volatile("st.shared.u8 [%0], %1;" :: "r"(a), "r"(v) : "memory");
}

constexpr int FT_CAP = 2 * (128 + 64);                         // open roots a 128 x 64 tile can have
#ifndef FT_NS
#define FT_NS 5
#endif
#ifndef FT_CTAS
#define FT_CTAS 2
#endif
constexpr int FT_CTAS_PER_SM = FT_CTAS;
constexpr int FT_NSTAGE = FT_NS;
#ifndef FT_PW
#define FT_PW 5
#endif
constexpr int FT_PROD_WARPS = FT_PW;
#ifndef FT_CH
#define FT_CH 4
#endif
// (a stage is filled by ONE producer warp, tile after tile: a waiter on an mbarrier phase may not run more than one phase ahead)
static_assert(FT_NSTAGE % FT_PROD_WARPS == 0, "stages per producer warp");
constexpr int FT_OFF_DEC = FT_TILE_BYTES;                      // the tile's own 256 decision words
constexpr int FT_OFF_LIST = FT_OFF_DEC + 1024;                 // its open roots: (tile-local index) | (decision << 15), uint16 each
constexpr int FT_OFF_N = FT_OFF_LIST + FT_CAP * 2;             // how many
constexpr int FT_STAGE_BYTES = (FT_OFF_N + 16 + 127) / 128 * 128;

// Warp-specialised, persistent: grid = (CTAs per lattice, nb), 256 consumer threads + FT_PROD_WARPS producer warps, dynamic shared
// memory = FT_NSTAGE * FT_STAGE_BYTES + 128.  A CTA owns the tiles blockIdx.x, blockIdx.x + gridDim.x, ...; tile j of its
// sequence goes through stage j % FT_NSTAGE.
//   producer warp p (tiles j = p, p + FT_PROD_WARPS, ...): waits until the consumers have released the stage, lane 0 issues two TMA
//     box loads into it -- the 128 x 64 box of 16-bit roots and the 4 x 64 box of the tile's own decision words -- and the
//     whole warp meanwhile resolves the tile's open roots: the chain of dependent loads open-root count -> node -> root
//     node -> decision word, four chains per lane in flight, result (tile-local index | decision << 15) written into the
//     stage; lane 0 then arrives on the stage's `full` barrier with the boxes' byte count (mbarrier complete_tx).
//   consumers: wait on `full`, build one decision BYTE per tile root in shared memory (own words, then the open roots'
//     list), look every site's byte up by its 16-bit root from the staged box, store a byte per 8 sites, release the stage.
// The consumers never wait on global memory; the producers' chains run up to FT_NSTAGE - 1 tiles ahead.  The nodes that are roots are the
// clusters that span tiles: counted, and their sizes maximised, by the producers.
__global__ void __launch_bounds__(256 + 32 * FT_PROD_WARPS, FT_CTAS_PER_SM)
k_flip16_tma(const __grid_constant__ CUtensorMap tm_lab, const __grid_constant__ CUtensorMap tm_dec,
             uint32_t* __restrict__ sbits, const uint32_t* __restrict__ D, const int4* __restrict__ nodes,
             const int* __restrict__ ocount, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
             DivL dv, int L, int N, int words, int nb, int tiles) {
    pdl_wait();
    constexpr int NW = 4, TH = 64, TW = 128, OSTEPS = 4, LOG_TW = 7;
    extern __shared__ __align__(128) uint8_t stage_mem[];
    __shared__ __align__(8) uint64_t full[FT_NSTAGE], empty[FT_NSTAGE];
    __shared__ __align__(16) uint8_t dec8[2][TH * TW];             // one decision BYTE per tile root (double-buffered)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int tilesX = L / TW;
    const uint32_t stage_s = ((uint32_t)__cvta_generic_to_shared(stage_mem) + 127u) & ~127u;   // (the launch adds 128 bytes for this)
    const uint32_t full_s = (uint32_t)__cvta_generic_to_shared(full), empty_s = (uint32_t)__cvta_generic_to_shared(empty);
    const int ntile = (tiles - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;     // tiles of this CTA

    if (tid == 0) {
        for (int s = 0; s < FT_NSTAGE; ++s) { mbar_init(full_s + 8u * s, 1u); mbar_init(empty_s + 8u * s, 8u); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp >= 8) {
        // ===== producers =====
        const int p = warp - 8;
        const uint32_t* d = D + (size_t)blockIdx.y * words;
        const size_t lb = (size_t)blockIdx.y * tiles * FT_CAP;
        int nroot = 0, big = 0;
        constexpr int CH = FT_CH;                                       // chains per lane in flight
        int n_next = p < ntile ? ocount[(size_t)blockIdx.y * tiles + blockIdx.x + p * gridDim.x] : 0;
        for (int j = p; j < ntile; j += FT_PROD_WARPS) {
            const int s = j % FT_NSTAGE;
            const int tile = blockIdx.x + j * gridDim.x;
            const int ty = tile / tilesX, tx = tile - ty * tilesX;
            const int tilebase = ty * TH * L + tx * TW;
            const uint32_t dst = stage_s + (uint32_t)s * FT_STAGE_BYTES;
            if (j >= FT_NSTAGE) mbar_wait(empty_s + 8u * s, (uint32_t)((j / FT_NSTAGE - 1) & 1));   // the consumers are done with tile j - FT_NSTAGE
            if (lane == 0) {
                asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
                tma_load_2d(dst, &tm_lab, tx * TW, blockIdx.y * L + ty * TH, full_s + 8u * s);
                tma_load_2d(dst + FT_OFF_DEC, &tm_dec, tx * NW, blockIdx.y * L + ty * TH, full_s + 8u * s);
            }
            const int n = n_next;                                      // (loaded a tile ahead: one dependent load less per tile)
            if (j + FT_PROD_WARPS < ntile) n_next = ocount[(size_t)blockIdx.y * tiles + tile + FT_PROD_WARPS * gridDim.x];
            for (int e0 = lane; e0 < n; e0 += 32 * CH) {               // CH independent chains per lane and round
                int4 me[CH]; int R[CH];
#pragma unroll
                for (int u = 0; u < CH; ++u) if (e0 + 32 * u < n) me[u] = nodes[lb + tile * FT_CAP + e0 + 32 * u];
#pragma unroll
                for (int u = 0; u < CH; ++u) if (e0 + 32 * u < n) {
                    const int id = tile * FT_CAP + e0 + 32 * u;        // (root node, size, min site, site of the tile root)
                    R[u] = me[u].x == id ? me[u].z : nodes[lb + me[u].x].z;
                    if (me[u].x == id) { ++nroot; big = max(big, me[u].y); }
                }
#pragma unroll
                for (int u = 0; u < CH; ++u) if (e0 + 32 * u < n) {
                    const uint32_t up = (__ldg(d + (R[u] >> 5)) >> (R[u] & 31)) & 1u;
                    const int delta = me[u].w - tilebase;
                    const int ry = div_l(delta, dv);
                    sts_u16(dst + FT_OFF_LIST + 2u * (e0 + 32 * u), (uint32_t)(ry * TW + (delta - ry * L)) | (up << 15));
                }
            }
            if (lane == 0) asm volatile("st.shared.u32 [%0], %1;" :: "r"(dst + FT_OFF_N), "r"(n) : "memory");
            __syncwarp();
            if (lane == 0) mbar_expect_tx(full_s + 8u * s, FT_TILE_BYTES + 1024);     // (arrive: the list is written; the boxes complete the count)
        }
        nroot = warp_sum_i(nroot); big = warp_max_i(big);
        if (lane == 0 && (nroot | big)) {
            Rec* r = rec + (size_t)ctl->slot * nb + blockIdx.y;
            if (nroot) atomic_add_ll(&r->ncl, nroot);
            if (big) atomic_max_ll(&r->maxcl, big);
        }
        return;
    }

    // ===== consumers (threads 0 .. 255) =====
    for (int k = 0; k < ntile; ++k) {
        const int s = k % FT_NSTAGE;
        const int tile = blockIdx.x + k * gridDim.x;
        const int ty = tile / tilesX, tx = tile - ty * tilesX;
        const int y0 = ty * TH, x0 = tx * TW;
        const uint32_t dc_s = (uint32_t)__cvta_generic_to_shared(dec8[k & 1]);
        mbar_wait(full_s + 8u * s, (uint32_t)((k / FT_NSTAGE) & 1));
        const uint32_t base = stage_s + (uint32_t)s * FT_STAGE_BYTES;
        // one decision byte per tile root: the tile's own words of the decision plane, a bit spread into a byte (a nibble
        // times 0x00204081 puts bit j at bit 8 j); open roots take their cluster root's.  A byte table costs 16 KB against
        // 2 KB of bits, and makes the per-site lookup a byte load and a multiply-add instead of eight ALU instructions.
        {
            const uint32_t w = lds_u32(base + FT_OFF_DEC + 4u * tid);      // (box rows are 4 words: word (row, wx) at 4 row + wx)
            uint32_t e[8];
#pragma unroll
            for (int g = 0; g < 8; ++g) e[g] = (((w >> (4 * g)) & 0xFu) * 0x00204081u) & 0x01010101u;
            sts_u128(dc_s + 32u * tid, make_uint4(e[0], e[1], e[2], e[3]));
            sts_u128(dc_s + 32u * tid + 16u, make_uint4(e[4], e[5], e[6], e[7]));
        }
        const int n = (int)lds_u32(base + FT_OFF_N);
        bar_consumers();
        for (int e = tid; e < n; e += 256) {
            const uint32_t v = lds_u16(base + FT_OFF_LIST + 2u * e);
            sts_u8(dc_s + (v & 0x1FFFu), v >> 15);
        }
        bar_consumers();
#pragma unroll
        for (int q = 0; q < OSTEPS; ++q) {
            const int l = 8 * (q * 256 + tid);
            const uint4 v = lds_u128(base + 2u * l);                       // (the box is row-major: site l at byte 2 l)
            const uint32_t w4[4] = { v.x, v.y, v.z, v.w };
            uint32_t b8 = 0;                                               // bit u: site l + u goes up
            uint32_t pr = 0xFFFFFFFFu, pb = 0;                             // (a site often has its left neighbour's root: no second lookup)
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint32_t r = (u & 1) ? (w4[u >> 1] >> 16) : (w4[u >> 1] & 0xFFFFu);
                if (r != pr) pb = lds_u8(dc_s + r);
                pr = r;
                b8 += pb << u;
            }
            const size_t gsite = (size_t)blockIdx.y * N + (size_t)(y0 + (l >> LOG_TW)) * L + x0 + (l & (TW - 1));
            reinterpret_cast<uint8_t*>(sbits)[gsite >> 3] = (uint8_t)b8;
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_s + 8u * s);                       // this warp is done with the stage
    }
}

} // namespace sw
