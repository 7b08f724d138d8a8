// sw_generic.cuh -- any-L kernels (L >= 2, any batch): the correct-first path and the fallback for
// lattice sides that are not a multiple of the tile.  Global union-find, no tiles.
// Batch lattice b = blockIdx.y everywhere; site / word index from blockIdx.x.
#pragma once
#include "sw_common.cuh"

namespace sw {

constexpr int GEN_THREADS = 256;

// ---- start configuration: spins[i] = bit_INIT(i) ? +1 : -1 (Fig. 1) ----------
// one thread per 32 sites (one word of the TAG_INIT bit field)
__global__ void __launch_bounds__(GEN_THREADS)
k_init_random(int8_t* __restrict__ spins, const Lat* __restrict__ lat, int N, int words) {
    const int w = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (w >= words) return;
    const Lat la = lat[blockIdx.y];
    const PhiloxKey key(la.key0, la.key1);
    const uint4 r = philox4x32_10((uint32_t)(w >> 2), 0u, 0u, TAG_INIT, key);
    const uint32_t bits = (w & 3) == 0 ? r.x : (w & 3) == 1 ? r.y : (w & 3) == 2 ? r.z : r.w;
    int8_t* s = spins + (size_t)blockIdx.y * N + (size_t)w * 32;
    const int n = min(32, N - w * 32);
    for (int k = 0; k < n; ++k) s[k] = ((bits >> k) & 1u) ? (int8_t)1 : (int8_t)-1;
}

__global__ void __launch_bounds__(GEN_THREADS)
k_fill_i8(int8_t* __restrict__ p, size_t n, int8_t v) {
    const size_t i = (size_t)blockIdx.x * GEN_THREADS + threadIdx.x;
    if (i < n) p[i] = v;
}

// ---- a1 bond formation: one thread per bit-plane word = 32 sites = 16 Philox calls
__global__ void __launch_bounds__(GEN_THREADS)
k_bond_generic(const int8_t* __restrict__ spins, uint32_t* __restrict__ bondE, uint32_t* __restrict__ bondS,
               const Lat* __restrict__ lat, const Ctl* __restrict__ ctl, int L, int N, int words) {
    const int w = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (w >= words) return;
    const Lat la = lat[blockIdx.y];
    const PhiloxKey key(la.key0, la.key1);
    const unsigned long long t = ctl->t;
    const uint32_t tlo = (uint32_t)t, thi = (uint32_t)(t >> 32);
    const int8_t* s = spins + (size_t)blockIdx.y * N;
    uint32_t e = 0, so = 0;
    const int i0 = w * 32;
#pragma unroll 4
    for (int c = 0; c < 16; ++c) {
        const int i = i0 + 2 * c;
        if (i >= N) break;
        const uint4 r = philox4x32_10((uint32_t)(i >> 1), tlo, thi, TAG_BOND, key);
#pragma unroll
        for (int j = 0; j < 2; ++j) {
            const int ii = i + j;
            if (ii < N) {
                const int y = ii / L, x = ii - y * L;
                const int ie = y * L + (x + 1 == L ? 0 : x + 1);
                const int is = (y + 1 == L ? 0 : y + 1) * L + x;
                const int8_t v = s[ii];
                const uint32_t we = j ? r.z : r.x, ws = j ? r.w : r.y;
                if (v == s[ie] && we < la.thr) e  |= 1u << (2 * c + j);
                if (v == s[is] && ws < la.thr) so |= 1u << (2 * c + j);
            }
        }
    }
    bondE[(size_t)blockIdx.y * words + w] = e;
    bondS[(size_t)blockIdx.y * words + w] = so;
}

// ---- a2-a4 labelling, generic: label[i] = i; one thread per site unites along its two bonds ----
__global__ void __launch_bounds__(GEN_THREADS)
k_label_init(int* __restrict__ label, int N) {
    const int i = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (i < N) label[(size_t)blockIdx.y * N + i] = i;
}

__global__ void __launch_bounds__(GEN_THREADS)
k_union_generic(int* label, const uint32_t* __restrict__ bondE, const uint32_t* __restrict__ bondS,
                int L, int N, int words) {
    const int i = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (i >= N) return;
    int* lab = label + (size_t)blockIdx.y * N;
    const uint32_t e  = bondE[(size_t)blockIdx.y * words + (i >> 5)] >> (i & 31);
    const uint32_t so = bondS[(size_t)blockIdx.y * words + (i >> 5)] >> (i & 31);
    if (!((e | so) & 1u)) return;
    const int y = i / L, x = i - y * L;
    if (e & 1u)  uf_union(lab, i, y * L + (x + 1 == L ? 0 : x + 1));
    if (so & 1u) uf_union(lab, i, (y + 1 == L ? 0 : y + 1) * L + x);
}

// label[i] = find(i); counts roots; accumulates cluster sizes into gsize[root] (generic path only)
__global__ void __launch_bounds__(GEN_THREADS)
k_compress_generic(int* label, int* __restrict__ gsize, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
                   int N, int nb) {
    const int i = blockIdx.x * GEN_THREADS + threadIdx.x;
    int isroot = 0;
    const unsigned act = __ballot_sync(0xffffffffu, i < N);
    if (i < N) {
        int* lab = label + (size_t)blockIdx.y * N;
        const int r = uf_find(lab, i);
        lab[i] = r;
        isroot = (r == i);
        const unsigned grp = __match_any_sync(act, r);          // lanes of one cluster add their count once
        if ((threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(gsize + (size_t)blockIdx.y * N + r, __popc(grp));
    }
    isroot = warp_sum_i(isroot);
    if ((threadIdx.x & 31) == 0 && isroot)
        atomic_add_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].ncl, isroot);
}

// largest cluster from gsize (zeroed by a memset before the sizes are counted).  A CTA covers MAXSIZE_SPAN sites (several
// independent loads per thread) and sends one maximum.
constexpr int MAXSIZE_SPAN = 16 * GEN_THREADS;
__global__ void __launch_bounds__(GEN_THREADS)
k_maxsize_generic(const int* __restrict__ label, const int* __restrict__ gsize, Rec* __restrict__ rec,
                  const Ctl* __restrict__ ctl, int N, int nb) {
    const int first = blockIdx.x * MAXSIZE_SPAN + threadIdx.x;
    const int* lab = label + (size_t)blockIdx.y * N;
    const int* gs = gsize + (size_t)blockIdx.y * N;
    int m = 0;
#pragma unroll
    for (int k = 0; k < MAXSIZE_SPAN / GEN_THREADS; ++k) {
        const int i = first + k * GEN_THREADS;
        if (i < N && lab[i] == i) m = max(m, gs[i]);
    }
    __shared__ int s_m;
    if (threadIdx.x == 0) s_m = 0;
    __syncthreads();
    m = warp_max_i(m);
    if ((threadIdx.x & 31) == 0 && m) atomicMax(&s_m, m);
    __syncthreads();
    if (threadIdx.x == 0 && s_m) atomic_max_ll(&rec[(size_t)ctl->slot * nb + blockIdx.y].maxcl, s_m);
}

// ---- a5 flip-bit plane: D word w = Philox(ctr = (w>>2, t, TAG_FLIP))[w&3];
//      one thread per call = 4 words = 128 candidate root decisions ------------------------------
__global__ void __launch_bounds__(GEN_THREADS)
k_flipbits(uint32_t* __restrict__ D, const Lat* __restrict__ lat, const Ctl* __restrict__ ctl, int words) {
    pdl_wait();
    const int c = blockIdx.x * GEN_THREADS + threadIdx.x;      // call index
    if (c * 4 >= words) return;
    const Lat la = lat[blockIdx.y];
    const PhiloxKey key(la.key0, la.key1);
    const unsigned long long t = ctl->t;
    const uint4 r = philox4x32_10((uint32_t)c, (uint32_t)t, (uint32_t)(t >> 32), TAG_FLIP, key);
    uint32_t* d = D + (size_t)blockIdx.y * words + (size_t)c * 4;
    if (c * 4 + 3 < words && (words & 3) == 0) {
        *reinterpret_cast<uint4*>(d) = r;
    } else {
        const uint32_t v[4] = { r.x, r.y, r.z, r.w };
        for (int k = 0; k < 4 && c * 4 + k < words; ++k) d[k] = v[k];
    }
}

// ---- a6 assignment: spins[i] = D bit at label[i] ? +1 : -1 (labels flat) -----------
__global__ void __launch_bounds__(GEN_THREADS)
k_flip_generic(int8_t* __restrict__ spins, const int* __restrict__ label, const uint32_t* __restrict__ D,
               int N, int words) {
    const int i = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (i >= N) return;
    const int r = label[(size_t)blockIdx.y * N + i];
    const uint32_t d = D[(size_t)blockIdx.y * words + (r >> 5)];
    spins[(size_t)blockIdx.y * N + i] = ((d >> (r & 31)) & 1u) ? (int8_t)1 : (int8_t)-1;
}

// ---- a7 observables: E = -sum_i s_i (s_E + s_S), M = sum_i s_i ----------------------
// rec_base points at the nb records to accumulate into (a series slot, or the "now" scratch record)
__global__ void __launch_bounds__(GEN_THREADS)
k_observe_generic(const int8_t* __restrict__ spins, Rec* __restrict__ rec, const Ctl* __restrict__ ctl,
                  int use_slot, int L, int N, int nb) {
    const int i = blockIdx.x * GEN_THREADS + threadIdx.x;
    int e = 0, m = 0;
    if (i < N) {
        const int8_t* s = spins + (size_t)blockIdx.y * N;
        const int y = i / L, x = i - y * L;
        const int v = s[i];
        e = -v * ((int)s[y * L + (x + 1 == L ? 0 : x + 1)] + (int)s[(y + 1 == L ? 0 : y + 1) * L + x]);
        m = v;
    }
    e = warp_sum_i(e); m = warp_sum_i(m);
    __shared__ int se[GEN_THREADS / 32], sm[GEN_THREADS / 32];
    if ((threadIdx.x & 31) == 0) { se[threadIdx.x >> 5] = e; sm[threadIdx.x >> 5] = m; }
    __syncthreads();
    if (threadIdx.x == 0) {
        int te = 0, tm = 0;
        for (int k = 0; k < GEN_THREADS / 32; ++k) { te += se[k]; tm += sm[k]; }
        Rec* r = rec + (use_slot ? (size_t)ctl->slot * nb : 0) + blockIdx.y;
        if (te) atomic_add_ll(&r->E, te);
        if (tm) atomic_add_ll(&r->M, tm);
    }
}

// ---- bit-packed host interface (north_star: "int8 or bit-packed spins"): word w holds sites 32w .. 32w+31 of a
//      lattice, bit = 1 for spin +1; 8x fewer bytes over PCIe than the int8 plane -------------------------------
__global__ void __launch_bounds__(GEN_THREADS)
k_unpack_spins(int8_t* __restrict__ spins, const uint32_t* __restrict__ bits, int N, int words) {
    const int w = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (w >= words) return;
    const uint32_t b = bits[(size_t)blockIdx.y * words + w];
    int8_t* s = spins + (size_t)blockIdx.y * N + (size_t)w * 32;
    if ((N & 31) == 0) {                              // whole words, 16-byte aligned rows of 32 sites
        reinterpret_cast<uint4*>(s)[0] = make_uint4(spin_bytes4(b & 15u), spin_bytes4((b >> 4) & 15u),
                                                    spin_bytes4((b >> 8) & 15u), spin_bytes4((b >> 12) & 15u));
        reinterpret_cast<uint4*>(s)[1] = make_uint4(spin_bytes4((b >> 16) & 15u), spin_bytes4((b >> 20) & 15u),
                                                    spin_bytes4((b >> 24) & 15u), spin_bytes4(b >> 28));
    } else {
        const int n = min(32, N - w * 32);
        for (int k = 0; k < n; ++k) s[k] = ((b >> k) & 1u) ? (int8_t)1 : (int8_t)-1;
    }
}
__global__ void __launch_bounds__(GEN_THREADS)
k_pack_spins(const int8_t* __restrict__ spins, uint32_t* __restrict__ bits, int N, int words) {
    const int w = blockIdx.x * GEN_THREADS + threadIdx.x;
    if (w >= words) return;
    const int8_t* s = spins + (size_t)blockIdx.y * N + (size_t)w * 32;
    uint32_t b = 0;
    if ((N & 31) == 0) {
        b = ~neg_mask32(reinterpret_cast<const uint4*>(s)[0], reinterpret_cast<const uint4*>(s)[1]);
    } else {
        const int n = min(32, N - w * 32);
        for (int k = 0; k < n; ++k) b |= (s[k] > 0 ? 1u : 0u) << k;
    }
    bits[(size_t)blockIdx.y * words + w] = b;
}

// ---- the ALU ceiling of the bond stage: the Philox4x32-10 draws of a sweep and nothing else.
//      One thread per 32-site word = 16 calls, as in the bond kernels; the words are XOR-reduced and stored once per
//      warp (so the calls cannot be removed), no other memory traffic ------------------------------------------------
__global__ void __launch_bounds__(GEN_THREADS)
k_philox_only(uint32_t* __restrict__ sink, uint32_t key0, uint32_t key1, uint32_t tlo, long long words) {
    const long long w = (long long)blockIdx.x * GEN_THREADS + threadIdx.x;
    uint32_t acc = 0;
    if (w < words) {
        const PhiloxKey key(key0, key1);
#pragma unroll
        for (int c = 0; c < 16; ++c) {
            const uint4 r = philox4x32_10((uint32_t)w * 16u + c, tlo, 0u, TAG_BOND, key);
            acc ^= r.x ^ r.y ^ r.z ^ r.w;
        }
    }
    acc = __reduce_xor_sync(0xffffffffu, acc);
    if ((threadIdx.x & 31) == 0) sink[w >> 5] = acc;
}

// ---- sweep control -------------------------------------------------------------------------------
__global__ void k_set_ctl(Ctl* ctl, unsigned long long t, uint32_t slot, uint32_t cap) {
    pdl_wait();
    ctl->t = t; ctl->slot = slot; ctl->cap = cap; ctl->done = 0; ctl->pad = 0;
}
// end of a sweep: t += 1, move to the next series slot and zero it.  acc: which record feeds the running
// moments -- 1: this sweep's (its E, M are complete), 2: the previous sweep's (scan path: E, M of a sweep
// arrive with the next sweep's bond test), 0: none.  One thread per lattice: sweep order, fixed arithmetic.
__device__ __forceinline__ void advance_sweep(Ctl* ctl, Rec* rec, int nb, Mom* mom, int N, int acc) {   // (a whole block)
    const uint32_t cur = ctl->slot;
    const uint32_t next = (cur + 1 == ctl->cap) ? 0u : cur + 1;
    const uint32_t from = acc == 2 ? (cur == 0 ? ctl->cap - 1 : cur - 1) : cur;
    for (int b = threadIdx.x; b < nb; b += blockDim.x) {
        if (acc) {
            const Rec r = rec[(size_t)from * nb + b];
            Mom m = mom[b];
            mom_add(m, r.E, r.M, N);
            mom[b] = m;
        }
        rec[(size_t)next * nb + b] = Rec{0, 0, 0, 0};
    }
    __syncthreads();
    if (threadIdx.x == 0) { ctl->t += 1; ctl->slot = next; }
}
__global__ void k_advance(Ctl* ctl, Rec* rec, int nb, Mom* mom, int N, int acc) { advance_sweep(ctl, rec, nb, mom, N, acc); }
// scan path, end of a sw_sweep call (after k_observe_rows): the last sweep's record, now complete
__global__ void k_moments_last(const Ctl* ctl, const Rec* rec, int nb, Mom* mom, int N) {
    pdl_wait();
    pdl_wait();
    const uint32_t from = ctl->slot == 0 ? ctl->cap - 1 : ctl->slot - 1;
    for (int b = threadIdx.x; b < nb; b += blockDim.x) {
        const Rec r = rec[(size_t)from * nb + b];
        Mom m = mom[b];
        mom_add(m, r.E, r.M, N);
        mom[b] = m;
    }
}

// ---- test hook: Philox on the device ---------------------------------------------------------------
__global__ void k_test_philox(const uint32_t* __restrict__ ctr, const uint32_t* __restrict__ key,
                              uint32_t* __restrict__ out, long long n) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const PhiloxKey k(key[2 * i], key[2 * i + 1]);
    const uint4 r = philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], k);
    out[4 * i] = r.x; out[4 * i + 1] = r.y; out[4 * i + 2] = r.z; out[4 * i + 3] = r.w;
}

} // namespace sw
