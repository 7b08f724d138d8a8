// sw_common.cuh -- device-side types and helpers shared by the kernels of libsw_b200.so.
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace sw {

// Philox stream tags: counter = (block, t_lo, t_hi, TAG)
constexpr uint32_t TAG_INIT = 0u, TAG_BOND = 1u, TAG_FLIP = 2u;

// per-lattice parameters (device array of nb entries)
struct Lat {
    uint32_t key0, key1;   // Philox key = (seed & 0xffffffff, seed >> 32)
    uint32_t thr;          // floor((1 - exp(-2/T)) * 2^32), clamped to 2^32 - 1
    uint32_t pad;
};

// device-resident sweep control: lets one captured launch sequence serve every sweep
struct Ctl {
    unsigned long long t;  // sweep index the next sweep uses
    uint32_t slot;         // series slot the running sweep accumulates into
    uint32_t cap;          // number of series slots (ring)
    uint32_t done;         // CTAs of the sweep's last kernel that have finished (k_flip16<FUSED>: the last one advances the sweep)
    uint32_t pad;
};

// one per (series slot, lattice); accumulated with atomics during the sweep
struct Rec {
    long long E, M, ncl, maxcl;
};

// running sums of the per-sweep observables of one lattice (sw_moments):
// e = E / N, a = |M| / N per configuration, summed one sweep at a time in double, in sweep
// order, with no fused operations -- the same arithmetic in the same order as the oracle's definition.
struct Mom {
    double s_e, s_e2, s_am, s_m2, s_m4;
    long long n;
};
__device__ __forceinline__ void mom_add(Mom& m, long long E, long long M, int N) {
    const double fN = (double)N;
    const double e = __ddiv_rn((double)E, fN);
    const double a = fabs(__ddiv_rn((double)M, fN));
    const double a2 = __dmul_rn(a, a);
    m.s_e = __dadd_rn(m.s_e, e);
    m.s_e2 = __dadd_rn(m.s_e2, __dmul_rn(e, e));
    m.s_am = __dadd_rn(m.s_am, a);
    m.s_m2 = __dadd_rn(m.s_m2, a2);
    m.s_m4 = __dadd_rn(m.s_m4, __dmul_rn(a2, a2));
    m.n += 1;
}

// programmatic dependent launch: the kernels of a sweep are launched with the "programmatic stream serialization" attribute, so
// that the next kernel's launch overlaps the tail of the running one; a kernel waits HERE -- before it reads anything an
// earlier kernel of the stream wrote -- until that kernel has completed and its writes are visible (a no-op in a kernel that was
// launched the ordinary way)
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// bit-plane layout shared by the bond planes and the decision plane D: bit (i & 31) of word (i >> 5)
__device__ __forceinline__ uint32_t get_bit(const uint32_t* __restrict__ plane, int i) {
    return (plane[i >> 5] >> (i & 31)) & 1u;
}

// ------------------------------------------------------------------------------------------
// Philox4x32-10.  mul.wide.u32 -> one IMAD.WIDE per multiply; the xor of three terms -> one LOP3.
// ------------------------------------------------------------------------------------------
constexpr uint32_t PHILOX_M0 = 0xD2511F53u, PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u, PHILOX_W1 = 0xBB67AE85u;

struct PhiloxKey {          // the ten round keys, expanded once per thread
    uint32_t k0[10], k1[10];
    __device__ __forceinline__ PhiloxKey(uint32_t key0, uint32_t key1) {
#pragma unroll
        for (int r = 0; r < 10; ++r) { k0[r] = key0 + (uint32_t)r * PHILOX_W0; k1[r] = key1 + (uint32_t)r * PHILOX_W1; }
    }
};

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const PhiloxKey& k) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)PHILOX_M0 * c0;
        const unsigned long long p1 = (unsigned long long)PHILOX_M1 * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k.k1[r];
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

// the 32 East and 32 South draw bits of bit-plane word w (sites 32w .. 32w+31): call c covers sites
// 2c, 2c+1; words x,y = East,South of the even site, z,w of the odd one.
__device__ __forceinline__ void bond_draws(uint32_t w, uint32_t tlo, uint32_t thi, uint32_t thr,
                                           const PhiloxKey& key, uint32_t& dE, uint32_t& dS) {
    dE = 0; dS = 0;
#pragma unroll
    for (int c = 0; c < 16; ++c) {
        const uint4 r = philox4x32_10(w * 16u + c, tlo, thi, TAG_BOND, key);
        dE |= (r.x < thr ? 1u : 0u) << (2 * c) | (r.z < thr ? 1u : 0u) << (2 * c + 1);
        dS |= (r.y < thr ? 1u : 0u) << (2 * c) | (r.w < thr ? 1u : 0u) << (2 * c + 1);
    }
}

// position of the highest set bit, 0xffffffff for 0 (one FLO)
__device__ __forceinline__ int bfind_u32(uint32_t x) {
    int r; asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x)); return r;
}

// shared-memory add with no return value, predicated (no branch around it)
// (addr: address in the shared window, from __cvta_generic_to_shared)
__device__ __forceinline__ void red_shared_add_if(uint32_t addr, uint32_t v, bool c) {
    asm volatile("{ .reg .pred q; setp.ne.u32 q, %2, 0; @q red.shared.add.u32 [%0], %1; }"
                 :: "r"(addr), "r"(v), "r"((uint32_t)c) : "memory");
}

// ------------------------------------------------------------------------------------------
// memory helpers
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int ld_cg(const int* p) {            // L2-coherent load (labels under atomics)
    int v; asm volatile("ld.global.cg.s32 %0, [%1];" : "=r"(v) : "l"(p)); return v;
}
__device__ __forceinline__ unsigned long long ld_cg64(const unsigned long long* p) {
    unsigned long long v; asm volatile("ld.global.cg.u64 %0, [%1];" : "=l"(v) : "l"(p)); return v;
}
__device__ __forceinline__ uint4 ld_stream_u4(const void* p) {   // read-once data: do not pollute L1
    uint4 v; asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
                          : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p)); return v;
}
__device__ __forceinline__ void st_stream_u4(void* p, uint4 v) {
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1,%2,%3,%4};"
                 :: "l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// sign bits of four int8 spins (+1 = 0x01, -1 = 0xFF) gathered into a nibble: bit k = (spin k == -1)
__device__ __forceinline__ uint32_t neg_nibble(uint32_t q) {
    return (((q >> 7) & 0x01010101u) * 0x01020408u) >> 24;
}
// 32 spins held as two uint4 -> 32-bit mask, bit k = (spin k == -1)
__device__ __forceinline__ uint32_t neg_mask32(uint4 a, uint4 b) {
    return  neg_nibble(a.x)        | (neg_nibble(a.y) << 4)  | (neg_nibble(a.z) << 8)  | (neg_nibble(a.w) << 12)
         | (neg_nibble(b.x) << 16) | (neg_nibble(b.y) << 20) | (neg_nibble(b.z) << 24) | (neg_nibble(b.w) << 28);
}
// four spin bits (bit = 1: +1) -> four int8 bytes (+1 = 0x01, -1 = 0xFF)
__device__ __forceinline__ uint32_t spin_bytes4(uint32_t nib) {
    const uint32_t up = (nib * 0x00204081u) & 0x01010101u;       // bit k -> byte k (0x01 where up)
    return up | ((up ^ 0x01010101u) * 0xFFu);                    // 0xFF where down
}

// block-wide sums / max into one atomic per block
__device__ __forceinline__ long long warp_sum_ll(long long v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ int warp_sum_i(int v) { return __reduce_add_sync(0xffffffffu, v); }
__device__ __forceinline__ int warp_max_i(int v) { return __reduce_max_sync(0xffffffffu, v); }
__device__ __forceinline__ void atomic_add_ll(long long* p, long long v) {
    atomicAdd(reinterpret_cast<unsigned long long*>(p), (unsigned long long)v);
}
__device__ __forceinline__ void atomic_max_ll(long long* p, long long v) {   // values are >= 0
    atomicMax(reinterpret_cast<unsigned long long*>(p), (unsigned long long)v);
}

// ------------------------------------------------------------------------------------------
// lock-free union-find on a global int32 parent array (generic path); label[x] <= x, roots have
// label[r] == r.  Hooking is "larger root under smaller" with atomicMin, so the surviving root of a
// component is its minimum site index whatever the race order (north_star stage 2).
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ int uf_find(const int* lab, int x) {
    int p = ld_cg(lab + x);
    while (p != x) { x = p; p = ld_cg(lab + x); }
    return x;
}
// the same walk through L1 (ld.global.ca).  A stale line can only show an older parent, which is still an
// ancestor, so the walk ends at a node that was a root when its line was fetched; callers either run when no
// root changes any more (k_roots_nodes) or let an atomic on the result arbitrate (uf_union_l1).  At T_c one
// cluster owns ~1/3 of all sites: its root's line would otherwise be fetched from one L2 slice by every walker.
__device__ __forceinline__ int ld_ca(const int* p) {
    int v; asm volatile("ld.global.ca.s32 %0, [%1];" : "=r"(v) : "l"(p)); return v;
}
__device__ __forceinline__ int uf_find_l1(const int* lab, int x) {
    int p = ld_ca(lab + x);
    while (p != x) { x = p; p = ld_ca(lab + x); }
    return x;
}
__device__ __forceinline__ void uf_union_l1(int* lab, int a, int b) {
    a = uf_find_l1(lab, a); b = uf_find_l1(lab, b);
    while (a != b) {
        if (a < b) { int s = a; a = b; b = s; }           // a is the larger
        const int old = atomicMin(lab + a, b);            // L2 decides whether a still is a root
        if (old == a) break;
        a = old;
    }
}
// find with one-shot compression of the starting node when the walk was longer than one hop
// (only ever writes a smaller ancestor: safe under races)
__device__ __forceinline__ int uf_find_compress(int* lab, int x) {
    const int x0 = x;
    int p = ld_cg(lab + x);
    if (p == x) return x;
    int q = ld_cg(lab + p);
    if (q == p) return p;
    x = q; p = ld_cg(lab + x);
    while (p != x) { x = p; p = ld_cg(lab + x); }
    atomicMin(lab + x0, x);
    return x;
}
__device__ __forceinline__ void uf_union(int* lab, int a, int b) {
    a = uf_find_compress(lab, a); b = uf_find_compress(lab, b);
    while (a != b) {
        if (a < b) { int s = a; a = b; b = s; }           // a is the larger
        const int old = atomicMin(lab + a, b);
        if (old == a) break;                               // a was a root and now hangs under b
        a = old;                                           // a already had a parent: unite that with b
    }
}

} // namespace sw
