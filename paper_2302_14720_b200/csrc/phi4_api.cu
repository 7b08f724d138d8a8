// phi4_api.cu -- the Wolff-type embedded cluster update for the O(4) phi^4 theory in four dimensions (include/phi4.h;
// PAPER.md:93-109, section 3, Eq. 2-3): kernels and the extern "C" boundary.
// Product code (CUDA path).  No CPU fallback.  Shares the device Philox and the lock-free union-find with the Ising path
// (sw_common.cuh); nothing with oracle/.
//
// One update = 4 launches on one stream, no host synchronisation (the sweep index lives on the device, so the sequence is
// replayed from a CUDA graph):
//   (k4_direction  first update of a call only: the update's direction r, rejection from the cube to the ball, IEEE-exact
//                  operations; afterwards the block that closes an update draws the next one's)
//   k4_bonds       thread per site: projections, Eq. 2 thresholds, 4 Philox words -> bond byte; label[x] = x
//   k4_union       thread per site: lock-free union-find over its bonds (atomicMin hooking: the root is the minimum index)
//   k4_reflect     thread per site: root (stored: flat labels), cluster sizes, selection bit of the root, Eq. 3
//   k4_observe     link and magnetisation sums of the new field (fixed tree inside a block, partials per block); the block that
//                  finishes last sums the partials in block order, writes the record, advances t and draws the next direction
// The lattices of the paper (L = 16 .. 28: 2 .. 20 MB of field) live in L2; the update is bound by launch latency and the
// dependent walks of the union-find, not by HBM.
#include "../../include/phi4.h"
#include "sw_common.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace sw;

namespace {

thread_local std::string g_err4 = "";
void set_err4(const char* fmt, ...) __attribute__((format(printf, 1, 2)));
void set_err4(const char* fmt, ...) {
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
    g_err4 = buf;
}
#define P4_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            set_err4("CUDA error %s at %s:%d: %s", cudaGetErrorName(e_), __FILE__, __LINE__,       \
                     cudaGetErrorString(e_));                                                      \
            return PHI4_ECUDA;                                                                     \
        }                                                                                          \
    } while (0)

constexpr uint32_t TAG_INIT4 = 16u, TAG_DIR = 17u, TAG_BOND4 = 18u, TAG_SEL = 19u;
constexpr int P4_THREADS = 256;
constexpr int64_t P4_SERIES_CAP = 4096;

struct Ctl4 { unsigned long long t; uint32_t slot, cap; };
struct Rec4 { double link, m[4]; long long ncl, maxcl, nbonds; };
struct Geo { int L, L2, L3, V; };

// uniform in (0, 1) from a 32-bit word; v = 2 u - 1 (separately rounded: the oracle's order)
__device__ __forceinline__ double unif(uint32_t w) { return __dmul_rn(__dadd_rn((double)w, 0.5), 1.0 / 4294967296.0); }
__device__ __forceinline__ double sym(uint32_t w) { return __dsub_rn(__dmul_rn(2.0, unif(w)), 1.0); }

__device__ __forceinline__ uint4 draw4(uint32_t index, unsigned long long t, uint32_t tag, uint32_t key0, uint32_t key1) {
    const PhiloxKey k(key0, key1);
    return philox4x32_10(index, (uint32_t)t, (uint32_t)(t >> 32), tag, k);
}
// phi_x . r = ((p0 r0 + p1 r1) + p2 r2) + p3 r3, every operation rounded on its own
__device__ __forceinline__ double proj(const double2 a, const double2 b, const double* r) {
    return __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(a.x, r[0]), __dmul_rn(a.y, r[1])), __dmul_rn(b.x, r[2])), __dmul_rn(b.y, r[3]));
}
__device__ __forceinline__ int fwd(const Geo g, int x, int mu) {
    const int stride = mu == 0 ? 1 : mu == 1 ? g.L : mu == 2 ? g.L2 : g.L3;
    const int c = (x / stride) % g.L;
    return c + 1 == g.L ? x - (g.L - 1) * stride : x + stride;
}

__global__ void k4_init(double* __restrict__ phi, int V, uint32_t key0, uint32_t key1) {
    const int x = blockIdx.x * P4_THREADS + threadIdx.x;
    if (x >= V) return;
    const uint4 w = draw4((uint32_t)x, 0ull, TAG_INIT4, key0, key1);
    reinterpret_cast<double2*>(phi)[2 * x] = make_double2(sym(w.x), sym(w.y));
    reinterpret_cast<double2*>(phi)[2 * x + 1] = make_double2(sym(w.z), sym(w.w));
}

__global__ void k4_set_ctl(Ctl4* ctl, unsigned long long t, uint32_t slot, uint32_t cap) { ctl->t = t; ctl->slot = slot; ctl->cap = cap; }

// step 1: the direction of the update with sweep index t, r . r = 1 (one thread)
__device__ __forceinline__ void draw_direction(double* __restrict__ r, unsigned long long t, uint32_t key0, uint32_t key1) {
    for (uint32_t j = 0; ; ++j) {
        const uint4 w = draw4(j, t, TAG_DIR, key0, key1);
        const double v0 = sym(w.x), v1 = sym(w.y), v2 = sym(w.z), v3 = sym(w.w);
        const double n2 = __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(v0, v0), __dmul_rn(v1, v1)), __dmul_rn(v2, v2)), __dmul_rn(v3, v3));
        if (n2 <= 1.0 && n2 >= 1e-4) {
            const double n = __dsqrt_rn(n2);
            r[0] = __ddiv_rn(v0, n); r[1] = __ddiv_rn(v1, n); r[2] = __ddiv_rn(v2, n); r[3] = __ddiv_rn(v3, n);
            return;
        }
    }
}
// first update of a phi4_sweep call: its direction, and the integer accumulators of its record cleared (the following
// updates get both from the end of the update before them: k4_observe)
__global__ void k4_direction(double* __restrict__ r, const Ctl4* __restrict__ ctl, long long* __restrict__ iacc,
                             uint32_t key0, uint32_t key1) {
    if (threadIdx.x != 0) return;
    iacc[0] = 0; iacc[1] = 0; iacc[2] = 0; iacc[3] = 0;
    draw_direction(r, ctl->t, key0, key1);
}

// Eq. 2 as an integer threshold on a 32-bit word
__device__ __forceinline__ uint32_t threshold4(double m4kappa, double sx, double sy) {
    const double arg = __dmul_rn(m4kappa, __dmul_rn(sx, sy));
    if (!(arg < 0.0)) return 0u;
    const double v = floor(__dmul_rn(-expm1(arg), 4294967296.0));
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

// step 2: bonds of site x to its four forward neighbours; label[x] = x for the union-find
__global__ void __launch_bounds__(P4_THREADS)
k4_bonds(const double* __restrict__ phi, const double* __restrict__ r, uint8_t* __restrict__ bonds, int* __restrict__ label,
         int* __restrict__ gsize, const Ctl4* __restrict__ ctl, long long* __restrict__ iacc, Geo g, double m4kappa,
         uint32_t key0, uint32_t key1) {
    const int x = blockIdx.x * P4_THREADS + threadIdx.x;
    int nb = 0;
    if (x < g.V) {
        const double rr[4] = { r[0], r[1], r[2], r[3] };
        const double2* p = reinterpret_cast<const double2*>(phi);
        const double sx = proj(p[2 * x], p[2 * x + 1], rr);
        const uint4 w = draw4((uint32_t)x, ctl->t, TAG_BOND4, key0, key1);
        const uint32_t ww[4] = { w.x, w.y, w.z, w.w };
        uint32_t b = 0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const int y = fwd(g, x, mu);
            const double sy = proj(p[2 * y], p[2 * y + 1], rr);
            if (ww[mu] < threshold4(m4kappa, sx, sy)) b |= 1u << mu;
        }
        bonds[x] = (uint8_t)b;
        label[x] = x;
        gsize[x] = 0;
        nb = __popc(b);
    }
    nb = warp_sum_i(nb);
    if ((threadIdx.x & 31) == 0 && nb) atomic_add_ll(&iacc[2], nb);
}

// step 3a: clusters -- lock-free union-find on the 4D index space, "larger root under smaller" with atomicMin
__global__ void __launch_bounds__(P4_THREADS)
k4_union(int* label, const uint8_t* __restrict__ bonds, Geo g) {
    const int x = blockIdx.x * P4_THREADS + threadIdx.x;
    if (x >= g.V) return;
    const uint32_t b = bonds[x];
#pragma unroll
    for (int mu = 0; mu < 4; ++mu)
        if ((b >> mu) & 1u) uf_union(label, x, fwd(g, x, mu));
}

// step 3b: flat labels, cluster sizes, selection with probability 1/2, reflection Eq. 3
__global__ void __launch_bounds__(P4_THREADS)
k4_reflect(double* __restrict__ phi, const double* __restrict__ r, int* label, int* __restrict__ gsize,
           const Ctl4* __restrict__ ctl, long long* __restrict__ iacc, Geo g, uint32_t key0, uint32_t key1) {
    const int x = blockIdx.x * P4_THREADS + threadIdx.x;
    int isroot = 0;
    int root = -1 - (int)(threadIdx.x & 31);                // (lanes past the end: distinct keys)
    if (x < g.V) root = uf_find(label, x);
    {   // sizes: one add per root and warp -- at kappa = 0.304 one cluster holds most of the lattice, and a site-by-site add
        // would send every one of its sites to the same address
        const unsigned grp = __match_any_sync(0xffffffffu, root);
        if (x < g.V && (int)(threadIdx.x & 31) == __ffs(grp) - 1) atomicAdd(gsize + root, __popc(grp));
    }
    if (x < g.V) {
        if (root != x) label[x] = root;                     // (only ever an ancestor: safe while others walk)
        isroot = root == x;
        const uint4 w = draw4((uint32_t)root >> 7, ctl->t, TAG_SEL, key0, key1);
        const uint32_t ww[4] = { w.x, w.y, w.z, w.w };
        if ((ww[(root >> 5) & 3] >> (root & 31)) & 1u) {
            const double rr[4] = { r[0], r[1], r[2], r[3] };
            double2* p = reinterpret_cast<double2*>(phi);
            const double2 a = p[2 * x], b = p[2 * x + 1];
            const double two_s = __dmul_rn(2.0, proj(a, b, rr));
            p[2 * x] = make_double2(__dsub_rn(a.x, __dmul_rn(two_s, rr[0])), __dsub_rn(a.y, __dmul_rn(two_s, rr[1])));
            p[2 * x + 1] = make_double2(__dsub_rn(b.x, __dmul_rn(two_s, rr[2])), __dsub_rn(b.y, __dmul_rn(two_s, rr[3])));
        }
    }
    isroot = warp_sum_i(isroot);
    if ((threadIdx.x & 31) == 0 && isroot) atomic_add_ll(&iacc[0], isroot);
}

// the block's partial sums in block order (fixed strided tree: the result does not depend on which block runs this), the
// record of the update, t += 1; with `advance` also the NEXT update's direction and cleared accumulators (r_last keeps the
// direction this update used, for phi4_direction)
__device__ void finish_update(const double* __restrict__ partial, int nblocks, Rec4* __restrict__ rec, Ctl4* ctl,
                              long long* __restrict__ iacc, double* __restrict__ r, double* __restrict__ r_last,
                              uint32_t key0, uint32_t key1, int advance, double (*sh)[P4_THREADS]) {
    double v[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
    for (int b = threadIdx.x; b < nblocks; b += P4_THREADS)
#pragma unroll
        for (int k = 0; k < 5; ++k) v[k] = __dadd_rn(v[k], __ldcg(partial + (size_t)b * 5 + k));
#pragma unroll
    for (int k = 0; k < 5; ++k) sh[k][threadIdx.x] = v[k];
    __syncthreads();
    for (int s = P4_THREADS / 2; s > 0; s >>= 1) {
        if (threadIdx.x < s)
#pragma unroll
            for (int k = 0; k < 5; ++k) sh[k][threadIdx.x] = __dadd_rn(sh[k][threadIdx.x], sh[k][threadIdx.x + s]);
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        Rec4 rc;
        rc.link = sh[0][0]; rc.m[0] = sh[1][0]; rc.m[1] = sh[2][0]; rc.m[2] = sh[3][0]; rc.m[3] = sh[4][0];
        rc.ncl = advance ? iacc[0] : 0; rc.maxcl = advance ? iacc[1] : 0; rc.nbonds = advance ? iacc[2] : 0;
        rec[advance ? ctl->slot : ctl->cap] = rc;                // (slot `cap` = the scratch record of phi4_observables)
        if (advance) {
            ctl->t += 1; ctl->slot = ctl->slot + 1 == ctl->cap ? 0u : ctl->slot + 1;
            r_last[0] = r[0]; r_last[1] = r[1]; r_last[2] = r[2]; r_last[3] = r[3];
            iacc[0] = 0; iacc[1] = 0; iacc[2] = 0;
            draw_direction(r, ctl->t, key0, key1);
        }
    }
}

// observables of the new field: per block a fixed tree over its sites -> partial[block][5]; largest cluster; the block
// that finishes last closes the update (finish_update)
__global__ void __launch_bounds__(P4_THREADS)
k4_observe(const double* __restrict__ phi, const int* __restrict__ gsize, double* __restrict__ partial,
           long long* __restrict__ iacc, Geo g, int with_sizes, Rec4* __restrict__ rec, Ctl4* ctl,
           double* __restrict__ r, double* __restrict__ r_last, uint32_t key0, uint32_t key1, int advance) {
    const int x = blockIdx.x * P4_THREADS + threadIdx.x;
    double v[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
    int big = 0;
    if (x < g.V) {
        const double2* p = reinterpret_cast<const double2*>(phi);
        const double2 a = p[2 * x], b = p[2 * x + 1];
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) {
            const int y = fwd(g, x, mu);
            const double2 c = p[2 * y], d = p[2 * y + 1];
            v[0] = __dadd_rn(v[0], __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(a.x, c.x), __dmul_rn(a.y, c.y)), __dmul_rn(b.x, d.x)), __dmul_rn(b.y, d.y)));
        }
        v[1] = a.x; v[2] = a.y; v[3] = b.x; v[4] = b.y;
        if (with_sizes) big = gsize[x];
    }
    __shared__ double sh[5][P4_THREADS];
    __shared__ int s_last;
#pragma unroll
    for (int k = 0; k < 5; ++k) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] = __dadd_rn(v[k], __shfl_xor_sync(0xffffffffu, v[k], o));
        if ((threadIdx.x & 31) == 0) sh[k][threadIdx.x >> 5] = v[k];
    }
    big = warp_max_i(big);
    if ((threadIdx.x & 31) == 0 && big) atomic_max_ll(&iacc[1], big);
    __syncthreads();
    if (threadIdx.x < 5) {
        double tot = 0.0;
        for (int w = 0; w < P4_THREADS / 32; ++w) tot = __dadd_rn(tot, sh[threadIdx.x][w]);
        partial[(size_t)blockIdx.x * 5 + threadIdx.x] = tot;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        s_last = atomicAdd(reinterpret_cast<unsigned long long*>(&iacc[3]), 1ull) == (unsigned long long)gridDim.x - 1;
    }
    __syncthreads();
    if (s_last) {                                           // (every other block's partials and maximum are in)
        __threadfence();
        if (threadIdx.x == 0) iacc[3] = 0;
        finish_update(partial, (int)gridDim.x, rec, ctl, iacc, r, r_last, key0, key1, advance, sh);
    }
}

struct DevGuard4 {
    int prev = -1; bool switched = false;
    explicit DevGuard4(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess; }
    ~DevGuard4() { if (switched) cudaSetDevice(prev); }
    DevGuard4(const DevGuard4&) = delete; DevGuard4& operator=(const DevGuard4&) = delete;
};

} // namespace

struct phi4_handle {
    int L = 0, V = 0, dev = 0, nblocks = 0;
    double kappa = 0.0;
    uint32_t key0 = 0, key1 = 0;
    Geo g{};
    double* phi = nullptr; double* r = nullptr; double* partial = nullptr;      // r: [0..3] the running update's direction, [4..7] the last one's
    uint8_t* bonds = nullptr; int* label = nullptr; int* gsize = nullptr;
    long long* iacc = nullptr; Ctl4* ctl = nullptr; Rec4* rec = nullptr;      // rec: P4_SERIES_CAP ring + 1 scratch
    uint64_t t = 0;
    int64_t last_n = 0, launches = 0;
    bool have_sweep = false, rec_valid = false;
    cudaStream_t stream = nullptr;
    bool use_graphs = true, graph_failed = false;
    cudaStream_t gstream = nullptr; cudaEvent_t gev[2] = { nullptr, nullptr };
    cudaGraphExec_t gexec = nullptr;
};

namespace {

int launch_update(phi4_handle* h, bool first) {
    const unsigned nb = (unsigned)h->nblocks;
    if (first) { k4_direction<<<1, 32, 0, h->stream>>>(h->r, h->ctl, h->iacc, h->key0, h->key1); h->launches += 1; }
    k4_bonds<<<nb, P4_THREADS, 0, h->stream>>>(h->phi, h->r, h->bonds, h->label, h->gsize, h->ctl, h->iacc, h->g,
                                               -4.0 * h->kappa, h->key0, h->key1);
    k4_union<<<nb, P4_THREADS, 0, h->stream>>>(h->label, h->bonds, h->g);
    k4_reflect<<<nb, P4_THREADS, 0, h->stream>>>(h->phi, h->r, h->label, h->gsize, h->ctl, h->iacc, h->g, h->key0, h->key1);
    k4_observe<<<nb, P4_THREADS, 0, h->stream>>>(h->phi, h->gsize, h->partial, h->iacc, h->g, 1, h->rec, h->ctl, h->r, h->r + 4,
                                                 h->key0, h->key1, 1);
    P4_CUDA(cudaGetLastError());
    h->launches += 4;
    return PHI4_OK;
}

void fill_obs4(const phi4_handle* h, const Rec4& r, uint64_t sweep, phi4_obs* o) {
    o->link = r.link;
    for (int a = 0; a < 4; ++a) o->m[a] = r.m[a];
    o->n_clusters = r.ncl; o->largest_cluster = r.maxcl; o->n_bonds = r.nbonds; o->sweep = sweep;
    o->link_per_link = r.link / (4.0 * (double)h->V);
    o->abs_m_per_site = std::sqrt(((r.m[0] * r.m[0] + r.m[1] * r.m[1]) + r.m[2] * r.m[2]) + r.m[3] * r.m[3]) / (double)h->V;
}

} // namespace

extern "C" {

const char* phi4_last_error(void) { return g_err4.c_str(); }

phi4_handle* phi4_create(int32_t L, double kappa, uint64_t seed) {
    if (L < 2 || L > PHI4_MAX_L || !(kappa >= 0.0) || !std::isfinite(kappa)) {
        set_err4("phi4_create: invalid argument (L = %d must be 2 .. %d, kappa = %g finite and >= 0)", L, PHI4_MAX_L, kappa);
        return nullptr;
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        set_err4("phi4_create: no usable CUDA device (%s); this library has no CPU path", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return nullptr;
    }
    phi4_handle* h = new (std::nothrow) phi4_handle();
    if (!h) { set_err4("phi4_create: out of host memory"); return nullptr; }
    h->L = L; h->V = L * L * L * L; h->kappa = kappa;
    h->g = Geo{ L, L * L, L * L * L, h->V };
    h->key0 = (uint32_t)(seed & 0xFFFFFFFFu); h->key1 = (uint32_t)(seed >> 32);
    h->nblocks = (h->V + P4_THREADS - 1) / P4_THREADS;
    bool ok = cudaGetDevice(&h->dev) == cudaSuccess;
    const size_t V = (size_t)h->V;
    ok = ok && cudaMalloc((void**)&h->phi, V * 4 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->r, 8 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->partial, (size_t)h->nblocks * 5 * sizeof(double)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->bonds, V) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->label, V * sizeof(int)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->gsize, V * sizeof(int)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->iacc, 4 * sizeof(long long)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->ctl, sizeof(Ctl4)) == cudaSuccess;
    ok = ok && cudaMalloc((void**)&h->rec, (size_t)(P4_SERIES_CAP + 1) * sizeof(Rec4)) == cudaSuccess;
    if (ok) {
        k4_init<<<(unsigned)h->nblocks, P4_THREADS>>>(h->phi, h->V, h->key0, h->key1);
        k4_set_ctl<<<1, 1>>>(h->ctl, 0ull, 0u, (uint32_t)P4_SERIES_CAP);
        ok = cudaMemset(h->r, 0, 8 * sizeof(double)) == cudaSuccess && cudaMemset(h->iacc, 0, 4 * sizeof(long long)) == cudaSuccess &&
             cudaDeviceSynchronize() == cudaSuccess;
    }
    if (!ok) {
        set_err4("phi4_create: device allocation or initialisation failed: %s", cudaGetErrorString(cudaGetLastError()));
        phi4_destroy(h);
        return nullptr;
    }
    return h;
}

void phi4_destroy(phi4_handle* h) {
    if (!h) return;
    DevGuard4 dg(h->dev);
    cudaStreamSynchronize(h->stream);
    if (h->gexec) cudaGraphExecDestroy(h->gexec);
    for (cudaEvent_t e : h->gev) if (e) cudaEventDestroy(e);
    if (h->gstream) cudaStreamDestroy(h->gstream);
    cudaFree(h->phi); cudaFree(h->r); cudaFree(h->partial); cudaFree(h->bonds); cudaFree(h->label); cudaFree(h->gsize);
    cudaFree(h->iacc); cudaFree(h->ctl); cudaFree(h->rec);
    (void)cudaGetLastError();
    delete h;
}

int phi4_sweep(phi4_handle* h, int64_t n) {
    if (!h || n < 0) { set_err4("phi4_sweep: invalid argument"); return PHI4_EINVAL; }
    DevGuard4 dg(h->dev);
    if (n == 0) return PHI4_OK;
    h->launches = 0;
    cudaStream_t const user = h->stream;
    struct StreamBack {
        phi4_handle* h; cudaStream_t user;
        ~StreamBack() {
            if (h->stream == user) return;
            if (h->gev[1] && cudaEventRecord(h->gev[1], h->stream) == cudaSuccess) cudaStreamWaitEvent(user, h->gev[1], 0);
            h->stream = user;
        }
    } back{h, user};
    bool graphs = h->use_graphs && !h->graph_failed && n >= 4;
    if (graphs && !h->gstream) {
        if (cudaStreamCreateWithFlags(&h->gstream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->gev[0], cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->gev[1], cudaEventDisableTiming) != cudaSuccess) {
            (void)cudaGetLastError(); h->graph_failed = true; graphs = false;
        }
    }
    if (graphs) {
        P4_CUDA(cudaEventRecord(h->gev[0], user));
        P4_CUDA(cudaStreamWaitEvent(h->gstream, h->gev[0], 0));
        h->stream = h->gstream;
    }
    k4_set_ctl<<<1, 1, 0, h->stream>>>(h->ctl, (unsigned long long)h->t, 0u, (uint32_t)P4_SERIES_CAP);
    h->launches += 1;
    { int rc = launch_update(h, true); if (rc) return rc; }
    int64_t k = 1;
    if (graphs && !h->gexec) {
        cudaGraph_t graph = nullptr;
        const int64_t keep = h->launches;
        bool ok = cudaStreamBeginCapture(h->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        if (ok) {
            const int rc = launch_update(h, false);
            ok = cudaStreamEndCapture(h->stream, &graph) == cudaSuccess && rc == PHI4_OK && graph;
        }
        if (ok) ok = cudaGraphInstantiate(&h->gexec, graph, 0) == cudaSuccess;
        if (graph) cudaGraphDestroy(graph);
        h->launches = keep;
        if (!ok) { (void)cudaGetLastError(); h->gexec = nullptr; h->graph_failed = true; graphs = false; }
    }
    if (graphs)
        for (; k < n; ++k) { P4_CUDA(cudaGraphLaunch(h->gexec, h->stream)); h->launches += 4; }
    for (; k < n; ++k) { int rc = launch_update(h, false); if (rc) return rc; }
    P4_CUDA(cudaGetLastError());
    h->t += (uint64_t)n; h->last_n = n; h->have_sweep = true; h->rec_valid = true;
    return PHI4_OK;
}

const double* phi4_field(phi4_handle* h) { if (!h) { set_err4("phi4_field: null handle"); return nullptr; } return h->phi; }
const int32_t* phi4_labels(phi4_handle* h) {
    if (!h) { set_err4("phi4_labels: null handle"); return nullptr; }
    if (!h->have_sweep) { set_err4("phi4_labels: no update has run yet"); return nullptr; }
    return h->label;
}
const uint8_t* phi4_bonds(phi4_handle* h) {
    if (!h) { set_err4("phi4_bonds: null handle"); return nullptr; }
    if (!h->have_sweep) { set_err4("phi4_bonds: no update has run yet"); return nullptr; }
    return h->bonds;
}
int phi4_direction(phi4_handle* h, double r[4]) {
    if (!h || !r) { set_err4("phi4_direction: null argument"); return PHI4_EINVAL; }
    if (!h->have_sweep) { set_err4("phi4_direction: no update has run yet"); return PHI4_ESTATE; }
    DevGuard4 dg(h->dev);
    P4_CUDA(cudaMemcpyAsync(r, h->r + 4, 4 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    P4_CUDA(cudaStreamSynchronize(h->stream));
    return PHI4_OK;
}

int phi4_observables(phi4_handle* h, phi4_obs* out) {
    if (!h || !out) { set_err4("phi4_observables: null argument"); return PHI4_EINVAL; }
    DevGuard4 dg(h->dev);
    Rec4 r;
    if (h->rec_valid) {
        const int64_t slot = (h->last_n - 1) % P4_SERIES_CAP;
        P4_CUDA(cudaMemcpyAsync(&r, h->rec + slot, sizeof(Rec4), cudaMemcpyDeviceToHost, h->stream));
    } else {
        k4_observe<<<(unsigned)h->nblocks, P4_THREADS, 0, h->stream>>>(h->phi, h->gsize, h->partial, h->iacc, h->g, 0, h->rec, h->ctl,
                                                                       h->r, h->r + 4, h->key0, h->key1, 0);
        P4_CUDA(cudaGetLastError());
        P4_CUDA(cudaMemcpyAsync(&r, h->rec + P4_SERIES_CAP, sizeof(Rec4), cudaMemcpyDeviceToHost, h->stream));
    }
    P4_CUDA(cudaStreamSynchronize(h->stream));
    fill_obs4(h, r, h->t, out);
    return PHI4_OK;
}

int64_t phi4_series(phi4_handle* h, phi4_obs* out, int64_t cap) {
    if (!h || !out || cap < 0) { set_err4("phi4_series: invalid argument"); return PHI4_EINVAL; }
    if (!h->rec_valid) return 0;
    DevGuard4 dg(h->dev);
    const int64_t kept = std::min<int64_t>(h->last_n, P4_SERIES_CAP), give = std::min(kept, cap);
    std::vector<Rec4> r((size_t)P4_SERIES_CAP);
    P4_CUDA(cudaMemcpyAsync(r.data(), h->rec, r.size() * sizeof(Rec4), cudaMemcpyDeviceToHost, h->stream));
    P4_CUDA(cudaStreamSynchronize(h->stream));
    const int64_t first = h->last_n - kept;
    for (int64_t k = 0; k < give; ++k)
        fill_obs4(h, r[(size_t)((first + k) % P4_SERIES_CAP)], h->t - (uint64_t)h->last_n + (uint64_t)(first + k) + 1, out + k);
    return kept;
}

int phi4_set_field(phi4_handle* h, const double* phi, int is_host) {
    if (!h || !phi) { set_err4("phi4_set_field: null argument"); return PHI4_EINVAL; }
    DevGuard4 dg(h->dev);
    P4_CUDA(cudaMemcpyAsync(h->phi, phi, (size_t)h->V * 4 * sizeof(double), is_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, h->stream));
    if (is_host) P4_CUDA(cudaStreamSynchronize(h->stream));
    h->have_sweep = false; h->rec_valid = false;
    return PHI4_OK;
}
int phi4_get_field(phi4_handle* h, double* out_host) {
    if (!h || !out_host) { set_err4("phi4_get_field: null argument"); return PHI4_EINVAL; }
    DevGuard4 dg(h->dev);
    P4_CUDA(cudaMemcpyAsync(out_host, h->phi, (size_t)h->V * 4 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    P4_CUDA(cudaStreamSynchronize(h->stream));
    return PHI4_OK;
}
int phi4_get_labels(phi4_handle* h, int32_t* out_host) {
    if (!h || !out_host) { set_err4("phi4_get_labels: null argument"); return PHI4_EINVAL; }
    if (!h->have_sweep) { set_err4("phi4_get_labels: no update has run yet"); return PHI4_ESTATE; }
    DevGuard4 dg(h->dev);
    P4_CUDA(cudaMemcpyAsync(out_host, h->label, (size_t)h->V * sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    P4_CUDA(cudaStreamSynchronize(h->stream));
    return PHI4_OK;
}
int phi4_get_bonds(phi4_handle* h, uint8_t* out_host) {
    if (!h || !out_host) { set_err4("phi4_get_bonds: null argument"); return PHI4_EINVAL; }
    if (!h->have_sweep) { set_err4("phi4_get_bonds: no update has run yet"); return PHI4_ESTATE; }
    DevGuard4 dg(h->dev);
    P4_CUDA(cudaMemcpyAsync(out_host, h->bonds, (size_t)h->V, cudaMemcpyDeviceToHost, h->stream));
    P4_CUDA(cudaStreamSynchronize(h->stream));
    return PHI4_OK;
}
int phi4_set_sweep_index(phi4_handle* h, uint64_t t) {
    if (!h) { set_err4("phi4_set_sweep_index: null handle"); return PHI4_EINVAL; }
    h->t = t;
    return PHI4_OK;
}
uint64_t phi4_sweep_index(const phi4_handle* h) { return h ? h->t : 0; }
int phi4_set_stream(phi4_handle* h, void* cuda_stream) {
    if (!h) { set_err4("phi4_set_stream: null handle"); return PHI4_EINVAL; }
    DevGuard4 dg(h->dev);
    P4_CUDA(cudaStreamSynchronize(h->stream));
    h->stream = (cudaStream_t)cuda_stream;
    return PHI4_OK;
}
int phi4_set_graphs(phi4_handle* h, int on) {
    if (!h) { set_err4("phi4_set_graphs: null handle"); return PHI4_EINVAL; }
    h->use_graphs = on != 0;
    return PHI4_OK;
}
int32_t phi4_L(const phi4_handle* h) { return h ? h->L : 0; }
int64_t phi4_last_launch_count(const phi4_handle* h) { return h ? h->launches : 0; }

} // extern "C"
