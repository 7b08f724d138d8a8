// sw_api.cu -- host logic and the extern "C" boundary of libsw_b200.so (see include/sw.h).
// Product code (CUDA path).  No CPU fallback: every compute entry point needs a CUDA device.
#include "../../include/sw.h"
#include "sw_common.cuh"
#include "sw_generic.cuh"
#include "sw_tiled.cuh"
#include "sw_scan.cuh"
#include "sw_flip_tma.cuh"
#include "sw_cluster.cuh"
#include "sw_equiv.cuh"
#include "sw_potts.cuh"
#include "sw_series.cuh"

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <string>
#include <vector>

using namespace sw;

namespace {

thread_local std::string g_err = "";

void set_err(const char* fmt, ...) __attribute__((format(printf, 1, 2)));
void set_err(const char* fmt, ...) {
    char buf[512];
    va_list ap; va_start(ap, fmt); vsnprintf(buf, sizeof buf, fmt, ap); va_end(ap);
    g_err = buf;
}

#define SW_CUDA(call)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (call);                                                                   \
        if (e_ != cudaSuccess) {                                                                   \
            set_err("CUDA error %s at %s:%d: %s", cudaGetErrorName(e_), __FILE__, __LINE__,        \
                    cudaGetErrorString(e_));                                                       \
            return SW_ECUDA;                                                                       \
        }                                                                                          \
    } while (0)

constexpr size_t ALIGN = 256;
constexpr int64_t DEFAULT_SERIES_CAP = 4096;
constexpr int MAX_TIMED_SWEEPS = 1024;
// kernel slots for per-kernel event timing (sw_kernel_ms); one event before each launch + one at the end
enum Kid { K_BOND = 0, K_TILE, K_MERGE, K_COMPRESS, K_SIZES, K_SIZES_RESET, K_FLIPBITS, K_FLIP, K_ENERGY, K_ADVANCE,
           K_BONDLABEL, K_FLIPTILE, K_COUNT };
const char* const KERNEL_NAMES[K_COUNT] = { "bond", "tile_label", "merge", "compress", "roots_open", "sizes_reset",
                                            "flipbits", "flip", "energy", "advance", "bond_label", "flip16" };
// stage of each kernel: bond, label, flip, observe.  The fused kernels are booked under the stage that
// dominates them: bond_label (a1 + a2) under "label", flip16 (a4 + a6) under "flip".
const int KERNEL_STAGE[K_COUNT] = { 0, 1, 1, 1, 1, 1, 2, 2, 3, 3, 1, 2 };
constexpr int EV_PER_SWEEP = K_COUNT + 1;

inline size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

// tile shapes of the fast path
// ROWS64: row kernels on the int8 plane + flat labels (path 11); SCAN_2: 64 x 32 tiles (L a multiple of 64 only);
// SCAN_4x64: 128 x 64 tiles (L a multiple of 128: the headline shape)
enum TileKind { TILE_NONE = 0, ROWS64 = 1, SCAN_2 = 3, SCAN_4x64 = 7 };
// width in 32-site words of the tiles the scan-line kernel and k_flip16 share (0: not a scan tile)
inline int scan_nw(TileKind k) { return k == SCAN_2 ? 2 : k == SCAN_4x64 ? 4 : 0; }
constexpr int SMALL_L = 1024;          // up to this side the fast path runs on 64 x 32 tiles
constexpr int MAX_DEV = 64;            // per-device "attribute set" flags of the kernels with opt-in shared memory

struct Layout {        // byte offsets into the workspace
    size_t spins, sbits, bondE, bondS, D, lab16, ocount, nodes, bslot, lat, ctl, rec_now, mom, series, total;
};

size_t node_entries(int L) {           // per lattice: CAP = 2 (TW + TH) entries per tile of the shape this L runs on
    const size_t N = (size_t)L * L;
    if (L % 128 == 0 && L > SMALL_L) return N / (128 * 64) * (size_t)(2 * (128 + 64));
    if (L % 64 == 0) return N / (64 * 32) * (size_t)(2 * (64 + 32));
    return 0;
}
size_t tiles_max(int L) { return (L % 128 == 0 && L > SMALL_L) ? (size_t)L * L / (128 * 64) : L % 64 == 0 ? (size_t)L * L / (64 * 32) : 0; }

DivL make_div(int d) {          // q = (v * m) >> p is exact for 0 <= v < 2^30 (error term < 1/d)
    int k = 0; while ((1 << k) < d) ++k;
    DivL D; D.p = 30 + k; D.d = d;
    D.m = (uint32_t)(((1ull << D.p) + (uint64_t)d - 1) / (uint64_t)d);
    return D;
}

Layout make_layout(int L, int nb) {
    const size_t N = (size_t)L * L, words = (N + 31) / 32;
    Layout o; size_t p = 0;
    o.spins = p;   p = align_up(p + (size_t)nb * N);
    o.sbits = p;   p = align_up(p + (size_t)nb * words * 4);     // bit-packed spins (fused scan path, packed host interface)
    o.bondE = p;   p = align_up(p + (size_t)nb * words * 4);
    o.bondS = p;   p = align_up(p + (size_t)nb * words * 4);
    o.D = p;       p = align_up(p + (size_t)nb * ((words + 3) / 4 * 4) * 4);
    // (the flat int32 labels and the generic paths' size array, 4 B/site each, are allocated on first use: need_label)
    o.lab16 = p;   p = align_up(p + (L % 64 == 0 ? (size_t)nb * N * 2 : 0));
    o.ocount = p;  p = align_up(p + (size_t)nb * tiles_max(L) * 4);
    o.nodes = p;   p = align_up(p + (size_t)nb * node_entries(L) * 16);     // node array of the scan path
    o.bslot = p;   p = align_up(p + (size_t)nb * node_entries(L) * 2);
    o.lat = p;     p = align_up(p + (size_t)nb * sizeof(Lat));
    o.ctl = p;     p = align_up(p + sizeof(Ctl));
    o.rec_now = p; p = align_up(p + (size_t)nb * sizeof(Rec));
    o.mom = p;     p = align_up(p + (size_t)nb * sizeof(Mom));
    o.series = p;  p = align_up(p + (size_t)(DEFAULT_SERIES_CAP + 1) * nb * sizeof(Rec));
    o.total = p;
    return o;
}

bool valid_dims(int32_t L, int32_t nb) {
    return L >= 2 && L <= SW_MAX_L && nb >= 1 && nb <= 65535 && (uint64_t)L * L * (uint64_t)nb <= (1ull << 40);
}

uint32_t host_threshold(double T) {
    // thr = min(floor(p 2^32), 2^32 - 1), p = 1 - exp(-2/T) via expm1
    const double p = -std::expm1(-2.0 / T);
    const double v = std::floor(p * 4294967296.0);
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

uint32_t host_threshold_potts(double T) {
    // Potts: p = 1 - exp(-1/T) (H = -sum delta; for q = 2 the Ising rule at T_Ising = 2 T)
    const double p = -std::expm1(-1.0 / T);
    const double v = std::floor(p * 4294967296.0);
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

} // namespace

struct sw_handle {
    int L = 0, nb = 0, N = 0, words = 0;
    int dev = 0;                     // the CUDA device the handle lives on: every entry point switches to it
    bool owns_ws = false;
    char* ws = nullptr; size_t ws_bytes = 0;
    uint32_t* sbits = nullptr;       // bit-packed spins: bit 1 = +1.  The fused scan path keeps the state HERE
    bool i8_valid = true, bits_valid = false;      // which of the two spin planes holds the current configuration
    int8_t* spins = nullptr; uint32_t *bondE = nullptr, *bondS = nullptr, *D = nullptr;
    int *label = nullptr, *gsize = nullptr;          // flat labels / cluster sizes, 4 B/site each: allocated on first use
    int* ocount = nullptr;
    uint16_t* lab16 = nullptr;       // tile-local root index of every site (scan path)
    int4* nodes = nullptr;           // union-find over open tile roots: (parent, size, min site, site)
    uint16_t* bslot = nullptr;       // per tile: slot of the root of each border site
    int q = 0;                       // 0: Ising (spins +-1); >= 2: q-state Potts (colours 0 .. q-1), sw_potts.cuh
    int* potts_cnt = nullptr;        // [nb][q] sites per colour (Potts observables)
    int* eq_ref = nullptr; int* eq_flags = nullptr;   // path 11 (label equivalence): allocated on first use
    bool eq_ran = false;
    Lat* lat = nullptr; Ctl* ctl = nullptr; Rec* rec_now = nullptr; Mom* mom = nullptr;
    std::vector<double> hT;          // temperatures (sw_moments: specific heat, susceptibility)
    Rec* series = nullptr; Rec* series_owned = nullptr;
    int64_t series_cap = DEFAULT_SERIES_CAP;       // sweeps retained; the ring has series_cap + 1 slots
    int64_t ring() const { return series_cap + 1; }  // (the slot after the last sweep is already zeroed)
    std::vector<Lat> hlat;
    uint64_t t = 0;
    cudaStream_t stream = nullptr;
    bool have_sweep = false;       // labels / bonds / cluster observables of a sweep exist
    bool labels_flat = false;      // label[] holds roots (else: site -> tile root -> global root)
    bool eager_labels = false;     // the flip kernel also stores the flat labels every sweep
    bool rec_valid = false;        // the last series slot holds E, M of the current spins
    int64_t last_n = 0;
    int path = 0; TileKind tile = TILE_NONE;
    TileKind lab_tile = TILE_NONE;  // tile shape of the sweep whose 16-bit roots are pending (flattened on demand)
    bool timing = false; std::vector<cudaEvent_t> ev; int64_t timed_sweeps = 0;
    cudaEvent_t ev_tail[2] = { nullptr, nullptr };   // around the trailing k_observe_rows of a call
    // CUDA graphs of the steady sweep (every sweep of a call but the first launches the same kernels with the
    // same arguments: the sweep index lives on the device).  Replayed on an internal stream ordered after /
    // before the caller's stream by events, because the legacy default stream cannot be captured.
    bool use_graphs = true, graph_failed = false;
    cudaStream_t gstream = nullptr; cudaEvent_t gev[2] = { nullptr, nullptr };
    cudaGraphExec_t gexec[2] = { nullptr, nullptr };  // GRAPH_UNROLL sweeps, 1 sweep
    const void* gkey_series = nullptr; int gkey_path = -1, gkey_eager = -1; int64_t glaunches = 0;
    int ev_cursor = 0; std::vector<int> ev_seq;   // kernel ids in launch order within one sweep
    int64_t cur_sweep = 0;
    int64_t launches = 0;
    // TMA staging of the 16-bit root plane in the assignment kernel (sw_flip_tma.cuh): tensor map of lab16, made on first use
    CUtensorMap tmap, tmap_d; int tmap_state = 0;   // 0: not tried, 1: ready, -1: unavailable (k_flip16 is used)
    bool use_tma = true;
    // lattices of at most 8 tiles: the whole sw_sweep call inside one kernel, one thread-block cluster per lattice (sw_cluster.cuh)
    bool use_cluster = true, cluster_failed = false;
    // side branch of the sweep: the decision plane depends on nothing but the sweep index, so k_flipbits runs beside the labelling
    cudaStream_t side = nullptr; cudaEvent_t ev_fork = nullptr, ev_join = nullptr; bool side_failed = false;
};

namespace {

// paths: 0 the fast path (fused bond + scan-line labelling on 128 x 64 tiles when L is a multiple of 128, on 64 x 32
// tiles when it is a multiple of 64, generic kernels otherwise); 1 generic kernels; 6 the fast path's tiles with a
// stand-alone bond kernel on the int8 plane (per-stage timing); 11 the paper's label-equivalence labelling
TileKind pick_tile(int L, int path) {
    if (path == 1) return TILE_NONE;
    if (path == 11) return L % 64 == 0 ? ROWS64 : TILE_NONE;          // row kernels for bond / flip / energy; labels: sw_equiv.cuh
    // small lattices wait for the latency of ONE tile: 64 x 32 tiles (8 warps each on 32 x 8 blocks) up to L = 1024
    if (L % 128 == 0 && L > SMALL_L) return SCAN_4x64;
    if (L % 64 == 0) return SCAN_2;
    return TILE_NONE;
}
bool valid_path(int path) { return path == 0 || path == 1 || path == 6 || path == 11; }

// Potts handles: the scan-line path on 128 x 64 tiles when L allows it (path 0), else the generic kernels
TileKind potts_tile(int L, int path) { return (path == 0 && L % 128 == 0) ? SCAN_4x64 : TILE_NONE; }

inline dim3 grid1(size_t n, int threads, int nb) { return dim3((unsigned)((n + threads - 1) / threads), (unsigned)nb); }

// every entry point runs on the handle's device, whatever device is current in the calling thread
struct DevGuard {
    int prev = -1; bool switched = false;
    explicit DevGuard(int dev) {
        if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) switched = cudaSetDevice(dev) == cudaSuccess;
    }
    ~DevGuard() { if (switched) cudaSetDevice(prev); }
    DevGuard(const DevGuard&) = delete; DevGuard& operator=(const DevGuard&) = delete;
};

// flat int32 labels (sw_labels, generic / path-11 labelling) and the generic paths' cluster-size array: 4 B/site each,
// allocated the first time a path needs them, so that the fast path's footprint stays at ~4.5 B/site
int need_label(sw_handle* h) {
    if (h->label) return SW_OK;
    cudaError_t e = cudaMalloc((void**)&h->label, (size_t)h->nb * h->N * sizeof(int));
    if (e != cudaSuccess) { (void)cudaGetLastError(); set_err("cudaMalloc of the label array (%zu bytes) failed: %s", (size_t)h->nb * h->N * sizeof(int), cudaGetErrorString(e)); h->label = nullptr; return SW_ENOMEM; }
    return SW_OK;
}
int need_gsize(sw_handle* h) {
    if (h->gsize) return SW_OK;
    cudaError_t e = cudaMalloc((void**)&h->gsize, (size_t)h->nb * h->N * sizeof(int));
    if (e != cudaSuccess) { (void)cudaGetLastError(); set_err("cudaMalloc of the size array (%zu bytes) failed: %s", (size_t)h->nb * h->N * sizeof(int), cudaGetErrorString(e)); h->gsize = nullptr; return SW_ENOMEM; }
    return SW_OK;
}

// the two spin planes: the fused scan path sweeps on the bit plane, everything else on the int8 plane
bool sweeps_on_bits(const sw_handle* h) { return scan_nw(h->tile) && h->path != 6 && !h->q; }
int ensure_i8(sw_handle* h) {
    if (h->i8_valid) return SW_OK;
    k_unpack_spins<<<grid1(h->words, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(h->spins, h->sbits, h->N, h->words);
    SW_CUDA(cudaGetLastError());
    h->i8_valid = true;
    return SW_OK;
}
int ensure_bits(sw_handle* h) {
    if (h->bits_valid) return SW_OK;
    k_pack_spins<<<grid1(h->words, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(h->spins, h->sbits, h->N, h->words);
    SW_CUDA(cudaGetLastError());
    h->bits_valid = true;
    return SW_OK;
}

// timing mode: an event before kernel `kid` of sweep h->cur_sweep (kid == K_COUNT closes the sweep)
int mark(sw_handle* h, int kid) {
    if (!h->timing || h->cur_sweep >= MAX_TIMED_SWEEPS) return SW_OK;
    if (h->cur_sweep == 0) h->ev_seq.push_back(kid);
    SW_CUDA(cudaEventRecord(h->ev[(size_t)h->cur_sweep * EV_PER_SWEEP + h->ev_cursor++], h->stream));
    return SW_OK;
}
#define SW_MARK(h, kid) do { int rc_ = mark((h), (kid)); if (rc_) return rc_; } while (0)

// k_roots_nodes: 4 warps per tile while the whole batch has fewer tiles than the GPU holds warps
#ifndef ROOTS_WPT
#define ROOTS_WPT 1
#endif
inline int roots_warps_per_tile(const sw_handle* h, int tiles) { return (long long)tiles * h->nb < 4096 ? 4 : ROOTS_WPT; }

// launch with programmatic stream serialization (see pdl_wait in sw_common.cuh): the kernels of the fast path's sweep.
// Not with per-kernel timing: an event between two overlapping launches does not separate them (sw_sweep sets t_pdl).
thread_local bool t_pdl = true;
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = t_pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

// opt-in dynamic shared memory, once per kernel and device
template <typename K>
int opt_in_smem(K kernel, size_t smem, bool* done, int dev) {
    if (dev < 0 || dev >= MAX_DEV || !done[dev]) {
        SW_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (dev >= 0 && dev < MAX_DEV) done[dev] = true;
    }
    return SW_OK;
}

// fast path: fused bond + scan-line tile labelling, global merge, open roots (a1-a3)
template <int NW, int TH, int BAND_T = 32>
int launch_bond_label_scan(sw_handle* h, bool fused, bool obs_prev) {
    constexpr int TW = 32 * NW, CAP = 2 * (TW + TH), THREADS = NW * TH * (32 / BAND_T);
    const int tiles = h->N / (TW * TH);
    constexpr size_t smem = bond_label_smem(TW * TH);                 // the parent array + the list of hooked nodes (dynamic: 34 KB at 128 x 64)
    static bool done[2][MAX_DEV];
    { int rc = opt_in_smem(k_bond_label<NW, TH, true, false, BAND_T>, smem, done[0], h->dev); if (rc) return rc; }
    { int rc = opt_in_smem(k_bond_label<NW, TH, false, false, BAND_T>, smem, done[1], h->dev); if (rc) return rc; }
    if (fused) {
        SW_MARK(h, K_BONDLABEL);
        SW_CUDA(launch_pdl(k_bond_label<NW, TH, true, false, BAND_T>, dim3(tiles, h->nb), dim3(THREADS), smem, h->stream,
            h->sbits, h->bondE, h->bondS, h->lab16, h->nodes, h->ocount, h->bslot,
            h->series, h->lat, h->ctl,
            h->L, h->N, h->words, h->nb, obs_prev ? 1 : 0));
    } else {
        SW_MARK(h, K_TILE);
        k_bond_label<NW, TH, false, false, BAND_T><<<dim3(tiles, h->nb), THREADS, smem, h->stream>>>(
            nullptr, h->bondE, h->bondS, h->lab16, h->nodes, h->ocount, h->bslot,
            h->series, h->lat, h->ctl,
            h->L, h->N, h->words, h->nb, obs_prev ? 1 : 0);
    }
    const size_t nedge = (size_t)h->L * (h->L / TW + h->L / TH);
    SW_MARK(h, K_MERGE);
    SW_CUDA(launch_pdl(k_merge_nodes<TW, TH>, grid1(nedge, 256, h->nb), dim3(256), 0, h->stream,
        h->nodes, h->bslot, h->L / TW, h->L / TH, make_div(h->L / TW)));
    SW_MARK(h, K_SIZES);
    const int wpt = roots_warps_per_tile(h, tiles);
    SW_CUDA(launch_pdl(k_roots_nodes<CAP>, grid1((size_t)tiles * wpt * 32, 256, h->nb), dim3(256), 0, h->stream,
        h->nodes, h->ocount, tiles, wpt));
    h->launches += 3;
    return SW_OK;
}
// a4 for the scan path: open tile roots take their cluster's label, then two hops per site
template <int NW, int TH>
int launch_flatten_scan(sw_handle* h) {
    constexpr int TW = 32 * NW;
    const int tiles = h->N / (TW * TH);
    constexpr size_t smem = (size_t)TW * TH * sizeof(int);
    static bool done[MAX_DEV];
    { int rc = opt_in_smem(k_labels16<NW, TH>, smem, done, h->dev); if (rc) return rc; }
    { int rc = need_label(h); if (rc) return rc; }
    k_labels16<NW, TH><<<dim3(tiles, h->nb), NW * TH, smem, h->stream>>>(
        h->label, h->lab16, h->nodes, h->ocount, make_div(h->L), h->L, h->N);
    h->launches += 1;
    return SW_OK;
}
int flatten_scan(sw_handle* h, TileKind tile) {
    switch (tile) {
        case SCAN_2:    return launch_flatten_scan<2, 32>(h);
        case SCAN_4x64: return launch_flatten_scan<4, 64>(h);
        default:        return SW_ESTATE;
    }
}
// tensor map of the 16-bit root plane: [nb * L rows][L columns] uint16, boxes of 128 x 64 (one tile)
bool make_lab16_tmap(sw_handle* h) {
    if (h->tmap_state) return h->tmap_state > 0;
    h->tmap_state = -1;
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn || qr != cudaDriverEntryPointSuccess) {
        (void)cudaGetLastError();
        return false;
    }
    const cuuint64_t dims[2] = { (cuuint64_t)h->L, (cuuint64_t)h->L * (cuuint64_t)h->nb };
    const cuuint64_t strides[1] = { (cuuint64_t)h->L * 2 };
    const cuuint32_t box[2] = { 128, 64 }, estr[2] = { 1, 1 };
    if (((EncodeFn)fn)(&h->tmap, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, h->lab16, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                       CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    // the decision plane: [nb * L rows][L / 32 words] uint32, boxes of 4 x 64 (a tile's own words)
    const cuuint64_t ddims[2] = { (cuuint64_t)(h->L / 32), (cuuint64_t)h->L * (cuuint64_t)h->nb };
    const cuuint64_t dstrides[1] = { (cuuint64_t)(h->L / 32) * 4 };
    const cuuint32_t dbox[2] = { 4, 64 };
    if (((size_t)h->words * 4) % 16 != 0 ||
        ((EncodeFn)fn)(&h->tmap_d, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, h->D, ddims, dstrides, dbox, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                       CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return false;
    h->tmap_state = 1;
    return true;
}

// a4-a6 fused (+ count and largest of the clusters that span tiles)
// small lattices on 64 x 32 tiles: decision words drawn inside the assignment kernel, sweep advanced by its last CTA
bool flip_fused(const sw_handle* h) { return h->tile == SCAN_2 && sweeps_on_bits(h); }

template <int NW, int TH>
int launch_flip_scan(sw_handle* h, int adv_acc) {
    constexpr int TW = 32 * NW;
    const int tiles = h->N / (TW * TH);
    SW_MARK(h, K_FLIPTILE);
    if (NW == 4 && TH == 64 && sweeps_on_bits(h) && h->use_tma && tiles >= 512 && make_lab16_tmap(h)) {
        constexpr size_t smem = (size_t)FT_NSTAGE * FT_STAGE_BYTES + 128;
        static bool done[MAX_DEV];
        { int rc = opt_in_smem(k_flip16_tma, smem, done, h->dev); if (rc) return rc; }
        static int sms[MAX_DEV];
        int& nsm = sms[h->dev >= 0 && h->dev < MAX_DEV ? h->dev : 0];
        if (!nsm) SW_CUDA(cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, h->dev));
        const int ctas = std::max(1, std::min(tiles, FT_CTAS_PER_SM * nsm / std::max(1, std::min(h->nb, FT_CTAS_PER_SM))));   // persistent: FT_CTAS_PER_SM CTAs per SM in all
        SW_CUDA(launch_pdl(k_flip16_tma, dim3(ctas, h->nb), dim3(256 + 32 * FT_PROD_WARPS), smem, h->stream,
            h->tmap, h->tmap_d, h->sbits, h->D, h->nodes, h->ocount, h->series, h->ctl, make_div(h->L), h->L, h->N, h->words, h->nb, tiles));
    } else if (flip_fused(h))
        SW_CUDA(launch_pdl(k_flip16<NW, TH, true, true>, dim3(tiles, h->nb), dim3(NW * TH), 0, h->stream,
            h->spins, h->sbits, h->lab16, nullptr, h->nodes, h->ocount, h->series, h->ctl, h->lat, h->mom, adv_acc,
            make_div(h->L), h->L, h->N, h->words, h->nb));
    else if (sweeps_on_bits(h))
        k_flip16<NW, TH, true><<<dim3(tiles, h->nb), NW * TH, 0, h->stream>>>(
            h->spins, h->sbits, h->lab16, h->D, h->nodes, h->ocount, h->series, h->ctl, h->lat, h->mom, adv_acc,
            make_div(h->L), h->L, h->N, h->words, h->nb);
    else
        k_flip16<NW, TH, false><<<dim3(tiles, h->nb), NW * TH, 0, h->stream>>>(
            h->spins, h->sbits, h->lab16, h->D, h->nodes, h->ocount, h->series, h->ctl, h->lat, h->mom, adv_acc,
            make_div(h->L), h->L, h->N, h->words, h->nb);
    h->launches += 1;
    if (h->eager_labels) {                          // a4 every sweep instead of on demand
        SW_MARK(h, K_COMPRESS);
        return launch_flatten_scan<NW, TH>(h);
    }
    return SW_OK;
}

int launch_label_generic(sw_handle* h) {
    SW_MARK(h, K_TILE);
    k_label_init<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(h->label, h->N);
    SW_MARK(h, K_MERGE);
    k_union_generic<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
        h->label, h->bondE, h->bondS, h->L, h->N, h->words);
    SW_MARK(h, K_COMPRESS);
    SW_CUDA(cudaMemsetAsync(h->gsize, 0, (size_t)h->nb * h->N * sizeof(int), h->stream));
    k_compress_generic<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
        h->label, h->gsize, h->series, h->ctl, h->N, h->nb);
    SW_MARK(h, K_SIZES);
    k_maxsize_generic<<<grid1(h->N, MAXSIZE_SPAN, h->nb), GEN_THREADS, 0, h->stream>>>(
        h->label, h->gsize, h->series, h->ctl, h->N, h->nb);
    h->launches += 4;
    return SW_OK;
}

// a2-a4 the paper's way: one cooperative kernel runs the label-equivalence passes to convergence
int launch_label_equiv(sw_handle* h) {
    static int max_blocks[MAX_DEV];
    int& mb = max_blocks[h->dev >= 0 && h->dev < MAX_DEV ? h->dev : 0];
    if (!mb) {
        int sms = 0, per_sm = 0, coop = 0;
        SW_CUDA(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->dev));
        if (!coop) { set_err("path 11: the device does not support cooperative launches"); return SW_ECUDA; }
        SW_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, h->dev));
        SW_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, k_label_equiv, EQ_THREADS, 0));
        if (per_sm < 1) { set_err("path 11: k_label_equiv does not fit on an SM"); return SW_ECUDA; }
        mb = sms * per_sm;
    }
    if (!h->eq_ref) {
        SW_CUDA(cudaMalloc(&h->eq_ref, (size_t)h->nb * h->N * sizeof(int)));
        SW_CUDA(cudaMalloc(&h->eq_flags, (size_t)(EQ_MAX_PASSES + 1) * sizeof(int)));
    }
    SW_CUDA(cudaMemsetAsync(h->eq_flags, 0, (size_t)(EQ_MAX_PASSES + 1) * sizeof(int), h->stream));
    const int blocks = std::max(1, std::min(mb, (h->N + EQ_THREADS - 1) / EQ_THREADS));
    DivL dv = make_div(h->L);
    void* args[] = { &h->label, &h->eq_ref, &h->bondE, &h->bondS, &h->eq_flags, &dv, &h->L, &h->N, &h->words, &h->nb };
    SW_MARK(h, K_TILE);
    SW_CUDA(cudaLaunchCooperativeKernel((const void*)k_label_equiv, dim3(blocks), dim3(EQ_THREADS), args, 0, h->stream));
    // cluster count and largest cluster from the flat labels
    SW_MARK(h, K_COMPRESS);
    SW_CUDA(cudaMemsetAsync(h->gsize, 0, (size_t)h->nb * h->N * sizeof(int), h->stream));
    k_count_flat<<<grid1(h->N, EQ_COUNT_SPAN, h->nb), EQ_THREADS, 0, h->stream>>>(
        h->label, h->gsize, h->series, h->ctl, h->N, h->nb);
    SW_MARK(h, K_SIZES);
    k_maxsize_generic<<<grid1(h->N, MAXSIZE_SPAN, h->nb), GEN_THREADS, 0, h->stream>>>(
        h->label, h->gsize, h->series, h->ctl, h->N, h->nb);
    h->launches += 3;
    h->eq_ran = true;
    return SW_OK;
}

// labelling alone from the bond planes, leaving flat labels (the unfused order; sw_test_label)
template <int NW, int TH>
int launch_label_scan(sw_handle* h) {
    int rc = NW == 2 ? launch_bond_label_scan<NW, TH, 8>(h, false, false) : launch_bond_label_scan<NW, TH>(h, false, false);
    if (rc) return rc;
    SW_MARK(h, K_COMPRESS);
    return launch_flatten_scan<NW, TH>(h);
}

int launch_label(sw_handle* h) {
    if (!scan_nw(h->tile)) {                        // flat labels + the size array: allocated on first use
        int rc = need_label(h); if (rc) return rc;
        rc = need_gsize(h); if (rc) return rc;
    }
    if (h->path == 11) return launch_label_equiv(h);
    switch (h->tile) {
        case SCAN_2:      return launch_label_scan<2, 32>(h);
        case SCAN_4x64:   return launch_label_scan<4, 64>(h);
        default:          return launch_label_generic(h);
    }
}

// Potts fast path: k_bond_label<4, 64, FUSE, POTTS> (equal-colour masks from the int8 plane), then the node merge
// Potts fast path with few colours: E of a sweep from the next sweep's bond test, colour counts (for M) from the assignment kernel
bool potts_folded(const sw_handle* h) { return h->q && h->q <= 8 && h->tile == SCAN_4x64; }

int launch_bond_label_potts(sw_handle* h, bool obs_prev) {
    constexpr int NW = 4, TH = 64, TW = 32 * NW, CAP = 2 * (TW + TH);
    const int tiles = h->N / (TW * TH);
    constexpr size_t smem = bond_label_smem(TW * TH);
    static bool done[MAX_DEV];
    { int rc = opt_in_smem(k_bond_label<NW, TH, true, true>, smem, done, h->dev); if (rc) return rc; }
    SW_MARK(h, K_BONDLABEL);
    k_bond_label<NW, TH, true, true><<<dim3(tiles, h->nb), NW * TH, smem, h->stream>>>(
        reinterpret_cast<const uint32_t*>(h->spins), h->bondE, h->bondS, h->lab16, h->nodes, h->ocount, h->bslot,
        h->series, h->lat, h->ctl, h->L, h->N, h->words, h->nb, obs_prev ? 1 : 0);
    const size_t nedge = (size_t)h->L * (h->L / TW + h->L / TH);
    SW_MARK(h, K_MERGE);
    k_merge_nodes<TW, TH><<<grid1(nedge, 256, h->nb), 256, 0, h->stream>>>(h->nodes, h->bslot, h->L / TW, h->L / TH, make_div(h->L / TW));
    SW_MARK(h, K_SIZES);
    const int wpt = roots_warps_per_tile(h, tiles);
    k_roots_nodes<CAP><<<grid1((size_t)tiles * wpt * 32, 256, h->nb), 256, 0, h->stream>>>(h->nodes, h->ocount, tiles, wpt);
    h->launches += 3;
    return SW_OK;
}

// Potts sweep (sw_potts.cuh): bonds between equal colours, labels (generic union-find, or path 11), a colour per
// cluster, observables
int launch_sweep_potts(sw_handle* h, int64_t k) {
    int rc;
    h->cur_sweep = k; h->ev_cursor = 0;
    if (h->tile != SCAN_4x64) {
        SW_MARK(h, K_BOND);
        k_bond_generic<<<grid1(h->words, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
            h->spins, h->bondE, h->bondS, h->lat, h->ctl, h->L, h->N, h->words);
        h->launches += 1;
    }
    if (h->tile == SCAN_4x64) {
        // fast path: fused bond draw + scan-line tile labelling, node merge, colour per tile root
        const bool folded = potts_folded(h);          // E with the next sweep's bond test, colour counts in the assignment
        if ((rc = launch_bond_label_potts(h, folded && k > 0))) return rc;
        SW_MARK(h, K_FLIPTILE);
        k_assign16_potts<4, 64><<<dim3(h->N / (128 * 64), h->nb), 256, 0, h->stream>>>(
            h->spins, h->lab16, h->nodes, h->ocount, h->series, h->lat, h->ctl, make_div(h->L), h->q, h->L, h->N, h->nb,
            folded ? h->potts_cnt : nullptr);
        SW_MARK(h, K_ENERGY);
        if (!folded) {
            k_observe_potts_rows<<<grid1((size_t)h->N / 16, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
                h->spins, h->series, h->potts_cnt, h->ctl, 1, h->q, h->L, h->N, h->nb);
            h->launches += 1;
        }
        k_potts_finish<<<1, 64, 0, h->stream>>>(h->series, h->potts_cnt, h->ctl, 1, h->q, h->N, h->nb);
        SW_MARK(h, K_ADVANCE);
        k_advance<<<1, 64, 0, h->stream>>>(h->ctl, h->series, h->nb, h->mom, h->N, folded ? (k > 0 ? 2 : 0) : 1);
        h->launches += 3;
        SW_MARK(h, K_COUNT);
        h->labels_flat = false;                      // int32 labels on demand (k_labels16)
        h->lab_tile = h->tile;
        return SW_OK;
    }
    h->labels_flat = true;
    if ((rc = launch_label(h))) return rc;
    SW_MARK(h, K_FLIP);
    k_assign_potts<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
        h->spins, h->label, h->lat, h->ctl, h->q, h->N);
    SW_MARK(h, K_ENERGY);
    k_observe_potts<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
        h->spins, h->series, h->potts_cnt, h->ctl, 1, h->q, h->L, h->N, h->nb);
    k_potts_finish<<<1, 64, 0, h->stream>>>(h->series, h->potts_cnt, h->ctl, 1, h->q, h->N, h->nb);
    SW_MARK(h, K_ADVANCE);
    k_advance<<<1, 64, 0, h->stream>>>(h->ctl, h->series, h->nb, h->mom, h->N, 1);
    h->launches += 4;
    SW_MARK(h, K_COUNT);
    return SW_OK;
}

// Small lattices (sw_cluster.cuh): tiles per lattice when the whole call can run inside k_sweeps_cluster, else 0.  Not with
// per-kernel timing or eager labels (they need the kernels apart), nor on the unfused path.
constexpr int CLUSTER_MAX_TILES = 8;                // (the portable cluster size)
int cluster_tiles(const sw_handle* h) {
    if (!h->use_cluster || h->cluster_failed || !sweeps_on_bits(h) || h->timing || h->eager_labels) return 0;
    if (scan_nw(h->tile) != 2) return 0;            // (64 x 32 tiles: L = 64 -> 2 tiles, L = 128 -> 8)
    const int tiles = h->N / (64 * 32);
    return tiles <= CLUSTER_MAX_TILES ? tiles : 0;
}
template <int NW, int TH, int BAND_T>
cudaError_t launch_sweeps_cluster(sw_handle* h, int64_t n, int tiles) {
    constexpr int THREADS = NW * TH * (32 / BAND_T);
    constexpr size_t smem = bond_label_smem(32 * NW * TH);
    static bool done[MAX_DEV];
    if (opt_in_smem(k_sweeps_cluster<NW, TH, BAND_T>, smem, done, h->dev)) return cudaErrorUnknown;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(tiles, h->nb); cfg.blockDim = dim3(THREADS); cfg.dynamicSmemBytes = smem; cfg.stream = h->stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = tiles; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, k_sweeps_cluster<NW, TH, BAND_T>, h->sbits, h->bondE, h->bondS, h->lab16, h->nodes, h->ocount, h->bslot,
                              h->series, (const Lat*)h->lat, h->mom, (unsigned long long)h->t, (uint32_t)h->ring(), (long long)n, 0,
                              make_div(h->L), h->L, h->N, h->words, h->nb);
}

// one full sweep on h->stream; the sweep index and series slot are read on the device from h->ctl
int launch_sweep(sw_handle* h, int64_t k) {
    if (h->q) return launch_sweep_potts(h, k);
    int rc;
    h->cur_sweep = k; h->ev_cursor = 0;
    if (const int nw = scan_nw(h->tile)) {
        const bool fused = h->path != 6;
        const bool obs_prev = k > 0;                    // E, M of sweep k - 1 come out of this sweep's bond test
        // the decision plane on a side branch (fork here, join before the assignment): under capture this becomes a parallel
        // branch of the graph.  Not with per-kernel timing (the events of the split assume one stream).
        bool side = fused && !flip_fused(h) && !h->timing && !h->side_failed;
        if (side && !h->side) {
            if (cudaStreamCreateWithFlags(&h->side, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming) != cudaSuccess) {
                (void)cudaGetLastError(); h->side_failed = true; side = false;
            }
        }
        if (side) {
            SW_CUDA(cudaEventRecord(h->ev_fork, h->stream));
            SW_CUDA(cudaStreamWaitEvent(h->side, h->ev_fork, 0));
            k_flipbits<<<grid1(((size_t)h->words + 3) / 4, GEN_THREADS, h->nb), GEN_THREADS, 0, h->side>>>(
                h->D, h->lat, h->ctl, h->words);
            SW_CUDA(cudaEventRecord(h->ev_join, h->side));
            h->launches += 1;
        }
        if (!fused) {                                   // stand-alone a1 for the per-stage split
            SW_MARK(h, K_BOND);
            k_bond_rows<<<grid1(h->words, ROW_THREADS, h->nb), ROW_THREADS, 0, h->stream>>>(
                h->spins, h->bondE, h->bondS, h->lat, h->ctl, h->L, h->N, h->words, h->series, h->nb, obs_prev ? 1 : 0);
            h->launches += 1;
        }
        // (64 x 32 tiles: 8 warps per tile, each scanning 32 x 8 sites -- the latency of one tile is what small lattices wait for)
        rc = nw == 4 ? launch_bond_label_scan<4, 64>(h, fused, obs_prev) : launch_bond_label_scan<2, 32, 8>(h, fused, obs_prev);
        if (rc) return rc;
        const int adv_acc = k > 0 ? 2 : 0;              // (E, M of a sweep arrive with the next sweep's bond test)
        const bool ff = flip_fused(h);
        if (side) SW_CUDA(cudaStreamWaitEvent(h->stream, h->ev_join, 0));
        if (!ff && !side) {
            SW_MARK(h, K_FLIPBITS);
            SW_CUDA(launch_pdl(k_flipbits, grid1(((size_t)h->words + 3) / 4, GEN_THREADS, h->nb), dim3(GEN_THREADS), 0, h->stream,
                h->D, h->lat, h->ctl, h->words));
            h->launches += 1;
        }
        rc = nw == 4 ? launch_flip_scan<4, 64>(h, adv_acc) : launch_flip_scan<2, 32>(h, adv_acc);
        if (rc) return rc;
        if (!ff) {
            SW_MARK(h, K_ADVANCE);
            SW_CUDA(launch_pdl(k_advance, dim3(1), dim3(64), 0, h->stream, h->ctl, h->series, h->nb, h->mom, h->N, adv_acc));
            h->launches += 1;
        }
        SW_MARK(h, K_COUNT);
        h->labels_flat = h->eager_labels;
        h->lab_tile = h->tile;                          // the tile shape lab16 / nodes were written with
        return SW_OK;
    }
    h->labels_flat = true;
    // a1 bonds
    SW_MARK(h, K_BOND);
    if (h->tile != TILE_NONE)
        k_bond_rows<<<grid1(h->words, ROW_THREADS, h->nb), ROW_THREADS, 0, h->stream>>>(
            h->spins, h->bondE, h->bondS, h->lat, h->ctl, h->L, h->N, h->words, h->series, h->nb, 0);
    else
        k_bond_generic<<<grid1(h->words, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
            h->spins, h->bondE, h->bondS, h->lat, h->ctl, h->L, h->N, h->words);
    h->launches += 1;
    // a2-a4 labels (+ cluster count, largest cluster)
    if ((rc = launch_label(h))) return rc;
    // a5-a6 assignment
    SW_MARK(h, K_FLIPBITS);
    k_flipbits<<<grid1(((size_t)h->words + 3) / 4, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
        h->D, h->lat, h->ctl, h->words);
    SW_MARK(h, K_FLIP);
    if (h->tile != TILE_NONE)
        k_flip_rows<<<grid1((size_t)h->N / 16, ROW_THREADS, h->nb), ROW_THREADS, 0, h->stream>>>(
            h->spins, h->label, h->D, h->series, h->ctl, h->N, h->words, h->nb);
    else
        k_flip_generic<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
            h->spins, h->label, h->D, h->N, h->words);
    h->launches += 2;
    // a7 observables of the new configuration
    SW_MARK(h, K_ENERGY);
    if (h->tile != TILE_NONE)
        k_energy_rows<<<grid1(h->words, ROW_THREADS, h->nb), ROW_THREADS, 0, h->stream>>>(
            h->spins, h->series, h->ctl, h->L, h->N, h->words, h->nb);
    else
        k_observe_generic<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
            h->spins, h->series, h->ctl, 1, h->L, h->N, h->nb);
    SW_MARK(h, K_ADVANCE);
    k_advance<<<1, 64, 0, h->stream>>>(h->ctl, h->series, h->nb, h->mom, h->N, 1);
    h->launches += 2;
    SW_MARK(h, K_COUNT);
    return SW_OK;
}

int init_handle(sw_handle* h, const double* T, const uint64_t* seed) {
    const Layout o = make_layout(h->L, h->nb);
    char* w = h->ws;
    h->spins = (int8_t*)(w + o.spins);
    h->sbits = (uint32_t*)(w + o.sbits);
    h->bondE = (uint32_t*)(w + o.bondE); h->bondS = (uint32_t*)(w + o.bondS); h->D = (uint32_t*)(w + o.D);
    h->lab16 = (uint16_t*)(w + o.lab16);
    h->nodes = (int4*)(w + o.nodes); h->bslot = (uint16_t*)(w + o.bslot);
    h->ocount = (int*)(w + o.ocount);
    h->lat = (Lat*)(w + o.lat); h->ctl = (Ctl*)(w + o.ctl); h->rec_now = (Rec*)(w + o.rec_now); h->mom = (Mom*)(w + o.mom);
    h->hT.assign(T, T + h->nb);
    h->series = (Rec*)(w + o.series);
    h->hlat.resize(h->nb);
    for (int b = 0; b < h->nb; ++b) {
        h->hlat[b].key0 = (uint32_t)(seed[b] & 0xFFFFFFFFu);
        h->hlat[b].key1 = (uint32_t)(seed[b] >> 32);
        h->hlat[b].thr = h->q ? host_threshold_potts(T[b]) : host_threshold(T[b]);
        h->hlat[b].pad = 0;
    }
    SW_CUDA(cudaMemcpyAsync(h->lat, h->hlat.data(), sizeof(Lat) * h->nb, cudaMemcpyHostToDevice, h->stream));
    SW_CUDA(cudaMemsetAsync(h->series, 0, (size_t)h->ring() * h->nb * sizeof(Rec), h->stream));
    SW_CUDA(cudaMemsetAsync(h->mom, 0, (size_t)h->nb * sizeof(Mom), h->stream));
    k_set_ctl<<<1, 1, 0, h->stream>>>(h->ctl, 0ull, 0u, (uint32_t)h->ring());
    if (h->q) {
        SW_CUDA(cudaMalloc(&h->potts_cnt, (size_t)h->nb * h->q * sizeof(int)));
        SW_CUDA(cudaMemsetAsync(h->potts_cnt, 0, (size_t)h->nb * h->q * sizeof(int), h->stream));
        k_init_potts<<<grid1(((size_t)h->N + 3) / 4, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(h->spins, h->lat, h->q, h->N);
    } else {
        k_init_random<<<grid1(h->words, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(h->spins, h->lat, h->N, h->words);
    }
    SW_CUDA(cudaGetLastError());
    SW_CUDA(cudaStreamSynchronize(h->stream));       // hlat is read by the async copy
    h->tile = h->q ? potts_tile(h->L, h->path) : pick_tile(h->L, h->path);
    return SW_OK;
}

sw_handle* create_common(void* ws, uint64_t ws_bytes, int32_t L, int32_t nb, const double* T, const uint64_t* seed, int q = 0) {
    if (q != 0 && (q < 2 || q > POTTS_MAX_Q)) { set_err("sw_create_potts: q = %d is not in 2 .. %d", q, POTTS_MAX_Q); return nullptr; }
    if (!valid_dims(L, nb) || !T || !seed) { set_err("sw_create: invalid argument (L=%d, nb=%d)", L, nb); return nullptr; }
    for (int b = 0; b < nb; ++b)
        if (!(T[b] > 0.0) || !std::isfinite(T[b])) { set_err("sw_create: T[%d] = %g is not a positive finite number", b, T[b]); return nullptr; }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0) {
        set_err("sw_create: no usable CUDA device (%s); this library has no CPU path", cudaGetErrorString(e));
        (void)cudaGetLastError();
        return nullptr;
    }
    sw_handle* h = new (std::nothrow) sw_handle();
    if (!h) { set_err("sw_create: out of host memory"); return nullptr; }
    h->L = L; h->nb = nb; h->N = L * L; h->words = (h->N + 31) / 32; h->q = q;
    if (cudaGetDevice(&h->dev) != cudaSuccess) { (void)cudaGetLastError(); set_err("sw_create: cudaGetDevice failed"); delete h; return nullptr; }
    const size_t need = make_layout(L, nb).total;
    if (ws) {
        if (ws_bytes < need || ((uintptr_t)ws % ALIGN) != 0) {
            set_err("sw_create_in: workspace of %llu bytes (need %llu, %zu-byte aligned)",
                    (unsigned long long)ws_bytes, (unsigned long long)need, ALIGN);
            delete h; return nullptr;
        }
        h->ws = (char*)ws; h->ws_bytes = ws_bytes; h->owns_ws = false;
    } else {
        void* p = nullptr;
        e = cudaMalloc(&p, need);
        if (e != cudaSuccess) { set_err("sw_create: cudaMalloc(%zu) failed: %s", need, cudaGetErrorString(e)); (void)cudaGetLastError(); delete h; return nullptr; }
        h->ws = (char*)p; h->ws_bytes = need; h->owns_ws = true;
    }
    if (init_handle(h, T, seed) != SW_OK) { if (h->potts_cnt) cudaFree(h->potts_cnt); if (h->owns_ws) cudaFree(h->ws); delete h; return nullptr; }
    return h;
}

void fill_obs(const sw_handle* h, const Rec& r, uint64_t sweep, sw_obs* o) {
    o->energy = r.E; o->magnetisation = r.M; o->n_clusters = r.ncl; o->largest_cluster = r.maxcl;
    o->sweep = sweep;
    o->e_per_site = (double)r.E / (double)h->N;
    o->abs_m_per_site = (double)(r.M < 0 ? -r.M : r.M) / (double)h->N;
}

} // namespace

// =================================================================================================
// ---- sw_bins_noalloc: binning with no allocation (include/sw.h) ------------------------------------------
// The bin means -- scratch between k_series_bins and k_series_binerr, which sw_bins takes from cudaMalloc -- live in a
// file-scope device array: every GPU that loads the library holds these 512 KiB until the process exits.  In host code the
// array's NAME is a host-side stand-in, not a device address (a kernel given it would fault or, where the GPU can reach
// host memory, silently use the wrong memory): the address comes from cudaGetSymbolAddress, once per device, with that
// device current.  Every call shares the array; calls that overlap on a GPU race on it.
static __device__ __align__(256) double g_bins_scratch[SW_BINS_NOALLOC_MAX];
namespace {
double* g_bins_scratch_ptr[MAX_DEV];   // per device; written once (a race between two first calls stores the same value)
int bins_scratch(int dev, double** out) {
    if (dev < 0 || dev >= MAX_DEV) { set_err("sw_bins_noalloc: device %d is outside the per-device table (0 .. %d)", dev, MAX_DEV - 1); return SW_EINVAL; }
    if (!g_bins_scratch_ptr[dev]) {
        double* p = nullptr;
        SW_CUDA(cudaGetSymbolAddress((void**)&p, g_bins_scratch));     // (the current device is `dev`: DevGuard of the caller)
        if (!p) { set_err("sw_bins_noalloc: cudaGetSymbolAddress returned a null address"); return SW_ECUDA; }
        g_bins_scratch_ptr[dev] = p;
    }
    *out = g_bins_scratch_ptr[dev];
    return SW_OK;
}
} // namespace

extern "C" {

const char* sw_last_error(void) { return g_err.c_str(); }
const char* sw_version(void) { return "sw-b200 0.1 (sm_100a)"; }

uint64_t sw_workspace_bytes(int32_t L, int32_t nb) {
    if (!valid_dims(L, nb)) return 0;
    return make_layout(L, nb).total;
}

sw_handle* sw_create(int32_t L, double T, uint64_t seed) { return create_common(nullptr, 0, L, 1, &T, &seed); }
sw_handle* sw_create_batch(int32_t L, int32_t nb, const double* T, const uint64_t* seed) {
    return create_common(nullptr, 0, L, nb, T, seed);
}
sw_handle* sw_create_potts(int32_t L, int32_t q, double T, uint64_t seed) {
    if (q < 2) { set_err("sw_create_potts: q = %d is not in 2 .. %d", q, POTTS_MAX_Q); return nullptr; }
    return create_common(nullptr, 0, L, 1, &T, &seed, q);
}
sw_handle* sw_create_potts_in(void* workspace, uint64_t workspace_bytes, int32_t L, int32_t q, int32_t nb,
                              const double* T, const uint64_t* seed) {
    if (!workspace) { set_err("sw_create_potts_in: null workspace"); return nullptr; }
    if (q < 2) { set_err("sw_create_potts_in: q = %d is not in 2 .. %d", q, POTTS_MAX_Q); return nullptr; }
    return create_common(workspace, workspace_bytes, L, nb, T, seed, q);
}
int32_t sw_q(const sw_handle* h) { return h ? h->q : 0; }
sw_handle* sw_create_in(void* workspace, uint64_t workspace_bytes, int32_t L, int32_t nb,
                        const double* T, const uint64_t* seed) {
    if (!workspace) { set_err("sw_create_in: null workspace"); return nullptr; }
    return create_common(workspace, workspace_bytes, L, nb, T, seed);
}

void sw_destroy(sw_handle* h) {
    if (!h) return;
    DevGuard dg(h->dev);
    cudaStreamSynchronize(h->stream);
    for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
    for (cudaEvent_t e : h->ev_tail) if (e) cudaEventDestroy(e);
    for (cudaGraphExec_t g : h->gexec) if (g) cudaGraphExecDestroy(g);
    for (cudaEvent_t e : h->gev) if (e) cudaEventDestroy(e);
    if (h->gstream) cudaStreamDestroy(h->gstream);
    if (h->ev_fork) cudaEventDestroy(h->ev_fork);
    if (h->ev_join) cudaEventDestroy(h->ev_join);
    if (h->side) cudaStreamDestroy(h->side);
    if (h->series_owned) cudaFree(h->series_owned);
    if (h->potts_cnt) cudaFree(h->potts_cnt);
    if (h->eq_ref) cudaFree(h->eq_ref);
    if (h->eq_flags) cudaFree(h->eq_flags);
    if (h->label) cudaFree(h->label);
    if (h->gsize) cudaFree(h->gsize);
    if (h->owns_ws) cudaFree(h->ws);
    (void)cudaGetLastError();
    delete h;
}

namespace {
constexpr int GRAPH_UNROLL = 8;

// (re)build the graphs of the steady sweep on h->gstream; on any failure the handle falls back to plain launches
bool build_graphs(sw_handle* h) {
    if (h->gexec[0] && h->gkey_series == h->series && h->gkey_path == h->path && h->gkey_eager == (int)h->eager_labels)
        return true;
    for (cudaGraphExec_t& g : h->gexec) if (g) { cudaGraphExecDestroy(g); g = nullptr; }
    const int64_t keep = h->launches;
    for (int v = 0; v < 2; ++v) {
        const int reps = v == 0 ? GRAPH_UNROLL : 1;
        cudaGraph_t graph = nullptr;
        if (cudaStreamBeginCapture(h->gstream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) { (void)cudaGetLastError(); return false; }
        h->launches = 0;
        int rc = SW_OK;
        for (int u = 0; u < reps && rc == SW_OK; ++u) rc = launch_sweep(h, 1);
        const cudaError_t e = cudaStreamEndCapture(h->gstream, &graph);
        if (rc != SW_OK || e != cudaSuccess || !graph) { (void)cudaGetLastError(); if (graph) cudaGraphDestroy(graph); h->launches = keep; return false; }
        h->glaunches = h->launches / reps;
        const cudaError_t ei = cudaGraphInstantiate(&h->gexec[v], graph, 0);
        cudaGraphDestroy(graph);
        if (ei != cudaSuccess) { (void)cudaGetLastError(); h->gexec[v] = nullptr; h->launches = keep; return false; }
    }
    h->launches = keep;
    h->gkey_series = h->series; h->gkey_path = h->path; h->gkey_eager = (int)h->eager_labels;
    return true;
}
} // namespace

int sw_sweep(sw_handle* h, int64_t n) {
    if (!h || n < 0) { set_err("sw_sweep: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (n == 0) return SW_OK;
    h->launches = 0;
    t_pdl = !h->timing;
    {   // the configuration must sit in the plane this path sweeps on
        const int rc = sweeps_on_bits(h) ? ensure_bits(h) : ensure_i8(h);
        if (rc) return rc;
    }
    // graph replay: scan path, no per-kernel timing, enough sweeps to pay for the two stream hops
    cudaStream_t const user = h->stream;
    struct StreamBack {                                 // whatever the exit: the handle goes back to the caller's stream,
        sw_handle* h; cudaStream_t user;                // ordered after what ran on the internal one
        ~StreamBack() {
            if (h->stream == user) return;
            if (h->gev[1] && cudaEventRecord(h->gev[1], h->stream) == cudaSuccess) cudaStreamWaitEvent(user, h->gev[1], 0);
            h->stream = user;
        }
    } stream_back{h, user};
    int ctiles = cluster_tiles(h);
    bool graphs = h->use_graphs && !h->graph_failed && !h->timing && scan_nw(h->tile) && n >= 4 && !h->q && !ctiles;
    if (graphs) {
        if (!h->gstream) {
            if (cudaStreamCreateWithFlags(&h->gstream, cudaStreamNonBlocking) != cudaSuccess ||
                cudaEventCreateWithFlags(&h->gev[0], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&h->gev[1], cudaEventDisableTiming) != cudaSuccess) {
                (void)cudaGetLastError(); h->graph_failed = true; graphs = false;
            }
        }
    }
    if (graphs) {
        SW_CUDA(cudaEventRecord(h->gev[0], user));
        SW_CUDA(cudaStreamWaitEvent(h->gstream, h->gev[0], 0));
        h->stream = h->gstream;                         // everything below runs on the internal stream
    }
    if (h->timing) {
        for (int i = 0; i < 2; ++i)
            if (!h->ev_tail[i]) SW_CUDA(cudaEventCreate(&h->ev_tail[i]));
        const size_t need = (size_t)std::min<int64_t>(n, MAX_TIMED_SWEEPS) * EV_PER_SWEEP;
        while (h->ev.size() < need) {
            cudaEvent_t e; SW_CUDA(cudaEventCreate(&e));
            h->ev.push_back(e);
        }
        h->ev_seq.clear();
    }
    SW_CUDA(cudaMemsetAsync(h->series, 0, (size_t)h->nb * sizeof(Rec), h->stream));
    int64_t k = 0;
    if (ctiles) {                                       // the whole call inside one kernel, a cluster per lattice
        const cudaError_t e = launch_sweeps_cluster<2, 32, 8>(h, n, ctiles);
        if (e != cudaSuccess) { (void)cudaGetLastError(); h->cluster_failed = true; ctiles = 0; }   // (nothing ran: take the kernels one by one)
        else {
            // Ctl as the sweeps below would have left it: the next sweep index, the slot after the last sweep (cleared)
            k_set_ctl<<<1, 1, 0, h->stream>>>(h->ctl, (unsigned long long)h->t + (unsigned long long)n, (uint32_t)(n % h->ring()), (uint32_t)h->ring());
            h->launches += 2;
            h->labels_flat = false; h->lab_tile = h->tile;
            k = n;
        }
    }
    if (!ctiles) {
        k_set_ctl<<<1, 1, 0, h->stream>>>(h->ctl, (unsigned long long)h->t, 0u, (uint32_t)h->ring());
        h->launches += 1;
        int rc = launch_sweep(h, 0);                    // (also sets the kernels' attributes before any capture)
        if (rc) return rc;
        k = 1;
    }
    if (graphs && !build_graphs(h)) { h->graph_failed = true; graphs = false; }
    if (graphs) {
        for (; k + GRAPH_UNROLL <= n; k += GRAPH_UNROLL) {
            SW_CUDA(cudaGraphLaunch(h->gexec[0], h->stream));
            h->launches += h->glaunches * GRAPH_UNROLL;
        }
        for (; k < n; ++k) {
            SW_CUDA(cudaGraphLaunch(h->gexec[1], h->stream));
            h->launches += h->glaunches;
        }
    }
    for (; k < n; ++k) {
        int rc = launch_sweep(h, k);
        if (rc) return rc;
    }
    if (potts_folded(h)) {                              // Potts fast path: E of the configuration the call ends with
        if (h->timing) SW_CUDA(cudaEventRecord(h->ev_tail[0], h->stream));
        k_observe_potts_rows<<<grid1((size_t)h->N / 16, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
            h->spins, h->series, h->potts_cnt, h->ctl, 2, h->q, h->L, h->N, h->nb);
        k_moments_last<<<1, 64, 0, h->stream>>>(h->ctl, h->series, h->nb, h->mom, h->N);
        if (h->timing) SW_CUDA(cudaEventRecord(h->ev_tail[1], h->stream));
        h->launches += 2;
    }
    if (scan_nw(h->tile) && !h->q) {                    // a7 of the configuration the call ends with
        if (h->timing) SW_CUDA(cudaEventRecord(h->ev_tail[0], h->stream));
        if (sweeps_on_bits(h))
            k_observe_bits<<<grid1(h->words, 256, h->nb), 256, 0, h->stream>>>(
                h->sbits, h->series, h->ctl, h->L, h->N, h->words, h->nb);
        else
        k_observe_rows<<<grid1(h->words, 256, h->nb), 256, 0, h->stream>>>(
            h->spins, h->series, h->ctl, h->L, h->N, h->words, h->nb);
        k_moments_last<<<1, 64, 0, h->stream>>>(h->ctl, h->series, h->nb, h->mom, h->N);
        if (h->timing) SW_CUDA(cudaEventRecord(h->ev_tail[1], h->stream));
        h->launches += 2;
    }
    if (h->stream != user) {                            // hand the result back to the caller's stream
        SW_CUDA(cudaEventRecord(h->gev[1], h->stream));
        SW_CUDA(cudaStreamWaitEvent(user, h->gev[1], 0));
        h->stream = user;
    }
    SW_CUDA(cudaGetLastError());
    h->t += (uint64_t)n;
    h->last_n = n;
    h->timed_sweeps = h->timing ? std::min<int64_t>(n, MAX_TIMED_SWEEPS) : 0;
    h->have_sweep = true; h->rec_valid = true;
    if (sweeps_on_bits(h)) { h->bits_valid = true; h->i8_valid = false; }
    else                   { h->i8_valid = true; h->bits_valid = false; }
    return SW_OK;
}

const int32_t* sw_labels(sw_handle* h) {
    if (!h) { set_err("sw_labels: null handle"); return nullptr; }
    DevGuard dg(h->dev);
    if (!h->have_sweep) { set_err("sw_labels: no sweep has run yet"); return nullptr; }
    if (!h->labels_flat) {      // the fast path leaves site -> tile root -> cluster root: flatten on demand (a4)
        if (flatten_scan(h, h->lab_tile) != SW_OK || cudaGetLastError() != cudaSuccess) { set_err("sw_labels: flatten launch failed"); return nullptr; }
        h->labels_flat = true;
    }
    return h->label;
}

int sw_bonds(sw_handle* h, const uint32_t** bondE, const uint32_t** bondS) {
    if (!h || !bondE || !bondS) { set_err("sw_bonds: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (!h->have_sweep) { set_err("sw_bonds: no sweep has run yet"); return SW_ESTATE; }
    *bondE = h->bondE; *bondS = h->bondS;
    return SW_OK;
}

const int8_t* sw_spins(sw_handle* h) {
    if (!h) { set_err("sw_spins: null handle"); return nullptr; }
    DevGuard dg(h->dev);
    if (ensure_i8(h) != SW_OK) return nullptr;         // the fused path sweeps on the bit plane: int8 on demand
    return h->spins;
}

int sw_observables(sw_handle* h, sw_obs* out) {
    if (!h || !out) { set_err("sw_observables: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    std::vector<Rec> r(h->nb);
    if (h->rec_valid) {
        const int64_t slot = (h->last_n - 1) % h->ring();
        SW_CUDA(cudaMemcpyAsync(r.data(), h->series + (size_t)slot * h->nb, sizeof(Rec) * h->nb,
                                cudaMemcpyDeviceToHost, h->stream));
    } else {
        { const int rc = ensure_i8(h); if (rc) return rc; }
        SW_CUDA(cudaMemsetAsync(h->rec_now, 0, sizeof(Rec) * h->nb, h->stream));
        if (h->q) {
            k_observe_potts<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
                h->spins, h->rec_now, h->potts_cnt, h->ctl, 0, h->q, h->L, h->N, h->nb);
            k_potts_finish<<<1, 64, 0, h->stream>>>(h->rec_now, h->potts_cnt, h->ctl, 0, h->q, h->N, h->nb);
        } else
        k_observe_generic<<<grid1(h->N, GEN_THREADS, h->nb), GEN_THREADS, 0, h->stream>>>(
            h->spins, h->rec_now, h->ctl, 0, h->L, h->N, h->nb);
        SW_CUDA(cudaGetLastError());
        SW_CUDA(cudaMemcpyAsync(r.data(), h->rec_now, sizeof(Rec) * h->nb, cudaMemcpyDeviceToHost, h->stream));
    }
    SW_CUDA(cudaStreamSynchronize(h->stream));
    for (int b = 0; b < h->nb; ++b) fill_obs(h, r[b], h->t, out + b);
    return SW_OK;
}

int64_t sw_series(sw_handle* h, sw_obs* out, int64_t cap) {
    if (!h || !out || cap < 0) { set_err("sw_series: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (!h->rec_valid) return 0;
    const int64_t kept = std::min(h->last_n, h->series_cap);
    const int64_t give = std::min(kept, cap);
    std::vector<Rec> r((size_t)h->ring() * h->nb);
    SW_CUDA(cudaMemcpyAsync(r.data(), h->series, r.size() * sizeof(Rec), cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    const int64_t first = h->last_n - kept;          // index (within the call) of the oldest retained sweep
    for (int64_t k = 0; k < give; ++k) {
        const int64_t slot = (first + k) % h->ring();
        for (int b = 0; b < h->nb; ++b)
            fill_obs(h, r[(size_t)slot * h->nb + b], h->t - (uint64_t)h->last_n + (uint64_t)(first + k) + 1,
                     out + (size_t)k * h->nb + b);
    }
    return kept;
}

int sw_moments(sw_handle* h, sw_mom* out) {
    if (!h || !out) { set_err("sw_moments: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    std::vector<Mom> m(h->nb);
    SW_CUDA(cudaMemcpyAsync(m.data(), h->mom, sizeof(Mom) * h->nb, cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    for (int b = 0; b < h->nb; ++b) {
        sw_mom* o = out + b;
        std::memset(o, 0, sizeof *o);
        o->n = m[b].n;
        if (m[b].n == 0) continue;
        const double fn = (double)m[b].n, fN = (double)h->N, T = h->hT[b];
        const double e = m[b].s_e / fn, e2 = m[b].s_e2 / fn, am = m[b].s_am / fn, m2 = m[b].s_m2 / fn, m4 = m[b].s_m4 / fn;
        o->e_mean = e; o->e2_mean = e2; o->absm_mean = am; o->m2_mean = m2; o->m4_mean = m4;
        o->specific_heat = fN * (e2 - e * e) / (T * T);
        o->susceptibility = fN * (m2 - am * am) / T;
        o->binder = m2 > 0.0 ? 1.0 - m4 / (3.0 * (m2 * m2)) : 0.0;
    }
    return SW_OK;
}

int sw_moments_reset(sw_handle* h) {
    if (!h) { set_err("sw_moments_reset: null handle"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    SW_CUDA(cudaMemsetAsync(h->mom, 0, (size_t)h->nb * sizeof(Mom), h->stream));
    return SW_OK;
}

namespace {
// the retained sweeps of the last sw_sweep call, as the kernels of sw_series.cuh see them
bool series_view(const sw_handle* h, int32_t which, SeriesView* v) {
    if (!h->rec_valid || h->last_n <= 0) return false;
    const int64_t kept = std::min(h->last_n, h->series_cap);
    v->rec = h->series; v->first = h->last_n - kept; v->ring = h->ring(); v->n = kept; v->nb = h->nb; v->which = which;
    return true;
}
struct DevBuf {                 // scratch of one analysis call, freed on every exit
    void* p = nullptr;
    ~DevBuf() { if (p) cudaFree(p); }
    cudaError_t alloc(size_t bytes) { return cudaMalloc(&p, bytes ? bytes : 1); }
};
} // namespace

int sw_bins(sw_handle* h, int32_t which, int64_t bin_len, double* bin_means, int64_t cap, sw_binstat* out) {
    if (!h || !out || (which != 0 && which != 1) || bin_len < 1 || cap < 0) { set_err("sw_bins: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    SeriesView v;
    if (!series_view(h, which, &v)) { set_err("sw_bins: no series (no sw_sweep since the last state change)"); return SW_ESTATE; }
    const long long nbins = v.n / bin_len;
    DevBuf bins, stat;
    if (bins.alloc((size_t)h->nb * nbins * sizeof(double)) != cudaSuccess || stat.alloc((size_t)h->nb * sizeof(BinStat)) != cudaSuccess) {
        (void)cudaGetLastError(); set_err("sw_bins: cudaMalloc failed"); return SW_ENOMEM;
    }
    if (nbins > 0)
        k_series_bins<<<grid1((size_t)nbins, 256, h->nb), 256, 0, h->stream>>>(v, (double*)bins.p, bin_len, nbins, h->N);
    k_series_binerr<<<(h->nb + 63) / 64, 64, 0, h->stream>>>((const double*)bins.p, (BinStat*)stat.p, nbins, h->nb);
    SW_CUDA(cudaGetLastError());
    std::vector<BinStat> hs(h->nb);
    SW_CUDA(cudaMemcpyAsync(hs.data(), stat.p, sizeof(BinStat) * h->nb, cudaMemcpyDeviceToHost, h->stream));
    std::vector<double> hb;
    if (bin_means && nbins > 0) {
        hb.resize((size_t)h->nb * nbins);
        SW_CUDA(cudaMemcpyAsync(hb.data(), bins.p, hb.size() * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    }
    SW_CUDA(cudaStreamSynchronize(h->stream));
    const int64_t give = std::min<int64_t>(nbins, cap);
    for (int b = 0; b < h->nb; ++b) {
        out[b].n_bins = hs[b].n_bins; out[b].mean = hs[b].mean; out[b].err = hs[b].err;
        if (bin_means) for (int64_t j = 0; j < give; ++j) bin_means[(size_t)b * cap + j] = hb[(size_t)b * nbins + j];
    }
    return SW_OK;
}

int sw_autocorr(sw_handle* h, int32_t which, int64_t tmax, double c, double* rho, sw_taustat* out) {
    if (!h || !out || (which != 0 && which != 1) || tmax < 0 || !(c > 0.0)) { set_err("sw_autocorr: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    SeriesView v;
    if (!series_view(h, which, &v)) { set_err("sw_autocorr: no series (no sw_sweep since the last state change)"); return SW_ESTATE; }
    const long long tm = std::min<long long>(tmax, v.n - 1);            // (rho is still written with stride tmax + 1)
    DevBuf x, xbar, C, R, stat;
    if (x.alloc((size_t)h->nb * v.n * sizeof(double)) != cudaSuccess || xbar.alloc((size_t)h->nb * sizeof(double)) != cudaSuccess ||
        C.alloc((size_t)h->nb * (tm + 1) * sizeof(double)) != cudaSuccess || R.alloc((size_t)h->nb * (tm + 1) * sizeof(double)) != cudaSuccess ||
        stat.alloc((size_t)h->nb * sizeof(TauStat)) != cudaSuccess) {
        (void)cudaGetLastError(); set_err("sw_autocorr: cudaMalloc failed"); return SW_ENOMEM;
    }
    k_series_x<<<grid1((size_t)v.n, 256, h->nb), 256, 0, h->stream>>>(v, (double*)x.p, h->N);
    k_series_mean<<<(h->nb + 63) / 64, 64, 0, h->stream>>>((const double*)x.p, (double*)xbar.p, v.n, h->nb);
    k_series_autocov<<<grid1((size_t)(tm + 1), 128, h->nb), 128, 0, h->stream>>>((const double*)x.p, (const double*)xbar.p, (double*)C.p, v.n, tm);
    k_series_tau<<<(h->nb + 63) / 64, 64, 0, h->stream>>>((const double*)C.p, (double*)R.p, (TauStat*)stat.p, tm, c, h->nb);
    SW_CUDA(cudaGetLastError());
    std::vector<TauStat> hs(h->nb);
    SW_CUDA(cudaMemcpyAsync(hs.data(), stat.p, sizeof(TauStat) * h->nb, cudaMemcpyDeviceToHost, h->stream));
    std::vector<double> hr;
    if (rho) {
        hr.resize((size_t)h->nb * (tm + 1));
        SW_CUDA(cudaMemcpyAsync(hr.data(), R.p, hr.size() * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    }
    SW_CUDA(cudaStreamSynchronize(h->stream));
    for (int b = 0; b < h->nb; ++b) {
        out[b].tau_int = hs[b].tau_int; out[b].window = hs[b].window; out[b].tmax = hs[b].tmax; out[b].c0 = hs[b].c0;
        if (rho) for (int64_t t = 0; t <= tmax; ++t) rho[(size_t)b * (tmax + 1) + t] = t <= tm ? hr[(size_t)b * (tm + 1) + t] : 0.0;
    }
    return SW_OK;
}

int sw_set_series_capacity(sw_handle* h, int64_t sweeps) {
    if (!h || sweeps < 1 || sweeps > (1ll << 26)) { set_err("sw_set_series_capacity: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    SW_CUDA(cudaStreamSynchronize(h->stream));
    Rec* p = nullptr;
    cudaError_t e = cudaMalloc((void**)&p, (size_t)(sweeps + 1) * h->nb * sizeof(Rec));
    if (e != cudaSuccess) { (void)cudaGetLastError(); set_err("sw_set_series_capacity: cudaMalloc failed"); return SW_ENOMEM; }
    if (h->series_owned) cudaFree(h->series_owned);
    h->series_owned = p; h->series = p; h->series_cap = sweeps;
    h->rec_valid = false;
    return SW_OK;
}

int sw_set_spins(sw_handle* h, const int8_t* spins, int is_host) {
    if (!h || !spins) { set_err("sw_set_spins: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    SW_CUDA(cudaMemcpyAsync(h->spins, spins, (size_t)h->nb * h->N,
                            is_host ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice, h->stream));
    if (is_host) SW_CUDA(cudaStreamSynchronize(h->stream));
    h->i8_valid = true; h->bits_valid = false;
    h->have_sweep = false; h->rec_valid = false;
    return SW_OK;
}

int sw_set_cold(sw_handle* h) {
    if (!h) { set_err("sw_set_cold: null handle"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    const size_t n = (size_t)h->nb * h->N;
    k_fill_i8<<<(unsigned)((n + GEN_THREADS - 1) / GEN_THREADS), GEN_THREADS, 0, h->stream>>>(h->spins, n, (int8_t)(h->q ? 0 : 1));
    SW_CUDA(cudaGetLastError());
    h->i8_valid = true; h->bits_valid = false;
    h->have_sweep = false; h->rec_valid = false;
    return SW_OK;
}

// bit-packed host interface: straight into / out of the bit plane the fused path sweeps on
int sw_set_spins_bits(sw_handle* h, const uint32_t* bits_host) {
    if (!h || !bits_host) { set_err("sw_set_spins_bits: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (h->q) { set_err("sw_set_spins_bits: Ising handles only (a Potts colour does not fit a bit)"); return SW_ESTATE; }
    SW_CUDA(cudaMemcpyAsync(h->sbits, bits_host, (size_t)h->nb * h->words * 4, cudaMemcpyHostToDevice, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));          // the caller may reuse its buffer
    h->bits_valid = true; h->i8_valid = false;
    h->have_sweep = false; h->rec_valid = false;
    return SW_OK;
}

int sw_get_spins_bits(sw_handle* h, uint32_t* out_host) {
    if (!h || !out_host) { set_err("sw_get_spins_bits: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (h->q) { set_err("sw_get_spins_bits: Ising handles only"); return SW_ESTATE; }
    { const int rc = ensure_bits(h); if (rc) return rc; }
    SW_CUDA(cudaMemcpyAsync(out_host, h->sbits, (size_t)h->nb * h->words * 4, cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    return SW_OK;
}

int sw_get_spins(sw_handle* h, int8_t* out_host) {
    if (!h || !out_host) { set_err("sw_get_spins: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    { const int rc = ensure_i8(h); if (rc) return rc; }
    SW_CUDA(cudaMemcpyAsync(out_host, h->spins, (size_t)h->nb * h->N, cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    return SW_OK;
}

int sw_get_labels(sw_handle* h, int32_t* out_host) {
    if (!h || !out_host) { set_err("sw_get_labels: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    const int32_t* l = sw_labels(h);
    if (!l) return SW_ESTATE;
    SW_CUDA(cudaMemcpyAsync(out_host, l, (size_t)h->nb * h->N * 4, cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    return SW_OK;
}

int sw_set_sweep_index(sw_handle* h, uint64_t t) {
    if (!h) { set_err("sw_set_sweep_index: null handle"); return SW_EINVAL; }
    h->t = t;                   // written to the device at the start of the next sw_sweep
    return SW_OK;
}
uint64_t sw_sweep_index(const sw_handle* h) { return h ? h->t : 0; }

int sw_set_stream(sw_handle* h, void* cuda_stream) {
    if (!h) { set_err("sw_set_stream: null handle"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    SW_CUDA(cudaStreamSynchronize(h->stream));
    h->stream = (cudaStream_t)cuda_stream;
    return SW_OK;
}

int sw_set_stage_timing(sw_handle* h, int on) {
    if (!h) { set_err("sw_set_stage_timing: null handle"); return SW_EINVAL; }
    h->timing = on != 0;
    if (!h->timing) h->timed_sweeps = 0;
    return SW_OK;
}

int sw_kernel_ms(sw_handle* h, float* out, int32_t cap) {
    if (!h || !out || cap < 0) { set_err("sw_kernel_ms: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    for (int i = 0; i < cap; ++i) out[i] = 0.f;
    if (h->timed_sweeps == 0) { set_err("sw_kernel_ms: the last sw_sweep ran without stage timing"); return SW_ESTATE; }
    SW_CUDA(cudaStreamSynchronize(h->stream));
    const int ns = (int)h->ev_seq.size();            // launches per sweep + the closing mark
    for (int64_t k = 0; k < h->timed_sweeps; ++k)
        for (int j = 0; j + 1 < ns; ++j) {
            float ms = 0.f;
            SW_CUDA(cudaEventElapsedTime(&ms, h->ev[(size_t)k * EV_PER_SWEEP + j], h->ev[(size_t)k * EV_PER_SWEEP + j + 1]));
            if (h->ev_seq[j] < cap) out[h->ev_seq[j]] += ms;
        }
    if (scan_nw(h->tile) && (!h->q || potts_folded(h)) && K_ENERGY < cap) {  // the trailing observables pass of the call
        float ms = 0.f;
        SW_CUDA(cudaEventElapsedTime(&ms, h->ev_tail[0], h->ev_tail[1]));
        out[K_ENERGY] += ms;
    }
    return K_COUNT;
}

int64_t sw_sweep_ms(sw_handle* h, float* out, int64_t cap) {
    if (!h || !out || cap < 0) { set_err("sw_sweep_ms: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (h->timed_sweeps == 0) { set_err("sw_sweep_ms: the last sw_sweep ran without stage timing"); return SW_ESTATE; }
    SW_CUDA(cudaStreamSynchronize(h->stream));
    const int ns = (int)h->ev_seq.size();            // marks per sweep, the closing one included
    const int64_t n = std::min<int64_t>(h->timed_sweeps, cap);
    for (int64_t k = 0; k < n; ++k)
        SW_CUDA(cudaEventElapsedTime(out + k, h->ev[(size_t)k * EV_PER_SWEEP], h->ev[(size_t)k * EV_PER_SWEEP + ns - 1]));
    return h->timed_sweeps;
}

const char* sw_kernel_name(int32_t i) { return (i >= 0 && i < K_COUNT) ? KERNEL_NAMES[i] : ""; }

int sw_stage_ms(sw_handle* h, float out[4]) {
    if (!h || !out) { set_err("sw_stage_ms: null argument"); return SW_EINVAL; }
    out[0] = out[1] = out[2] = out[3] = 0.f;
    float k[K_COUNT];
    const int rc = sw_kernel_ms(h, k, K_COUNT);
    if (rc < 0) return rc;
    for (int i = 0; i < K_COUNT; ++i) out[KERNEL_STAGE[i]] += k[i];
    return SW_OK;
}

int sw_set_path(sw_handle* h, int path) {
    if (!h || !valid_path(path)) { set_err("sw_set_path: path %d is not one of 0 (fast path), 1 (generic kernels), 6 (unfused stages), 11 (label equivalence)", path); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (h->q && path == 6) { set_err("sw_set_path: a Potts handle runs on paths 0 (128 x 64 tiles when L allows, else generic), 1 (generic) and 11"); return SW_EINVAL; }
    h->path = path;
    h->eq_ran = false;
    // (16-bit roots of a sweep on the previous path stay valid: sw_labels flattens them with the tile shape that wrote them)
    h->tile = h->q ? potts_tile(h->L, path) : pick_tile(h->L, path);
    return SW_OK;
}

int sw_set_graphs(sw_handle* h, int on) {
    if (!h) { set_err("sw_set_graphs: null handle"); return SW_EINVAL; }
    h->use_graphs = on != 0;
    return SW_OK;
}

int sw_set_tma(sw_handle* h, int on) {
    if (!h) { set_err("sw_set_tma: null handle"); return SW_EINVAL; }
    h->use_tma = on != 0;
    h->gkey_path = -1;                              // (the captured sweep holds the other kernel: capture again)
    return SW_OK;
}

int sw_set_cluster(sw_handle* h, int on) {
    if (!h) { set_err("sw_set_cluster: null handle"); return SW_EINVAL; }
    h->use_cluster = on != 0;
    return SW_OK;
}

int sw_set_eager_labels(sw_handle* h, int on) {
    if (!h) { set_err("sw_set_eager_labels: null handle"); return SW_EINVAL; }
    h->eager_labels = on != 0;
    return SW_OK;
}

int64_t sw_last_launch_count(const sw_handle* h) { return h ? h->launches : 0; }
uint32_t sw_threshold(const sw_handle* h, int32_t b) { return (h && b >= 0 && b < h->nb) ? h->hlat[b].thr : 0u; }
int32_t sw_L(const sw_handle* h) { return h ? h->L : 0; }
int32_t sw_batch(const sw_handle* h) { return h ? h->nb : 0; }

int sw_test_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int64_t n) {
    if (!ctr || !key || !out || n < 0) { set_err("sw_test_philox: invalid argument"); return SW_EINVAL; }
    if (n == 0) return SW_OK;
    struct Bufs {                                       // freed on every exit
        uint32_t *dc = nullptr, *dk = nullptr, *dout = nullptr;
        ~Bufs() { cudaFree(dc); cudaFree(dk); cudaFree(dout); }
    } b;
    SW_CUDA(cudaMalloc((void**)&b.dc, (size_t)n * 16));
    SW_CUDA(cudaMalloc((void**)&b.dk, (size_t)n * 8));
    SW_CUDA(cudaMalloc((void**)&b.dout, (size_t)n * 16));
    SW_CUDA(cudaMemcpy(b.dc, ctr, (size_t)n * 16, cudaMemcpyHostToDevice));
    SW_CUDA(cudaMemcpy(b.dk, key, (size_t)n * 8, cudaMemcpyHostToDevice));
    k_test_philox<<<(unsigned)((n + 255) / 256), 256>>>(b.dc, b.dk, b.dout, n);
    SW_CUDA(cudaGetLastError());
    SW_CUDA(cudaMemcpy(out, b.dout, (size_t)n * 16, cudaMemcpyDeviceToHost));
    return SW_OK;
}

int sw_label_passes(sw_handle* h, int32_t* passes) {
    if (!h || !passes) { set_err("sw_label_passes: null argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    if (h->path != 11 || !h->eq_ran) { set_err("sw_label_passes: no labelling has run on path 11 yet"); return SW_ESTATE; }
    int tail[2] = { 0, 0 };
    SW_CUDA(cudaMemcpyAsync(&tail[1], h->eq_flags + EQ_MAX_PASSES, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    if (tail[1] < 1 || tail[1] > EQ_MAX_PASSES) { set_err("sw_label_passes: bad pass count %d", tail[1]); return SW_ESTATE; }
    SW_CUDA(cudaMemcpyAsync(&tail[0], h->eq_flags + tail[1] - 1, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    if (tail[0]) { set_err("sw_label_passes: no convergence within %d passes", EQ_MAX_PASSES); return SW_ESTATE; }
    *passes = tail[1];
    return SW_OK;
}

int sw_test_philox_ceiling(int64_t sites, int32_t reps, float* ms_out) {
    if (sites < 32 || sites > (1ll << 40) || reps < 1 || !ms_out) { set_err("sw_test_philox_ceiling: invalid argument"); return SW_EINVAL; }
    const long long words = sites / 32;
    const long long blocks = (words + GEN_THREADS - 1) / GEN_THREADS;
    if (blocks > 0x7fffffffll) { set_err("sw_test_philox_ceiling: too many sites"); return SW_EINVAL; }
    uint32_t* sink = nullptr;
    SW_CUDA(cudaMalloc((void**)&sink, (size_t)(blocks * GEN_THREADS / 32) * 4));
    cudaEvent_t e0, e1;
    SW_CUDA(cudaEventCreate(&e0)); SW_CUDA(cudaEventCreate(&e1));
    for (int i = 0; i < 3; ++i) k_philox_only<<<(unsigned)blocks, GEN_THREADS>>>(sink, 6u, 0u, (uint32_t)i, words);
    SW_CUDA(cudaEventRecord(e0));
    for (int i = 0; i < reps; ++i) k_philox_only<<<(unsigned)blocks, GEN_THREADS>>>(sink, 6u, 0u, 100u + (uint32_t)i, words);
    SW_CUDA(cudaEventRecord(e1));
    SW_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f;
    SW_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    *ms_out = ms / (float)reps;
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(sink);
    SW_CUDA(cudaGetLastError());
    return SW_OK;
}

int sw_test_label(sw_handle* h, const uint32_t* bondE, const uint32_t* bondS, int32_t* labels_out) {
    if (!h || !bondE || !bondS || !labels_out || h->nb != 1) { set_err("sw_test_label: invalid argument"); return SW_EINVAL; }
    DevGuard dg(h->dev);
    SW_CUDA(cudaMemcpyAsync(h->bondE, bondE, (size_t)h->words * 4, cudaMemcpyHostToDevice, h->stream));
    SW_CUDA(cudaMemcpyAsync(h->bondS, bondS, (size_t)h->words * 4, cudaMemcpyHostToDevice, h->stream));
    SW_CUDA(cudaMemsetAsync(h->series, 0, sizeof(Rec), h->stream));
    k_set_ctl<<<1, 1, 0, h->stream>>>(h->ctl, (unsigned long long)h->t, 0u, (uint32_t)h->ring());
    int rc = launch_label(h);
    if (rc) return rc;
    SW_CUDA(cudaGetLastError());
    SW_CUDA(cudaMemcpyAsync(labels_out, h->label, (size_t)h->N * 4, cudaMemcpyDeviceToHost, h->stream));
    SW_CUDA(cudaStreamSynchronize(h->stream));
    h->have_sweep = false; h->rec_valid = false;
    return SW_OK;
}

int sw_bins_noalloc(sw_handle* h, int32_t which, int64_t bin_len, sw_binstat* out_dev) {
    if (!h || !out_dev || (which != 0 && which != 1) || bin_len < 1) { set_err("sw_bins_noalloc: invalid argument"); return SW_EINVAL; }
    static_assert(sizeof(BinStat) == sizeof(sw_binstat), "the kernel's record is the header's");
    DevGuard dg(h->dev);
    SeriesView v;
    if (!series_view(h, which, &v)) { set_err("sw_bins_noalloc: no series (no sw_sweep since the last state change)"); return SW_ESTATE; }
    const long long nbins = v.n / bin_len;
    if ((long long)h->nb * nbins > (long long)SW_BINS_NOALLOC_MAX) {
        set_err("sw_bins_noalloc: %d lattices x %lld bins = %lld bin means exceed the static scratch of SW_BINS_NOALLOC_MAX = %d; "
                "use a longer bin_len, or sw_bins", h->nb, nbins, (long long)h->nb * nbins, (int)SW_BINS_NOALLOC_MAX);
        return SW_EINVAL;
    }
    double* scratch = nullptr;
    { const int rc = bins_scratch(h->dev, &scratch); if (rc) return rc; }
    // (nothing in the scratch has to start at zero: k_series_bins writes every entry k_series_binerr reads)
    if (nbins > 0)
        k_series_bins<<<grid1((size_t)nbins, 256, h->nb), 256, 0, h->stream>>>(v, scratch, bin_len, nbins, h->N);
    k_series_binerr<<<(h->nb + 63) / 64, 64, 0, h->stream>>>(scratch, reinterpret_cast<BinStat*>(out_dev), nbins, h->nb);
    SW_CUDA(cudaGetLastError());
    return SW_OK;
}

} // extern "C"
