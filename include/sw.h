/*
 * sw.h -- C ABI of the B200 Swendsen-Wang library (libsw_b200.so).
 *
 * One thing is built here: the full Swendsen-Wang sweep on the 2D square-lattice Ising model with
 * periodic boundaries (arxiv 2302.14720, Protzman & Giedt; "five steps ... of which
 * three require computation"), as hand-written CUDA for sm_100a.  There is no CPU fallback: every
 * entry point that needs the GPU fails with SW_ECUDA when no usable device is present.
 *
 * Conventions:
 *   site i = y*L + x, 0 <= x,y < L; East(i) = y*L + (x+1) mod L; South(i) = ((y+1) mod L)*L + x;
 *   N = L*L; spins are int8 +1 / -1; J = 1, k_B = 1;
 *   bond probability  p = 1 - exp(-2/T)  -- the paper prints p = 1 - exp(-1/k_B T)
 *   in its own units; with H = -sum s_i s_j and the critical point its figures show
 *   near k_B T ~ 2.25 this is 1 - exp(-2J/T) with J = 1.  T_c = 2/ln(1+sqrt 2).
 *
 * One sweep with sweep index t (the k-th sweep since creation uses t = k, from 0):
 *   1 bonds   (section 2.1)  w = Philox4x32-10(ctr = (i>>1, t_lo, t_hi, 1), key = seed);
 *             bondE[i] = spins[i]==spins[East(i)]  && w[2*(i&1)]   < thr
 *             bondS[i] = spins[i]==spins[South(i)] && w[2*(i&1)+1] < thr,  thr = floor(p * 2^32) (<= 2^32-1)
 *   2 labels  (section 2.3)  label[i] = minimum site index of i's connected component
 *             of the bond graph ("lowest value label", labels "incrementing from zero")
 *   3 assign  (section 2.4)     spins[i] = bit(label[i]) ? +1 : -1, where
 *             bit(r) = (Philox(ctr = (r>>7, t_lo, t_hi, 2), key = seed)[(r>>5)&3] >> (r&31)) & 1
 *   observables (section 2.5)   E = -sum_i s_i (s_East(i) + s_South(i)), M = sum_i s_i.
 * The random start is spins[i] = bit_INIT(i) ? +1 : -1 with tag 0 and t = 0.
 *
 * Memory: the handle owns its device buffers (or carves them from a caller-supplied workspace,
 * sw_create_in).  Pointers returned by sw_spins / sw_labels / sw_bonds are DEVICE pointers,
 * borrowed: valid until the next sw_sweep, sw_set_* or sw_destroy on that handle.  All `out`
 * arguments are HOST memory owned by the caller unless stated.
 *
 * Streams: all work of a handle is issued on one CUDA stream (default: the legacy default stream;
 * sw_set_stream installs another, e.g. torch.cuda.current_stream().cuda_stream).  sw_sweep is
 * asynchronous; sw_observables / sw_series / sw_stage_ms / sw_get_spins synchronise that stream.
 *
 * Errors: no exceptions, no abort.  int functions return SW_OK (0) or a negative code; pointer
 * functions return NULL; sw_last_error() gives the text for the calling thread.
 */
#ifndef SW_B200_H
#define SW_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SW_OK       0
#define SW_EINVAL  -1   /* L < 2, L > 32768, T <= 0 or not finite, n < 0, nb < 1, null pointer, bad size */
#define SW_ENOMEM  -2   /* host or device allocation failed / workspace too small */
#define SW_ECUDA   -3   /* CUDA error; text in sw_last_error() */
#define SW_ESTATE  -4   /* labels / bonds asked for before the first sweep, etc. */

#define SW_MAX_L   32768      /* int32 labels: N <= 2^30 */

typedef struct sw_handle sw_handle;   /* opaque */

/* Observables of one lattice.  E and M are of the CURRENT spins; n_clusters / largest_cluster are of
 * the LAST sweep's bond graph (0 before any sweep); `sweep` = number of sweeps completed.
 * e_per_site = energy / N, abs_m_per_site = |magnetisation| / N, in double. */
typedef struct {
    int64_t  energy;
    int64_t  magnetisation;
    int64_t  n_clusters;
    int64_t  largest_cluster;
    uint64_t sweep;
    double   e_per_site;
    double   abs_m_per_site;
} sw_obs;

/* ---- creation (Fig. 1: the first configuration assigns a random spin to each site) ---- */

/* One L x L lattice at temperature T, random start from `seed` (Philox tag 0).  NULL on error. */
sw_handle* sw_create(int32_t L, double T, uint64_t seed);

/* nb independent L x L lattices (BASELINE config 5: temperature scan), lattice b at T[b] with seed[b];
 * every stage is ONE launch for the whole batch.  T, seed: HOST arrays of nb entries. */
sw_handle* sw_create_batch(int32_t L, int32_t nb, const double* T, const uint64_t* seed);

/* Bytes of device workspace a handle for (L, nb) needs; 0 on invalid arguments. */
uint64_t   sw_workspace_bytes(int32_t L, int32_t nb);

/* As sw_create_batch, but every device buffer is carved from `workspace` (DEVICE pointer, 256-byte
 * aligned, >= sw_workspace_bytes(L, nb) bytes, owned by the caller and kept alive until sw_destroy).
 * This is how the Python binding lets PyTorch own the memory. */
sw_handle* sw_create_in(void* workspace, uint64_t workspace_bytes,
                        int32_t L, int32_t nb, const double* T, const uint64_t* seed);

void       sw_destroy(sw_handle* h);                       /* NULL is a no-op */

/* ---- q-state Potts model on the same sweep ----
 * PAPER.md:33 ("The approach can be generalized to other discrete spin systems").  The paper gives no
 * formulas; the textbook readings are taken: colours 0 .. q-1 in the int8 plane sw_spins returns,
 * H = -sum_<ij> delta(c_i, c_j) with J = 1, a bond between EQUAL colours with p = 1 - exp(-1/T) (drawn exactly as for
 * the Ising model: same Philox words, same East / South ownership), the same labelling, and every cluster assigned the
 * colour floor(word * q / 2^32), word = 32-bit field `label` of the TAG_FLIP stream of the sweep (Philox call
 * label >> 2, word label & 3); random start: the same with TAG_INIT, t = 0, field = site index.
 * q in 2 .. 127.  A Potts handle answers every call of this header; differences: sw_obs.energy = -#(equal East /
 * South pairs), sw_obs.magnetisation = q * max_c n_c - N (n_c = sites of colour c), abs_m_per_site =
 * magnetisation / N; sw_set_cold sets colour 0; sw_set_spins takes colours; paths 0 (128 x 64 tiles when L is a
 * multiple of 128, else the generic kernels), 1 (generic kernels) and 11 only.  sw_create_potts allocates its own workspace; sw_create_potts_in takes one of sw_workspace_bytes(L, nb)
 * bytes like sw_create_in (plus nb*q*4 bytes the library allocates itself for the colour counts).
 * NULL + error text on invalid arguments (q outside 2 .. 127, and as for sw_create). */
sw_handle* sw_create_potts(int32_t L, int32_t q, double T, uint64_t seed);
sw_handle* sw_create_potts_in(void* workspace, uint64_t workspace_bytes, int32_t L, int32_t q, int32_t nb,
                              const double* T, const uint64_t* seed);
int32_t    sw_q(const sw_handle* h);                       /* 0 for an Ising handle */

/* ---- the hot path ---- */

/* n >= 0 full sweeps (bonds -> labels -> assignment -> observables) on the handle's stream;
 * asynchronous.  PAPER.md:33 (the five-step iteration). */
int        sw_sweep(sw_handle* h, int64_t n);

/* DEVICE pointer to nb*N int32: flat minimum-index labels of the last sweep, each lattice indexed
 * within itself.  Flattens lazily (one extra kernel on the handle's stream) if the last sweep left the
 * two-level forest site -> tile root -> cluster root; sw_set_eager_labels(h, 1) stores them every sweep instead.  NULL + SW_ESTATE text
 * before the first sweep.  PAPER.md:51. */
const int32_t* sw_labels(sw_handle* h);

/* Synchronises; fills out[0..nb-1] (HOST).  PAPER.md:63. */
int        sw_observables(sw_handle* h, sw_obs* out);

/* ---- extras the configurations and the parity tests need ---- */

const int8_t* sw_spins(sw_handle* h);                      /* DEVICE ptr, nb*N int8 (+1/-1) */

/* DEVICE pointers to the canonical bond bit-planes of the last sweep: bit (i&31) of uint32 word
 * (i>>5), i the site index; lattice b starts at word b*words_per_lattice, words_per_lattice =
 * ceil(N/32).  SW_ESTATE before the first sweep.  PAPER.md:39, Fig. 2. */
int        sw_bonds(sw_handle* h, const uint32_t** bondE, const uint32_t** bondS);
int        sw_set_eager_labels(sw_handle* h, int on);       /* default 0 */
/* Default 1: on the fast path, sw_sweep(h, n >= 4) replays CUDA graphs of the steady sweep (the sweep index lives
 * on the device, so every sweep but the first of a call launches the same kernels with the same arguments)
 * on an internal stream ordered after / before the handle's stream by events.  0: plain launches.  Results are
 * identical either way; graphs remove most of the launch overhead that dominates small lattices. */
int        sw_set_graphs(sw_handle* h, int on);

/* Replace the spins (cold start, injected states).  `spins`: nb*N int8 of +1/-1, on the device
 * (is_host = 0) or on the host (is_host = 1).  Values are not validated. */
int        sw_set_spins(sw_handle* h, const int8_t* spins, int is_host);
int        sw_set_cold(sw_handle* h);                      /* all +1 (BASELINE config 3) */
int        sw_get_spins(sw_handle* h, int8_t* out_host);   /* synchronising copy, nb*N bytes */
/* The same two transfers with BIT-PACKED host buffers (north_star: "int8 or bit-packed spins"): nb * ceil(N/32)
 * uint32 words, lattice b at word b*ceil(N/32), site i of a lattice in bit (i & 31) of its word (i >> 5), bit 1 = spin +1,
 * padding bits of the last word ignored / zero.  1/8 of the bytes of the int8 plane cross PCIe; packing and unpacking
 * run on the device.  Both synchronise.  Ising handles only (SW_ESTATE for a Potts handle).  PAPER.md:71 (Fig. 1). */
int        sw_set_spins_bits(sw_handle* h, const uint32_t* bits_host);
int        sw_get_spins_bits(sw_handle* h, uint32_t* out_host);
int        sw_get_labels(sw_handle* h, int32_t* out_host); /* synchronising copy, nb*N int32 */

/* Next sweep uses sweep index t (checkpoint / resume, one-step parity at large L). */
int        sw_set_sweep_index(sw_handle* h, uint64_t t);
uint64_t   sw_sweep_index(const sw_handle* h);

int        sw_set_stream(sw_handle* h, void* cuda_stream); /* a cudaStream_t; NULL = default stream */

/* Per-sweep history of the LAST sw_sweep call, oldest first: record (k*nb + b) is lattice b after the
 * k-th retained sweep.  `cap` counts SWEEPS: `out` (HOST) must hold cap * nb records, and min(retained, cap) * nb
 * are written; returns the number of sweeps retained (<= the series capacity, default 4096 sweeps, see
 * sw_set_series_capacity) or a negative code. */
int64_t    sw_series(sw_handle* h, sw_obs* out, int64_t cap);
int        sw_set_series_capacity(sw_handle* h, int64_t sweeps);

/* Moments of the per-sweep observables over every sweep since creation or the last sw_moments_reset
 * (the paper validates on E, the specific heat and M against T: PAPER.md:113-123,
 * section 4, Figs. 5-7).  Per configuration e = E/N, a = |M|/N; summed on the device one
 * sweep at a time in double, in sweep order, unfused.  e_mean = <e>, e2_mean = <e^2>, absm_mean = <|m|>,
 * m2_mean = <m^2>, m4_mean = <m^4>; specific_heat = N (<e^2> - <e>^2) / T^2; susceptibility =
 * N (<m^2> - <|m|>^2) / T; binder = 1 - <m^4> / (3 <m^2>^2).  n = 0 (all fields 0) before any sweep.
 * sw_moments synchronises and fills out[0..nb-1] (HOST); discard thermalisation with sw_moments_reset
 * (asynchronous on the handle's stream).  Sweeps are counted whatever the start state was set to. */
typedef struct {
    int64_t n;
    double  e_mean, e2_mean, absm_mean, m2_mean, m4_mean;
    double  specific_heat, susceptibility, binder;
} sw_mom;
int        sw_moments(sw_handle* h, sw_mom* out);
int        sw_moments_reset(sw_handle* h);

/* Error analysis of the per-sweep series the LAST sw_sweep call left on the device (the sweeps sw_series returns),
 * binning and the integrated autocorrelation time -- the quantity the paper's motivation is
 * about (tau ~ |g - g*|^(-z) for local updates; cluster updates keep it small; section 4).
 * The paper gives no formulas; the textbook definitions are taken:
 *   series x_k = E_k / N (which = 0) or |M_k| / N (which = 1), retained sweeps in order, n of them;
 *   sw_bins: n_bins = floor(n / bin_len) bins of consecutive sweeps (a remainder at the end is dropped); a bin mean is
 *     the exact integer sum of its E_k (or |M_k|) divided once by bin_len * N; mean = mean of the bin means;
 *     err = sqrt( sum (b_j - mean)^2 / (n_bins (n_bins - 1)) ), 0 with fewer than two bins;
 *   sw_autocorr: C(t) = (1/(n-t)) sum_k (x_k - xbar)(x_{k+t} - xbar), rho(t) = C(t) / C(0), t = 0 .. min(tmax, n-1);
 *     tau_int = 1/2 + sum_{t=1}^{W} rho(t) with the self-consistent window W = smallest W >= 1 with W >= c * tau(W)
 *     (c = 6 is customary), else the last lag; a constant series has rho = 0, tau_int = 1/2, window = 0.
 * All sums run on the device in index order in double with unfused operations.  Both calls synchronise.
 * out[0..nb-1] (HOST).  bin_means: NULL or HOST [nb][cap] (the first min(n_bins, cap) bin means of each lattice);
 * rho: NULL or HOST [nb][tmax + 1] (0 beyond lag n - 1); sw_taustat.tmax = the last lag computed, c0 = C(0).
 * SW_ESTATE when there is no series (no sweep since the state was set), SW_EINVAL on bad arguments. */
typedef struct { int64_t n_bins; double mean, err; } sw_binstat;
typedef struct { double tau_int; int64_t window, tmax; double c0; } sw_taustat;
int        sw_bins(sw_handle* h, int32_t which, int64_t bin_len, double* bin_means, int64_t cap, sw_binstat* out);
int        sw_autocorr(sw_handle* h, int32_t which, int64_t tmax, double c, double* rho, sw_taustat* out);

/* sw_bins for callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid
 * cudaMalloc): the same binning, the same kernels, no cudaMalloc / cudaFree / host copy / synchronisation.  The bin means
 * -- scratch between the two kernels -- live in a static device array of SW_BINS_NOALLOC_MAX doubles (512 KiB that every
 * GPU which loads the library holds until the process exits), so nb * floor(n / bin_len) may not exceed
 * SW_BINS_NOALLOC_MAX: beyond it the call returns SW_EINVAL and says so in sw_last_error (take a longer bin_len, or sw_bins).
 * out_dev: DEVICE, nb records (n_bins, mean, err), written asynchronously on the handle's stream -- the caller orders its
 * reads after it on that stream.  All calls on a GPU share the scratch array: calls that overlap on the GPU (handles on
 * different streams) race on it; calls on one stream do not.  It keeps the last call's contents; nothing in it has to be
 * cleared (every entry read is written first).  The first call on a device resolves the array's address
 * (cudaGetSymbolAddress, no allocation): make one call before starting a graph capture.  Errors as sw_bins. */
#define SW_BINS_NOALLOC_MAX 65536
int        sw_bins_noalloc(sw_handle* h, int32_t which, int64_t bin_len, sw_binstat* out_dev);

/* Per-stage device time in ms, summed over the sweeps of the last sw_sweep call that ran with stage
 * timing on: out = {bond, label, flip, observe}.  Stage timing brackets each stage with CUDA events
 * (it serialises nothing but adds event records; off by default).  BASELINE config 3. */
int        sw_set_stage_timing(sw_handle* h, int on);
int        sw_stage_ms(sw_handle* h, float out[4]);
/* The same measurement per kernel: out[i] = ms of kernel slot i summed over the timed sweeps (at most the
 * first 1024 sweeps of the call), i < cap; returns the number of kernel slots (or a negative code).
 * sw_kernel_name(i) names slot i ("bond", "tile_label", "merge", "roots_open", "compress", "bond_label" (a1 + a2 fused),
 * "flip16" (a4 + a6 fused), ...; "" past the end). */
int        sw_kernel_ms(sw_handle* h, float* out, int32_t cap);
const char* sw_kernel_name(int32_t i);
/* The same measurement per SWEEP, as a time series (a random start is not equilibrated quickly, so the
 * cost of a sweep drifts): out[k] = ms from the first to the last event of timed sweep k, k < min(cap, timed sweeps);
 * returns the number of timed sweeps of the last call (or a negative code). */
int64_t    sw_sweep_ms(sw_handle* h, float* out, int64_t cap);

/* Select the kernel path.  Results are identical on every path.
 *   0  the fast path: fused bond draw + scan-line tile labelling on 128 x 64 tiles when L is a multiple of 128, on
 *      64 x 32 tiles when it is a multiple of 64, the generic kernels otherwise
 *   1  generic any-L path (global union-find, no tiles)
 *   6  as 0 but UNFUSED, on the int8 spin plane: stand-alone bond kernel, then labelling from the bond planes
 *      (per-stage timing of bond / label / flip, BASELINE config 3); Ising handles only
 *   11 the paper's own labelling (section 2.3): the label-equivalence iteration scan -> collapse
 *      -> relabel, repeated until a scan forms no reference, run to convergence by ONE cooperative kernel (in
 *      place of the paper's dynamic-parallelism maintenance kernel); any L; kept for A/B timing
 *      against the union-find paths.  Allocates nb*N*4 extra bytes with cudaMalloc on first use (freed by
 *      sw_destroy).
 * Any other value: SW_EINVAL.  (The flat int32 labels of sw_labels and the size array of paths 1 / 11, nb*N*4 bytes
 * each, are allocated by the library on first use, outside a caller-supplied workspace, and freed by sw_destroy.) */
int        sw_set_path(sw_handle* h, int path);

/* Default 1: on the fast path with 128 x 64 tiles the assignment kernel stages the 16-bit root plane through the TMA
 * engine (cp.async.bulk.tensor.2d boxes of one tile into a ring of shared-memory stages, persistent CTAs:
 * k_flip16_tma); 0: the direct-load kernel k_flip16 (also used when the driver cannot encode the tensor map, and for
 * lattices of fewer than 8 tiles).  Same results. */
int        sw_set_tma(sw_handle* h, int on);

/* Default 1: a lattice of at most 8 tiles of 64 x 32 sites (L = 64, 128) runs a whole
 * sw_sweep(h, n) call inside ONE kernel, one thread-block cluster per lattice of the batch, the steps of a sweep separated
 * by the cluster's hardware barrier instead of by kernel boundaries (k_sweeps_cluster; the paper's own sizes,
 * PAPER.md:133-142).  0: the kernels of the fast path one by one, as for larger lattices (also taken with per-kernel
 * timing, eager labels, path 6, and when the cluster launch fails).  Same results. */
int        sw_set_cluster(sw_handle* h, int on);

/* Path 11 only: number of passes (scans, including the last one that formed no reference) the label-equivalence
 * iteration of the last sweep / sw_test_label took -- a deterministic function of the bond graph (PAPER.md:53
 * reports "5 or 6" for 512 x 512).  Synchronises.  SW_ESTATE on another path, before any labelling, or if the
 * iteration did not converge within 1024 passes. */
int        sw_label_passes(sw_handle* h, int32_t* passes);

/* Number of kernel launches issued by the last sw_sweep call (for bench.py's gpu_launches). */
int64_t    sw_last_launch_count(const sw_handle* h);

uint32_t   sw_threshold(const sw_handle* h, int32_t b);    /* integer bond threshold of lattice b */
int32_t    sw_L(const sw_handle* h);
int32_t    sw_batch(const sw_handle* h);

/* Stand-alone pieces for tests (device work on the default stream, synchronising):
 * Philox4x32-10 of n (ctr, key) pairs, HOST arrays ctr[4n], key[2n] -> out[4n], computed ON THE GPU
 * by the same device function the kernels use. */
int        sw_test_philox(const uint32_t* ctr, const uint32_t* key, uint32_t* out, int64_t n);
/* The measured integer-ALU ceiling of the bond stage: ms per launch (mean of `reps`, after 3 warm-up
 * launches, CUDA events on the default stream) of a kernel that makes the sites/2 Philox4x32-10 calls of one sweep of
 * `sites` sites -- 16 per thread, as the bond kernels do -- XOR-reduces the words and stores one word per warp: no
 * other memory traffic.  Synchronises. */
int        sw_test_philox_ceiling(int64_t sites, int32_t reps, float* ms_out);
/* Label injected bond planes: bondE/bondS HOST canonical bit-planes of one L x L lattice ->
 * labels_out[N] (HOST), through the handle's labelling kernels (h must have the same L, nb = 1). */
int        sw_test_label(sw_handle* h, const uint32_t* bondE, const uint32_t* bondS, int32_t* labels_out);

const char* sw_last_error(void);                           /* thread-local text, never NULL */
const char* sw_version(void);

#ifdef __cplusplus
}
#endif
#endif /* SW_B200_H */
