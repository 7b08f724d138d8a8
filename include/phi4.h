/*
 * phi4.h -- C ABI of the second workload of arxiv 2302.14720: the Wolff-type embedded cluster update for the O(4)
 * symmetric phi^4 theory on a four-dimensional periodic lattice, hand-written CUDA for sm_100a (libsw_b200.so).
 * SURVEY.md 8(f) NEXT-4.  The operation is PAPER.md:93-109 (section 3): per update
 *   1. a random direction r on the unit sphere S^3;
 *   2. for every site x and direction mu = 0..3 a bond with probability
 *        p = 1 - exp{ min(0, -4 kappa (phi_x . r)(phi_{x+mu} . r)) }                      (Eq. 2)
 *   3. the clusters of the bond graph (labelled by their minimum site index); each is selected with probability 1/2,
 *      and the selected ones are reflected: phi_x -> phi_x - 2 (phi_x . r) r            (Eq. 3)
 * Only this cluster update is built (it is all the paper states): |phi_x| never changes; kappa is the hopping parameter
 * of S = sum_x [ -2 kappa sum_mu phi_x . phi_{x+mu} + phi_x^2 + lambda (phi_x^2 - 1)^2 ].  Readings:
 * site x = ((x3 L + x2) L + x1) L + x0, direction mu raises x_mu by one (periodic); field phi[4 x + a] in double;
 * Philox4x32-10 keyed by the seed, counter = (index, t lo, t hi, TAG), tags 16 start / 17 direction / 18 bonds /
 * 19 selection; a word w is the uniform (w + 1/2) 2^-32; the direction is the first point of the cube (-1, 1)^4 with
 * 1e-4 <= |v|^2 <= 1, normalised; a bond forms iff word_mu of call (x, t) < floor(-expm1(arg) 2^32) (clamped), arg =
 * (-4 kappa)((phi_x . r)(phi_y . r)) < 0; a cluster is selected iff bit `label` of the 128-bit fields of call
 * (label >> 7, t) is set.  Projections, the reflection and the direction use separately rounded IEEE operations in a fixed
 * order (no fused multiply-add), so the field is reproducible bit for bit; only expm1 is a library function.
 *
 * Pointers marked DEVICE point into the handle's device memory (valid until the next phi4_sweep / phi4_destroy);
 * everything else is HOST.  Calls return PHI4_OK (0) or a negative code; phi4_last_error() has the text (thread-local).
 * There is no CPU path: phi4_create fails when no CUDA device is present.  A handle lives on the device that was current
 * when it was created; every call switches to it.
 */
#ifndef PHI4_B200_H
#define PHI4_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PHI4_OK       0
#define PHI4_EINVAL  -1   /* L < 2, L > PHI4_MAX_L, kappa not finite or < 0, n < 0, null pointer */
#define PHI4_ENOMEM  -2
#define PHI4_ECUDA   -3
#define PHI4_ESTATE  -4   /* labels / bonds / direction asked for before the first update */

#define PHI4_MAX_L   128      /* V = L^4 <= 2^28 sites (int32 labels, 32-bit Philox counters) */

typedef struct phi4_handle phi4_handle;   /* opaque */

/* Observables: link = sum_x sum_mu phi_x . phi_{x+mu} and m[a] = sum_x phi_x[a] of the CURRENT field (deterministic
 * tree sums on the device); n_clusters / largest_cluster / n_bonds of the LAST update's bond graph (0 before any);
 * sweep = updates completed; link_per_link = link / (4 V); abs_m_per_site = |m| / V. */
typedef struct {
    double   link, m[4];
    int64_t  n_clusters, largest_cluster, n_bonds;
    uint64_t sweep;
    double   link_per_link, abs_m_per_site;
} phi4_obs;

const char* phi4_last_error(void);

/* L^4 lattice, hopping parameter kappa >= 0, Philox seed; start: every component uniform in (-1, 1) (tag 16).  NULL on error. */
phi4_handle* phi4_create(int32_t L, double kappa, uint64_t seed);
void         phi4_destroy(phi4_handle* h);                  /* NULL is a no-op */

/* n updates (sweep indices t .. t + n - 1), asynchronous on the handle's stream; from the second update of a call on the
 * launch sequence is replayed from a CUDA graph (the sweep index lives on the device). */
int          phi4_sweep(phi4_handle* h, int64_t n);

const double*  phi4_field(phi4_handle* h);                  /* DEVICE, 4 V doubles, phi[4 x + a] */
const int32_t* phi4_labels(phi4_handle* h);                 /* DEVICE, V int32: minimum site index of the site's cluster (last update) */
const uint8_t* phi4_bonds(phi4_handle* h);                  /* DEVICE, V bytes: bit mu = bond to the neighbour in direction mu (last update) */
int          phi4_direction(phi4_handle* h, double r[4]);   /* the last update's direction; synchronises */
int          phi4_observables(phi4_handle* h, phi4_obs* out);                 /* synchronises */
/* per-update history of the LAST phi4_sweep call, oldest first; `out` holds `cap` records; returns the number retained
 * (<= 4096) or a negative code */
int64_t      phi4_series(phi4_handle* h, phi4_obs* out, int64_t cap);

int          phi4_set_field(phi4_handle* h, const double* phi, int is_host);  /* 4 V doubles */
int          phi4_get_field(phi4_handle* h, double* out_host);                /* synchronising copy */
int          phi4_get_labels(phi4_handle* h, int32_t* out_host);
int          phi4_get_bonds(phi4_handle* h, uint8_t* out_host);
int          phi4_set_sweep_index(phi4_handle* h, uint64_t t);
uint64_t     phi4_sweep_index(const phi4_handle* h);
int          phi4_set_stream(phi4_handle* h, void* cuda_stream);              /* a cudaStream_t; NULL = default stream */
int          phi4_set_graphs(phi4_handle* h, int on);                         /* default 1 */
int32_t      phi4_L(const phi4_handle* h);
int64_t      phi4_last_launch_count(const phi4_handle* h);

#ifdef __cplusplus
}
#endif
#endif
