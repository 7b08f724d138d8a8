/*
 * sw_oracle.c -- serial CPU Swendsen-Wang for the 2D periodic Ising model.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, link or call this
 * file.  It shares no code, header, table or helper with the CUDA path under
 * paper_2302_14720_b200/csrc/ and neither includes the other.
 *
 * What it is: the plain, slow, one-site-at-a-time statement of the sweep of
 *   PAPER.md:33-63 (section 2, steps 2.1-2.5), in the order the paper gives it,
 *   under the readings SURVEY.md section 8(c) fixes (listed in DESIGN.md):
 *     - J = 1, k_B = 1, spins +-1, periodic in both directions (c-2);
 *     - bond probability p = 1 - exp(-2/T) (c-1: the paper prints
 *       1 - exp(-1/k_B T), in units where its own figures put
 *       the critical point at k_B T ~ 2.25);
 *     - one draw per undirected edge, owned by its West / North end
 *       ("checks the sites to East and South"; c-3);
 *     - site i = y*L + x, East = x+1, South = y+1 ("below and to the right",
 *       PAPER.md:83; c-4);
 *     - random numbers: Philox4x32-10, counter based (c-5);
 *     - a cluster is named by its minimum site index ("unique integer
 *       incrementing from zero", "lowest value label"; c-8);
 *     - each cluster is ASSIGNED a new spin, up or down with probability 1/2
 *       (c-7).
 *   Labelling is written as the definition (breadth-first search over the bond
 *   graph, components visited in increasing index order), not as the paper's
 *   label-equivalence iteration: both reach the same unique result.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known answers,
 *   thresholds against 50-digit arithmetic, exact enumeration of the 4x4
 *   lattice, Kaufman's finite-lattice energy, Onsager/Yang, per-sweep cluster
 *   invariants checked by independent numpy/scipy code, SURVEY golden vectors.
 *   No function here is "parity unpinned" except <|m|> at and above T_c for
 *   L > 4, which has no exact value (SURVEY.md 8(c) pin 5); that quantity is
 *   covered only by GPU<->oracle bit-exactness.
 *
 * Plain C99, no threads, no SIMD intrinsics, no blocking.  Never tuned.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORC_TAG_INIT 0u
#define ORC_TAG_BOND 1u
#define ORC_TAG_FLIP 2u

/* ---- Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), SURVEY.md 8(c) ---- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2],
                       uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * (uint64_t)c0;
        uint64_t p1 = (uint64_t)M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;           /* key bumped after each round */
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* one generator call: key from the lattice seed, counter (block, t, TAG) */
static void orc_draw(uint64_t seed, uint64_t t, uint32_t tag, uint32_t block,
                     uint32_t out[4])
{
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { block, (uint32_t)(t & 0xFFFFFFFFu), (uint32_t)(t >> 32), tag };
    orc_philox4x32_10(ctr, key, out);
}

/* bit(idx, t, TAG): 128 site-bits per call */
int orc_bit(uint64_t seed, uint64_t t, uint32_t tag, int64_t idx)
{
    uint32_t w[4];
    orc_draw(seed, t, tag, (uint32_t)(idx >> 7), w);
    return (int)((w[(idx >> 5) & 3] >> (idx & 31)) & 1u);
}

/* thr = min(floor(p * 2^32), 0xFFFFFFFF), p = 1 - exp(-2/T) = -expm1(-2/T) (c-6) */
uint32_t orc_threshold(double T)
{
    double p = -expm1(-2.0 / T);
    double v = floor(p * 4294967296.0);
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

/* ---- start configurations (Fig. 1; cold start: BASELINE config 3) ---- */
void orc_init_random(int32_t L, uint64_t seed, int8_t *spins)
{
    int64_t N = (int64_t)L * L;
    for (int64_t i = 0; i < N; ++i)
        spins[i] = orc_bit(seed, 0, ORC_TAG_INIT, i) ? (int8_t)1 : (int8_t)-1;
}

void orc_init_cold(int32_t L, int8_t *spins)
{
    int64_t N = (int64_t)L * L;
    for (int64_t i = 0; i < N; ++i) spins[i] = 1;
}

static int64_t east_of(int32_t L, int64_t i)
{
    int64_t y = i / L, x = i % L;
    return y * L + (x + 1) % L;
}
static int64_t south_of(int32_t L, int64_t i)
{
    int64_t y = i / L, x = i % L;
    return ((y + 1) % L) * L + x;
}
static int64_t west_of(int32_t L, int64_t i)
{
    int64_t y = i / L, x = i % L;
    return y * L + (x + L - 1) % L;
}
static int64_t north_of(int32_t L, int64_t i)
{
    int64_t y = i / L, x = i % L;
    return ((y + L - 1) % L) * L + x;
}

/* ---- step 1: bond formation, PAPER.md:37-39 (section 2.1), Fig. 2 ---- */
void orc_bonds(int32_t L, uint32_t thr, uint64_t seed, uint64_t t,
               const int8_t *spins, uint8_t *bondE, uint8_t *bondS)
{
    int64_t N = (int64_t)L * L;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t w[4];
        orc_draw(seed, t, ORC_TAG_BOND, (uint32_t)(i >> 1), w);
        int j = (int)(i & 1);
        bondE[i] = (uint8_t)(spins[i] == spins[east_of(L, i)]  && w[2 * j]     < thr);
        bondS[i] = (uint8_t)(spins[i] == spins[south_of(L, i)] && w[2 * j + 1] < thr);
    }
}

/* ---- step 3: clusters = connected components of the bond graph,
 *      PAPER.md:49-51 (section 2.3); label = minimum site index (c-8).
 *      Breadth-first search; components are discovered in increasing index
 *      order, so the first site of each one is its minimum.               ---- */
int orc_labels(int32_t L, const uint8_t *bondE, const uint8_t *bondS,
               int32_t *label)
{
    int64_t N = (int64_t)L * L;
    int64_t *queue = (int64_t *)malloc((size_t)N * sizeof(int64_t));
    if (!queue) return -1;
    for (int64_t i = 0; i < N; ++i) label[i] = -1;
    for (int64_t s = 0; s < N; ++s) {
        if (label[s] >= 0) continue;
        int64_t head = 0, tail = 0;
        label[s] = (int32_t)s;
        queue[tail++] = s;
        while (head < tail) {
            int64_t i = queue[head++];
            int64_t e = east_of(L, i), so = south_of(L, i);
            int64_t w = west_of(L, i), n = north_of(L, i);
            if (bondE[i] && label[e] < 0)  { label[e]  = (int32_t)s; queue[tail++] = e;  }
            if (bondS[i] && label[so] < 0) { label[so] = (int32_t)s; queue[tail++] = so; }
            if (bondE[w] && label[w] < 0)  { label[w]  = (int32_t)s; queue[tail++] = w;  }
            if (bondS[n] && label[n] < 0)  { label[n]  = (int32_t)s; queue[tail++] = n;  }
        }
    }
    free(queue);
    return 0;
}

/* ---- step 4: every cluster is assigned a new spin, PAPER.md:57 (section 2.4) ---- */
void orc_assign(int32_t L, uint64_t seed, uint64_t t, const int32_t *label,
                int8_t *spins)
{
    int64_t N = (int64_t)L * L;
    for (int64_t i = 0; i < N; ++i)
        spins[i] = orc_bit(seed, t, ORC_TAG_FLIP, (int64_t)label[i]) ? (int8_t)1 : (int8_t)-1;
}

/* ---- observables, PAPER.md:63 (section 2.5): E = H = -sum_<ij> s_i s_j,
 *      M = sum_i s_i (the paper's M times N); cluster count and largest
 *      cluster (c-12).  out = {E, M, ncl, maxcl}; label may be NULL.      ---- */
int orc_observables(int32_t L, const int8_t *spins, const int32_t *label,
                    int64_t out[4])
{
    int64_t N = (int64_t)L * L;
    int64_t E = 0, M = 0, ncl = 0, maxcl = 0;
    for (int64_t i = 0; i < N; ++i) {
        E -= (int64_t)spins[i] * ((int64_t)spins[east_of(L, i)] + (int64_t)spins[south_of(L, i)]);
        M += spins[i];
    }
    if (label) {
        int64_t *size = (int64_t *)calloc((size_t)N, sizeof(int64_t));
        if (!size) return -1;
        for (int64_t i = 0; i < N; ++i) {
            if (label[i] == (int32_t)i) ++ncl;
            size[label[i]] += 1;
        }
        for (int64_t i = 0; i < N; ++i)
            if (size[i] > maxcl) maxcl = size[i];
        free(size);
    }
    out[0] = E; out[1] = M; out[2] = ncl; out[3] = maxcl;
    return 0;
}

/* ---- one sweep with sweep index t, steps 1-5 of PAPER.md:33.
 *      Steps 2 and 5 (erasure of spins / bonds) need no code. ---- */
int orc_sweep(int32_t L, uint32_t thr, uint64_t seed, uint64_t t,
              int8_t *spins, uint8_t *bondE, uint8_t *bondS, int32_t *label,
              int64_t obs[4])
{
    orc_bonds(L, thr, seed, t, spins, bondE, bondS);
    if (orc_labels(L, bondE, bondS, label) != 0) return -1;
    orc_assign(L, seed, t, label, spins);
    if (obs) return orc_observables(L, spins, label, obs);
    return 0;
}

/* ---- n sweeps t0 .. t0+n-1 from the given spins; series (may be NULL) gets
 *      4 int64 per sweep.  Work arrays are allocated here.                 ---- */
int orc_run(int32_t L, double T, uint64_t seed, uint64_t t0, int64_t n,
            int8_t *spins, int64_t *series)
{
    int64_t N = (int64_t)L * L;
    uint32_t thr = orc_threshold(T);
    uint8_t *bE = (uint8_t *)malloc((size_t)N);
    uint8_t *bS = (uint8_t *)malloc((size_t)N);
    int32_t *lab = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int rc = 0;
    if (!bE || !bS || !lab) rc = -1;
    for (int64_t k = 0; rc == 0 && k < n; ++k)
        rc = orc_sweep(L, thr, seed, t0 + (uint64_t)k, spins, bE, bS, lab,
                       series ? series + 4 * k : NULL);
    free(bE); free(bS); free(lab);
    return rc;
}

/* ==========================================================================
 * q-state Potts model, SURVEY.md 8(f) NEXT-3.  PAPER.md:33: "The approach can
 * be generalized to other discrete spin systems" (and section 6).
 * The paper gives no formulas for it; the readings are the textbook ones
 * (Swendsen & Wang's algorithm was stated for the Potts model), DESIGN.md 7d:
 *   - colours c_i in {0 .. q-1}, H = -J sum_<ij> delta(c_i, c_j), J = 1;
 *   - bond between equal colours with p = 1 - exp(-J/T) (for q = 2 this is the
 *     Ising rule at T_Ising = 2 T); same draws as orc_bonds (the rule there
 *     is "equal values AND word < thr", so orc_bonds serves unchanged);
 *   - clusters and labels as before (orc_labels);
 *   - every cluster is assigned a colour uniform in {0 .. q-1}:
 *       colour = floor(word * q / 2^32), word = 32-bit field `idx` of the
 *       generator (call idx >> 2, word idx & 3), idx = the cluster's label;
 *       start configuration: the same with TAG_INIT, t = 0, idx = site;
 *   - observables: E = -#(equal East / South pairs), M = q max_c n_c - N
 *     (n_c = sites of colour c; M / ((q-1) N) is the usual order parameter;
 *     q = 2: M = |n_0 - n_1|), cluster count, largest cluster.
 * Pins (tests/test_oracle_potts.py): exact enumeration of all 3^9 states of
 * the 3x3 three-state lattice and of the 2^16 states of the 4x4 two-state one
 * (= the Ising table at T_Ising = 2 T), the exact critical energy
 * -(1 + 1/sqrt q) per site at T_c = 1/ln(1 + sqrt q), invariants.
 * ========================================================================== */
uint32_t orc_potts_threshold(double T)
{
    double p = -expm1(-1.0 / T);
    double v = floor(p * 4294967296.0);
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

int orc_potts_colour(uint64_t seed, uint64_t t, uint32_t tag, int64_t idx, int32_t q)
{
    uint32_t w[4];
    orc_draw(seed, t, tag, (uint32_t)(idx >> 2), w);
    return (int)(((uint64_t)w[idx & 3] * (uint64_t)(uint32_t)q) >> 32);
}

void orc_potts_init_random(int32_t L, int32_t q, uint64_t seed, int8_t *colours)
{
    int64_t N = (int64_t)L * L;
    for (int64_t i = 0; i < N; ++i)
        colours[i] = (int8_t)orc_potts_colour(seed, 0, ORC_TAG_INIT, i, q);
}

void orc_potts_assign(int32_t L, int32_t q, uint64_t seed, uint64_t t,
                      const int32_t *label, int8_t *colours)
{
    int64_t N = (int64_t)L * L;
    for (int64_t i = 0; i < N; ++i)
        colours[i] = (int8_t)orc_potts_colour(seed, t, ORC_TAG_FLIP, (int64_t)label[i], q);
}

/* out = {E, M, ncl, maxcl}; counts (may be NULL) gets n_0 .. n_{q-1} */
int orc_potts_observables(int32_t L, int32_t q, const int8_t *colours,
                          const int32_t *label, int64_t out[4], int64_t *counts)
{
    int64_t N = (int64_t)L * L;
    int64_t E = 0, ncl = 0, maxcl = 0, nmax = 0;
    int64_t n[128];
    if (q < 2 || q > 127) return -2;
    for (int c = 0; c < q; ++c) n[c] = 0;
    for (int64_t i = 0; i < N; ++i) {
        if (colours[i] == colours[east_of(L, i)]) E -= 1;
        if (colours[i] == colours[south_of(L, i)]) E -= 1;
        n[colours[i]] += 1;
    }
    for (int c = 0; c < q; ++c) {
        if (n[c] > nmax) nmax = n[c];
        if (counts) counts[c] = n[c];
    }
    if (label) {
        int64_t *size = (int64_t *)calloc((size_t)N, sizeof(int64_t));
        if (!size) return -1;
        for (int64_t i = 0; i < N; ++i) {
            if (label[i] == (int32_t)i) ++ncl;
            size[label[i]] += 1;
        }
        for (int64_t i = 0; i < N; ++i)
            if (size[i] > maxcl) maxcl = size[i];
        free(size);
    }
    out[0] = E; out[1] = (int64_t)q * nmax - N; out[2] = ncl; out[3] = maxcl;
    return 0;
}

int orc_potts_sweep(int32_t L, int32_t q, uint32_t thr, uint64_t seed, uint64_t t,
                    int8_t *colours, uint8_t *bondE, uint8_t *bondS, int32_t *label,
                    int64_t obs[4])
{
    orc_bonds(L, thr, seed, t, colours, bondE, bondS);
    if (orc_labels(L, bondE, bondS, label) != 0) return -1;
    orc_potts_assign(L, q, seed, t, label, colours);
    if (obs) return orc_potts_observables(L, q, colours, label, obs, NULL);
    return 0;
}

int orc_potts_run(int32_t L, int32_t q, double T, uint64_t seed, uint64_t t0, int64_t n,
                  int8_t *colours, int64_t *series)
{
    int64_t N = (int64_t)L * L;
    uint32_t thr = orc_potts_threshold(T);
    uint8_t *bE = (uint8_t *)malloc((size_t)N);
    uint8_t *bS = (uint8_t *)malloc((size_t)N);
    int32_t *lab = (int32_t *)malloc((size_t)N * sizeof(int32_t));
    int rc = 0;
    if (!bE || !bS || !lab) rc = -1;
    for (int64_t k = 0; rc == 0 && k < n; ++k)
        rc = orc_potts_sweep(L, q, thr, seed, t0 + (uint64_t)k, colours, bE, bS, lab,
                             series ? series + 4 * k : NULL);
    free(bE); free(bS); free(lab);
    return rc;
}
