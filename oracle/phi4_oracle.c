/*
 * phi4_oracle.c -- serial CPU statement of the Wolff-type embedded cluster update for the O(4)
 * symmetric phi^4 theory on a four-dimensional periodic lattice.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/ and bench.py's cpu_baseline leg may build,
 * link or call this file.  It shares no code, header, table or helper with the CUDA path under
 * paper_2302_14720_b200/csrc/; the one thing it takes from outside is the oracle's own Philox
 * (orc_philox4x32_10 of sw_oracle.c, pinned by published known answers).
 *
 * What it is: PAPER.md:93-109 (section 3), one site at a time, in the paper's order:
 *   1. a random four-component direction r, r.r = 1;
 *   2. for every site x and every direction mu = 0..3 ("each site now checks the next index for
 *      each of the four array elements") a bond with probability
 *          p = 1 - exp{ min(0, -4 kappa (phi_x . r)(phi_{x+mu} . r)) }          (Eq. 2)
 *   3. the clusters of the bond graph; each is selected with probability 1/2 and the selected ones
 *      are reflected, phi_x -> phi_x - 2 (phi_x . r) r                          (Eq. 3)
 * Readings (the paper gives Eq. 2 and Eq. 3 and nothing else; DESIGN.md 7e lists these):
 *   - lattice L^4, periodic; site x = ((x3 L + x2) L + x1) L + x0; direction mu raises x_mu by one;
 *     field phi[4 x + a], a = 0..3, double precision; for L = 2 the two links between a pair of
 *     sites are independent (as for the 2D lattice);
 *   - only the cluster update is stated by the paper, so only it is built: |phi_x| never changes
 *     (a full phi^4 simulation adds a local update of the moduli, which the paper does not describe);
 *     kappa is the hopping parameter of the usual lattice action
 *     S = sum_x [ -2 kappa sum_mu phi_x . phi_{x+mu} + phi_x^2 + lambda (phi_x^2 - 1)^2 ];
 *   - random numbers: Philox4x32-10, key = seed, counter = (index, t lo, t hi, TAG) with tags
 *     16 (start), 17 (direction), 18 (bonds), 19 (selection), disjoint from the Ising tags;
 *     a 32-bit word w gives the uniform u = (w + 1/2) 2^-32 in (0, 1);
 *   - direction: attempt j = 0, 1, ... draws call (j, t, TAG_DIR), v_a = 2 u_a - 1; the first
 *     attempt with 1e-4 <= |v|^2 <= 1 is kept, r = v / |v| (rejection from the cube to the ball makes
 *     the direction uniform on the sphere; only +, *, /, sqrt: exact in IEEE arithmetic);
 *   - bonds: call (x, t, TAG_BOND4), word mu for direction mu; s_x = ((phi0 r0 + phi1 r1) + phi2 r2)
 *     + phi3 r3; arg = (-4 kappa) (s_x s_y); no bond for arg >= 0; else thr = min(floor(-expm1(arg)
 *     2^32), 2^32 - 1) and the bond forms iff word < thr; bonds[x] holds bit mu;
 *   - a cluster is named by its minimum site index; it is selected iff bit `label` of the 128-bit
 *     fields of (label >> 7, t, TAG_SEL) is 1 (the Ising oracle's bit-field layout);
 *   - reflection: phi_a <- phi_a - (2 s) r_a with the s above;
 *   - observables of the new configuration: link = sum_x sum_mu phi_x . phi_{x+mu},
 *     M_a = sum_x phi_x[a], both summed in index order; clusters, largest cluster, bonds of the sweep.
 * Pins (tests/test_oracle_phi4.py): uniformity of r on the sphere (second and fourth moments), Eq. 2's
 * probability on a constant field against 1 - exp(-4 kappa s^2) computed apart, no bonds where the
 * projections have opposite signs or kappa = 0, clusters against scipy on an independently built 4D
 * graph, reflections that keep |phi_x| and phi_x . phi_y inside a cluster, selection rate 1/2, and the
 * link energy of the O(4) model at fixed moduli against a Metropolis simulation of the same Boltzmann
 * weight written with numpy (2^4 and 3^4 lattices, unit and unequal moduli) within 4 sigma.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);   /* sw_oracle.c */

enum { TAG_INIT4 = 16, TAG_DIR = 17, TAG_BOND4 = 18, TAG_SEL = 19 };

static void draw4(uint64_t seed, uint64_t t, uint32_t tag, uint32_t index, uint32_t out[4])
{
    uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { index, (uint32_t)(t & 0xFFFFFFFFu), (uint32_t)(t >> 32), tag };
    orc_philox4x32_10(ctr, key, out);
}
static double unif(uint32_t w) { return ((double)w + 0.5) * (1.0 / 4294967296.0); }

static int64_t volume(int32_t L) { return (int64_t)L * L * L * L; }

/* neighbour of x in direction mu (coordinate mu + 1, periodic) */
static int64_t fwd(int32_t L, int64_t x, int mu)
{
    int64_t stride = 1;
    for (int k = 0; k < mu; ++k) stride *= L;
    int64_t c = (x / stride) % L;
    return c + 1 == L ? x - (int64_t)(L - 1) * stride : x + stride;
}
static int64_t bwd(int32_t L, int64_t x, int mu)
{
    int64_t stride = 1;
    for (int k = 0; k < mu; ++k) stride *= L;
    int64_t c = (x / stride) % L;
    return c == 0 ? x + (int64_t)(L - 1) * stride : x - stride;
}

/* start: every component uniform in (-1, 1) */
void orc4_init(int32_t L, uint64_t seed, double *phi)
{
    int64_t V = volume(L);
    for (int64_t x = 0; x < V; ++x) {
        uint32_t w[4];
        draw4(seed, 0, TAG_INIT4, (uint32_t)x, w);
        for (int a = 0; a < 4; ++a) phi[4 * x + a] = 2.0 * unif(w[a]) - 1.0;
    }
}

/* step 1: the sweep's direction; returns the number of attempts it took */
int orc4_direction(uint64_t seed, uint64_t t, double r[4])
{
    for (uint32_t j = 0; ; ++j) {
        uint32_t w[4];
        double v[4];
        draw4(seed, t, TAG_DIR, j, w);
        for (int a = 0; a < 4; ++a) v[a] = 2.0 * unif(w[a]) - 1.0;
        double n2 = ((v[0] * v[0] + v[1] * v[1]) + v[2] * v[2]) + v[3] * v[3];
        if (n2 <= 1.0 && n2 >= 1e-4) {
            double n = sqrt(n2);
            for (int a = 0; a < 4; ++a) r[a] = v[a] / n;
            return (int)j + 1;
        }
    }
}

static double proj(const double *p, const double r[4])
{
    return ((p[0] * r[0] + p[1] * r[1]) + p[2] * r[2]) + p[3] * r[3];
}

/* Eq. 2 as an integer threshold on a 32-bit word */
uint32_t orc4_threshold(double kappa, double sx, double sy)
{
    double arg = (-4.0 * kappa) * (sx * sy);
    if (!(arg < 0.0)) return 0u;
    double v = floor(-expm1(arg) * 4294967296.0);
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

/* step 2: bonds[x] bit mu = bond between x and its neighbour in direction mu */
void orc4_bonds(int32_t L, double kappa, uint64_t seed, uint64_t t, const double *phi,
                const double r[4], uint8_t *bonds)
{
    int64_t V = volume(L);
    for (int64_t x = 0; x < V; ++x) {
        uint32_t w[4];
        draw4(seed, t, TAG_BOND4, (uint32_t)x, w);
        double sx = proj(phi + 4 * x, r);
        uint8_t b = 0;
        for (int mu = 0; mu < 4; ++mu) {
            double sy = proj(phi + 4 * fwd(L, x, mu), r);
            if (w[mu] < orc4_threshold(kappa, sx, sy)) b |= (uint8_t)(1u << mu);
        }
        bonds[x] = b;
    }
}

/* step 3a: clusters by breadth-first search, components visited in increasing index order, so
 * label[x] = the minimum site index of x's cluster */
int orc4_labels(int32_t L, const uint8_t *bonds, int32_t *label)
{
    int64_t V = volume(L);
    int32_t *queue = (int32_t *)malloc((size_t)V * sizeof(int32_t));
    if (!queue) return -1;
    for (int64_t x = 0; x < V; ++x) label[x] = -1;
    for (int64_t s = 0; s < V; ++s) {
        if (label[s] >= 0) continue;
        int64_t head = 0, tail = 0;
        queue[tail++] = (int32_t)s; label[s] = (int32_t)s;
        while (head < tail) {
            int64_t x = queue[head++];
            for (int mu = 0; mu < 4; ++mu) {
                int64_t y = fwd(L, x, mu);
                if (((bonds[x] >> mu) & 1u) && label[y] < 0) { label[y] = (int32_t)s; queue[tail++] = (int32_t)y; }
                int64_t z = bwd(L, x, mu);
                if (((bonds[z] >> mu) & 1u) && label[z] < 0) { label[z] = (int32_t)s; queue[tail++] = (int32_t)z; }
            }
        }
    }
    free(queue);
    return 0;
}

int orc4_selected(uint64_t seed, uint64_t t, int64_t label)
{
    uint32_t w[4];
    draw4(seed, t, TAG_SEL, (uint32_t)(label >> 7), w);
    return (int)((w[(label >> 5) & 3] >> (label & 31)) & 1u);
}

/* step 3b: reflect the selected clusters, Eq. 3 */
void orc4_reflect(int32_t L, uint64_t seed, uint64_t t, const int32_t *label, const double r[4], double *phi)
{
    int64_t V = volume(L);
    for (int64_t x = 0; x < V; ++x) {
        if (!orc4_selected(seed, t, label[x])) continue;
        double two_s = 2.0 * proj(phi + 4 * x, r);
        for (int a = 0; a < 4; ++a) phi[4 * x + a] = phi[4 * x + a] - two_s * r[a];
    }
}

/* dout = {link, M0, M1, M2, M3}; iout = {clusters, largest cluster, bonds} (label / bonds may be NULL: zeros) */
int orc4_observables(int32_t L, const double *phi, const int32_t *label, const uint8_t *bonds,
                     double dout[5], int64_t iout[3])
{
    int64_t V = volume(L);
    double link = 0.0, M[4] = { 0.0, 0.0, 0.0, 0.0 };
    for (int64_t x = 0; x < V; ++x) {
        for (int mu = 0; mu < 4; ++mu) {
            const double *p = phi + 4 * x, *q = phi + 4 * fwd(L, x, mu);
            link = link + (((p[0] * q[0] + p[1] * q[1]) + p[2] * q[2]) + p[3] * q[3]);
        }
        for (int a = 0; a < 4; ++a) M[a] = M[a] + phi[4 * x + a];
    }
    dout[0] = link;
    for (int a = 0; a < 4; ++a) dout[1 + a] = M[a];
    iout[0] = iout[1] = iout[2] = 0;
    if (label) {
        int64_t *size = (int64_t *)calloc((size_t)V, sizeof(int64_t));
        if (!size) return -1;
        for (int64_t x = 0; x < V; ++x) size[label[x]] += 1;
        for (int64_t x = 0; x < V; ++x) {
            if (label[x] == x) iout[0] += 1;
            if (size[x] > iout[1]) iout[1] = size[x];
        }
        free(size);
    }
    if (bonds)
        for (int64_t x = 0; x < V; ++x)
            for (int mu = 0; mu < 4; ++mu) iout[2] += (bonds[x] >> mu) & 1u;
    return 0;
}

/* one full update with sweep index t; phi is updated in place */
int orc4_sweep(int32_t L, double kappa, uint64_t seed, uint64_t t, double *phi, double r[4],
               uint8_t *bonds, int32_t *label, double dout[5], int64_t iout[3])
{
    orc4_direction(seed, t, r);
    orc4_bonds(L, kappa, seed, t, phi, r, bonds);
    if (orc4_labels(L, bonds, label)) return -1;
    orc4_reflect(L, seed, t, label, r, phi);
    return orc4_observables(L, phi, label, bonds, dout, iout);
}

/* n updates t0 .. t0 + n - 1; series (may be NULL) gets dout (5 doubles) per sweep, iseries iout (3 int64) */
int orc4_run(int32_t L, double kappa, uint64_t seed, uint64_t t0, int64_t n, double *phi,
             double *series, int64_t *iseries)
{
    int64_t V = volume(L);
    uint8_t *bonds = (uint8_t *)malloc((size_t)V);
    int32_t *label = (int32_t *)malloc((size_t)V * sizeof(int32_t));
    if (!bonds || !label) { free(bonds); free(label); return -1; }
    for (int64_t k = 0; k < n; ++k) {
        double r[4], d[5];
        int64_t i3[3];
        if (orc4_sweep(L, kappa, seed, t0 + (uint64_t)k, phi, r, bonds, label, d, i3)) { free(bonds); free(label); return -1; }
        if (series) for (int a = 0; a < 5; ++a) series[5 * k + a] = d[a];
        if (iseries) for (int a = 0; a < 3; ++a) iseries[3 * k + a] = i3[a];
    }
    free(bonds); free(label);
    return 0;
}
