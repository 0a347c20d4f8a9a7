/*
 * tm_inputs/gen.c -- seeded, counter-based synthetic input generators.
 *
 * DATA ONLY: this file holds none of the method's arithmetic (no gamma matrices,
 * no hopping term, no solver, no contraction, no device layout).  It produces the
 * synthetic stand-ins for the paper's inputs, in the canonical host layout:
 *
 *   gauge   U[site][mu][row][col][re,im]   fp64, site = x + X*(y + Y*(z + Z*t)), mu = 0..3 = x,y,z,t
 *   spinor  psi[site][spin][colour][re,im] fp64
 *
 * Recipe (BASELINE.json configs[0]):
 *   links  = Gram-Schmidt SU(3) projection of (w*1 + eps*G), G_ij = g1 + i*g2, g ~ N(0,1)
 *   noise  = Z2 (x) iZ2 ("Z4" in BASELINE.json): (+-1 +- i)/sqrt(2) per (site, spin, colour)
 *            (section II.A lists Z2, Z4 and Z2 (x) iZ2 noise)
 *
 * Every value is a pure function of (seed, stream, global index, draw number), so any
 * traversal order / slab decomposition / site sampling gives the same field.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

static inline uint64_t splitmix64(uint64_t z)
{
    z += 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

/* counter-based hash: three chained splitmix64 rounds over (seed, stream, idx, draw) */
static inline uint64_t ctr_hash(uint64_t seed, uint64_t stream, uint64_t idx, uint64_t draw)
{
    uint64_t z = splitmix64(seed ^ (stream * 0xD6E8FEB86659FD93ULL));
    z = splitmix64(z ^ (idx * 0xA0761D6478BD642FULL));
    z = splitmix64(z ^ (draw * 0xE7037ED1A0B428DBULL));
    return z;
}

/* uniform in (0, 1] */
static inline double u01(uint64_t h) { return ((double)(h >> 11) + 1.0) * (1.0 / 9007199254740992.0); }

/* one Box-Muller pair from two hashes */
static inline void gauss_pair(uint64_t h1, uint64_t h2, double* g1, double* g2)
{
    const double r = sqrt(-2.0 * log(u01(h1)));
    const double ph = 6.283185307179586476925286766559 * u01(h2);
    *g1 = r * cos(ph);
    *g2 = r * sin(ph);
}

enum { STREAM_GAUGE = 1, STREAM_Z4 = 2, STREAM_GAUSS = 3 };

/* one SU(3) matrix: Gram-Schmidt of (w*1 + eps*G); out[3][3][2] row-major */
static void su3_from_hash(uint64_t seed, uint64_t stream, uint64_t linkidx, double w, double eps, double* out)
{
    double a[3][3][2];
    for (int k = 0; k < 9; ++k) {
        double g1, g2;
        gauss_pair(ctr_hash(seed, stream, linkidx, 2 * k), ctr_hash(seed, stream, linkidx, 2 * k + 1), &g1, &g2);
        a[k / 3][k % 3][0] = eps * g1 + ((k / 3 == k % 3) ? w : 0.0);
        a[k / 3][k % 3][1] = eps * g2;
    }
    /* r1 = a0 / |a0| */
    double n = 0;
    for (int j = 0; j < 3; ++j) n += a[0][j][0] * a[0][j][0] + a[0][j][1] * a[0][j][1];
    n = 1.0 / sqrt(n);
    for (int j = 0; j < 3; ++j) { a[0][j][0] *= n; a[0][j][1] *= n; }
    /* r2 = a1 - (r1^dagger . a1) r1, normalised */
    double pr = 0, pi = 0;
    for (int j = 0; j < 3; ++j) {
        pr += a[0][j][0] * a[1][j][0] + a[0][j][1] * a[1][j][1];
        pi += a[0][j][0] * a[1][j][1] - a[0][j][1] * a[1][j][0];
    }
    for (int j = 0; j < 3; ++j) {
        a[1][j][0] -= pr * a[0][j][0] - pi * a[0][j][1];
        a[1][j][1] -= pr * a[0][j][1] + pi * a[0][j][0];
    }
    n = 0;
    for (int j = 0; j < 3; ++j) n += a[1][j][0] * a[1][j][0] + a[1][j][1] * a[1][j][1];
    n = 1.0 / sqrt(n);
    for (int j = 0; j < 3; ++j) { a[1][j][0] *= n; a[1][j][1] *= n; }
    /* r3 = conj(r1 x r2) */
    for (int j = 0; j < 3; ++j) {
        const int j1 = (j + 1) % 3, j2 = (j + 2) % 3;
        const double cr = (a[0][j1][0] * a[1][j2][0] - a[0][j1][1] * a[1][j2][1]) -
                          (a[0][j2][0] * a[1][j1][0] - a[0][j2][1] * a[1][j1][1]);
        const double ci = (a[0][j1][0] * a[1][j2][1] + a[0][j1][1] * a[1][j2][0]) -
                          (a[0][j2][0] * a[1][j1][1] + a[0][j2][1] * a[1][j1][0]);
        a[2][j][0] = cr;
        a[2][j][1] = -ci;
    }
    for (int k = 0; k < 18; ++k) out[k] = (&a[0][0][0])[k];
}

/* links of the sites [site0, site1) (global lexicographic indices); out[(site-site0)][4][3][3][2] */
void tmi_gauge_range(uint64_t seed, double w, double eps, int64_t site0, int64_t site1, double* out)
{
#pragma omp parallel for schedule(static)
    for (int64_t s = site0; s < site1; ++s)
        for (int mu = 0; mu < 4; ++mu)
            su3_from_hash(seed, STREAM_GAUGE, (uint64_t)s * 4 + mu, w, eps, out + ((s - site0) * 4 + mu) * 18);
}

/* links of an arbitrary list of sites; out[n][4][3][3][2] */
void tmi_gauge_sites(uint64_t seed, double w, double eps, int64_t n, const int64_t* sites, double* out)
{
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k)
        for (int mu = 0; mu < 4; ++mu)
            su3_from_hash(seed, STREAM_GAUGE, (uint64_t)sites[k] * 4 + mu, w, eps, out + (k * 4 + mu) * 18);
}

/* one SU(3) matrix per site (used as a random gauge transformation g(x)); out[n][3][3][2] */
void tmi_su3_range(uint64_t seed, double w, double eps, int64_t site0, int64_t site1, double* out)
{
#pragma omp parallel for schedule(static)
    for (int64_t s = site0; s < site1; ++s)
        su3_from_hash(seed, STREAM_GAUGE + 16, (uint64_t)s, w, eps, out + (s - site0) * 18);
}

/* Z2 (x) iZ2 noise code of component comp (= spin*3 + colour) at a site: bit0 -> sign of re, bit1 -> sign of im */
static inline unsigned z4_code(uint64_t seed, uint64_t site, int comp)
{
    return (unsigned)(ctr_hash(seed, STREAM_Z4, site * 12 + comp, 0) >> 62);
}

/* codes[(site-site0)][12] as bytes 0..3 */
void tmi_z4_codes_range(uint64_t seed, int64_t site0, int64_t site1, uint8_t* codes)
{
#pragma omp parallel for schedule(static)
    for (int64_t s = site0; s < site1; ++s)
        for (int c = 0; c < 12; ++c) codes[(s - site0) * 12 + c] = (uint8_t)z4_code(seed, (uint64_t)s, c);
}

/* psi[(site-site0)][4][3][2] = (+-1 +- i)/sqrt(2) */
void tmi_z4_range(uint64_t seed, int64_t site0, int64_t site1, double* psi)
{
    const double r = 0.70710678118654752440084436210485;
#pragma omp parallel for schedule(static)
    for (int64_t s = site0; s < site1; ++s)
        for (int c = 0; c < 12; ++c) {
            const unsigned code = z4_code(seed, (uint64_t)s, c);
            psi[((s - site0) * 12 + c) * 2 + 0] = (code & 1u) ? -r : r;
            psi[((s - site0) * 12 + c) * 2 + 1] = (code & 2u) ? -r : r;
        }
}

void tmi_z4_sites(uint64_t seed, int64_t n, const int64_t* sites, double* psi)
{
    const double r = 0.70710678118654752440084436210485;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k)
        for (int c = 0; c < 12; ++c) {
            const unsigned code = z4_code(seed, (uint64_t)sites[k], c);
            psi[(k * 12 + c) * 2 + 0] = (code & 1u) ? -r : r;
            psi[(k * 12 + c) * 2 + 1] = (code & 2u) ? -r : r;
        }
}

/* complex Gaussian spinor, unit variance per real component; psi[(site-site0)][4][3][2] */
void tmi_gauss_range(uint64_t seed, int64_t site0, int64_t site1, double* psi)
{
#pragma omp parallel for schedule(static)
    for (int64_t s = site0; s < site1; ++s)
        for (int c = 0; c < 12; ++c) {
            double g1, g2;
            gauss_pair(ctr_hash(seed, STREAM_GAUSS, (uint64_t)s * 12 + c, 0),
                       ctr_hash(seed, STREAM_GAUSS, (uint64_t)s * 12 + c, 1), &g1, &g2);
            psi[((s - site0) * 12 + c) * 2 + 0] = g1;
            psi[((s - site0) * 12 + c) * 2 + 1] = g2;
        }
}
