/* Seeded random sequential addition (RSA) of non-overlapping spheres in a cubic periodic box.
 *
 * Input generator ONLY: this file holds none of the method's arithmetic (no Ewald sums, no
 * Gaussians, no mobility couplings).  It serves both the CPU oracle and the CUDA path by producing
 * the particle configurations of BASELINE.json's configs ("uniform random non-overlapping positions
 * (seeded rejection sampling) in cubic periodic box"), standing in for the paper's random hard-sphere
 * suspensions ("random bidisperse hard-sphere system", L552).
 *
 * Algorithm: particles are inserted in the order given (callers pass descending radii); a candidate
 * centre is drawn uniformly in [0,L)^3 from a xoshiro256** stream seeded by splitmix64(seed) and
 * accepted when its minimum-image distance to every placed sphere j satisfies |x - x_j| >= a + a_j.
 * A uniform cell grid (cell edge >= a_min + a_max) bounds the overlap search.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static uint64_t rotl64(uint64_t x, int k) { return (x << k) | (x >> (64 - k)); }

typedef struct { uint64_t s[4]; } xoshiro;

static uint64_t splitmix64(uint64_t *state)
{
    uint64_t z = (*state += 0x9E3779B97F4A7C15ULL);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

static uint64_t xoshiro_next(xoshiro *g)
{
    uint64_t *s = g->s;
    uint64_t result = rotl64(s[1] * 5, 7) * 9;
    uint64_t t = s[1] << 17;
    s[2] ^= s[0]; s[3] ^= s[1]; s[1] ^= s[2]; s[0] ^= s[3];
    s[2] ^= t; s[3] = rotl64(s[3], 45);
    return result;
}

static double uniform01(xoshiro *g) { return (double)(xoshiro_next(g) >> 11) * (1.0 / 9007199254740992.0); }

/* Returns 0 on success, 1 when a particle could not be placed within max_attempts proposals,
 * 2 on allocation failure.  pos is [N][3] row-major, written in insertion order. */
int rsa_generate(int64_t N, double L, const double *radii, uint64_t seed, int64_t max_attempts,
                 double *pos, int64_t *total_attempts)
{
    double amin = radii[0], amax = radii[0];
    for (int64_t i = 1; i < N; ++i) {
        if (radii[i] < amin) amin = radii[i];
        if (radii[i] > amax) amax = radii[i];
    }
    int64_t nc = (int64_t)floor(L / (amin + amax));
    if (nc < 1) nc = 1;
    if (nc > 512) nc = 512;
    const double h = L / (double)nc;
    const int64_t ncell = nc * nc * nc;
    int64_t *head = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell);
    int64_t *next = (int64_t *)malloc(sizeof(int64_t) * (size_t)N);
    if (!head || !next) { free(head); free(next); return 2; }
    for (int64_t c = 0; c < ncell; ++c) head[c] = -1;

    uint64_t sm = seed;
    xoshiro g;
    for (int k = 0; k < 4; ++k) g.s[k] = splitmix64(&sm);

    int64_t attempts_all = 0;
    int status = 0;
    for (int64_t i = 0; i < N && status == 0; ++i) {
        const double a = radii[i];
        const int reach = (int)ceil((a + amax) / h);
        int placed = 0;
        for (int64_t att = 0; att < max_attempts && !placed; ++att) {
            ++attempts_all;
            double x[3];
            int64_t c[3];
            for (int d = 0; d < 3; ++d) {
                x[d] = L * uniform01(&g);
                c[d] = (int64_t)floor(x[d] / h);
                if (c[d] >= nc) c[d] = nc - 1;
            }
            int ok = 1;
            /* when 2*reach+1 >= nc every cell is visited once: clamp the loop to nc cells per axis */
            int lo = -reach, hi = reach;
            if (2 * reach + 1 >= nc) { lo = 0; hi = (int)nc - 1; }
            for (int dx = lo; dx <= hi && ok; ++dx)
            for (int dy = lo; dy <= hi && ok; ++dy)
            for (int dz = lo; dz <= hi && ok; ++dz) {
                int64_t cx = (2 * reach + 1 >= nc) ? dx : ((c[0] + dx) % nc + nc) % nc;
                int64_t cy = (2 * reach + 1 >= nc) ? dy : ((c[1] + dy) % nc + nc) % nc;
                int64_t cz = (2 * reach + 1 >= nc) ? dz : ((c[2] + dz) % nc + nc) % nc;
                for (int64_t j = head[(cx * nc + cy) * nc + cz]; j >= 0; j = next[j]) {
                    double r2 = 0.0;
                    for (int d = 0; d < 3; ++d) {
                        double dd = x[d] - pos[3 * j + d];
                        dd -= L * nearbyint(dd / L);
                        r2 += dd * dd;
                    }
                    const double s = a + radii[j];
                    if (r2 < s * s) { ok = 0; break; }
                }
            }
            if (ok) {
                for (int d = 0; d < 3; ++d) pos[3 * i + d] = x[d];
                int64_t ci = (c[0] * nc + c[1]) * nc + c[2];
                next[i] = head[ci];
                head[ci] = i;
                placed = 1;
            }
        }
        if (!placed) status = 1;
    }
    if (total_attempts) *total_attempts = attempts_all;
    free(head); free(next);
    return status;
}
