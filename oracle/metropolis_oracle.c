/*
 * metropolis_oracle.c -- independent textbook Metropolis for the 3D +-J
 * Edwards-Anderson model.  TEST INFRASTRUCTURE (see micsa_oracle.c header):
 * it exists only to pin the MicSA oracle's equilibrium energies in the
 * paramagnetic phase (BASELINE.json north_star; "if a fresh
 * value of the n were drawn for every spin-flip attempt, our elementary move
 * would become the textbook Metropolis update").
 *
 * Deliberately written differently from micsa_oracle.c: neighbour tables
 * instead of inline wraps, sequential (typewriter) site order instead of the
 * checkerboard, a splitmix64 stream instead of Philox, floating-point
 * acceptance min(1, exp(-beta dH)) instead of demons.  Canonical layouts are
 * the ones documented in micsa_oracle.c.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static inline uint64_t splitmix64(uint64_t *state)
{
    uint64_t z = (*state += 0x9E3779B97F4A7C15ull);
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static inline double uniform01(uint64_t *state)
{
    return (double)(splitmix64(state) >> 11) * (1.0 / 9007199254740992.0);
}

/* H_EA of one system, Eq. (1), each bond once. */
static double energy_per_spin(int64_t N, const int64_t *nbr_plus,
                              const int8_t *s, const int8_t *J)
{
    int64_t e = 0;
    for (int d = 0; d < 3; ++d)
        for (int64_t i = 0; i < N; ++i)
            e -= (int64_t)J[d * N + i] * s[i] * s[nbr_plus[d * N + i]];
    return (double)e / (double)N;
}

void metropolis_run(int L, int n_samples, int n_replicas, double T,
                    int n_sweeps, uint64_t seed, int8_t *s, const int8_t *J,
                    double *e_out /* [n_sweeps][n_sys] */)
{
    const int64_t N = (int64_t)L * L * L;
    const int n_sys = n_samples * n_replicas;
    const double beta = 1.0 / T;
    int64_t *nbr_plus  = (int64_t *)malloc(sizeof(int64_t) * 3 * N);
    int64_t *nbr_minus = (int64_t *)malloc(sizeof(int64_t) * 3 * N);
    for (int64_t i = 0; i < N; ++i) {
        const int c[3] = { (int)(i % L), (int)((i / L) % L), (int)(i / ((int64_t)L * L)) };
        const int64_t stride[3] = { 1, L, (int64_t)L * L };
        for (int d = 0; d < 3; ++d) {
            const int up = (c[d] + 1 == L) ? 0 : c[d] + 1;
            const int dn = (c[d] == 0) ? L - 1 : c[d] - 1;
            nbr_plus[d * N + i]  = i + (up - c[d]) * stride[d];
            nbr_minus[d * N + i] = i + (dn - c[d]) * stride[d];
        }
    }
    /* Boltzmann factors for dH = 4, 8, 12 */
    const double w[4] = { 1.0, exp(-4.0 * beta), exp(-8.0 * beta), exp(-12.0 * beta) };

#pragma omp parallel for schedule(static)
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas;
        int8_t *ss = s + (int64_t)sys * N;
        const int8_t *Js = J + (int64_t)sample * 3 * N;
        uint64_t rng = seed * 0xD1342543DE82EF95ull + (uint64_t)sys * 0x2545F4914F6CDD1Dull + 1u;
        for (int t = 0; t < n_sweeps; ++t) {
            for (int64_t i = 0; i < N; ++i) {
                int h = 0;
                for (int d = 0; d < 3; ++d) {
                    const int64_t ip = nbr_plus[d * N + i], im = nbr_minus[d * N + i];
                    h += Js[d * N + i] * ss[ip] + Js[d * N + im] * ss[im];
                }
                const int dH = 2 * ss[i] * h;
                if (dH <= 0 || uniform01(&rng) < w[dH / 4])
                    ss[i] = (int8_t)(-ss[i]);
            }
            e_out[(int64_t)t * n_sys + sys] = energy_per_spin(N, nbr_plus, ss, Js);
        }
    }
    free(nbr_plus);
    free(nbr_minus);
}
