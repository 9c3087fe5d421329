/*
 * gauss_oracle.c -- CPU ORACLE for the continuous-daemon form of the method
 * (SURVEY.md 8(f) rank 4): real-valued daemons / walkers n >= 0 with Gaussian
 * couplings, PAPER.md:136-140 (Sec. 2.4, Eq. 9) and :436-454 (Appendix C).
 *
 * THIS FILE IS TEST INFRASTRUCTURE (same rules as micsa_oracle.c): only
 * tests/, __graft_entry__.smoke() and bench.py's cpu legs may build or call
 * it; it shares no code with paper_2506_16240_b200/csrc/.
 *
 * State, canonical unpacked layout (site i = x + L*(y + L*z), periodic):
 *   s[(sample*R + replica)*N + i]   int8  in {-1,+1}
 *   n[(sample*R + replica)*N + i]   float64 >= 0, the daemon / walker energy
 *   J[(sample*3 + d)*N + i]         float64, bond from site i to its +d neighbour
 *                                   (J ~ N(0,1) in Appendix C; replicas share it)
 *
 * Elementary move (Eq. 8, with NO cap -- "we do not need to
 * limit the capacity of the walkers as in Sec. 2.5, but we can take a step
 * back and use the elementary move described in Sec. 2.3"):
 *   dH = 2 s_x sum_y J_xy s_y;  n' = n - dH;  legal iff n' >= 0; then s_x <- -s_x,
 *   n <- n'.
 * Readings (R18-R21): all arithmetic in IEEE float64 without fused
 * multiply-add; the local field is summed in the fixed order
 *   h = ((((J(+x) s(+x) + J(-x) s(-x)) + J(+y) s(+y)) + J(-y) s(-y)) + J(+z) s(+z)) + J(-z) s(-z)
 * (each product is +-J exactly), dH = (2 s_x) * h, n' = n - dH, accept iff
 * n' >= 0.0.  Refresh (Eq. 9: Prob(0 < n < R) = 1 - exp(-R/T)): one 32-bit
 * Philox word x per daemon, u = (x + 0.5) * 2^-32 in (0,1), n = -T * log(u);
 * counter (i, global sample, (5 << 24) | replica, step), output word 0.
 *
 * Pins (tests/test_oracle_gauss.py): Kolmogorov-Smirnov of the refreshed n
 * against Eq. (9), mean T and variance T^2; conservation of H_EA + sum n to
 * rounding, and EXACT conservation / involution when J = +-1 and n integer;
 * reduction to the capped integer oracle whenever the cap never binds;
 * 2x2x2 Boltzmann average by enumeration with Gaussian J; equilibrium energy
 * against an independent numpy Metropolis; wandering period L.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);   /* micsa_oracle.c */

enum { TAG_GAUSS_REFRESH = 5 };

static inline int wrapg(int a, int L) { return (a + L) % L; }

/* Eq. (9) refresh of every daemon at temperature T, refresh index `step`. */
int oracle_gauss_refresh(int L, int n_samples, int n_replicas, uint64_t seed, double T,
                         uint32_t step, int sample_offset, double *n)
{
    if (!(T > 0.0) || !isfinite(T)) return -1;
    const int64_t N = (int64_t)L * L * L;
    const uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    const int n_sys = n_samples * n_replicas;
#pragma omp parallel for schedule(static)
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas, rep = sys % n_replicas;
        for (int64_t i = 0; i < N; ++i) {
            const uint32_t ctr[4] = { (uint32_t)i, (uint32_t)(sample_offset + sample),
                                      ((uint32_t)TAG_GAUSS_REFRESH << 24) | (uint32_t)rep, step };
            uint32_t out[4];
            oracle_philox4x32_10(ctr, key, out);
            const double u = ((double)out[0] + 0.5) * (1.0 / 4294967296.0);
            n[(int64_t)sys * N + i] = -T * log(u);
        }
    }
    return 0;
}

/* The uniform a daemon's refresh is built on (for the pins). */
double oracle_gauss_uniform(int64_t i, int gsample, int rep, uint32_t step, uint64_t seed)
{
    const uint32_t key[2] = { (uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32) };
    const uint32_t ctr[4] = { (uint32_t)i, (uint32_t)gsample, ((uint32_t)TAG_GAUSS_REFRESH << 24) | (uint32_t)rep, step };
    uint32_t out[4];
    oracle_philox4x32_10(ctr, key, out);
    return ((double)out[0] + 0.5) * (1.0 / 4294967296.0);
}

/* One half-sweep: the elementary move on every site of parity p (PAPER.md:132:
 * the order inside a parity class is immaterial). */
void oracle_gauss_half_sweep(int L, int n_samples, int n_replicas, int8_t *s, double *n,
                             const double *J, int parity)
{
    const int64_t N = (int64_t)L * L * L;
    const int n_sys = n_samples * n_replicas;
#pragma omp parallel for schedule(static)
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas;
        int8_t *S = s + (int64_t)sys * N;
        double *D = n + (int64_t)sys * N;
        const double *Jx = J + ((int64_t)sample * 3 + 0) * N;
        const double *Jy = J + ((int64_t)sample * 3 + 1) * N;
        const double *Jz = J + ((int64_t)sample * 3 + 2) * N;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != parity) continue;
                    const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t ixp = wrapg(x + 1, L) + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t ixm = wrapg(x - 1, L) + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t iyp = x + (int64_t)L * (wrapg(y + 1, L) + (int64_t)L * z);
                    const int64_t iym = x + (int64_t)L * (wrapg(y - 1, L) + (int64_t)L * z);
                    const int64_t izp = x + (int64_t)L * (y + (int64_t)L * wrapg(z + 1, L));
                    const int64_t izm = x + (int64_t)L * (y + (int64_t)L * wrapg(z - 1, L));
                    double h = Jx[i] * (double)S[ixp];
                    h = h + Jx[ixm] * (double)S[ixm];
                    h = h + Jy[i] * (double)S[iyp];
                    h = h + Jy[iym] * (double)S[iym];
                    h = h + Jz[i] * (double)S[izp];
                    h = h + Jz[izm] * (double)S[izm];
                    const double dH = (2.0 * (double)S[i]) * h;     /* change of H_EA if s_i flips (Eq. 1) */
                    const double nn = D[i] - dH;                    /* Eq. (8) */
                    if (nn >= 0.0) { S[i] = (int8_t)(-S[i]); D[i] = nn; }
                }
    }
}

/* Wandering half-cycle: walkers on sites of parity `parity`
 * exchange with their neighbour at +sign along `axis`. */
void oracle_gauss_wander(int L, int n_samples, int n_replicas, double *n, int axis, int sign, int parity)
{
    const int64_t N = (int64_t)L * L * L;
    const int n_sys = n_samples * n_replicas;
#pragma omp parallel for schedule(static)
    for (int sys = 0; sys < n_sys; ++sys) {
        double *D = n + (int64_t)sys * N;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != parity) continue;
                    int c[3] = { x, y, z };
                    c[axis] = wrapg(c[axis] + sign, L);
                    const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t j = c[0] + (int64_t)L * (c[1] + (int64_t)L * c[2]);
                    const double t = D[i]; D[i] = D[j]; D[j] = t;
                }
    }
}

/* E = H_EA of Eq. (1) summed site by site (i ascending, d = x, y, z inside),
 * E_daemon = sum of n (Eq. 4), Q = sum_x s^a s^b for the replica pairs a < b. */
void oracle_gauss_measure(int L, int n_samples, int n_replicas, const int8_t *s, const double *n,
                          const double *J, double *E, double *Edem, int64_t *Q)
{
    const int64_t N = (int64_t)L * L * L;
    const int n_sys = n_samples * n_replicas;
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas;
        const int8_t *S = s + (int64_t)sys * N;
        double e = 0.0, ed = 0.0;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t nb[3] = { wrapg(x + 1, L) + (int64_t)L * (y + (int64_t)L * z),
                                            x + (int64_t)L * (wrapg(y + 1, L) + (int64_t)L * z),
                                            x + (int64_t)L * (y + (int64_t)L * wrapg(z + 1, L)) };
                    for (int d = 0; d < 3; ++d)
                        e -= J[((int64_t)sample * 3 + d) * N + i] * (double)S[i] * (double)S[nb[d]];
                    ed += n[(int64_t)sys * N + i];
                }
        if (E) E[sys] = e;
        if (Edem) Edem[sys] = ed;
    }
    if (Q) {
        int64_t k = 0;
        for (int sample = 0; sample < n_samples; ++sample)
            for (int a = 0; a < n_replicas; ++a)
                for (int b = a + 1; b < n_replicas; ++b) {
                    const int8_t *A = s + ((int64_t)sample * n_replicas + a) * N;
                    const int8_t *B = s + ((int64_t)sample * n_replicas + b) * N;
                    int64_t q = 0;
                    for (int64_t i = 0; i < N; ++i) q += (int64_t)A[i] * (int64_t)B[i];
                    Q[k++] = q;
                }
    }
}
