/*
 * micsa_oracle.c — CPU ORACLE for microcanonical simulated annealing (MicSA).
 *
 * THIS FILE IS TEST INFRASTRUCTURE.  It is a plain, slow, obviously-correct
 * restatement of arxiv/paper_2506_16240 for the 3D +-J
 * Edwards-Anderson spin glass with one capped demon per site.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call it.  It shares no code with the CUDA library in
 * paper_2506_16240_b200/csrc/ and neither includes the other.
 *
 * State, in the canonical unpacked layout used at the C-ABI boundary:
 *   s[(sample*R + replica)*N + i]  in {-1,+1}   spins
 *   m[(sample*R + replica)*N + i]  in {0,1,2,3} demon level, n = 4m
 *
 *   J[(sample*3 + d)*N + i]        in {-1,+1}   bond from site i to its +d
 *                                               neighbour, d = 0,1,2 = x,y,z;
 *                                               replicas share it
 *   site i = x + L*(y + L*z), 0-based, periodic boundaries,
 *   parity (x+y+z) mod 2, parity 0 = "even".
 *
 * No blocking, packing or reordering: every function is the paper's
 * definition written out with serial loops.  The OpenMP pragma only spreads
 * *independent systems* (sample, replica) over host threads; inside a system
 * everything is serial.
 *
 * Pins (tests/test_oracle_*.py, all -m "not gpu"):
 *   philox4x32_10      vs cuRAND's host PHILOX4_32_10 generator (library)
 *   half_sweep         exact conservation of H_EA + H_aux,
 *                      involution, incremental == from-scratch
 *                      energy, all 28 (U, m) cases of Eq. (8)+(10),
 *                      brute-force Boltzmann average on the 2x2x2 lattice,
 *                      agreement with the independent Metropolis oracle
 *   measure            vs an independent numpy (np.roll) evaluation of Eq. (1)
 *   thresholds/refresh histogram vs Eq. (11), mean vs Eq. (12) closed forms
 *   wander             period L, involution, conservation, 2x2x2
 *                      Boltzmann average with walkers
 *   refresh_alpha      family 0 == refresh, families uncorrelated, conservation and the
 *                      2x2x2 Boltzmann average with gamma = 2, 6 daemons and 6 walkers
 *   metropolis_*       acceptance rates exp(-dH/T), 2x2x2 Boltzmann average, the
 *                      independent typewriter Metropolis (metropolis_oracle.c)
 *   c4                 np.roll, line-sum identity, S(r) = S(L-r), special replicas
 * Unpinned by the paper: low-temperature quench curves (configs 3, 4) and the
 * final annealed energies (config 5) -- see DESIGN.md "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ------------------------------------------------------------------ */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw 2011; public algorithm).   */
/* DESIGN.md reading R8.  ctr = 128-bit counter, key = 64-bit key.       */
/* ------------------------------------------------------------------ */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2],
                          uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;              /* key schedule: bumped after each round */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Domain tags of the counter word c2 (R8). */
enum { TAG_REFRESH = 0, TAG_SPIN_INIT = 1, TAG_BOND_INIT = 2, TAG_METROPOLIS = 3 };

static inline void seed_key(uint64_t seed, uint32_t key[2])
{
    key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
    key[1] = (uint32_t)(seed >> 32);
}

static inline int wrap(int a, int L) { return (a + L) % L; }

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ------------------------------------------------------------------ */
/* a0  Initial state (PAPER.md:73 couplings +-1 w.p. 1/2; PAPER.md:223  */
/* "fully disordered" start).  One random bit per spin / bond:          */
/*   spin : ctr = (i, gsample>>7, (1<<24)|replica, 0)                    */
/*   bond : ctr = (i, gsample>>7, (2<<24)|d,       0)                    */
/*   bit (gsample & 31) of output word (gsample>>5)&3; bit 1 <=> -1.     */
/* gsample = sample_offset + sample is the *global* sample index so that */
/* a run sharded by sample over several GPUs reproduces the unsharded    */
/* run (multi-GPU).                                           */
/* ------------------------------------------------------------------ */
void oracle_init_spins(int L, int n_samples, int n_replicas, uint64_t seed,
                       int sample_offset, int8_t *s)
{
    const int64_t N = (int64_t)L * L * L;
    uint32_t key[2]; seed_key(seed, key);
    for (int sample = 0; sample < n_samples; ++sample)
        for (int rep = 0; rep < n_replicas; ++rep)
            for (int64_t i = 0; i < N; ++i) {
                uint32_t g = (uint32_t)(sample_offset + sample);
                uint32_t ctr[4] = { (uint32_t)i, g >> 7,
                                    ((uint32_t)TAG_SPIN_INIT << 24) | (uint32_t)rep, 0u };
                uint32_t out[4];
                oracle_philox4x32_10(ctr, key, out);
                uint32_t bit = (out[(g >> 5) & 3] >> (g & 31)) & 1u;
                s[((int64_t)sample * n_replicas + rep) * N + i] = bit ? -1 : +1;
            }
}

void oracle_init_bonds(int L, int n_samples, uint64_t seed, int sample_offset,
                       int8_t *J)
{
    const int64_t N = (int64_t)L * L * L;
    uint32_t key[2]; seed_key(seed, key);
    for (int sample = 0; sample < n_samples; ++sample)
        for (int d = 0; d < 3; ++d)
            for (int64_t i = 0; i < N; ++i) {
                uint32_t g = (uint32_t)(sample_offset + sample);
                uint32_t ctr[4] = { (uint32_t)i, g >> 7,
                                    ((uint32_t)TAG_BOND_INIT << 24) | (uint32_t)d, 0u };
                uint32_t out[4];
                oracle_philox4x32_10(ctr, key, out);
                uint32_t bit = (out[(g >> 5) & 3] >> (g & 31)) & 1u;
                J[((int64_t)sample * 3 + d) * N + i] = bit ? -1 : +1;
            }
}

/* ------------------------------------------------------------------ */
/* a1/a2  Half-sweep on one lattice parity.     */
/* For every site x of the given parity, in any order:    */
/*   h      = sum over the 6 neighbours y of J_xy s_y       (Eq. 1)       */
/*   dH     = H_EA(after flip) - H_EA(before) = 2 s_x h                   */
/*   n_new  = n_x - dH                                      (Eq. 8)       */
/*   flip s_x and set n_x = n_new iff 0 <= n_new <= 12      (Eq. 10)      */
/* Returns, per system, the number of accepted flips and the sum of dH   */
/* over accepted flips (the incremental energy, pin P4).                 */
/* ------------------------------------------------------------------ */
void oracle_half_sweep(int L, int n_samples, int n_replicas, int parity,
                       int8_t *s, uint8_t *m, const int8_t *J,
                       int64_t *accepted /* [n_sys] or NULL */,
                       int64_t *dE       /* [n_sys] or NULL */)
{
    const int64_t N = (int64_t)L * L * L;
    const int n_sys = n_samples * n_replicas;
#pragma omp parallel for schedule(static) if (N * n_sys > 65536)
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas;
        int8_t  *ss = s + (int64_t)sys * N;
        uint8_t *mm = m + (int64_t)sys * N;
        const int8_t *Jx = J + ((int64_t)sample * 3 + 0) * N;
        const int8_t *Jy = J + ((int64_t)sample * 3 + 1) * N;
        const int8_t *Jz = J + ((int64_t)sample * 3 + 2) * N;
        int64_t acc = 0, de = 0;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != parity) continue;
                    const int64_t i   = x + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t ixp = wrap(x + 1, L) + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t ixm = wrap(x - 1, L) + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t iyp = x + (int64_t)L * (wrap(y + 1, L) + (int64_t)L * z);
                    const int64_t iym = x + (int64_t)L * (wrap(y - 1, L) + (int64_t)L * z);
                    const int64_t izp = x + (int64_t)L * (y + (int64_t)L * wrap(z + 1, L));
                    const int64_t izm = x + (int64_t)L * (y + (int64_t)L * wrap(z - 1, L));
                    /* the bond to the -d neighbour is that neighbour's +d bond */
                    const int h = Jx[i]   * ss[ixp] + Jx[ixm] * ss[ixm]
                                + Jy[i]   * ss[iyp] + Jy[iym] * ss[iym]
                                + Jz[i]   * ss[izp] + Jz[izm] * ss[izm];
                    const int dH = 2 * ss[i] * h;              /* in {0,+-4,+-8,+-12} */
                    const int n_new = 4 * (int)mm[i] - dH;     /* Eq. (8) */
                    if (0 <= n_new && n_new <= 12) {           /* Eq. (10) */
                        ss[i] = (int8_t)(-ss[i]);
                        mm[i] = (uint8_t)(n_new / 4);
                        ++acc; de += dH;
                    }
                }
        if (accepted) accepted[sys] = acc;
        if (dE) dE[sys] = de;
    }
}

/* Sweep = even half-sweep, then odd half-sweep. gamma = 1. */
void oracle_sweep(int L, int n_samples, int n_replicas, int n_sweeps,
                  int8_t *s, uint8_t *m, const int8_t *J)
{
    for (int t = 0; t < n_sweeps; ++t) {
        oracle_half_sweep(L, n_samples, n_replicas, 0, s, m, J, NULL, NULL);
        oracle_half_sweep(L, n_samples, n_replicas, 1, s, m, J, NULL, NULL);
    }
}

/* ------------------------------------------------------------------ */
/* NEXT-1  Walkers (Sec. 2.6).  One half of the        */
/* two-timestep wandering cycle along axis d (0,1,2 = X,Y,Z), direction  */
/* sign (+1 forward, -1 backward): every walker sitting on a site of the */
/* given lattice parity exchanges its value with the walker on that      */
/* site's nearest neighbour along sign*d (periodic; the neighbour has    */
/* the other parity, L even).  PAPER.md:172-174: even sites exchange at  */
/* the first timestep of a cycle, odd sites at the second.  Spins are    */
/* not touched.                                                          */
/* ------------------------------------------------------------------ */
void oracle_wander(int L, int n_samples, int n_replicas, int axis, int sign,
                   int parity, uint8_t *m)
{
    const int64_t N = (int64_t)L * L * L;
    const int n_sys = n_samples * n_replicas;
    for (int sys = 0; sys < n_sys; ++sys) {
        uint8_t *mm = m + (int64_t)sys * N;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != parity) continue;
                    const int xn = (axis == 0) ? wrap(x + sign, L) : x;
                    const int yn = (axis == 1) ? wrap(y + sign, L) : y;
                    const int zn = (axis == 2) ? wrap(z + sign, L) : z;
                    const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t j = xn + (int64_t)L * (yn + (int64_t)L * zn);
                    const uint8_t tmp = mm[i]; mm[i] = mm[j]; mm[j] = tmp;
                }
    }
}

/* Timesteps with gamma = 1 walker per spin, forward-X wandering          */
/* (Sec. 2.8.1 step 3): each step = one sweep,     */
/* then the half of the wandering cycle dictated by the parity of the     */
/* time index t (even t: walkers on even sites exchange), then t += 1.    */
void oracle_timesteps_walkers(int L, int n_samples, int n_replicas, int n_steps,
                              int64_t t0, int8_t *s, uint8_t *m, const int8_t *J)
{
    for (int64_t t = t0; t < t0 + n_steps; ++t) {
        oracle_half_sweep(L, n_samples, n_replicas, 0, s, m, J, NULL, NULL);
        oracle_half_sweep(L, n_samples, n_replicas, 1, s, m, J, NULL, NULL);
        oracle_wander(L, n_samples, n_replicas, 0, +1, (int)(t & 1), m);
    }
}

/* ------------------------------------------------------------------ */
/* a3  Demon refresh (PAPER.md:154-157 Eq. 11, :190).                    */
/* Thresholds (R7), float64, this exact operation order:       */
/*   x = exp(-4/T); x2 = x*x; x3 = x2*x; Z = ((1 + x) + x2) + x3          */
/*   c0 = 1/Z; c1 = (1 + x)/Z; c2 = ((1 + x) + x2)/Z   (cumulative p)     */
/*   thr[k] = floor(c_k * 2^32) as uint64 in [0, 2^32]                    */
/* Draw: u = one 32-bit uniform per demon; m = #{k : u >= thr[k]}.        */
/* ------------------------------------------------------------------ */
int oracle_thresholds(double T, uint64_t thr[3])
{
    if (!(T > 0.0) || !isfinite(T)) return -1;
    const double x  = exp(-4.0 / T);
    const double x2 = x * x;
    const double x3 = x2 * x;
    const double Z  = ((1.0 + x) + x2) + x3;
    const double c[3] = { 1.0 / Z, (1.0 + x) / Z, ((1.0 + x) + x2) / Z };
    for (int k = 0; k < 3; ++k) {
        double t = floor(ldexp(c[k], 32));
        if (t > 4294967296.0) t = 4294967296.0;
        thr[k] = (uint64_t)t;
    }
    return 0;
}

/* The 32-bit uniform u of one demon (R8; the paper does not say
 * how the refresh draws its random numbers, north_star asks for Philox keyed
 * by seed, sample, site and refresh index).  u is assembled most significant
 * bit first from 32 random bit-planes; the planes of the 16 global samples
 * g with the same g>>4 (same site, replica, step) come from four Philox
 * calls c = 0..3 with
 *     ctr = (i, (g>>4) | (c<<28), (0<<24) | replica, step),  key = (seed lo, hi)
 * plane k = 8c + 2j + h is the 16-bit half h (0 = low, 1 = high) of output
 * word j of call c, and sample g owns bit (g & 15) of it:
 *     u = sum_k  bit_k * 2^(31-k).
 * Every bit of every output word is used by exactly one demon, so u is a
 * uniform 32-bit integer and distinct demons are independent. */
static uint32_t tagged_uniform(uint32_t tag, uint32_t i, uint32_t g, uint32_t rep,
                               uint32_t step, const uint32_t key[2])
{
    uint32_t u = 0;
    for (uint32_t c = 0; c < 4; ++c) {
        uint32_t ctr[4] = { i, (g >> 4) | (c << 28), (tag << 24) | rep, step };
        uint32_t out[4];
        oracle_philox4x32_10(ctr, key, out);
        for (uint32_t j = 0; j < 4; ++j)
            for (uint32_t h = 0; h < 2; ++h) {
                const uint32_t k = 8 * c + 2 * j + h;           /* 0 = most significant */
                const uint32_t bit = (out[j] >> (16 * h + (g & 15))) & 1u;
                u |= bit << (31 - k);
            }
    }
    return u;
}

static uint32_t refresh_uniform(uint32_t i, uint32_t g, uint32_t rep,
                                uint32_t step, const uint32_t key[2])
{
    return tagged_uniform((uint32_t)TAG_REFRESH, i, g, rep, step, key);
}

/* Debug/test hook: the uniform itself (pins: uniformity, bit independence). */
uint32_t oracle_refresh_uniform(uint32_t i, uint32_t g, uint32_t rep,
                                uint32_t step, uint64_t seed)
{
    uint32_t key[2]; seed_key(seed, key);
    return refresh_uniform(i, g, rep, step, key);
}

/* Refresh of the alpha-th family of auxiliary variables (PAPER.md:196-198:
 * gamma daemons n_{x,alpha} per spin): the same draw with alpha in bits 20..23
 * of the counter word that carries the replica (replica < 2^20), so that the
 * gamma families are independent and alpha = 0 is the single-daemon refresh. */
int oracle_refresh_alpha(int L, int n_samples, int n_replicas, uint64_t seed,
                         int sample_offset, double T, uint32_t step, int alpha, uint8_t *m)
{
    const int64_t N = (int64_t)L * L * L;
    uint64_t thr[3];
    if (oracle_thresholds(T, thr) != 0 || alpha < 0 || alpha > 15) return -1;
    uint32_t key[2]; seed_key(seed, key);
    const int n_sys = n_samples * n_replicas;
#pragma omp parallel for schedule(static) if (N * n_sys > 65536)
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas, rep = sys % n_replicas;
        const uint32_t g = (uint32_t)(sample_offset + sample);
        uint8_t *mm = m + (int64_t)sys * N;
        for (int64_t i = 0; i < N; ++i) {
            const uint64_t u = (uint64_t)refresh_uniform((uint32_t)i, g, ((uint32_t)alpha << 20) | (uint32_t)rep,
                                                         step, key);
            mm[i] = (uint8_t)((u >= thr[0]) + (u >= thr[1]) + (u >= thr[2]));
        }
    }
    return 0;
}

/* Refresh: every demon <- #{k : u >= thr[k]} with its own u (Eq. 11). */
int oracle_refresh(int L, int n_samples, int n_replicas, uint64_t seed,
                   int sample_offset, double T, uint32_t step, uint8_t *m)
{
    const int64_t N = (int64_t)L * L * L;
    uint64_t thr[3];
    if (oracle_thresholds(T, thr) != 0) return -1;
    uint32_t key[2]; seed_key(seed, key);
    const int n_sys = n_samples * n_replicas;
#pragma omp parallel for schedule(static) if (N * n_sys > 65536)
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas, rep = sys % n_replicas;
        const uint32_t g = (uint32_t)(sample_offset + sample);
        uint8_t *mm = m + (int64_t)sys * N;
        for (int64_t i = 0; i < N; ++i) {
            const uint64_t u = (uint64_t)refresh_uniform((uint32_t)i, g, (uint32_t)rep, step, key);
            mm[i] = (uint8_t)((u >= thr[0]) + (u >= thr[1]) + (u >= thr[2]));
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* NEXT-3  Canonical comparator: standard Metropolis on the same         */
/* checkerboard (Table 3; a fresh random   */
/* number per spin-flip attempt).  Flip s_x with probability             */
/* min(1, exp(-dH/T)), dH = 2 s_x h in {0,+-4,+-8,+-12}:                  */
/*   accept iff dH <= 0 or u < thr[dH/4 - 1],                             */
/*   thr[k] = floor(exp(-4/T)^(k+1) * 2^32), this operation order:        */
/*   x = exp(-4/T); x2 = x*x; x3 = x2*x; capped at 2^32                   */
/* u = the attempt's own 32-bit uniform: the bit-sliced map of the        */
/* refresh (R8) with domain tag 3 and the sweep index tau in    */
/* the counter word the refresh uses for its step -- every site is        */
/* attempted once per sweep, so (site, sample, replica, tau) is unique.   */
/* ------------------------------------------------------------------ */
int oracle_metropolis_thresholds(double T, uint64_t thr[3])
{
    if (!(T > 0.0) || !isfinite(T)) return -1;
    const double x  = exp(-4.0 / T);
    const double x2 = x * x;
    const double x3 = x2 * x;
    const double p[3] = { x, x2, x3 };
    for (int k = 0; k < 3; ++k) {
        double t = floor(ldexp(p[k], 32));
        if (t > 4294967296.0) t = 4294967296.0;
        thr[k] = (uint64_t)t;
    }
    return 0;
}

int oracle_metropolis_half_sweep(int L, int n_samples, int n_replicas, uint64_t seed,
                                 int sample_offset, double T, uint32_t tau, int parity,
                                 int8_t *s, const int8_t *J)
{
    const int64_t N = (int64_t)L * L * L;
    uint64_t thr[3];
    if (oracle_metropolis_thresholds(T, thr) != 0) return -1;
    uint32_t key[2]; seed_key(seed, key);
    const int n_sys = n_samples * n_replicas;
#pragma omp parallel for schedule(static) if (N * n_sys > 65536)
    for (int sys = 0; sys < n_sys; ++sys) {
        const int sample = sys / n_replicas, rep = sys % n_replicas;
        const uint32_t g = (uint32_t)(sample_offset + sample);
        int8_t *ss = s + (int64_t)sys * N;
        const int8_t *Jx = J + ((int64_t)sample * 3 + 0) * N;
        const int8_t *Jy = J + ((int64_t)sample * 3 + 1) * N;
        const int8_t *Jz = J + ((int64_t)sample * 3 + 2) * N;
        for (int z = 0; z < L; ++z)
            for (int y = 0; y < L; ++y)
                for (int x = 0; x < L; ++x) {
                    if (((x + y + z) & 1) != parity) continue;
                    const int64_t i   = x + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t ixp = wrap(x + 1, L) + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t ixm = wrap(x - 1, L) + (int64_t)L * (y + (int64_t)L * z);
                    const int64_t iyp = x + (int64_t)L * (wrap(y + 1, L) + (int64_t)L * z);
                    const int64_t iym = x + (int64_t)L * (wrap(y - 1, L) + (int64_t)L * z);
                    const int64_t izp = x + (int64_t)L * (y + (int64_t)L * wrap(z + 1, L));
                    const int64_t izm = x + (int64_t)L * (y + (int64_t)L * wrap(z - 1, L));
                    const int h = Jx[i]   * ss[ixp] + Jx[ixm] * ss[ixm]
                                + Jy[i]   * ss[iyp] + Jy[iym] * ss[iym]
                                + Jz[i]   * ss[izp] + Jz[izm] * ss[izm];
                    const int dH = 2 * ss[i] * h;
                    int accept = (dH <= 0);
                    if (!accept) {
                        const uint64_t u = (uint64_t)tagged_uniform((uint32_t)TAG_METROPOLIS, (uint32_t)i, g,
                                                                    (uint32_t)rep, tau, key);
                        accept = (u < thr[dH / 4 - 1]);
                    }
                    if (accept) ss[i] = (int8_t)(-ss[i]);
                }
    }
    return 0;
}

/* n Metropolis sweeps (even sites, then odd sites) with sweep indices tau0, tau0+1, ... */
int oracle_metropolis_sweep(int L, int n_samples, int n_replicas, uint64_t seed,
                            int sample_offset, double T, uint32_t tau0, int n_sweeps,
                            int8_t *s, const int8_t *J)
{
    for (int t = 0; t < n_sweeps; ++t)
        for (int parity = 0; parity < 2; ++parity)
            if (oracle_metropolis_half_sweep(L, n_samples, n_replicas, seed, sample_offset, T,
                                             tau0 + (uint32_t)t, parity, s, J) != 0) return -1;
    return 0;
}

/* ------------------------------------------------------------------ */
/* a4-a6  Measurements, exact integer sums.                              */
/*   E[sys]    = -sum_i sum_d J[d][i] s[i] s[i+d]      (Eq. 1)            */
/*   Edem[sys] = sum_i 4 m[i]                          (Eq. 4, n = 4m)    */
/*   Q[sample][pair(a<b)] = sum_i s^a[i] s^b[i]        (Eq. C.1 times N)  */
/* Pairs ordered (0,1),(0,2),...,(1,2),... lexicographically.            */
/* ------------------------------------------------------------------ */
void oracle_measure(int L, int n_samples, int n_replicas,
                    const int8_t *s, const uint8_t *m, const int8_t *J,
                    int64_t *E, int64_t *Edem, int64_t *Q)
{
    const int64_t N = (int64_t)L * L * L;
    const int n_sys = n_samples * n_replicas;
    if (E) {
#pragma omp parallel for schedule(static) if (N * n_sys > 65536)
        for (int sys = 0; sys < n_sys; ++sys) {
            const int sample = sys / n_replicas;
            const int8_t *ss = s + (int64_t)sys * N;
            int64_t e = 0;
            for (int z = 0; z < L; ++z)
                for (int y = 0; y < L; ++y)
                    for (int x = 0; x < L; ++x) {
                        const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
                        const int64_t nb[3] = {
                            wrap(x + 1, L) + (int64_t)L * (y + (int64_t)L * z),
                            x + (int64_t)L * (wrap(y + 1, L) + (int64_t)L * z),
                            x + (int64_t)L * (y + (int64_t)L * wrap(z + 1, L)) };
                        for (int d = 0; d < 3; ++d)
                            e -= (int64_t)J[((int64_t)sample * 3 + d) * N + i] * ss[i] * ss[nb[d]];
                    }
            E[sys] = e;
        }
    }
    if (Edem) {
        for (int sys = 0; sys < n_sys; ++sys) {
            const uint8_t *mm = m + (int64_t)sys * N;
            int64_t a = 0;
            for (int64_t i = 0; i < N; ++i) a += 4 * (int64_t)mm[i];
            Edem[sys] = a;
        }
    }
    if (Q) {
        int64_t k = 0;
        for (int sample = 0; sample < n_samples; ++sample)
            for (int a = 0; a < n_replicas; ++a)
                for (int b = a + 1; b < n_replicas; ++b) {
                    const int8_t *sa = s + ((int64_t)sample * n_replicas + a) * N;
                    const int8_t *sb = s + ((int64_t)sample * n_replicas + b) * N;
                    int64_t q = 0;
                    for (int64_t i = 0; i < N; ++i) q += (int64_t)sa[i] * sb[i];
                    Q[k++] = q;
                }
    }
}

/* ------------------------------------------------------------------ */
/* NEXT-2  Four-point replica correlation along the axes, Eq. (16)       */
/* before the normalisation and the average over      */
/* axes: for the replica pair (a<b) of a sample, axis d and r = 0..L/2,   */
/*   S[pair][d][r] = sum_x q_x q_{x + r e_d},  q_x = s^a_x s^b_x,          */
/* periodic.  C4(r) = (S[.][0][r] + S[.][1][r] + S[.][2][r]) / (3N) for    */
/* one pair.  Pairs ordered like Q in oracle_measure.                     */
/* ------------------------------------------------------------------ */
void oracle_c4(int L, int n_samples, int n_replicas, const int8_t *s, int64_t *S)
{
    const int64_t N = (int64_t)L * L * L;
    const int R = L / 2 + 1;
    int64_t k = 0;
    for (int sample = 0; sample < n_samples; ++sample)
        for (int a = 0; a < n_replicas; ++a)
            for (int b = a + 1; b < n_replicas; ++b, ++k) {
                const int8_t *sa = s + ((int64_t)sample * n_replicas + a) * N;
                const int8_t *sb = s + ((int64_t)sample * n_replicas + b) * N;
                for (int d = 0; d < 3; ++d)
                    for (int r = 0; r < R; ++r) {
                        int64_t acc = 0;
                        for (int z = 0; z < L; ++z)
                            for (int y = 0; y < L; ++y)
                                for (int x = 0; x < L; ++x) {
                                    const int xn = (d == 0) ? wrap(x + r, L) : x;
                                    const int yn = (d == 1) ? wrap(y + r, L) : y;
                                    const int zn = (d == 2) ? wrap(z + r, L) : z;
                                    const int64_t i = x + (int64_t)L * (y + (int64_t)L * z);
                                    const int64_t j = xn + (int64_t)L * (yn + (int64_t)L * zn);
                                    acc += (int64_t)(sa[i] * sb[i]) * (sa[j] * sb[j]);
                                }
                        S[(k * 3 + d) * R + r] = acc;
                    }
            }
}

