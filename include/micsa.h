/*
 * micsa.h -- C ABI of the B200-native MicSA library (libmicsa.so).
 *
 * Microcanonical simulated annealing for the 3D +-J Edwards-Anderson spin
 * glass, arxiv/paper_2506_16240 (citations are PAPER.md:<line>).  Capped
 * daemons n in {0,4,8,12}, one per spin by default (gamma = 1; up to 6
 * families and walkers: micsa_set_gamma, micsa_set_walkers); checkerboard
 * sweeps without random numbers; sporadic Philox-driven daemon refresh; E /
 * E_daemon / q reductions and C4; a Metropolis comparator on the same layout.
 * Every step runs in hand-written CUDA kernels for sm_100a; there
 * is no CPU fallback: every call fails with MICSA_ERR_CUDA when no device is
 * usable.
 *
 * Conventions
 *   N = L^3 sites, site i = x + L*(y + L*z), 0-based, periodic.
 *   parity(i) = (x+y+z) mod 2; parity 0 = "even" sublattice.
 *   system  = (sample, replica); sys = sample*n_replicas + replica;
 *             n_sys = n_samples*n_replicas.  Replicas of a sample share its
 *             couplings.
 *   Canonical (unpacked) host layouts -- the byte-for-byte parity surface:
 *     spins   int8   [n_samples][n_replicas][N]   values -1 / +1
 *     daemons uint8  [n_samples][n_replicas][N]   level m in 0..3, n = 4m
 *
 *     bonds   int8   [n_samples][3][N]            J[s][d][i] = coupling between
 *                                                 site i and its +d neighbour,
 *                                                 d = 0,1,2 = x,y,z
 *   On the device the state is bit-sliced across systems (1 bit per spin,
 *   2 bit-planes per daemon); that layout is private.
 *
 * Pointers: "host" = ordinary (pageable or pinned) host memory owned by the
 * caller; the library copies in/out and never keeps the pointer.  "device" =
 * CUDA device memory.  All calls on one context must come from one thread at
 * a time.  Work is queued on the context's stream; calls documented as
 * "synchronous" wait for it.
 *
 * Errors: every int-returning call gives MICSA_OK (0) or a negative code and
 * leaves the state unchanged on MICSA_ERR_INVALID.  CUDA errors are sticky on
 * the context.  Nothing is printed, nothing aborts.
 */
#ifndef MICSA_H
#define MICSA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MICSA_OK            0
#define MICSA_ERR_INVALID  (-1)   /* bad argument */
#define MICSA_ERR_NOMEM    (-2)   /* host or device allocation failed */
#define MICSA_ERR_CUDA     (-3)   /* CUDA runtime error (sticky) */

typedef struct micsa_ctx micsa_ctx;

/* One step of an annealing schedule (Sec. 2.8.1, with an
 * explicit list of steps instead of the 2^s rule):
 * refresh all daemons at temperature T, then n_sweeps sweeps (timesteps of
 * gamma sweeps plus wandering when micsa_set_gamma / micsa_set_walkers are in
 * force); after every measure_every-th of them (0 = never) one measurement row
 * is taken. */
typedef struct micsa_step {
    double  T;
    int32_t n_sweeps;
    int32_t measure_every;
} micsa_step;

/* Caller-owned host arrays receiving the measurement rows of micsa_anneal.
 * Row r holds the exact integer sums after global sweep number sweep[r]
 * (counted from 1 within the call).  Any array pointer may be NULL. */
typedef struct micsa_trace {
    int64_t  capacity;     /* in: rows the arrays can hold                      */
    int64_t  n_rows;       /* out: rows the schedule produced (may exceed
                              capacity; only the first `capacity` are stored)   */
    int64_t *sweep;        /* [capacity]                                        */
    double  *T;            /* [capacity]                                        */
    int64_t *E;            /* [capacity][n_sys]      H_EA, Eq. (1)              */
    int64_t *E_daemon;     /* [capacity][n_sys]      H_aux = sum of n, Eq. (4)  */
    int64_t *Q;            /* [capacity][n_pairs]    N*q, Eq. (C.1)             */
} micsa_trace;

/* Static description of the last error on this thread ("" if none). */
const char *micsa_last_error(void);

/* ---- life cycle ---------------------------------------------------------
 * micsa_create: allocates device state on the current CUDA device and the
 * default stream, then initialises it with Philox4x32-10 keyed by `seed`
 * (R8): spins i.i.d. +-1 ("fully disordered" start),
 * bonds i.i.d. +-1 with p = 1/2, daemons 0.
 * Errors (NULL returned, see micsa_last_error): L < 2 or L odd (checkerboard
 * with periodic boundaries needs even L), n_samples < 1,
 * n_replicas < 1, N*n_sys overflow, no device, out of memory.
 *
 * micsa_create_ex: same, with
 *   sample_offset  global index of this context's first sample; Philox
 *                  counters use sample_offset + sample, so a run sharded by
 *                  sample over several GPUs reproduces the unsharded run.
 *                  Must be a multiple of 16 (the sample block of the refresh,
 *                  DESIGN.md R8) and >= 0.
 *   dev_workspace  device memory of at least micsa_workspace_bytes(...) bytes,
 *                  256-byte aligned, owned by the caller (e.g. a torch tensor)
 *                  and kept alive until micsa_destroy; NULL = the library
 *                  allocates with cudaMalloc.
 *   cuda_stream    a cudaStream_t passed as void*; NULL = default stream.     */
micsa_ctx *micsa_create(int L, int n_samples, int n_replicas, uint64_t seed);
micsa_ctx *micsa_create_ex(int L, int n_samples, int n_replicas, uint64_t seed,
                           int sample_offset, void *dev_workspace,
                           size_t workspace_bytes, void *cuda_stream);
size_t     micsa_workspace_bytes(int L, int n_samples, int n_replicas);
int        micsa_destroy(micsa_ctx *ctx);            /* NULL is a no-op */
int        micsa_synchronize(micsa_ctx *ctx);        /* waits for the stream */

/* ---- state in / out (canonical layouts above; host pointers; synchronous) -
 * micsa_set_couplings: J = +-1 with replicas sharing the sample's bonds; any
 * other value -> MICSA_ERR_INVALID and the stored bonds are unchanged.
 * micsa_set_spins / micsa_set_daemons: same rule (values +-1 / 0..3).
 * micsa_get_state: any of s, m, J may be NULL.                               */
int micsa_set_couplings(micsa_ctx *ctx, const int8_t *J);
int micsa_set_spins(micsa_ctx *ctx, const int8_t *s);
int micsa_set_daemons(micsa_ctx *ctx, const uint8_t *m);
int micsa_set_demons(micsa_ctx *ctx, const uint8_t *m);   /* same call, SURVEY.md 8(b) spelling */
int micsa_get_state(micsa_ctx *ctx, int8_t *s, uint8_t *m, int8_t *J);

/* ---- the hot path ------------------------------------------------------
 * micsa_sweep: n full sweeps; one sweep = elementary move on all even sites,
 * then on all odd sites.  Elementary move on site x
 * (PAPER.md:119-124 Eq. 8, :150 Eq. 10): dH = change of H_EA if s_x flips;
 * if 0 <= n_x - dH <= 12 then s_x <- -s_x, n_x <- n_x - dH; else nothing.
 * No random numbers.  Asynchronous.  n < 0 -> MICSA_ERR_INVALID; n = 0 no-op.
 * micsa_half_sweep: the move on one parity only (0 even, 1 odd); applying it
 * twice restores the state.                                   */
int micsa_sweep(micsa_ctx *ctx, int n);
int micsa_half_sweep(micsa_ctx *ctx, int parity);

/* ---- walkers (PAPER.md:163-178 Sec. 2.6, :196-217 Sec. 2.8) ---------------
 * micsa_wander: one half of the two-timestep wandering cycle along axis
 * (0,1,2 = X,Y,Z) in direction sign (+1 forward, -1 backward): every walker
 * (auxiliary variable) on a site of lattice parity `parity` exchanges its
 * value with the walker on that site's neighbour along sign*axis, periodic.
 * Even sites exchange at the first timestep of a cycle, odd sites at the
 * second.  Spins untouched.  Asynchronous.
 *
 * micsa_set_walkers(mode): 0 (default) = the auxiliary variables are daemons
 * bound to their site; 1 = one forward-X walker per spin (the paper's gamma = 1
 * walker variant): micsa_sweep, micsa_sweep_measure and
 * micsa_anneal then run TIMESTEPS -- a sweep, then micsa_wander(0, +1, t & 1),
 * then t += 1.  t is the context's time index: sweeps done
 * through those calls since create (timesteps, when gamma > 1), settable with
 * micsa_set_time (a refresh does not reset it; micsa_half_sweep does not advance
 * it).  micsa_wander acts on the daemon family chosen with
 * micsa_select_daemon_set.  For gamma > 1 see micsa_set_gamma. */
/* gamma daemons per spin: micsa_set_gamma(gamma), gamma = 1..6
 * (the paper tests 1, 2, 4, 6), keeps gamma families n_{x,alpha} of auxiliary
 * variables; a new family starts at level 0.  micsa_sweep / micsa_sweep_measure
 * / micsa_anneal then run TIMESTEPS of gamma sweeps, the alpha-th sweep of a
 * timestep using family alpha; micsa_refresh_demons redraws every family (the
 * family index sits in bits 20..23 of the Philox counter word that carries the
 * replica, so family 0 is the gamma = 1 refresh and n_replicas < 2^20);
 * E_daemon sums over the families; a prefetched refresh covers every family.
 * micsa_set_daemons / micsa_get_state address the family chosen with
 * micsa_select_daemon_set(alpha) (default 0).  With walkers on
 * (micsa_set_walkers(1)) family alpha wanders along the alpha-th direction of
 * PAPER.md:204 Eq. (13) -- forward X, Y, Z, backward X, Y, Z -- after the gamma
 * sweeps of a timestep (the paper uses gamma = 6 for all six; smaller gamma
 * takes the first gamma rows).  Synchronises the stream. */
int micsa_set_gamma(micsa_ctx *ctx, int gamma);
int micsa_select_daemon_set(micsa_ctx *ctx, int alpha);
int micsa_wander(micsa_ctx *ctx, int axis, int sign, int parity);
int micsa_set_walkers(micsa_ctx *ctx, int mode);
int micsa_set_time(micsa_ctx *ctx, int64_t t);
int micsa_get_time(micsa_ctx *ctx, int64_t *t);

/* ---- canonical comparator (PAPER.md:339-350 Table 3, :130) -----------------
 * micsa_metropolis_sweep: n standard Metropolis sweeps (even sites, then odd
 * sites) at temperature T on the same spins and couplings: flip with
 * probability min(1, exp(-dH/T)); daemons are neither read nor written.  One
 * 32-bit uniform per attempt, defined bit-sliced like the refresh's (DESIGN.md
 * 2.1) with domain tag 3 and the sweep index tau0 + k where the refresh has its
 * step; accept iff dH <= 0 or u < floor(exp(-dH/T) * 2^32)
 * (micsa_debug_metropolis_thresholds gives the three integers for dH = 4, 8,
 * 12).  The caller chooses tau0 so that sweep indices never repeat.
 * micsa_metropolis_half_sweep: one parity, index tau.  Asynchronous. */
int micsa_metropolis_sweep(micsa_ctx *ctx, double T, uint32_t tau0, int n);
int micsa_metropolis_half_sweep(micsa_ctx *ctx, double T, uint32_t tau, int parity);
int micsa_debug_metropolis_thresholds(double T, uint64_t thr[3]);

/* micsa_refresh_demons: every daemon <- independent draw from Eq. (11),
 * p(n=4m) ~ exp(-4m/T), m = 0..3; spins untouched
 * (PAPER.md:190).  One 32-bit uniform u per daemon, compared with integer
 * thresholds floor(cdf_k * 2^32) computed on the host (R7).  u is
 * defined bit-sliced (R8): the 16 samples gs of block gs/16 share
 * four Philox4x32-10 calls c = 0..3, counter = (site i, gs/16 | c<<28,
 * replica, step), key = seed; bit-plane k = 8c+2j+h is the 16-bit half h of
 * output word j of call c, sample gs owns bit gs%16 and u = sum_k bit_k <<
 * (31-k).  Same (seed, step, T) => same daemons whatever happened before.
 * Asynchronous.  T must be finite and > 0. */
int micsa_refresh_demons(micsa_ctx *ctx, double T, uint32_t step);

/* micsa_prefetch_refresh: the refreshed levels depend only on (seed, T, step),
 * never on the state (PAPER.md:190 -- the old daemons are thrown away), so the
 * next refresh can be generated while the sweeps run, as the paper's own
 * implementation does on CPU threads.  This call queues the
 * generation of refresh (T, step) into a second pair of daemon planes on a
 * library-owned side stream; it starts when the context's stream reaches this
 * point.  A later micsa_refresh_demons with exactly the same (T, step) then
 * only waits for it and swaps plane pointers; any other (T, step) is generated
 * directly as usual, and the prefetched planes stay valid until consumed or
 * replaced by another prefetch.  Results are bit-identical either way.
 * micsa_anneal prefetches step k+1 under the sweeps of step k by itself when
 * the context's stream has a HIGHER priority than the default (bench.py and
 * run_configs create one): the side stream has the lowest priority, so the
 * generation then only fills what the sweeps leave idle.  On a stream of
 * default priority the two grids would take turns block by block (measured:
 * 366 us per step of config 4 instead of 243), so there micsa_anneal generates
 * its refreshes in line (251 us); large lattices only -- beside the clusters of
 * a small lattice most SMs are idle and the prefetch is always used.  With gamma > 1 every family gets its own staging
 * pair (allocated at the first prefetch: MICSA_ERR_NOMEM if that fails, nothing
 * changed).  Asynchronous.  T must be finite and > 0. */
int micsa_prefetch_refresh(micsa_ctx *ctx, double T, uint32_t step);

/* micsa_effective_temperature (host arithmetic only): the temperature at which
 * Eq. (12) gives the measured daemon energy per auxiliary
 * variable, <H_aux>/(gamma N) = E_daemon / (gamma N) -- the instantaneous
 * temperature of the daemons / walkers.  The argument must lie
 * strictly between 0 (T -> 0) and 6 (T -> infinity). */
int micsa_effective_temperature(double e_daemon_per_variable, double *T);

/* The thresholds micsa_refresh_demons uses: thr[k] = floor(cdf_k * 2^32),
 * k = 0,1,2, each in [0, 2^32]; level m = #{k : u >= thr[k]}.               */
int micsa_debug_thresholds(double T, uint64_t thr[3]);

/* Test hook (pin P6, R8): the library's own device Philox4x32-10.
 * counters = host array [n][4] of counter words (c0, c1, c2, c3), out = host
 * array [n][4] receiving the four output words of each; key = (seed low 32
 * bits, seed high 32 bits).  Synchronous, default stream, no context needed.
 * Errors: NULL pointer / n < 0 -> MICSA_ERR_INVALID; no device -> MICSA_ERR_CUDA. */
int micsa_debug_philox(uint64_t seed, const uint32_t *counters, int n, uint32_t *out);

/* micsa_measure_i64 (synchronous): exact integer sums into host arrays, any
 * may be NULL:
 *   E[n_sys]        H_EA = -sum_<xy> J s s                 (Eq. 1)
 *   E_daemon[n_sys] H_aux = sum_x n_x = 4 sum_x m_x        (Eq. 4)
 *   Q[n_samples * n_replicas(n_replicas-1)/2]  sum_x s^a_x s^b_x for replica
 *                   pairs a < b of each sample, pairs in lexicographic order
 *                                                          (PAPER.md:441 C.1)
 * micsa_measure: the same divided by N as float64 (e of Eq. 15, PAPER.md:255;
 * q of Eq. C.1).  Q != NULL with n_replicas < 2 -> MICSA_ERR_INVALID.        */
int micsa_measure_i64(micsa_ctx *ctx, int64_t *E, int64_t *E_daemon, int64_t *Q);

/* micsa_measure_c4 (synchronous): four-point replica correlation along the
 * lattice axes, Eq. (16), as exact integer sums for EVERY
 * replica pair a < b of every sample (pairs ordered like Q of micsa_measure;
 * n_replicas < 2 -> MICSA_ERR_INVALID):
 *   S[n_samples][n_replicas (n_replicas - 1) / 2][3][L/2 + 1],
 *   S[s][pair][d][r] = sum_x q_x q_{x + r e_d},  q = s^a s^b, periodic; d = 0,1,2 = x,y,z.
 * C4(r) of Eq. (16) for a sample = sum over its pairs and the three axes /
 * (3 N n_replicas (n_replicas - 1) / 2).  Caller-owned host array.
 *
 * micsa_xi (host arithmetic on L/2 + 1 numbers, no context): the integrals
 * I_n = int r^n C4(r) dr, n = 1, 2, 3 (Eq. 17) and the lengths
 * xi_12 = I_2 / I_1, xi_23 / xi_12 = I_3 I_1 / I_2^2 (Eq. 18).
 * The paper defers the estimation of I_n to its refs. [61, 46]; the reading
 * taken here (R22): C4[r] is given at r = 0 .. n_r - 1, trapezoidal
 * rule, integration stops before the first C4[r] <= c_min (the caller's noise
 * floor, e.g. three times the sample error), no tail.  I = double[3] or NULL.
 * Fewer than two points above the floor -> MICSA_ERR_INVALID. */
int micsa_measure_c4(micsa_ctx *ctx, int64_t *S);
int micsa_xi(const double *C4, int n_r, double c_min, double I[3], double *xi12,
             double *xi23_over_xi12);

/* The same measurement split in two, so that the caller can queue more work
 * (or stop a timer on the stream) before waiting: micsa_measure_begin queues
 * the reduction kernel and the device->host copy of the row into pinned memory
 * owned by the context and returns at once; micsa_measure_end waits for the
 * stream and copies the sums out (same arrays and rules as micsa_measure_i64;
 * MICSA_ERR_INVALID without a preceding _begin).  The row is the state at the
 * point of _begin in stream order. */
int micsa_measure_begin(micsa_ctx *ctx);
/* micsa_sweep_measure(n) == micsa_sweep(n) followed by micsa_measure_begin(),
 * with the counting done inside the two launches of the last sweep (after a
 * sweep every bond has exactly one odd end, whose half-sweep holds all its six
 * bonds in registers), so the state is not read a second time.  Falls back to
 * the separate measurement kernel when n == 0, n_replicas > 2, L % 8 != 0 or
 * another sweep kernel is selected.  Same bits either way. */
int micsa_sweep_measure(micsa_ctx *ctx, int n);
int micsa_measure_end(micsa_ctx *ctx, int64_t *E, int64_t *E_daemon, int64_t *Q);
int micsa_measure(micsa_ctx *ctx, double *energy, double *demon_energy,
                  double *q_overlap);

/* micsa_measure_noalloc: micsa_measure_i64 for callers that cannot allocate or
 * synchronise (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc).  The same kernels as micsa_measure_begin, but their
 * scratch -- the per-lane 64-bit counters and the ticket word -- lives in a
 * file-scope `static __device__` array of the library instead of the context's
 * workspace, and the row goes to a buffer the caller owns:
 *   ctx    input: the context's state at this point in stream order (created
 *          and filled beforehand; micsa_create* does allocate).
 *   d_row  output, DEVICE memory, int64 [2 n_sys + n_pairs]:
 *          E[n_sys] | E_daemon[n_sys] | Q[n_pairs], the sums and order of
 *          micsa_measure_i64 (E_daemon over all gamma families).  Anything but
 *          device / managed memory -> MICSA_ERR_INVALID.
 * Asynchronous on the context's stream; the call itself performs no cudaMalloc,
 * cudaFree, host allocation, memcpy or stream synchronisation (two
 * cudaMemsetAsync of the scratch and the measurement launches, nothing else).
 * Limit: the array holds MICSA_NOALLOC_MAX_COUNTERS counters (128 KiB + one
 * 256-byte ticket line, resident on every GPU that loads the library until
 * exit).  A context needs 64 per word lattice + 32 per (sample group, replica
 * pair): n_words = ceil(n_samples / (32 / rpw)) * n_replicas / rpw, rpw = 2
 * for even n_replicas, else 1 -- all five BASELINE configurations fit (96, 384,
 * 768, 96 and 2 048 counters); more -> MICSA_ERR_INVALID, nothing launched.
 * The array is shared by every context and stream on a device and keeps the
 * last call's contents: each call clears what it uses first, and two calls
 * that OVERLAP on the GPU (different streams, or graphs replayed
 * concurrently) race on it -- order them.  It does not touch the scratch of the
 * other measurement calls, which may run concurrently with it. */
#define MICSA_NOALLOC_MAX_COUNTERS 16384
int micsa_measure_noalloc(micsa_ctx *ctx, int64_t *d_row);

/* micsa_anneal: for k = 0..n_steps-1: refresh(T_k, step0 + k); n_sweeps_k
 * sweeps with measurement rows as micsa_step says.  The whole schedule is
 * queued without host synchronisation; rows are kept on the device and copied
 * once at the end (synchronous on return).
 *   min_energy  host [n_sys] or NULL: minimum over this call's rows of E/N
 *               (+inf if there was no row).
 *   trace       host struct or NULL.                                         */
int micsa_anneal(micsa_ctx *ctx, const micsa_step *sched, int n_steps,
                 uint32_t step0, double *min_energy, micsa_trace *trace);

/* Running totals since create: spin-flip attempts; 32-bit uniforms the
 * refreshes are defined on (one per daemon, R8) plus one per Metropolis
 * attempt; Philox4x32-10
 * blocks the refresh kernels actually evaluated.  The refresh compares
 * bit-plane by bit-plane and stops once every lane is decided, so the last is
 * data dependent (about half of the 1 block per 4 daemons a full evaluation
 * needs); it is counted on the device and asking for it synchronises the
 * stream.  Initialisation draws are not counted.  Any pointer may be NULL. */
int micsa_counters(micsa_ctx *ctx, uint64_t *attempts, uint64_t *rns_drawn,
                   uint64_t *philox_calls);

/* Geometry of the private device layout, for roofline accounting:
 * info[0] = bytes of packed state (spins + daemons + bonds),
 * info[1] = bytes one sweep must read+write at least once (compulsory),
 * info[2] = number of 32-bit spin words per site, info[3] = bits per bond word,
 * info[4] = kernel launches issued so far on this context.                   */
int micsa_layout_info(micsa_ctx *ctx, uint64_t info[5]);

/* Tuning / A-B switch, never needed for correctness (every setting gives the
 * same bits; tests/test_gpu_parity.py runs parity cases under each).  They
 * only matter when L % 8 == 0; other L always use the generic kernel.
 * key MICSA_TUNE_SWEEP_KERNEL: 1 = row-marching register kernel; 2 =
 *   software-pipelined row-marching kernel, one launch per half-sweep
 *   (default).
 * key MICSA_TUNE_PIPE_ROWS: rows per thread of kernel 2: 4 (default) or 8.
 * key MICSA_TUNE_PIPE_PLANES: lattice planes per CTA of kernel 2 (one warp
 *   each): 4 (default) or 1.
 * key MICSA_TUNE_FUSE_MEASURE: 1 (default) = micsa_sweep_measure and micsa_anneal count
 *   the observables inside the last sweep, 0 = separate measurement kernel.
 * key MICSA_TUNE_FUSE_WALK: 1 (default) = with walkers the wandering exchange is done by the odd
 *   half-sweep of kernel 2 itself, 0 = by a separate kernel after the sweep.
 * key MICSA_TUNE_L2_GROUPS: 1 (default) = when the packed state exceeds the L2 cache, a call of several
 *   sweeps runs all of them on one group of word lattices (independent systems) that fits in L2 before
 *   touching the next group, 0 = every half-sweep over all lattices.
 * key MICSA_TUNE_SMALL_PATH: 1 (default) = on small lattices (L a multiple of 8, L*L*L/8 <= 8192 quad rows,
 *   n_replicas <= 2, one daemon per spin) micsa_sweep, micsa_sweep_measure and up to eight consecutive schedule
 *   steps of micsa_anneal run as ONE launch in which each word lattice is walked by a thread-block cluster (all
 *   sweeps and the measurement rows; cluster barriers instead of kernel boundaries; the steps' refreshes are
 *   generated beforehand into staging planes, 2 x 8 plane pairs allocated at the first such micsa_anneal:
 *   MICSA_ERR_NOMEM if that fails), 0 = the general path.
 * key MICSA_TUNE_SMALL_ITEMS: quad rows per CTA and parity the small-lattice path aims at when it chooses the cluster
 *   size (1 .. 16 CTAs per word lattice): 0 = default, else 1 .. 1024.
 * key MICSA_TUNE_PDL: 1 (default) = kernel 2 is launched with programmatic
 *   stream serialization (the next half-sweep's grid is scheduled while this
 *   one drains and waits on the device for its completion), 0 = plain launches.
 * Unknown key or value: MICSA_ERR_INVALID, nothing changes. */
enum { MICSA_TUNE_SWEEP_KERNEL = 0, MICSA_TUNE_PIPE_ROWS = 2, MICSA_TUNE_PDL = 3,
       MICSA_TUNE_PIPE_PLANES = 4, MICSA_TUNE_FUSE_MEASURE = 5,
       MICSA_TUNE_FUSE_WALK = 6, MICSA_TUNE_L2_GROUPS = 7,
       MICSA_TUNE_SMALL_PATH = 8, MICSA_TUNE_SMALL_ITEMS = 9 };
int micsa_set_tuning(micsa_ctx *ctx, int key, int value);

/* ---- continuous daemons / walkers with real couplings -------------
 * PAPER.md:136-140 (Sec. 2.4, Eq. 9: in the continuous case the n are exponentially
 * distributed, Prob(0 < n < R) = 1 - exp(-R/T)) and :436-454 (Appendix C: Gaussian couplings
 * J ~ N(0,1), "continuous walker variables", no cap: the elementary move of Sec. 2.3,
 * n <- n - dH, legal iff n >= 0).  A context of its own; float64 arithmetic without fused
 * multiply-add in the order DESIGN.md R20 fixes, so that the accept decision is taken on the
 * same number as in the oracle.
 * Canonical host layouts (site i = x + L (y + L z)):
 *   s  int8    [n_samples][n_replicas][N]   spins +-1
 *   n  float64 [n_samples][n_replicas][N]   daemon / walker energies, >= 0
 *   J  float64 [n_samples][3][N]            bond from site i to its +d neighbour; replicas share it
 * micsa_gauss_create: spins = the Philox start of micsa_create (same seed, same counters), n = 0,
 *   J = 0 until micsa_gauss_set_couplings (the Gaussian couplings are an INPUT: a caller-owned host
 *   array, finite values; copied).  NULL on error (L odd or < 2, sizes, no device, out of memory).
 * micsa_gauss_set_state / get_state: any pointer may be NULL; spins must be +-1, n finite and >= 0
 *   (else MICSA_ERR_INVALID, state unchanged).  Synchronous.
 * micsa_gauss_refresh: every n <- -T log(u), u = (x + 1/2) 2^-32, x = word 0 of Philox4x32-10 at counter
 *   (i, sample_offset + sample, (5 << 24) | replica, step), key = seed (Eq. 9).  T finite and > 0.
 * micsa_gauss_sweep: n timesteps = even half-sweep, odd half-sweep and, with walkers
 *   (micsa_gauss_set_walkers(ctx, 1, t)), the forward-X wandering half-cycle of parity t mod 2 after each
 *   (Appendix C step 1(b); R15), t += 1.  Asynchronous on the context's stream.
 * micsa_gauss_wander: one half-cycle, walkers on sites of `parity` exchange with the neighbour at +sign along axis.
 * micsa_gauss_measure: E[n_sys] = H_EA (Eq. 1), E_daemon[n_sys] = sum of n (Eq. 4) as float64 sums (fixed
 *   summation tree: reproducible run to run; equal to the oracle's site-ordered sum to ~1e-13 relative),
 *   Q[n_samples * n_replicas (n_replicas - 1) / 2] = N q (exact); any pointer may be NULL.  Synchronises. */
typedef struct micsa_gauss_ctx micsa_gauss_ctx;
micsa_gauss_ctx *micsa_gauss_create(int L, int n_samples, int n_replicas, uint64_t seed,
                                    int sample_offset, void *cuda_stream);
int micsa_gauss_destroy(micsa_gauss_ctx *ctx);
int micsa_gauss_set_couplings(micsa_gauss_ctx *ctx, const double *J);
int micsa_gauss_set_state(micsa_gauss_ctx *ctx, const int8_t *s, const double *n);
int micsa_gauss_get_state(micsa_gauss_ctx *ctx, int8_t *s, double *n, double *J);
int micsa_gauss_refresh(micsa_gauss_ctx *ctx, double T, uint32_t step);
int micsa_gauss_sweep(micsa_gauss_ctx *ctx, int n);
int micsa_gauss_half_sweep(micsa_gauss_ctx *ctx, int parity);
int micsa_gauss_wander(micsa_gauss_ctx *ctx, int axis, int sign, int parity);
int micsa_gauss_set_walkers(micsa_gauss_ctx *ctx, int mode, int64_t t);
int micsa_gauss_measure(micsa_gauss_ctx *ctx, double *E, double *E_daemon, int64_t *Q);
int micsa_gauss_counters(micsa_gauss_ctx *ctx, uint64_t *attempts, uint64_t *rns_drawn);
int micsa_gauss_synchronize(micsa_gauss_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* MICSA_H */
