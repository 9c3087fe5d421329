// measure.cuh -- per-system reductions on bit-sliced data (SURVEY 8(a) rows
// a4-a6):
//   H_EA   = -sum_<xy> J s s = 2*U_tot - 3N   (Eq. 1), U_tot =
//            number of unsatisfied bonds, each of the 3N bonds counted once
//            at its owner site;
//   H_aux  = sum_x n_x = 4 sum_x m_x           (Eq. 4);
//   N q    = sum_x s^a_x s^b_x = N - 2 sum_x (sigma^a ^ sigma^b).
// One count per bit lane is needed, not a popcount of the word: every thread
// keeps a "vertical" counter (bit k of the count of lane l is bit l of plane
// k) fed through carry-save adders, the warp adds its 32 vertical counters
// with shuffles, lanes pick out their own count, and the block issues one
// 64-bit atomic per lane.
#pragma once
#include "layout.cuh"

namespace micsa {

__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c) {
    return (a & b) | (c & (a ^ b));
}

template <int NP> struct VCount {
    uint32_t c[NP];
    __device__ __forceinline__ void clear() {
#pragma unroll
        for (int k = 0; k < NP; ++k) c[k] = 0;
    }
    // add the bit-sliced number whose planes are b[0..K-1] (weights 1, 2, 4, ...)
    template <int K> __device__ __forceinline__ void add(const uint32_t (&b)[K]) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < NP; ++k) {
            const uint32_t x = (k < K) ? b[k] : 0u;
            const uint32_t s = c[k] ^ x ^ carry;
            carry = maj3(c[k], x, carry);
            c[k] = s;
        }
    }
};

constexpr int kThreadPlanes = 16;     // per-thread count < 65536 per lane
constexpr int kWarpPlanes   = 21;     // + 5 bits for the 32 threads of a warp
constexpr int kCountBlock   = 128;

// Adds the per-thread vertical counter over the block and accumulates the 32
// lane counts into out[0..31] (global, 64-bit).  Shuffle version, used by the
// general replica-pair kernel below.
__device__ __forceinline__ void block_lane_counts(const VCount<kThreadPlanes>& acc,
                                                  unsigned long long* out)
{
    __shared__ unsigned int s_cnt[32];
    if (threadIdx.x < 32) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    uint32_t c[kWarpPlanes];
#pragma unroll
    for (int k = 0; k < kWarpPlanes; ++k) c[k] = (k < kThreadPlanes) ? acc.c[k] : 0u;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < kWarpPlanes; ++k) {
            const uint32_t x = __shfl_down_sync(0xFFFFFFFFu, c[k], off);
            const uint32_t s = c[k] ^ x ^ carry;
            carry = maj3(c[k], x, carry);
            c[k] = s;
        }
    }
    const int lane = threadIdx.x & 31;
    unsigned int mine = 0;
#pragma unroll
    for (int k = 0; k < kWarpPlanes; ++k) {
        const uint32_t plane = __shfl_sync(0xFFFFFFFFu, c[k], 0);
        mine += ((plane >> lane) & 1u) << k;
    }
    atomicAdd(&s_cnt[lane], mine);
    __syncthreads();
    if (threadIdx.x < 32 && s_cnt[threadIdx.x])
        atomicAdd(&out[threadIdx.x], (unsigned long long)s_cnt[threadIdx.x]);
}

// Version for the one-pass kernel: P planes per thread, B threads.  The warp
// adds its 32 vertical counters with a shuffle butterfly (level l works on
// P + l planes only), every lane picks out its own count, the warps meet in
// shared-memory atomics and 32 threads issue the global ones.
template <int P, int B>
__device__ __forceinline__ void block_warp_lane_counts(const uint32_t (&acc)[P], unsigned int* s_cnt,
                                                       unsigned long long* out)
{
    uint32_t c[P + 5];
#pragma unroll
    for (int k = 0; k < P + 5; ++k) c[k] = (k < P) ? acc[k] : 0u;
#pragma unroll
    for (int l = 0; l < 5; ++l) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < P + 5; ++k) {
            if (k <= P + l) {                       // planes above P + l are still zero
                const uint32_t x = __shfl_xor_sync(0xFFFFFFFFu, c[k], 1 << l);
                const uint32_t s = c[k] ^ x ^ carry;
                carry = maj3(c[k], x, carry);
                c[k] = s;
            }
        }
    }
    const int lane = threadIdx.x & 31;
    unsigned int mine = 0;
#pragma unroll
    for (int k = 0; k < P + 5; ++k) mine += ((c[k] >> lane) & 1u) << k;
    if (threadIdx.x < 32) s_cnt[threadIdx.x] = 0;
    __syncthreads();
    if (mine) atomicAdd(&s_cnt[lane], mine);
    __syncthreads();
    if (threadIdx.x < 32 && s_cnt[threadIdx.x])
        atomicAdd(&out[threadIdx.x], (unsigned long long)s_cnt[threadIdx.x]);
    __syncthreads();
}

// Version for the measuring half-sweep launches (B = 128 threads, P planes per
// thread): the four warps leave their planes in shared memory, ONE warp adds the
// four vertical counters of each lane position (P + 2 planes), runs the shuffle
// butterfly over its 32 threads and issues the 32 global atomics.  The caller
// gives each of its counters to a different warp, so the block pays one butterfly
// per counter instead of one per counter and warp, and its tail is one butterfly
// long instead of three.  pl = [P][128] words of shared memory, filled by every
// thread before the barrier that precedes this call.
template <int P>
__device__ __forceinline__ void warp_sum_lane_counts(const uint32_t (*pl)[128], int lane, unsigned long long* out)
{
    uint32_t c[P + 7];
#pragma unroll
    for (int k = 0; k < P + 7; ++k) c[k] = (k < P) ? pl[k][lane] : 0u;
#pragma unroll
    for (int wv = 1; wv < 4; ++wv) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < P + 2; ++k) {
            const uint32_t x = (k < P) ? pl[k][wv * 32 + lane] : 0u;
            const uint32_t s = c[k] ^ x ^ carry;
            carry = maj3(c[k], x, carry);
            c[k] = s;
        }
    }
#pragma unroll
    for (int l = 0; l < 5; ++l) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < P + 7; ++k) {
            if (k <= P + 2 + l) {                   // planes above P + 2 + l are still zero
                const uint32_t x = __shfl_xor_sync(0xFFFFFFFFu, c[k], 1 << l);
                const uint32_t s = c[k] ^ x ^ carry;
                carry = maj3(c[k], x, carry);
                c[k] = s;
            }
        }
    }
    unsigned int mine = 0;
#pragma unroll
    for (int k = 0; k < P + 7; ++k) mine += ((c[k] >> lane) & 1u) << k;
    if (mine) atomicAdd(&out[lane], (unsigned long long)mine);
}

// The warp-level part of the above alone: the count of lane l of the word, summed over the warp's 32 vertical
// counters, returned to the thread whose lane index is l.
template <int P>
__device__ __forceinline__ unsigned int warp_lane_count(const uint32_t (&acc)[P])
{
    uint32_t c[P + 5];
#pragma unroll
    for (int k = 0; k < P + 5; ++k) c[k] = (k < P) ? acc[k] : 0u;
#pragma unroll
    for (int l = 0; l < 5; ++l) {
        uint32_t carry = 0;
#pragma unroll
        for (int k = 0; k < P + 5; ++k) {
            if (k <= P + l) {
                const uint32_t x = __shfl_xor_sync(0xFFFFFFFFu, c[k], 1 << l);
                const uint32_t s = c[k] ^ x ^ carry;
                carry = maj3(c[k], x, carry);
                c[k] = s;
            }
        }
    }
    const int lane = threadIdx.x & 31;
    unsigned int mine = 0;
#pragma unroll
    for (int k = 0; k < P + 5; ++k) mine += ((c[k] >> lane) & 1u) << k;
    return mine;
}

struct MeasureArgs {
    const uint32_t* spin; const uint32_t* m0; const uint32_t* m1; const void* J;
    int L, Lh, n_rg, n_replicas, n_samples;
    long long half;
    unsigned long long* cntU;    // [n_words][32]  unsatisfied bonds
    unsigned long long* cntM;    // [n_words][32]  sum of daemon levels
    unsigned long long* cntX;    // [n_sg][pairs_per_sample][32]  sum of sigma^a ^ sigma^b
};

// Replica overlap: differing spins of replicas (ra, rb) of every sample of
// sample group sg.  grid = (nblk, n_sg, pairs_per_sample).
template <int V, int RPW>
__global__ void __launch_bounds__(kCountBlock)
count_xor_kernel(MeasureArgs a)
{
    constexpr int SPW = 32 / RPW;
    const int sg = blockIdx.y;
    int ra = 0, rb = 1;
    for (int k = 0; k < (int)blockIdx.z; ++k) {          // k-th pair (a<b), lexicographic
        if (++rb == a.n_replicas) { ++ra; rb = ra + 1; }
    }
    const long long n = 2 * a.half, nvec = n / V;
    const uint32_t* pa = a.spin + ((long long)sg * a.n_rg + ra / RPW) * n;
    const uint32_t* pb = a.spin + ((long long)sg * a.n_rg + rb / RPW) * n;
    const int sha = (ra % RPW) * SPW, shb = (rb % RPW) * SPW;
    const uint32_t mask = (SPW == 32) ? 0xFFFFFFFFu : ((1u << (SPW & 31)) - 1u);
    VCount<kThreadPlanes> acc; acc.clear();
    for (long long iv = (long long)blockIdx.x * blockDim.x + threadIdx.x; iv < nvec;
         iv += (long long)gridDim.x * blockDim.x) {
        const Vec<V> x = ldg_vec<V>(pa + iv * V), y = ldg_vec<V>(pb + iv * V);
        VCount<4> loc; loc.clear();
#pragma unroll
        for (int k = 0; k < V; ++k) {
            const uint32_t b[1] = { ((x.v[k] >> sha) ^ (y.v[k] >> shb)) & mask };
            loc.add(b);
        }
        acc.add(loc.c);
    }
    block_lane_counts(acc, a.cntX + ((long long)sg * gridDim.z + blockIdx.z) * 32);
}

// Sum of the daemon levels of one more family (gamma > 1) into cntM.
// grid = (nblk, n_words); both parities of a lattice are contiguous (n words).
__global__ void __launch_bounds__(kCountBlock)
count_levels_kernel(const uint32_t* __restrict__ m0, const uint32_t* __restrict__ m1, long long n,
                    unsigned long long* __restrict__ cntM)
{
    const int w = blockIdx.y;
    const uint32_t* p0 = m0 + (long long)w * n;
    const uint32_t* p1 = m1 + (long long)w * n;
    VCount<kThreadPlanes> acc; acc.clear();
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const uint32_t b[2] = { p0[i], p1[i] };
        acc.add(b);
    }
    block_lane_counts(acc, cntM + (long long)w * 32);
}

struct FinalizeArgs {
    unsigned long long* cntU; unsigned long long* cntM; unsigned long long* cntX;
    long long cnt_words;   // length of the counter area starting at cntU (zeroed after use)
    unsigned int* ticket;  // blocks done so far (last one finalises and resets it)
    long long* row;        // [n_sys E | n_sys E_daemon | n_pairs Q]
    long long* min_E;      // [n_sys] running minimum, or nullptr
    int n_samples, n_replicas, n_rg, rpw, spw, pairs_per_sample;
    long long N;
};

// counts -> exact sums in canonical system order (run by one block)
__device__ __forceinline__ void finalize_rows(const FinalizeArgs& f)
{
    const int n_sys = f.n_samples * f.n_replicas;
    const int n_pairs = f.n_samples * f.pairs_per_sample;
    for (int t = threadIdx.x; t < n_sys; t += blockDim.x) {
        const int sample = t / f.n_replicas, rep = t - sample * f.n_replicas;
        const int sg = sample / f.spw, sl = sample - sg * f.spw;
        const int w = sg * f.n_rg + rep / f.rpw, lane = (rep % f.rpw) * f.spw + sl;
        const long long E = 2 * (long long)__ldcg(&f.cntU[(long long)w * 32 + lane]) - 3 * f.N;
        f.row[t] = E;
        f.row[n_sys + t] = 4 * (long long)__ldcg(&f.cntM[(long long)w * 32 + lane]);
        if (f.min_E && E < f.min_E[t]) f.min_E[t] = E;
    }
    for (int t = threadIdx.x; t < n_pairs; t += blockDim.x) {
        const int sample = t / f.pairs_per_sample, pr = t - sample * f.pairs_per_sample;
        const int sg = sample / f.spw, sl = sample - sg * f.spw;
        f.row[2 * n_sys + t] =
            f.N - 2 * (long long)__ldcg(&f.cntX[((long long)sg * f.pairs_per_sample + pr) * 32 + sl]);
    }
    __syncthreads();
    for (long long k = threadIdx.x; k < f.cnt_words; k += blockDim.x) f.cntU[k] = 0ull;   // ready for the next one
}

constexpr int kMeasureBlock = 256;
constexpr int kMeasurePlanes = 10;     // per-thread vertical counters
constexpr int kMeasureMaxItems = 84;   // per thread (even): 84 * 12 < 2^10

__device__ __forceinline__ void full_add(uint32_t a, uint32_t b, uint32_t c, uint32_t& s, uint32_t& cy) {
    s = a ^ b ^ c; cy = maj3(a, b, c);
}
__device__ __forceinline__ void half_add(uint32_t a, uint32_t b, uint32_t& s, uint32_t& cy) {
    s = a ^ b; cy = a & b;
}

// sum of four 1-bit lanes-wise numbers (weight 1) and four more of weight 2 -> 4 planes (<= 12)
__device__ __forceinline__ void csa_4x1_4x2(const uint32_t (&lo)[4], const uint32_t (&hi)[4], uint32_t (&o)[4]) {
    uint32_t a, b, b2, d, e4, f, g4, h4;
    full_add(lo[0], lo[1], lo[2], a, b);
    half_add(a, lo[3], o[0], b2);
    full_add(hi[0], hi[1], hi[2], d, e4);
    full_add(hi[3], b, b2, f, g4);
    half_add(d, f, o[1], h4);
    full_add(e4, g4, h4, o[2], o[3]);
}

// partial sums of one item: unsatisfied own bonds (<= 3V), daemon levels (<= 3V), differing replica lanes (<= V)
struct ItemSums { uint32_t u[4], m[4], x[3]; };

template <int V, int RPW, bool PAIR>
__device__ __forceinline__ void measure_item(ItemSums& r, uint32_t it, uint32_t items_p, uint32_t nxv, uint32_t L,
                                             uint32_t Lh, long long half, const uint32_t* s0, const uint32_t* d0,
                                             const uint32_t* d1, const typename BondT<RPW>::type* Jb)
{
    const uint32_t p = it >= items_p;
    const uint32_t iv = it - (p ? items_p : 0u);
    const uint32_t rowi = iv / nxv, xv = iv - rowi * nxv;
    const uint32_t z = rowi / L, y = rowi - z * L;
    const uint32_t yp = (y + 1 == L) ? 0 : y + 1, zp = (z + 1 == L) ? 0 : z + 1;
    const uint32_t xh0 = xv * V;
    const uint32_t row = rowi * Lh, h = row + xh0;       // < half < 2^31
    const uint32_t c = (y + z + p) & 1u;      // c=1: +x neighbour at xh+1, else same xh
    const uint32_t* sp = s0 + (p ? half : 0);
    const uint32_t* sq = s0 + (p ? 0 : half);
    const Vec<V> s = ldg_vec<V>(sp + h);
    const Vec<V> A = ldg_vec<V>(sq + h);
    const uint32_t e = sq[row + ((xh0 + V == Lh) ? 0 : xh0 + V)];
    const Vec<V> ny = ldg_vec<V>(sq + (z * L + yp) * Lh + xh0);
    const Vec<V> nz = ldg_vec<V>(sq + (zp * L + y) * Lh + xh0);
    const Vec<V> jx = ldg_bonds<V, RPW>(Jb + (0 * 2 + p) * half + h);
    const Vec<V> jy = ldg_bonds<V, RPW>(Jb + (1 * 2 + p) * half + h);
    const Vec<V> jz = ldg_bonds<V, RPW>(Jb + (2 * 2 + p) * half + h);
    const Vec<V> b0 = ldg_vec<V>(d0 + (p ? half : 0) + h);
    const Vec<V> b1 = ldg_vec<V>(d1 + (p ? half : 0) + h);
    uint32_t us[V], uc[V], xs[V];
#pragma unroll
    for (int k = 0; k < V; ++k) {
        const uint32_t up = (k + 1 < V) ? A.v[k + 1] : e;
        const uint32_t nx = c ? up : A.v[k];
        full_add(s.v[k] ^ nx ^ jx.v[k], s.v[k] ^ ny.v[k] ^ jy.v[k], s.v[k] ^ nz.v[k] ^ jz.v[k], us[k], uc[k]);
        xs[k] = PAIR ? ((s.v[k] ^ (s.v[k] >> 16)) & 0xFFFFu) : 0u;
    }
    if (V == 4) {                             // carry-save adder trees
        const uint32_t u_lo[4] = { us[0], us[1], us[2], us[3] }, u_hi[4] = { uc[0], uc[1], uc[2], uc[3] };
        csa_4x1_4x2(u_lo, u_hi, r.u);
        const uint32_t m_lo[4] = { b0.v[0], b0.v[1], b0.v[2], b0.v[3] }, m_hi[4] = { b1.v[0], b1.v[1], b1.v[2], b1.v[3] };
        csa_4x1_4x2(m_lo, m_hi, r.m);
        if (PAIR) {
            uint32_t a2, b2, b3;
            full_add(xs[0], xs[1], xs[2], a2, b2);
            half_add(a2, xs[3], r.x[0], b3);
            r.x[1] = b2 ^ b3; r.x[2] = b2 & b3;
        } else { r.x[0] = r.x[1] = r.x[2] = 0u; }
    } else {                                  // small odd-sized lattices: plain ripple adds
        VCount<4> locU, locM; locU.clear(); locM.clear();
        VCount<3> locX; locX.clear();
#pragma unroll
        for (int k = 0; k < V; ++k) {
            const uint32_t bu[2] = { us[k], uc[k] }; locU.add(bu);
            const uint32_t bm[2] = { b0.v[k], b1.v[k] }; locM.add(bm);
            const uint32_t bx[1] = { xs[k] }; locX.add(bx);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) { r.u[k] = locU.c[k]; r.m[k] = locM.c[k]; }
#pragma unroll
        for (int k = 0; k < 3; ++k) r.x[k] = locX.c[k];
    }
}

// a + b for K-plane numbers -> K+1 planes
template <int K>
__device__ __forceinline__ void add_planes(const uint32_t (&a)[K], const uint32_t (&b)[K], uint32_t (&o)[K + 1]) {
    uint32_t carry = 0;
#pragma unroll
    for (int k = 0; k < K; ++k) { o[k] = a[k] ^ b[k] ^ carry; carry = maj3(a[k], b[k], carry); }
    o[K] = carry;
}

// One pass over the state for all three observables.
// An item = V consecutive words of one row of one parity array; it counts the
// unsatisfied +x,+y,+z bonds of its sites (every bond once, at its owner), the
// daemon levels of its sites and -- when PAIR (n_replicas == 2, both replicas
// in the word) -- the lanes where the two replicas differ.  Other replica
// pairs are counted by count_xor_kernel before this kernel runs.  Per item the
// bits are compressed by carry-save adder trees; two items' sums are added
// before they enter the thread's 10-plane vertical counters.  The last block
// to finish turns the counts into the measurement row.
// grid = (nblk, n_words), block = kMeasureBlock; 32-bit item indices
// (half / V < 2^31 because L^3 < 2^31).
template <int V, int RPW, bool PAIR>
__global__ void __launch_bounds__(kMeasureBlock, 2)
measure_kernel(MeasureArgs a, FinalizeArgs f)
{
    typedef typename BondT<RPW>::type JT;
    __shared__ unsigned int sm[32];
    __shared__ unsigned int s_last;
    const int w = blockIdx.y;
    const uint32_t L = (uint32_t)a.L, Lh = (uint32_t)a.Lh, nxv = Lh / V;
    const long long half = a.half;
    const uint32_t items_p = (uint32_t)(half / V), n_items = 2u * items_p;
    const uint32_t* s0 = a.spin + (long long)w * 2 * half;
    const uint32_t* d0 = a.m0 + (long long)w * 2 * half;
    const uint32_t* d1 = a.m1 + (long long)w * 2 * half;
    const int sg = w / a.n_rg;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;

    VCount<kMeasurePlanes> accU, accM, accX; accU.clear(); accM.clear(); accX.clear();
    const uint32_t stride = gridDim.x * kMeasureBlock;
    for (uint32_t it = blockIdx.x * kMeasureBlock + threadIdx.x; it < n_items; it += 2u * stride) {
        ItemSums A0, A1;
        measure_item<V, RPW, PAIR>(A0, it, items_p, nxv, L, Lh, half, s0, d0, d1, Jb);
        if (it + stride < n_items) {
            measure_item<V, RPW, PAIR>(A1, it + stride, items_p, nxv, L, Lh, half, s0, d0, d1, Jb);
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) { A1.u[k] = 0u; A1.m[k] = 0u; }
#pragma unroll
            for (int k = 0; k < 3; ++k) A1.x[k] = 0u;
        }
        uint32_t su[5], sm5[5], sx[4];
        add_planes<4>(A0.u, A1.u, su);  accU.add(su);
        add_planes<4>(A0.m, A1.m, sm5); accM.add(sm5);
        if (PAIR) { add_planes<3>(A0.x, A1.x, sx); accX.add(sx); }
    }
    block_warp_lane_counts<kMeasurePlanes, kMeasureBlock>(accU.c, sm, a.cntU + (long long)w * 32);
    block_warp_lane_counts<kMeasurePlanes, kMeasureBlock>(accM.c, sm, a.cntM + (long long)w * 32);
    if (PAIR) block_warp_lane_counts<kMeasurePlanes, kMeasureBlock>(accX.c, sm, a.cntX + (long long)sg * 32);

    // the last block to arrive finalises (its reads see every block's atomics)
    __threadfence();
    if (threadIdx.x == 0) {
        const unsigned int total = gridDim.x * gridDim.y;
        s_last = (atomicAdd(f.ticket, 1u) == total - 1u);
    }
    __syncthreads();
    if (s_last) {
        __threadfence();
        finalize_rows(f);
        if (threadIdx.x == 0) *f.ticket = 0u;
    }
}

__global__ void fill_i64_kernel(long long* p, long long v, int n) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) p[t] = v;
}

}  // namespace micsa
