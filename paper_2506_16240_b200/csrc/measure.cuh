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
// lane counts into out[0..31] (global, 64-bit).
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

struct MeasureArgs {
    const uint32_t* spin; const uint32_t* m0; const uint32_t* m1; const void* J;
    int L, Lh, n_rg, n_replicas, n_samples;
    long long half;
    unsigned long long* cntU;    // [n_words][32]  unsatisfied bonds
    unsigned long long* cntM;    // [n_words][32]  sum of daemon levels
    unsigned long long* cntX;    // [n_sg][pairs_per_sample][32]  sum of sigma^a ^ sigma^b
};

// Unsatisfied bonds.  grid = (nblk, 2 parities, n_words); grid-stride over the
// V-word vectors of the parity array; a vector never straddles a row.
template <int V, int RPW>
__global__ void __launch_bounds__(kCountBlock)
count_unsat_kernel(MeasureArgs a)
{
    typedef typename BondT<RPW>::type JT;
    const int p = blockIdx.y, q = 1 - p, w = blockIdx.z;
    const int L = a.L, Lh = a.Lh, nxv = Lh / V;
    const long long half = a.half, nvec = half / V;
    const uint32_t* sp = a.spin + ((long long)w * 2 + p) * half;
    const uint32_t* sq = a.spin + ((long long)w * 2 + q) * half;
    const int sg = w / a.n_rg;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;
    const JT* Jx = Jb + (0 * 2 + p) * half;
    const JT* Jy = Jb + (1 * 2 + p) * half;
    const JT* Jz = Jb + (2 * 2 + p) * half;

    VCount<kThreadPlanes> acc; acc.clear();
    for (long long iv = (long long)blockIdx.x * blockDim.x + threadIdx.x; iv < nvec;
         iv += (long long)gridDim.x * blockDim.x) {
        const long long rowi = iv / nxv;
        const int xv = (int)(iv - rowi * nxv);
        const int z = (int)(rowi / L), y = (int)(rowi - (long long)z * L);
        const int yp = (y + 1 == L) ? 0 : y + 1, zp = (z + 1 == L) ? 0 : z + 1;
        const int xh0 = xv * V;
        const long long row = rowi * Lh, h = row + xh0;
        const int c = (y + z + p) & 1;        // c=1: +x neighbour at xh+1, else same xh
        const Vec<V> s = ldg_vec<V>(sp + h);
        const Vec<V> A = ldg_vec<V>(sq + h);
        const uint32_t e = sq[row + ((xh0 + V == Lh) ? 0 : xh0 + V)];
        const Vec<V> ny = ldg_vec<V>(sq + ((long long)z * L + yp) * Lh + xh0);
        const Vec<V> nz = ldg_vec<V>(sq + ((long long)zp * L + y) * Lh + xh0);
        const Vec<V> jx = ldg_bonds<V, RPW>(Jx + h);
        const Vec<V> jy = ldg_bonds<V, RPW>(Jy + h);
        const Vec<V> jz = ldg_bonds<V, RPW>(Jz + h);
        VCount<4> loc; loc.clear();
#pragma unroll
        for (int k = 0; k < V; ++k) {
            const uint32_t up = (k + 1 < V) ? A.v[k + 1] : e;
            const uint32_t nx = c ? up : A.v[k];
            const uint32_t ux = s.v[k] ^ nx ^ jx.v[k];
            const uint32_t uy = s.v[k] ^ ny.v[k] ^ jy.v[k];
            const uint32_t uz = s.v[k] ^ nz.v[k] ^ jz.v[k];
            const uint32_t b[2] = { ux ^ uy ^ uz, maj3(ux, uy, uz) };
            loc.add(b);
        }
        acc.add(loc.c);
    }
    block_lane_counts(acc, a.cntU + (long long)w * 32);
}

// Sum of daemon levels.  grid = (nblk, n_words); both parities are contiguous.
template <int V>
__global__ void __launch_bounds__(kCountBlock)
count_levels_kernel(MeasureArgs a)
{
    const int w = blockIdx.y;
    const long long n = 2 * a.half, nvec = n / V;
    const uint32_t* p0 = a.m0 + (long long)w * n;
    const uint32_t* p1 = a.m1 + (long long)w * n;
    VCount<kThreadPlanes> acc; acc.clear();
    for (long long iv = (long long)blockIdx.x * blockDim.x + threadIdx.x; iv < nvec;
         iv += (long long)gridDim.x * blockDim.x) {
        const Vec<V> b0 = ldg_vec<V>(p0 + iv * V), b1 = ldg_vec<V>(p1 + iv * V);
        VCount<4> loc; loc.clear();
#pragma unroll
        for (int k = 0; k < V; ++k) {
            const uint32_t b[2] = { b0.v[k], b1.v[k] };
            loc.add(b);
        }
        acc.add(loc.c);
    }
    block_lane_counts(acc, a.cntM + (long long)w * 32);
}

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

struct FinalizeArgs {
    const unsigned long long* cntU; const unsigned long long* cntM; const unsigned long long* cntX;
    long long* row;        // [n_sys E | n_sys E_daemon | n_pairs Q]
    long long* min_E;      // [n_sys] running minimum, or nullptr
    int n_samples, n_replicas, n_rg, rpw, spw, pairs_per_sample;
    long long N;
};

// counts -> exact sums in canonical system order; one thread per system / pair
__global__ void finalize_measure_kernel(FinalizeArgs f)
{
    const int n_sys = f.n_samples * f.n_replicas;
    const int n_pairs = f.n_samples * f.pairs_per_sample;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n_sys) {
        const int sample = t / f.n_replicas, rep = t - sample * f.n_replicas;
        const int sg = sample / f.spw, sl = sample - sg * f.spw;
        const int w = sg * f.n_rg + rep / f.rpw, lane = (rep % f.rpw) * f.spw + sl;
        const long long E = 2 * (long long)f.cntU[(long long)w * 32 + lane] - 3 * f.N;
        f.row[t] = E;
        f.row[n_sys + t] = 4 * (long long)f.cntM[(long long)w * 32 + lane];
        if (f.min_E && E < f.min_E[t]) f.min_E[t] = E;
    }
    if (t < n_pairs) {
        const int sample = t / f.pairs_per_sample, pr = t - sample * f.pairs_per_sample;
        const int sg = sample / f.spw, sl = sample - sg * f.spw;
        f.row[2 * n_sys + t] =
            f.N - 2 * (long long)f.cntX[((long long)sg * f.pairs_per_sample + pr) * 32 + sl];
    }
}

__global__ void fill_i64_kernel(long long* p, long long v, int n) {
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) p[t] = v;
}

}  // namespace micsa
