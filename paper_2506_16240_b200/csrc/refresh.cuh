// refresh.cuh -- daemon refresh and Philox initial state
// (row a0).
//
// Refresh, PAPER.md:154-157 (Eq. 11) and :190: every daemon is replaced by an
// independent draw with p(n=4m) ~ exp(-4m/T), m = 0..3; spins are untouched.
// It is the only consumer of random numbers.  DESIGN.md R7/R8:
// every daemon has its own 32-bit uniform u and
//     m = [u >= thr0] + [u >= thr1] + [u >= thr2],
// thr_k = floor(cdf_k * 2^32) in [1, 2^32] computed on the host.  u is defined
// bit-sliced: for the 16 global samples of block B = gs >> 4 (same site i,
// replica, step) four Philox4x32-10 calls c = 0..3 with
//     counter = (i, B | (c << 28), kTagRefresh | replica, step)
// give 32 random 16-lane bit-planes, plane k = 8c + 2j + h = half h of output
// word j of call c, and u(gs) = sum_k bit_{gs & 15}(plane k) << (31 - k).
//
// This is the layout of the state itself, so the kernel never builds u: it
// compares all 32 lanes of a word with the three thresholds plane by plane,
// most significant first (eq = lanes still equal to the threshold prefix,
// gt = lanes already above it), and STOPS as soon as no lane is undecided --
// the remaining planes cannot change any level, so they are never generated.
// After 16 planes a lane is undecided with probability 3 * 2^-16: almost every
// word needs 2 of the 4 call pairs.  The number of Philox calls actually made
// is counted on the device (micsa_counters).
#pragma once
#include "layout.cuh"
#include "philox.cuh"

namespace micsa {

struct SiteGrid {            // thread -> (plane index, z, lattice), see kernels
    int L, Lh, n_rg, n_samples, sample_offset;
    long long half;
    uint32_t inv_Lh;         // fastdiv_magic(Lh)
};

// lanes of word-lattice sample group sg that hold a real sample
template <int RPW>
__device__ __forceinline__ uint32_t valid_lane_mask(int n_samples, int sg) {
    constexpr int SPW = 32 / RPW;
    const int left = n_samples - sg * SPW;
    const uint32_t f = (left >= SPW) ? ((SPW == 32) ? 0xFFFFFFFFu : ((1u << (SPW & 31)) - 1u))
                                     : ((1u << left) - 1u);
    return (RPW == 2) ? (f | (f << 16)) : f;
}

// Thresholds as the kernel sees them: tb[k][p] = all-ones if bit (31-p) of
// thr_k is set, else 0 (plane p, most significant first), so the lane-parallel
// compare takes its threshold bit straight from the constant bank; never[k] =
// thr_k is 2^32 (level k+1 has probability < 2^-32 and is never reached).
struct RefreshThr { uint32_t tb[3][32]; uint32_t never[3]; };

// One chunk c (bit-planes 8c .. 8c+7, one Philox call per 16-lane stream) of the
// lane-parallel compare of a word's 32 uniforms with the three thresholds.
// Per threshold k:  ge = (u_chunk >= t_chunk), a borrow chain from the least
// significant plane of the chunk, eq = (u_chunk == t_chunk), one 3-input logic
// op per plane each; chunks combine most significant first:
//   gt |= EQ & ge & ~eq;  EQ &= eq        (EQ = lanes equal to thr so far).
struct RefreshWord {            // what identifies a word's two Philox streams
    uint32_t i, blk_a, blk_b, rep_a, rep_b;
    bool has_b;
};

template <int CC>      // CC >= 0: chunk index known at compile time (threshold bits become constant-bank operands)
__device__ __forceinline__ void refresh_chunk(uint32_t c_rt, const RefreshWord& wd, uint32_t step,
                                              uint32_t (&EQ)[3], uint32_t (&gt)[3],
                                              const RefreshThr& thr, const PhiloxKeys& ks)
{
    const uint32_t c = (CC >= 0) ? (uint32_t)CC : c_rt;
    const uint4 oa = philox4x32_10(wd.i, wd.blk_a | (c << 28), wd.rep_a, step, ks);
    uint4 ob = make_uint4(0u, 0u, 0u, 0u);
    if (wd.has_b) ob = philox4x32_10(wd.i, wd.blk_b | (c << 28), wd.rep_b, step, ks);
    const uint32_t wa[4] = { oa.x, oa.y, oa.z, oa.w };
    const uint32_t wb[4] = { ob.x, ob.y, ob.z, ob.w };
    uint32_t ge[3] = { ~0u, ~0u, ~0u }, eq[3] = { ~0u, ~0u, ~0u };
#pragma unroll
    for (int q = 7; q >= 0; --q) {            // least significant plane of the chunk first
        const int j = q >> 1, h = q & 1;
        const uint32_t r = __byte_perm(wa[j], wb[j], h ? 0x7632 : 0x5410);
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const uint32_t tb = thr.tb[k][8 * c + q];     // c is uniform over the block in every phase
            ge[k] = (r & ~tb) | (~(r ^ tb) & ge[k]);
            eq[k] &= ~(r ^ tb);
        }
    }
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        gt[k] |= EQ[k] & ge[k] & ~eq[k];
        EQ[k] &= eq[k];
    }
}

constexpr int kRefreshBlock = 128;
constexpr int kRefreshSub = 4;        // groups of kRefreshBlock words per block

// grid = (ceil(L*Lh/block), L, n_words*2); one thread = one site word in phase 0.
// A word holds two 16-lane Philox streams a (lanes 0-15) and b (lanes 16-31):
// RPW = 2: the same sample block, replicas 2rg and 2rg+1;
// RPW = 1: sample blocks 2sg and 2sg+1 of one replica.
// Phase 0: every thread runs chunk 0 of its words (kRefreshSub groups of kRefreshBlock words per block).  About a
// quarter of the words still have an undecided lane after 8 planes; they are queued in shared memory and phase 1
// runs chunk 1 for the queued words only, densely on the threads of the block (so whole warps drop out instead of
// idling beside one busy lane), and so on.  Measured at config 4: 93 us with every thread iterating by itself, 84 us
// with a queue per 128 words, 67 us with the block-wide queue (one barrier per phase and 512 words).
template <int RPW>
__global__ void __launch_bounds__(kRefreshBlock)
refresh_kernel(uint32_t* __restrict__ m0, uint32_t* __restrict__ m1, SiteGrid g,
               PhiloxKeys ks, uint32_t step, RefreshThr thr,
               unsigned long long* __restrict__ n_calls, uint32_t alpha_bits)
{
    constexpr int SPW = 32 / RPW;
    constexpr int kQ = kRefreshBlock * kRefreshSub;       // every word of the block may be queued
    __shared__ uint32_t q_tid[2][kQ];
    __shared__ uint32_t q_st[2][6][kQ];
    __shared__ int q_n[4];
    __shared__ unsigned int s_calls;
    if (threadIdx.x < 4) q_n[threadIdx.x] = 0;
    if (threadIdx.x == 0) s_calls = 0;
    __syncthreads();

    const int z = blockIdx.y;
    const int w = blockIdx.z >> 1, p = blockIdx.z & 1;
    const int sg = w / g.n_rg, rg = w - sg * g.n_rg;
    const uint32_t blk = (uint32_t)(g.sample_offset + sg * SPW) >> 4;
    const uint32_t vm = valid_lane_mask<RPW>(g.n_samples, sg);
    const long long plane0 = ((long long)blockIdx.z) * g.half + (long long)z * g.L * g.Lh;
    RefreshWord wd;
    wd.blk_a = blk; wd.blk_b = (RPW == 2) ? blk : blk + 1u;
    wd.rep_a = kTagRefresh | alpha_bits | (uint32_t)(rg * RPW);     // alpha_bits = daemon family << 20
    wd.rep_b = (RPW == 2) ? wd.rep_a + 1u : wd.rep_a;
    wd.has_b = (vm >> 16) != 0u;                  // block-uniform
    const unsigned per_chunk = wd.has_b ? 2u : 1u;
    unsigned int calls = 0;

    // Phase 0 for all kRefreshSub groups of kRefreshBlock words of this block, then ONE barrier; the words that are
    // still undecided (about a quarter) sit densely in the block-wide queue and phase c runs chunk c for them, a
    // barrier per phase: three barriers per kRefreshSub * 128 words instead of three per 128 (ncu: 37 % of the stall
    // samples of the one-group kernel were warps waiting at those barriers).
    const int n_plane = g.L * g.Lh;
    auto finish = [&](int word, const uint32_t (&EQ)[3], const uint32_t (&gt)[3]) {
        // lanes equal to a threshold in all 32 bits are >= it
        const uint32_t ge0 = gt[0] | EQ[0], ge1 = gt[1] | EQ[1], ge2 = gt[2] | EQ[2];
        m0[plane0 + word] = (ge0 ^ ge1 ^ ge2) & vm;       // level odd
        m1[plane0 + word] = ge1 & vm;                     // level >= 2
    };
    auto push = [&](int c, int word, const uint32_t (&EQ)[3], const uint32_t (&gt)[3]) {
        const int slot = atomicAdd(&q_n[c], 1);
        const int b = c & 1;
        q_tid[b][slot] = (uint32_t)word;
#pragma unroll
        for (int k = 0; k < 3; ++k) { q_st[b][k][slot] = EQ[k]; q_st[b][3 + k][slot] = gt[k]; }
    };
#pragma unroll 1
    for (int sub = 0; sub < kRefreshSub; ++sub) {
        const int word = ((int)blockIdx.x * kRefreshSub + sub) * kRefreshBlock + (int)threadIdx.x;
        if (word >= n_plane) break;
        uint32_t EQ[3], gt[3] = { 0u, 0u, 0u };
#pragma unroll
        for (int k = 0; k < 3; ++k) EQ[k] = thr.never[k] ? 0u : vm;
        const int y = (int)fastdiv((uint32_t)word, g.inv_Lh), xh = word - y * g.Lh;
        wd.i = canonical_site(g.L, p, z, y, xh);
        refresh_chunk<0>(0u, wd, step, EQ, gt, thr, ks);
        calls += per_chunk;
        if ((EQ[0] | EQ[1] | EQ[2]) != 0u) push(0, word, EQ, gt);      // a lane is still equal to a threshold prefix
        else finish(word, EQ, gt);
    }
#pragma unroll 1
    for (uint32_t c = 1; c < 4; ++c) {
        __syncthreads();                          // queue c-1 is complete
        const int n = q_n[c - 1];
        if (n == 0) break;                        // block-uniform
        const int b = (c - 1) & 1;
        for (int e = threadIdx.x; e < n; e += kRefreshBlock) {
            const int word = (int)q_tid[b][e];
            uint32_t EQ[3], gt[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) { EQ[k] = q_st[b][k][e]; gt[k] = q_st[b][3 + k][e]; }
            const int y = (int)fastdiv((uint32_t)word, g.inv_Lh), xh = word - y * g.Lh;
            wd.i = canonical_site(g.L, p, z, y, xh);
            refresh_chunk<-1>(c, wd, step, EQ, gt, thr, ks);
            calls += per_chunk;
            if (c < 3 && (EQ[0] | EQ[1] | EQ[2]) != 0u) push((int)c, word, EQ, gt);
            else finish(word, EQ, gt);
        }
    }
    // Philox calls made by this block -> one atomic
    calls = __reduce_add_sync(0xFFFFFFFFu, calls);
    if ((threadIdx.x & 31) == 0 && calls) atomicAdd(&s_calls, calls);
    __syncthreads();
    if (threadIdx.x == 0 && s_calls) atomicAdd(n_calls, (unsigned long long)s_calls);
}

// one random bit for global sample gs from the block (c0, gs>>7, c2, 0)
__device__ __forceinline__ uint32_t init_bit(uint32_t c0, uint32_t gs, uint32_t c2,
                                             const PhiloxKeys& ks, uint32_t& cached_blk,
                                             uint4& cached) {
    const uint32_t blk = gs >> 7;
    if (blk != cached_blk) { cached = philox4x32_10(c0, blk, c2, 0u, ks); cached_blk = blk; }
    const uint32_t sel = (gs >> 5) & 3u;
    const uint32_t wv = sel == 0 ? cached.x : sel == 1 ? cached.y : sel == 2 ? cached.z : cached.w;
    return (wv >> (gs & 31u)) & 1u;
}

// spins: counter (i, gs>>7, kTagSpinInit | replica, 0), bit gs&31 of word (gs>>5)&3
template <int RPW>
__global__ void __launch_bounds__(128)
init_spins_kernel(uint32_t* __restrict__ spin, SiteGrid g, PhiloxKeys ks)
{
    constexpr int SPW = 32 / RPW;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.L * g.Lh) return;
    const int y = t / g.Lh, xh = t - y * g.Lh;
    const int z = blockIdx.y;
    const int w = blockIdx.z >> 1, p = blockIdx.z & 1;
    const int sg = w / g.n_rg, rg = w - sg * g.n_rg;
    const uint32_t i = canonical_site(g.L, p, z, y, xh);
    uint32_t bits = 0;
    for (int r = 0; r < RPW; ++r) {
        uint32_t cached_blk = 0xFFFFFFFFu; uint4 cached = make_uint4(0, 0, 0, 0);
        for (int sl = 0; sl < SPW; ++sl) {
            const int sample = sg * SPW + sl;
            if (sample >= g.n_samples) break;
            const uint32_t gs = (uint32_t)(g.sample_offset + sample);
            bits |= init_bit(i, gs, kTagSpinInit | (uint32_t)(rg * RPW + r), ks, cached_blk, cached)
                    << (r * SPW + sl);
        }
    }
    spin[((long long)blockIdx.z) * g.half + ((long long)z * g.L + y) * g.Lh + xh] = bits;
}

// bonds: counter (i, gs>>7, kTagBondInit | d, 0); grid.z = n_sg*6 (sg, d, p)
template <int RPW>
__global__ void __launch_bounds__(128)
init_bonds_kernel(typename BondT<RPW>::type* __restrict__ J, SiteGrid g, PhiloxKeys ks)
{
    constexpr int SPW = 32 / RPW;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.L * g.Lh) return;
    const int y = t / g.Lh, xh = t - y * g.Lh;
    const int z = blockIdx.y;
    const int p = blockIdx.z & 1, d = (blockIdx.z >> 1) % 3, sg = blockIdx.z / 6;
    const uint32_t i = canonical_site(g.L, p, z, y, xh);
    uint32_t bits = 0;
    uint32_t cached_blk = 0xFFFFFFFFu; uint4 cached = make_uint4(0, 0, 0, 0);
    for (int sl = 0; sl < SPW; ++sl) {
        const int sample = sg * SPW + sl;
        if (sample >= g.n_samples) break;
        const uint32_t gs = (uint32_t)(g.sample_offset + sample);
        bits |= init_bit(i, gs, kTagBondInit | (uint32_t)d, ks, cached_blk, cached) << sl;
    }
    J[((long long)blockIdx.z) * g.half + ((long long)z * g.L + y) * g.Lh + xh] =
        (typename BondT<RPW>::type)bits;
}

}  // namespace micsa
