// refresh.cuh -- daemon refresh and Philox initial state
// (row a0).
//
// Refresh, PAPER.md:154-157 (Eq. 11) and :190: every daemon is replaced by an
// independent draw with p(n=4m) ~ exp(-4m/T), m = 0..3; spins are untouched.
// It is the only consumer of random numbers.  DESIGN.md R7/R8:
// one 32-bit Philox4x32-10 output u per daemon,
//     counter = (site i, global_sample >> 2, kTagRefresh | replica, step)
//     u       = output word (global_sample & 3)
//     m       = [u >= thr0] + [u >= thr1] + [u >= thr2]
// with thr_k = floor(cdf_k * 2^32) in [1, 2^32] computed on the host; the
// kernel receives thr_k - 1 (a uint32) and tests u > thr_k - 1.
#pragma once
#include "layout.cuh"
#include "philox.cuh"

namespace micsa {

struct SiteGrid {            // thread -> (plane index, z, lattice), see kernels
    int L, Lh, n_rg, n_samples, sample_offset;
    long long half;
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

// grid = (ceil(L*Lh/block), L, n_words*2); one thread = one site word
template <int RPW>
__global__ void __launch_bounds__(128)
refresh_kernel(uint32_t* __restrict__ m0, uint32_t* __restrict__ m1, SiteGrid g,
               PhiloxKeys ks, uint32_t step, uint32_t a0, uint32_t a1, uint32_t a2)
{
    constexpr int SPW = 32 / RPW;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.L * g.Lh) return;
    const int y = t / g.Lh, xh = t - y * g.Lh;
    const int z = blockIdx.y;
    const int w = blockIdx.z >> 1, p = blockIdx.z & 1;
    const int sg = w / g.n_rg, rg = w - sg * g.n_rg;
    const uint32_t i = canonical_site(g.L, p, z, y, xh);
    const uint32_t blk0 = (uint32_t)(g.sample_offset + sg * SPW) >> 2;

    uint32_t b0 = 0, b1 = 0;
#pragma unroll
    for (int r = 0; r < RPW; ++r) {
        const uint32_t rep = (uint32_t)(rg * RPW + r);
#pragma unroll
        for (int c = 0; c < SPW / 4; ++c) {
            const uint4 o = philox4x32_10(i, blk0 + c, kTagRefresh | rep, step, ks);
            const uint32_t u[4] = { o.x, o.y, o.z, o.w };
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const int lane = r * SPW + 4 * c + j;
                const uint32_t g1 = u[j] > a0, g2 = u[j] > a1, g3 = u[j] > a2;
                b0 |= (g1 ^ g2 ^ g3) << lane;      // level odd
                b1 |= g2 << lane;                  // level >= 2
            }
        }
    }
    const uint32_t vm = valid_lane_mask<RPW>(g.n_samples, sg);
    const long long h = ((long long)blockIdx.z) * g.half + ((long long)z * g.L + y) * g.Lh + xh;
    m0[h] = b0 & vm;
    m1[h] = b1 & vm;
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
