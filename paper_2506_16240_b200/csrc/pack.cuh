// pack.cuh -- conversion between the canonical unpacked layouts of micsa.h
// (int8 / uint8, system-major, site i = x + L(y + L z)) and the private
// bit-sliced device layout of layout.cuh.  Off the hot path: used by
// micsa_set_* / micsa_get_state (the byte-for-byte parity surface).
#pragma once
#include "layout.cuh"
#include "refresh.cuh"   // SiteGrid

namespace micsa {

// Values must be +-1 (kind 0) or 0..3 (kind 1); run before packing so that an
// invalid input leaves the device state untouched.
__global__ void validate_kernel(const int8_t* __restrict__ src, long long n, int kind, int* bad)
{
    bool ok = true;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const int v = src[i];
        ok = ok && (kind == 0 ? (v == 1 || v == -1) : (v >= 0 && v <= 3));
    }
    if (!ok) atomicExch(bad, 1);
}

// kind: 0 spins (+-1 -> bit = s<0), 1 daemon levels (0..3 -> two planes).
// grid = (ceil(L*Lh/block), L, n_words*2)
template <int RPW>
__global__ void __launch_bounds__(128)
pack_sys_kernel(const int8_t* __restrict__ src, uint32_t* __restrict__ d0,
                uint32_t* __restrict__ d1, SiteGrid g, int n_replicas, int kind)
{
    constexpr int SPW = 32 / RPW;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.L * g.Lh) return;
    const int y = t / g.Lh, xh = t - y * g.Lh;
    const int z = blockIdx.y;
    const int w = blockIdx.z >> 1, p = blockIdx.z & 1;
    const int sg = w / g.n_rg, rg = w - sg * g.n_rg;
    const long long N = (long long)g.L * g.L * g.L;
    const long long i = canonical_site(g.L, p, z, y, xh);
    uint32_t b0 = 0, b1 = 0;
    for (int r = 0; r < RPW; ++r)
        for (int sl = 0; sl < SPW; ++sl) {
            const int sample = sg * SPW + sl;
            if (sample >= g.n_samples) break;
            const long long sys = (long long)sample * n_replicas + rg * RPW + r;
            const int v = src[sys * N + i];
            const int lane = r * SPW + sl;
            if (kind == 0) {
                b0 |= (uint32_t)(v < 0) << lane;
            } else {
                b0 |= (uint32_t)(v & 1) << lane;
                b1 |= (uint32_t)((v >> 1) & 1) << lane;
            }
        }
    const long long h = ((long long)blockIdx.z) * g.half + ((long long)z * g.L + y) * g.Lh + xh;
    d0[h] = b0;
    if (kind == 1) d1[h] = b1;
}

template <int RPW>
__global__ void __launch_bounds__(128)
unpack_sys_kernel(int8_t* __restrict__ dst, const uint32_t* __restrict__ d0,
                  const uint32_t* __restrict__ d1, SiteGrid g, int n_replicas, int kind)
{
    constexpr int SPW = 32 / RPW;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.L * g.Lh) return;
    const int y = t / g.Lh, xh = t - y * g.Lh;
    const int z = blockIdx.y;
    const int w = blockIdx.z >> 1, p = blockIdx.z & 1;
    const int sg = w / g.n_rg, rg = w - sg * g.n_rg;
    const long long N = (long long)g.L * g.L * g.L;
    const long long i = canonical_site(g.L, p, z, y, xh);
    const long long h = ((long long)blockIdx.z) * g.half + ((long long)z * g.L + y) * g.Lh + xh;
    const uint32_t b0 = d0[h], b1 = (kind == 1) ? d1[h] : 0u;
    for (int r = 0; r < RPW; ++r)
        for (int sl = 0; sl < SPW; ++sl) {
            const int sample = sg * SPW + sl;
            if (sample >= g.n_samples) break;
            const long long sys = (long long)sample * n_replicas + rg * RPW + r;
            const int lane = r * SPW + sl;
            const int bit0 = (b0 >> lane) & 1, bit1 = (b1 >> lane) & 1;
            dst[sys * N + i] = (kind == 0) ? (int8_t)(1 - 2 * bit0) : (int8_t)(bit0 + 2 * bit1);
        }
}

// bonds: src/dst int8 [n_samples][3][N]; grid.z = n_sg*6 ((sg*3+d)*2+p)
template <int RPW>
__global__ void __launch_bounds__(128)
pack_bonds_kernel(const int8_t* __restrict__ src, typename BondT<RPW>::type* __restrict__ J,
                  SiteGrid g)
{
    constexpr int SPW = 32 / RPW;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.L * g.Lh) return;
    const int y = t / g.Lh, xh = t - y * g.Lh;
    const int z = blockIdx.y;
    const int p = blockIdx.z & 1, d = (blockIdx.z >> 1) % 3, sg = blockIdx.z / 6;
    const long long N = (long long)g.L * g.L * g.L;
    const long long i = canonical_site(g.L, p, z, y, xh);
    uint32_t b = 0;
    for (int sl = 0; sl < SPW; ++sl) {
        const int sample = sg * SPW + sl;
        if (sample >= g.n_samples) break;
        const int v = src[((long long)sample * 3 + d) * N + i];
        b |= (uint32_t)(v < 0) << sl;
    }
    J[((long long)blockIdx.z) * g.half + ((long long)z * g.L + y) * g.Lh + xh] =
        (typename BondT<RPW>::type)b;
}

template <int RPW>
__global__ void __launch_bounds__(128)
unpack_bonds_kernel(int8_t* __restrict__ dst, const typename BondT<RPW>::type* __restrict__ J,
                    SiteGrid g)
{
    constexpr int SPW = 32 / RPW;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= g.L * g.Lh) return;
    const int y = t / g.Lh, xh = t - y * g.Lh;
    const int z = blockIdx.y;
    const int p = blockIdx.z & 1, d = (blockIdx.z >> 1) % 3, sg = blockIdx.z / 6;
    const long long N = (long long)g.L * g.L * g.L;
    const long long i = canonical_site(g.L, p, z, y, xh);
    const uint32_t b = J[((long long)blockIdx.z) * g.half + ((long long)z * g.L + y) * g.Lh + xh];
    for (int sl = 0; sl < SPW; ++sl) {
        const int sample = sg * SPW + sl;
        if (sample >= g.n_samples) break;
        dst[((long long)sample * 3 + d) * N + i] = (int8_t)(1 - 2 * (int)((b >> sl) & 1u));
    }
}

}  // namespace micsa
