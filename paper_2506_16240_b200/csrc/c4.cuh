// c4.cuh -- four-point replica correlation along the lattice axes (SURVEY 8(f)
// rank 2; Eq. 16) for every replica pair a < b of every sample:
//   S[sample][pair][d][r] = sum_x q_x q_{x + r e_d},  q_x = s^a_x s^b_x,  r = 0..L/2,
// periodic; C4(r) = sum over pairs and axes / (3 N N_R (N_R - 1) / 2).
// Bit-sliced: X_x = sigma^a_x ^ sigma^b_x (one bit per sample) is first laid out
// in canonical site order, so a displacement is an index shift; then
// q_x q_y = 1 - 2 (X_x ^ X_y) and one block counts, per sample lane, the sites
// where X differs at distance r along d.  An occasional measurement (the paper
// takes it on a logarithmic time grid), not part of the timed step.
#pragma once
#include "layout.cuh"
#include "measure.cuh"

namespace micsa {

// Overlap field of one replica pair (a, b) for every sample of every sample group: replica a lives in word lattice
// sg * n_rg + rga at bit offset sha (0, or 16 for the second replica of a word), likewise b; mask = the sample lanes.
// grid = (ceil(L*Lh/128), L, n_sg*2)
__global__ void __launch_bounds__(128)
overlap_field_kernel(const uint32_t* __restrict__ spin, uint32_t* __restrict__ X, int L, int Lh, long long half,
                     int n_rg, int rga, int sha, int rgb, int shb, uint32_t mask)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= L * Lh) return;
    const int y = t / Lh, xh = t - y * Lh;
    const int z = blockIdx.y, sg = blockIdx.z >> 1, p = blockIdx.z & 1;
    const long long o = (long long)p * half + ((long long)z * L + y) * Lh + xh;
    const uint32_t sa = spin[((long long)(sg * n_rg + rga) * 2) * half + o];
    const uint32_t sb = spin[((long long)(sg * n_rg + rgb) * 2) * half + o];
    const long long N = 2 * half;
    X[(long long)sg * N + canonical_site(L, p, z, y, xh)] = ((sa >> sha) ^ (sb >> shb)) & mask;
}

// grid = (nblk, L/2 + 1, 3 * n_sg), block = kCountBlock; out[((sg*3 + d)*R + r)*32 + lane] += differing sites
__global__ void __launch_bounds__(kCountBlock)
c4_count_kernel(const uint32_t* __restrict__ X, unsigned long long* __restrict__ out, int L)
{
    const int r = blockIdx.y, d = blockIdx.z % 3, sg = blockIdx.z / 3;
    const uint32_t uL = (uint32_t)L, N = uL * uL * uL;
    const uint32_t* Xs = X + (long long)sg * N;
    const uint32_t stride[3] = { 1u, uL, uL * uL };
    VCount<kThreadPlanes> acc; acc.clear();
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < N; i += gridDim.x * blockDim.x) {
        const uint32_t x = i % uL, yz = i / uL, y = yz % uL, z = yz / uL;
        const uint32_t cd = (d == 0) ? x : (d == 1) ? y : z;
        const uint32_t cn = (cd + (uint32_t)r >= uL) ? cd + (uint32_t)r - uL : cd + (uint32_t)r;
        const uint32_t j = i + (cn - cd) * stride[d];            // mod 2^32 arithmetic: exact
        const uint32_t b[1] = { Xs[i] ^ Xs[j] };
        acc.add(b);
    }
    block_lane_counts(acc, out + (((long long)sg * 3 + d) * gridDim.y + r) * 32);
}

}  // namespace micsa
