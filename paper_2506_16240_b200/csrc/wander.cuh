// wander.cuh -- walkers (Sec. 2.6).
//
// One half of the two-timestep wandering cycle along `axis` (0,1,2 = X,Y,Z) in
// direction `sign`: every walker on a site of lattice parity p exchanges its
// value with the walker on the site's neighbour along sign*axis (periodic).
// The neighbour has the other parity, so in the parity-split layout this is
// an exchange between word h of the parity-p daemon planes and one word of the
// parity-(1-p) planes: the same row and xh, the row / plane next to it, or --
// along X -- xh or xh +- 1 depending on which of the two sites of the
// compressed x pair the source is (layout.cuh).  Each pair is touched by
// exactly one thread (the one of its parity-p member).  Spins are not touched.
#pragma once
#include "layout.cuh"

namespace micsa {

struct WanderArgs {
    uint32_t* m0; uint32_t* m1;
    int L, Lh;
    long long half;
};

// grid = (ceil(L*Lh/128), L, n_words); one thread per word of the parity-p planes
__global__ void __launch_bounds__(128)
wander_kernel(WanderArgs a, int axis, int sign, int p)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= a.L * a.Lh) return;
    const int L = a.L, Lh = a.Lh;
    const int y = t / Lh, xh = t - y * Lh;
    const int z = blockIdx.y, w = blockIdx.z, q = 1 - p;
    int yn = y, zn = z, xn = xh;
    if (axis == 0) {
        const int c = (y + z + p) & 1;            // x = 2*xh + c
        if (sign > 0) xn = c ? ((xh + 1 == Lh) ? 0 : xh + 1) : xh;     // x+1 = 2*xh' + (1-c)
        else          xn = c ? xh : ((xh == 0) ? Lh - 1 : xh - 1);
    } else if (axis == 1) {
        yn = (sign > 0) ? ((y + 1 == L) ? 0 : y + 1) : ((y == 0) ? L - 1 : y - 1);
    } else {
        zn = (sign > 0) ? ((z + 1 == L) ? 0 : z + 1) : ((z == 0) ? L - 1 : z - 1);
    }
    const long long hp = ((long long)w * 2 + p) * a.half + ((long long)z * L + y) * Lh + xh;
    const long long hq = ((long long)w * 2 + q) * a.half + ((long long)zn * L + yn) * Lh + xn;
    const uint32_t a0 = a.m0[hp], a1 = a.m1[hp];
    const uint32_t b0 = a.m0[hq], b1 = a.m1[hq];
    a.m0[hp] = b0; a.m1[hp] = b1;
    a.m0[hq] = a0; a.m1[hq] = a1;
}

}  // namespace micsa
