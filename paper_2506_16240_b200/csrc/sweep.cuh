// sweep.cuh -- the microcanonical half-sweep.
//
// Elementary move, PAPER.md:119-124 (Eq. 8) and :150 (Eq. 10), for every site
// of one parity and all 32 systems of a word at once, Boolean operations only
// (PAPER.md:152).  With U = number of unsatisfied bonds among the six of the
// site, dH = 12 - 4U and n = 4m, so n - dH = 4(m + U - 3): the flip is legal
// iff 3 <= m + U <= 6 and then m <- m + U - 3.
#pragma once
#include "layout.cuh"

namespace micsa {

// one word: six "unsatisfied" indicators + daemon planes -> new spin / planes
__device__ __forceinline__ void creutz_word(uint32_t u1, uint32_t u2, uint32_t u3,
                                            uint32_t u4, uint32_t u5, uint32_t u6,
                                            uint32_t& sigma, uint32_t& m0, uint32_t& m1) {
    // 6 -> 3 bit population count with full adders
    const uint32_t sa = u1 ^ u2 ^ u3, ca = (u1 & u2) | (u3 & (u1 ^ u2));
    const uint32_t sb = u4 ^ u5 ^ u6, cb = (u4 & u5) | (u6 & (u4 ^ u5));
    const uint32_t U0 = sa ^ sb, cc = sa & sb;
    const uint32_t U1 = ca ^ cb ^ cc, U2 = (ca & cb) | (cc & (ca ^ cb));
    // S = m + U  (4 bits, S3 only enters the accept test)
    const uint32_t S0 = m0 ^ U0, c0 = m0 & U0;
    const uint32_t S1 = m1 ^ U1 ^ c0, c1 = (m1 & U1) | (c0 & (m1 ^ U1));
    const uint32_t S2 = U2 ^ c1, S3 = U2 & c1;
    // accept iff 3 <= S <= 6  <=>  S3 == 0 and S2 != (S1 & S0)
    const uint32_t acc = ~S3 & (S2 ^ (S1 & S0));
    // new level S - 3 for S in {3,4,5,6}: bit0 = ~S0, bit1 = S2 & (S1 | S0)
    sigma ^= acc;
    m0 = (acc & ~S0) | (~acc & m0);
    m1 = (acc & (S2 & (S1 | S0))) | (~acc & m1);
}

struct SweepArgs {
    uint32_t* spin; uint32_t* m0; uint32_t* m1; const void* J;
    int L, Lh, n_rg;
    long long half;
};

// One thread updates V consecutive words of one row (y,z) of the parity-p
// array of word lattice w.  grid = (ceil(L*(Lh/V)/block), L, n_words).
template <int V, int RPW>
__global__ void __launch_bounds__(128)
half_sweep_kernel(SweepArgs a, int p)
{
    typedef typename BondT<RPW>::type JT;
    const int nxv = a.Lh / V;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= a.L * nxv) return;
    const int y = t / nxv, xv = t - y * nxv;
    const int z = blockIdx.y, w = blockIdx.z;
    const int L = a.L, Lh = a.Lh;
    const int q = 1 - p;
    const long long half = a.half;

    uint32_t* sp = a.spin + ((long long)w * 2 + p) * half;
    const uint32_t* sq = a.spin + ((long long)w * 2 + q) * half;
    uint32_t* m0p = a.m0 + ((long long)w * 2 + p) * half;
    uint32_t* m1p = a.m1 + ((long long)w * 2 + p) * half;
    const int sg = w / a.n_rg;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;
    const JT* Jxp = Jb + (0 * 2 + p) * half; const JT* Jxq = Jb + (0 * 2 + q) * half;
    const JT* Jyp = Jb + (1 * 2 + p) * half; const JT* Jyq = Jb + (1 * 2 + q) * half;
    const JT* Jzp = Jb + (2 * 2 + p) * half; const JT* Jzq = Jb + (2 * 2 + q) * half;

    const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    const long long row = ((long long)z * L + y) * Lh;
    const int xh0 = xv * V;
    const long long h = row + xh0;
    const long long h_yp = ((long long)z * L + yp) * Lh + xh0;
    const long long h_ym = ((long long)z * L + ym) * Lh + xh0;
    const long long h_zp = ((long long)zp * L + y) * Lh + xh0;
    const long long h_zm = ((long long)zm * L + y) * Lh + xh0;
    // c = 1: x = 2xh+1, the -x neighbour has the same xh, the +x one xh+1
    // c = 0: x = 2xh,   the +x neighbour has the same xh, the -x one xh-1
    const int c = (y + z + p) & 1;
    const uint32_t cm = c ? 0xFFFFFFFFu : 0u;
    const int xe = c ? ((xh0 + V == Lh) ? 0 : xh0 + V) : ((xh0 == 0) ? Lh - 1 : xh0 - 1);

    Vec<V> s  = ldg_vec<V>(sp + h);
    Vec<V> d0 = ldg_vec<V>(m0p + h);
    Vec<V> d1 = ldg_vec<V>(m1p + h);
    const Vec<V> A   = ldg_vec<V>(sq + h);          // x-neighbour with the same xh
    const uint32_t e = sq[row + xe];                // the other x-neighbour of the end word
    const Vec<V> nyp = ldg_vec<V>(sq + h_yp), nym = ldg_vec<V>(sq + h_ym);
    const Vec<V> nzp = ldg_vec<V>(sq + h_zp), nzm = ldg_vec<V>(sq + h_zm);
    const Vec<V> jxo = ldg_bonds<V, RPW>(Jxp + h);  // own +x bond
    const Vec<V> jyo = ldg_bonds<V, RPW>(Jyp + h);
    const Vec<V> jzo = ldg_bonds<V, RPW>(Jzp + h);
    const Vec<V> B   = ldg_bonds<V, RPW>(Jxq + h);  // +x bond of the same-xh neighbour
    const uint32_t eJ = bond_expand<RPW>(Jxq[row + xe]);
    const Vec<V> jym = ldg_bonds<V, RPW>(Jyq + h_ym);
    const Vec<V> jzm = ldg_bonds<V, RPW>(Jzq + h_zm);

#pragma unroll
    for (int k = 0; k < V; ++k) {
        // x-neighbours and the bond towards -x (owned by the -x neighbour)
        const uint32_t up   = (k + 1 < V) ? A.v[k + 1] : e;    // xh+1 (valid for c=1)
        const uint32_t down = (k > 0) ? A.v[k - 1] : e;        // xh-1 (valid for c=0)
        const uint32_t n_xp = (cm & up) | (~cm & A.v[k]);
        const uint32_t n_xm = (cm & A.v[k]) | (~cm & down);
        const uint32_t Bdn  = (k > 0) ? B.v[k - 1] : eJ;
        const uint32_t j_xm = (cm & B.v[k]) | (~cm & Bdn);
        const uint32_t sg_  = s.v[k];
        creutz_word(sg_ ^ n_xp ^ jxo.v[k], sg_ ^ n_xm ^ j_xm,
                    sg_ ^ nyp.v[k] ^ jyo.v[k], sg_ ^ nym.v[k] ^ jym.v[k],
                    sg_ ^ nzp.v[k] ^ jzo.v[k], sg_ ^ nzm.v[k] ^ jzm.v[k],
                    s.v[k], d0.v[k], d1.v[k]);
    }
    stg_vec<V>(sp + h, s);
    stg_vec<V>(m0p + h, d0);
    stg_vec<V>(m1p + h, d1);
}

}  // namespace micsa
