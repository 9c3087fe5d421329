// metropolis.cuh -- canonical comparator (PAPER.md:339-350
// Table 3, :130): standard Metropolis on the same checkerboard and the same
// bit-sliced layout, with a fresh random number per spin-flip attempt.
//
// Flip with probability min(1, exp(-dH/T)), dH = 12 - 4U for U unsatisfied
// bonds: always if U >= 3, else iff u < thr[2-U], thr[k] = floor(exp(-4(k+1)/T)
// * 2^32) from the host.  u is the attempt's own 32-bit uniform, defined
// bit-sliced exactly like the refresh's with domain tag 3 and
// the sweep index tau where the refresh has its step -- so the same
// lane-parallel, most-significant-plane-first compare applies (refresh_chunk)
// and planes that cannot change any decision are never generated: a lane only
// takes part in the compare with the one threshold its U selects, and not at
// all when dH <= 0.  No daemons are read or written.
#pragma once
#include "layout.cuh"
#include "philox.cuh"
#include "refresh.cuh"

namespace micsa {

struct MetropolisArgs {
    uint32_t* spin; const void* J;
    int L, Lh, n_rg, n_samples, sample_offset;
    long long half;
    uint32_t inv_Lh;         // fastdiv_magic(Lh)
};

constexpr int kMetroBlock = 128;
constexpr int kMetroSub = 4;          // groups of kMetroBlock words per block

// grid = (ceil(L*Lh / (128 * kMetroSub)), L, n_words).
// Phase 0: every thread gathers the six "unsatisfied" flags of its words (kMetroSub groups of 128 words per block)
// and runs chunk 0 (planes 0..7) of the compare.  About a quarter of the words still have a lane equal to its
// threshold prefix after 8 planes; they are queued in shared memory and phase c runs chunk c for the queued words
// only, densely on the threads of the block -- one barrier per phase and block (the scheme of refresh_kernel).
template <int RPW>
__global__ void __launch_bounds__(kMetroBlock)
metropolis_half_sweep_kernel(MetropolisArgs a, int p, PhiloxKeys ks, uint32_t tau, RefreshThr thr,
                             unsigned long long* __restrict__ n_calls)
{
    typedef typename BondT<RPW>::type JT;
    constexpr int SPW = 32 / RPW;
    constexpr int B = kMetroBlock, kQ = kMetroBlock * kMetroSub;
    __shared__ uint32_t q_word[2][kQ];            // word index inside the plane
    // per queued word: EQ[0]|EQ[1]|EQ[2], gt[0]|gt[1]|gt[2] (a lane belongs to at most one dH class, and EQ[k], gt[k] are
    // subsets of need[k], so the union loses nothing), need[3], spin word with the sure flips applied -- 6 words instead
    // of 10: 29 KB of queue per block instead of 45, six resident blocks per SM instead of five
    __shared__ uint32_t q_st[2][6][kQ];
    __shared__ int q_n[4];
    __shared__ unsigned int s_calls;
    if (threadIdx.x < 4) q_n[threadIdx.x] = 0;
    if (threadIdx.x == 0) s_calls = 0;
    __syncthreads();

    const int L = a.L, Lh = a.Lh, q = 1 - p;
    const int z = blockIdx.y, w = blockIdx.z;
    const long long half = a.half;
    uint32_t* sp = a.spin + ((long long)w * 2 + p) * half;
    const uint32_t* sq = a.spin + ((long long)w * 2 + q) * half;
    const int sg = w / a.n_rg, rg = w - sg * a.n_rg;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;
    const uint32_t vm = valid_lane_mask<RPW>(a.n_samples, sg);
    RefreshWord wd;
    const uint32_t blk = (uint32_t)(a.sample_offset + sg * SPW) >> 4;
    wd.blk_a = blk; wd.blk_b = (RPW == 2) ? blk : blk + 1u;
    wd.rep_a = kTagMetropolis | (uint32_t)(rg * RPW);
    wd.rep_b = (RPW == 2) ? wd.rep_a + 1u : wd.rep_a;
    wd.has_b = (vm >> 16) != 0u;
    const unsigned per_chunk = wd.has_b ? 2u : 1u;
    const uint32_t plane = (uint32_t)z * (uint32_t)L * (uint32_t)Lh;
    const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    unsigned int calls = 0;

    auto finish = [&](int word, const uint32_t (&EQ)[3], const uint32_t (&gt)[3], const uint32_t (&need)[3], uint32_t s_acc) {
        // u >= thr_k where the lane is above or equal in all planes seen; accept iff u < thr
        uint32_t acc = 0u;
#pragma unroll
        for (int k = 0; k < 3; ++k) acc |= need[k] & ~(gt[k] | EQ[k]);
        sp[plane + (uint32_t)word] = s_acc ^ (acc & vm);
    };
    auto push = [&](int c, int word, const uint32_t (&EQ)[3], const uint32_t (&gt)[3], const uint32_t (&need)[3], uint32_t s_acc) {
        const int slot = atomicAdd(&q_n[c], 1);
        const int b = c & 1;
        q_word[b][slot] = (uint32_t)word;
#pragma unroll
        for (int k = 0; k < 3; ++k) q_st[b][2 + k][slot] = need[k];
        q_st[b][0][slot] = EQ[0] | EQ[1] | EQ[2]; q_st[b][1][slot] = gt[0] | gt[1] | gt[2];
        q_st[b][5][slot] = s_acc;
    };

#pragma unroll 1
    for (int sub = 0; sub < kMetroSub; ++sub) {
        const int t = ((int)blockIdx.x * kMetroSub + sub) * B + (int)threadIdx.x;
        if (t >= L * Lh) break;
        const int y = (int)fastdiv((uint32_t)t, a.inv_Lh), xh = t - y * Lh;
        const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
        const uint32_t row = plane + (uint32_t)y * Lh, h = row + xh;
        const uint32_t h_yp = plane + (uint32_t)yp * Lh + xh, h_ym = plane + (uint32_t)ym * Lh + xh;
        const uint32_t h_zp = ((uint32_t)zp * L + y) * Lh + xh, h_zm = ((uint32_t)zm * L + y) * Lh + xh;
        // c = 1: x = 2xh+1, -x neighbour at xh (it owns the bond), +x neighbour at xh+1
        // c = 0: x = 2xh,   +x neighbour at xh, -x neighbour at xh-1 (it owns the bond)
        const int cx = (y + z + p) & 1;
        const int xo = cx ? ((xh + 1 == Lh) ? 0 : xh + 1) : ((xh == 0) ? Lh - 1 : xh - 1);
        const uint32_t s = sp[h];
        const uint32_t A = sq[h], E = sq[row + xo];
        const uint32_t n_xp = cx ? E : A, n_xm = cx ? A : E;
        const uint32_t j_xp = bond_expand<RPW>(Jb[(0 * 2 + p) * half + h]);
        const uint32_t j_xm = bond_expand<RPW>(Jb[(0 * 2 + q) * half + (cx ? h : row + xo)]);
        const uint32_t u1 = bond_flag(s, n_xp, j_xp), u2 = bond_flag(s, n_xm, j_xm);
        const uint32_t u3 = bond_flag(s, sq[h_yp], bond_expand<RPW>(Jb[(1 * 2 + p) * half + h]));
        const uint32_t u4 = bond_flag(s, sq[h_ym], bond_expand<RPW>(Jb[(1 * 2 + q) * half + h_ym]));
        const uint32_t u5 = bond_flag(s, sq[h_zp], bond_expand<RPW>(Jb[(2 * 2 + p) * half + h]));
        const uint32_t u6 = bond_flag(s, sq[h_zm], bond_expand<RPW>(Jb[(2 * 2 + q) * half + h_zm]));
        // U = number of unsatisfied bonds, 3 planes (each line one LOP3, sweep.cuh)
        const uint32_t sa = lop3<kXor3>(u1, u2, u3), ca = lop3<kMaj3>(u1, u2, u3);
        const uint32_t sb = lop3<kXor3>(u4, u5, u6), cb = lop3<kMaj3>(u4, u5, u6);
        const uint32_t U0 = sa ^ sb, cc = sa & sb;
        const uint32_t U1 = lop3<kXor3>(ca, cb, cc), U2 = lop3<kMaj3>(ca, cb, cc);
        const uint32_t always = U2 | (U1 & U0);                     // U >= 3: dH <= 0
        const uint32_t need[3] = { ~U2 & U1 & ~U0, ~U2 & ~U1 & U0, ~U2 & ~U1 & ~U0 };   // U = 2, 1, 0: dH = 4, 8, 12
        const uint32_t s_acc = s ^ (always & vm);
        uint32_t EQ[3], gt[3] = { 0u, 0u, 0u };
#pragma unroll
        for (int k = 0; k < 3; ++k) EQ[k] = thr.never[k] ? 0u : (need[k] & vm);
        bool more = (EQ[0] | EQ[1] | EQ[2]) != 0u;
        if (more) {
            wd.i = canonical_site(L, p, z, y, xh);
            refresh_chunk<0>(0u, wd, tau, EQ, gt, thr, ks);
            calls += per_chunk;
            more = (EQ[0] | EQ[1] | EQ[2]) != 0u;
        }
        if (more) push(0, t, EQ, gt, need, s_acc);
        else finish(t, EQ, gt, need, s_acc);
    }
#pragma unroll 1
    for (uint32_t c = 1; c < 4; ++c) {
        __syncthreads();                          // queue c-1 is complete
        const int n = q_n[c - 1];
        if (n == 0) break;                        // block-uniform
        const int b = (c - 1) & 1;
        for (int e = threadIdx.x; e < n; e += B) {
            const int word = (int)q_word[b][e];
            uint32_t EQ[3], gt[3], need[3];
#pragma unroll
            for (int k = 0; k < 3; ++k) need[k] = q_st[b][2 + k][e];
            const uint32_t EQa = q_st[b][0][e], gta = q_st[b][1][e];
#pragma unroll
            for (int k = 0; k < 3; ++k) { EQ[k] = EQa & need[k]; gt[k] = gta & need[k]; }
            const uint32_t s_acc = q_st[b][5][e];
            const int y = (int)fastdiv((uint32_t)word, a.inv_Lh), xh = word - y * Lh;
            wd.i = canonical_site(L, p, z, y, xh);
            refresh_chunk<-1>(c, wd, tau, EQ, gt, thr, ks);
            calls += per_chunk;
            if (c < 3 && (EQ[0] | EQ[1] | EQ[2]) != 0u) push((int)c, word, EQ, gt, need, s_acc);
            else finish(word, EQ, gt, need, s_acc);
        }
    }
    calls = __reduce_add_sync(0xFFFFFFFFu, calls);
    if ((threadIdx.x & 31) == 0 && calls) atomicAdd(&s_calls, calls);
    __syncthreads();
    if (threadIdx.x == 0 && s_calls) atomicAdd(n_calls, (unsigned long long)s_calls);
}

}  // namespace micsa
