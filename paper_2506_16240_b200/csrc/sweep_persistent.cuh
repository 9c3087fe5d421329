// sweep_persistent.cuh -- n half-sweeps in ONE launch (L % 8 == 0).
//
// Same elementary move and the same per-thread work as the pipelined
// row-marching kernel of sweep.cuh (PAPER.md:119-124 Eq. 8, :150 Eq. 10,
// order even -> odd -> even ... PAPER.md:198); what changes is who waits for
// whom.  A half-sweep of parity p only needs, around a site, the opposite
// parity's values of the PREVIOUS half-sweep: the
// dependence is local in space.  So instead of a kernel boundary (a full-chip
// barrier with its launch gap, ramp and tail) between half-sweeps, the lattice
// is cut into slabs of ZT planes, a slab into NSUB parts, and a task
//     (hs, w, slab, sub)  = half-sweep index, word lattice, slab, part
// may start as soon as all parts of the slabs slab-1, slab, slab+1 (periodic)
// of half-sweep hs-1 are done.  That covers both directions: their results are
// what this task reads, and they are the only readers of what it overwrites.
// Tasks are sized so that one half-sweep has (where the lattice allows) more
// than twice as many tasks as there are resident CTAs: then the tasks a CTA
// draws depend on tasks that finished long ago and nobody waits.
//
// CTAs are persistent and take tasks from a global ticket counter in
// lexicographic (hs, w, slab) order.  Every dependence of a ticket is a lower
// ticket, already claimed by a CTA that is running or done, so the lowest
// unfinished ticket can always proceed: no co-residency assumption, no
// deadlock.  Completion is published per slab as a monotone counter
// progress[w][slab] = number of finished tasks of that slab = NSUB * (base +
// half-sweeps done) between launches (release-add after a __threadfence by all
// writers + barrier); a consumer spins on it with ld.acquire, then the CTA
// barriers and reads with ordinary loads.
#pragma once
#include "sweep.cuh"

namespace micsa {

struct PersistArgs {
    SweepArgs a;
    int n_hs;                    // half-sweeps in this launch
    int p_first;                 // parity of the first one; then alternating
    int ZT, n_slabs;             // planes per slab, slabs per word lattice (L = ZT * n_slabs)
    int n_sub, sub_items;        // parts per slab, thread items per part (the last part may be short)
    int n_words;
    int base;                    // half-sweeps every slab had done at launch (progress = n_sub * base)
    int* progress;               // [n_words][n_slabs]
    unsigned long long* ticket;  // global task counter (monotone across launches)
    unsigned long long ticket0;  // its value at launch
};

__device__ __forceinline__ int ld_acquire_gpu(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void add_release_gpu(int* p, int v) {
    asm volatile("red.release.gpu.global.add.s32 [%0], %1;" :: "l"(p), "r"(v) : "memory");
}

constexpr int kPersistBlock = 256;

template <int RPW, int YC>
__global__ void __launch_bounds__(kPersistBlock, 2)
sweep_persistent_kernel(PersistArgs A)
{
    typedef typename Bond4<RPW>::elem JT;
    __shared__ unsigned long long s_ticket;
    const SweepArgs& a = A.a;
    const int L = a.L, Lh = a.Lh;
    const int nxv = Lh >> 2;
    const int items_per_plane = (L / YC) * nxv;
    const int items = A.ZT * items_per_plane;
    const long long half = a.half;
    const long long plane = (long long)L * Lh;
    const int tasks_per_word = A.n_slabs * A.n_sub;
    const unsigned long long tasks_per_hs = (unsigned long long)A.n_words * tasks_per_word;
    const unsigned long long total = tasks_per_hs * (unsigned long long)A.n_hs;

    for (;;) {
        __syncthreads();                                   // everyone has read the previous ticket
        if (threadIdx.x == 0) s_ticket = atomicAdd(A.ticket, 1ull) - A.ticket0;
        __syncthreads();
        const unsigned long long t = s_ticket;
        if (t >= total) break;
        const int hs = (int)(t / tasks_per_hs);
        const int r = (int)(t - (unsigned long long)hs * tasks_per_hs);
        const int w = r / tasks_per_word, r2 = r - w * tasks_per_word;
        const int slab = r2 / A.n_sub, sub = r2 - slab * A.n_sub;
        int* prog = A.progress + (long long)w * A.n_slabs;

        if (hs > 0 && threadIdx.x < 3) {                   // the three neighbour slabs, previous half-sweep
            int sn = slab - 1 + (int)threadIdx.x;
            sn = (sn < 0) ? sn + A.n_slabs : (sn >= A.n_slabs ? sn - A.n_slabs : sn);
            const int need = (A.base + hs) * A.n_sub;
            while (ld_acquire_gpu(prog + sn) < need) __nanosleep(32);
        }
        __syncthreads();

        const int p = A.p_first ^ (hs & 1), q = 1 - p;
        const int sg = w / a.n_rg;
        const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;
        uint32_t* spb = a.spin + ((long long)w * 2 + p) * half;
        uint32_t* m0b = a.m0 + ((long long)w * 2 + p) * half;
        uint32_t* m1b = a.m1 + ((long long)w * 2 + p) * half;
        const uint32_t* sqb = a.spin + ((long long)w * 2 + q) * half;

        const int item_end = min(items, (sub + 1) * A.sub_items);
        for (int item = sub * A.sub_items + threadIdx.x; item < item_end; item += blockDim.x) {
            const int lz = item / items_per_plane, it = item - lz * items_per_plane;
            const int chunk = it / nxv, xv = it - chunk * nxv;
            const int z = slab * A.ZT + lz;
            const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
            RowPtrs P;
            P.sp = spb + z * plane; P.m0 = m0b + z * plane; P.m1 = m1b + z * plane;
            P.sq = sqb + z * plane; P.sq_zp = sqb + zp * plane; P.sq_zm = sqb + zm * plane;
            P.jx = Jb + (0 * 2 + p) * half + z * plane;
            P.jy = Jb + (1 * 2 + p) * half + z * plane;
            P.jz = Jb + (2 * 2 + p) * half + z * plane;
            P.jxq = Jb + (0 * 2 + q) * half + z * plane;
            P.jyq = Jb + (1 * 2 + q) * half + z * plane;
            P.jzq_zm = Jb + (2 * 2 + q) * half + zm * plane;
            if ((z + p) & 1) march_rows_pipe<RPW, YC, 1>(P, L, Lh, chunk * YC, xv * 4);
            else             march_rows_pipe<RPW, YC, 0>(P, L, Lh, chunk * YC, xv * 4);
        }

        __threadfence();                                   // every writer: results visible device-wide ...
        __syncthreads();
        if (threadIdx.x == 0) add_release_gpu(prog + slab, 1);               // ... before the part is published
    }
}

}  // namespace micsa
