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
// CTAs are persistent and take the tasks of a lattice from its ticket counter
// in lexicographic (hs, slab, sub) order.  Every dependence of a ticket is a lower
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
    int n_groups;                // word lattices worked on at the same time (gridDim.x % n_groups == 0)
    int base;                    // half-sweeps every slab had done at launch (progress = n_sub * base)
    int* progress;               // [n_words][n_slabs]
    unsigned long long* ticket;  // [n_words] task counters (monotone across launches)
    unsigned long long ticket0;  // their common value at launch
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

// one task: items [item0, item1) of slab `slab` of lattice w, parity P (compile time)
template <int RPW, int YC, int P>
__device__ __forceinline__ void persistent_task(const PersistArgs& A, int w, int slab, int item0, int item1)
{
    const SweepArgs& a = A.a;
    const int L = a.L, Lh = a.Lh;
    const int nxv = Lh >> 2;
    const int items_per_plane = (L / YC) * nxv;
    const PipeBase B = pipe_base<RPW>(a, w, P);            // w comes from blockIdx: uniform registers
    // consecutive threads own consecutive items (quads of a row, rows one after the other)
    for (int item = item0 + (int)threadIdx.x; ; item += (int)blockDim.x) {
        const bool active = item < item1;
        const unsigned mask = __ballot_sync(0xFFFFFFFFu, active);
        if (mask == 0u) break;                              // the whole warp is past the end
        if (!active) continue;
        const int lz = item / items_per_plane, it = item - lz * items_per_plane;
        const int chunk = it / nxv, xv = it - chunk * nxv;
        const int z = slab * A.ZT + lz;
        // shuffles need one code path per warp: only when a task lies inside one plane
        const XNb nb = x_neighbours((int)threadIdx.x, xv, nxv, mask, A.ZT == 1);
        if ((z + P) & 1) march_rows_pipe<RPW, YC, 1>(B, L, Lh, z, chunk * YC, xv * 4, nb);
        else             march_rows_pipe<RPW, YC, 0>(B, L, Lh, z, chunk * YC, xv * 4, nb);
    }
}

// CTA b works for the lattices w = b % n_groups, + n_groups, ... one after the
// other, each for all n_hs half-sweeps (a lattice never interacts with
// another one, and finishing one before touching the next keeps its state in
// L2 for the whole launch when the full state does not fit).
template <int RPW, int YC>
__global__ void __launch_bounds__(kPersistBlock, 2)
sweep_persistent_kernel(PersistArgs A)
{
    __shared__ unsigned long long s_ticket;
    const int items = A.ZT * (A.a.L / YC) * (A.a.Lh >> 2);
    const int tasks_per_hs = A.n_slabs * A.n_sub;
    const unsigned long long total = (unsigned long long)tasks_per_hs * (unsigned long long)A.n_hs;

    for (int w = (int)blockIdx.x % A.n_groups; w < A.n_words; w += A.n_groups) {
        int* prog = A.progress + (long long)w * A.n_slabs;
        for (;;) {
            __syncthreads();                               // everyone has read the previous ticket
            if (threadIdx.x == 0) s_ticket = atomicAdd(A.ticket + w, 1ull) - A.ticket0;
            __syncthreads();
            const unsigned long long t = s_ticket;
            if (t >= total) break;
            const int hs = (int)(t / (unsigned)tasks_per_hs);
            const int r = (int)(t - (unsigned long long)hs * tasks_per_hs);
            const int slab = r / A.n_sub, sub = r - slab * A.n_sub;

            if (hs > 0 && threadIdx.x < 3) {               // the three neighbour slabs, previous half-sweep
                int sn = slab - 1 + (int)threadIdx.x;
                sn = (sn < 0) ? sn + A.n_slabs : (sn >= A.n_slabs ? sn - A.n_slabs : sn);
                const int need = (A.base + hs) * A.n_sub;
                while (ld_acquire_gpu(prog + sn) < need) __nanosleep(32);
            }
            __syncthreads();

            const int item0 = sub * A.sub_items, item1 = min(items, item0 + A.sub_items);
            if ((A.p_first ^ hs) & 1) persistent_task<RPW, YC, 1>(A, w, slab, item0, item1);
            else                      persistent_task<RPW, YC, 0>(A, w, slab, item0, item1);

            __threadfence();                               // every writer: results visible device-wide ...
            __syncthreads();
            if (threadIdx.x == 0) add_release_gpu(prog + slab, 1);   // ... before the part is published
        }
    }
}

}  // namespace micsa
