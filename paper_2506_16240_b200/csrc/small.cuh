// small.cuh -- small lattices (SURVEY.md 7 "Tiny lattices": BASELINE configs 1 and 2): a whole
// schedule step -- daemon refresh (Eq. 11), n sweeps (Eq. 8 + 10, even then odd sites)
// and the measurement rows (Eq. 1, 4, C.1) -- in ONE launch.
//
// A lattice of 8^3 .. 32^3 sites gives a half-sweep a few microseconds of work at most, less than
// a kernel boundary costs, so the launch-per-half-sweep path is bound by launch latency (config 2:
// 3 us per half-sweep for 0.5 us of work).  Word lattices are independent systems, so here every
// word lattice gets ONE THREAD-BLOCK CLUSTER (1, 2, 4 or 8 CTAs): the cluster walks through the
// whole step by itself and the hardware cluster barrier (barrier.cluster, release / acquire)
// replaces the kernel boundary between half-sweeps; no grid-wide synchronisation exists at all.
// The state stays in L2 (opposite-parity spins are read with ld.global.cg, everything else a
// thread reads in a half-sweep it wrote itself); the update is the same 20-operation Boolean
// core as the large-lattice kernels (creutz_word20, sweep.cuh), the refresh the same lazy
// bit-plane compare (refresh_chunk, refresh.cuh), the counting the same carry-save trees
// (measure_item, measure.cuh).
#pragma once
#include "measure.cuh"
#include "refresh.cuh"
#include "sweep.cuh"

namespace micsa {

struct SmallArgs {
    SweepArgs a;                 // state of all word lattices (w0 unused)
    SiteGrid sg;                 // refresh: sample offsets
    MeasureArgs ma;              // counters (cntU / cntM / cntX)
    long long* rows;             // measurement rows kept: [rows_cap][row_len]
    long long* scratch_row;      // rows beyond rows_cap land here
    long long* min_E;            // [n_sys] running minimum of E, or nullptr
    long long row_len, row0, rows_cap;      // first row index of this launch
    unsigned long long* n_calls; // Philox calls (device counter)
    int n_words, cs;             // word lattices, CTAs per cluster
    int do_refresh; uint32_t step; uint32_t alpha_bits;
    int n_sweeps, measure_every; // measure after every measure_every-th sweep (0 = never)
    int n_samples, n_replicas, rpw, spw;
    long long N;
};

__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
    __threadfence();       // gpu-scope fence: also drops whatever this SM's L1 still holds of other CTAs' words
}

__device__ __forceinline__ uint4 ldcg4(const uint32_t* p) { return __ldcg(reinterpret_cast<const uint4*>(p)); }

// one item = the quad xq of row (y, z) of the parity-p array of one lattice
template <int RPW>
__device__ __forceinline__ void small_update_item(const SweepArgs& a, int w, int p, int it)
{
    typedef typename BondT<RPW>::type JT;
    const int L = a.L, Lh = a.Lh, nq = Lh >> 2, q = 1 - p;
    const int xq = it % nq, yz = it / nq, y = yz % L, z = yz / L;
    const long long half = a.half;
    uint32_t* sp = a.spin + ((long long)w * 2 + p) * half;
    const uint32_t* sq = a.spin + ((long long)w * 2 + q) * half;
    uint32_t* m0p = a.m0 + ((long long)w * 2 + p) * half;
    uint32_t* m1p = a.m1 + ((long long)w * 2 + p) * half;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)(w / a.n_rg) * 6 * half;
    const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    const int xh0 = 4 * xq;
    const int row = (z * L + y) * Lh, h = row + xh0;
    const int h_yp = (z * L + yp) * Lh + xh0, h_ym = (z * L + ym) * Lh + xh0;
    const int h_zp = (zp * L + y) * Lh + xh0, h_zm = (zm * L + y) * Lh + xh0;
    // c = 1: x = 2xh+1, the -x neighbour has the same xh, the +x one xh+1;  c = 0: x = 2xh, +x same xh, -x at xh-1
    const int c = (y + z + p) & 1;
    const uint32_t cm = 0u - (uint32_t)c;
    const int xe = c ? ((xh0 + 4 == Lh) ? 0 : xh0 + 4) : ((xh0 == 0) ? Lh - 1 : xh0 - 1);

    Vec<4> s = ldg_vec<4>(sp + h), d0 = ldg_vec<4>(m0p + h), d1 = ldg_vec<4>(m1p + h);      // written by this thread
    const uint4 A4 = ldcg4(sq + h), yp4 = ldcg4(sq + h_yp), ym4 = ldcg4(sq + h_ym);           // written by other CTAs
    const uint4 zp4 = ldcg4(sq + h_zp), zm4 = ldcg4(sq + h_zm);
    const uint32_t e = __ldcg(sq + row + xe);
    const Vec<4> jxo = ldg_bonds<4, RPW>(Jb + (0 * 2 + p) * half + h);
    const Vec<4> jyo = ldg_bonds<4, RPW>(Jb + (1 * 2 + p) * half + h);
    const Vec<4> jzo = ldg_bonds<4, RPW>(Jb + (2 * 2 + p) * half + h);
    const Vec<4> B   = ldg_bonds<4, RPW>(Jb + (0 * 2 + q) * half + h);
    const uint32_t eJ = bond_expand<RPW>(Jb[(0 * 2 + q) * half + row + xe]);
    const Vec<4> jym = ldg_bonds<4, RPW>(Jb + (1 * 2 + q) * half + h_ym);
    const Vec<4> jzm = ldg_bonds<4, RPW>(Jb + (2 * 2 + q) * half + h_zm);
    const uint32_t aw[4] = { A4.x, A4.y, A4.z, A4.w };
    const uint32_t ypv[4] = { yp4.x, yp4.y, yp4.z, yp4.w }, ymv[4] = { ym4.x, ym4.y, ym4.z, ym4.w };
    const uint32_t zpv[4] = { zp4.x, zp4.y, zp4.z, zp4.w }, zmv[4] = { zm4.x, zm4.y, zm4.z, zm4.w };
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t up = (k < 3) ? aw[k + 1] : e, dn = (k > 0) ? aw[k - 1] : e;
        const uint32_t bdn = (k > 0) ? B.v[k - 1] : eJ;
        const uint32_t nxp = (cm & up) | (~cm & aw[k]);
        const uint32_t nxm = (cm & aw[k]) | (~cm & dn);
        const uint32_t jxm = (cm & B.v[k]) | (~cm & bdn);
        const uint32_t g = s.v[k];
        creutz_word20(g ^ nxp ^ jxo.v[k], g ^ nxm ^ jxm,
                      g ^ ypv[k] ^ jyo.v[k], g ^ ymv[k] ^ jym.v[k],
                      g ^ zpv[k] ^ jzo.v[k], g ^ zmv[k] ^ jzm.v[k],
                      s.v[k], d0.v[k], d1.v[k]);
    }
    stg_vec<4>(sp + h, s);
    stg_vec<4>(m0p + h, d0);
    stg_vec<4>(m1p + h, d1);
}

// Eq. (11) for one word: the lazy bit-plane compare of refresh.cuh, all chunks in this thread
template <int RPW>
__device__ __forceinline__ unsigned small_refresh_word(const SmallArgs& A, const PhiloxKeys& ks, const RefreshThr& thr,
                                                       int w, int p, int word)
{
    constexpr int SPW = 32 / RPW;
    const SiteGrid& g = A.sg;
    const int sg = w / g.n_rg, rg = w - sg * g.n_rg;
    const uint32_t blk = (uint32_t)(g.sample_offset + sg * SPW) >> 4;
    const uint32_t vm = valid_lane_mask<RPW>(g.n_samples, sg);
    RefreshWord wd;
    wd.blk_a = blk; wd.blk_b = (RPW == 2) ? blk : blk + 1u;
    wd.rep_a = kTagRefresh | A.alpha_bits | (uint32_t)(rg * RPW);
    wd.rep_b = (RPW == 2) ? wd.rep_a + 1u : wd.rep_a;
    wd.has_b = (vm >> 16) != 0u;
    const int rowi = word / g.Lh, xh = word - rowi * g.Lh, z = rowi / g.L, y = rowi - z * g.L;
    wd.i = canonical_site(g.L, p, z, y, xh);
    uint32_t EQ[3], gt[3] = { 0u, 0u, 0u };
#pragma unroll
    for (int k = 0; k < 3; ++k) EQ[k] = thr.never[k] ? 0u : vm;
    unsigned calls = 0;
#pragma unroll 1
    for (uint32_t c = 0; c < 4; ++c) {
        refresh_chunk<-1>(c, wd, A.step, EQ, gt, thr, ks);
        calls += wd.has_b ? 2u : 1u;
        if ((EQ[0] | EQ[1] | EQ[2]) == 0u) break;
    }
    const uint32_t ge0 = gt[0] | EQ[0], ge1 = gt[1] | EQ[1], ge2 = gt[2] | EQ[2];
    const long long o = ((long long)w * 2 + p) * g.half + word;
    A.a.m0[o] = (ge0 ^ ge1 ^ ge2) & vm;
    A.a.m1[o] = ge1 & vm;
    return calls;
}

// counts of one lattice -> its entries of a measurement row; the lattice's counters are zeroed for the next one
__device__ __forceinline__ void small_finalize_lattice(const SmallArgs& A, int w, long long* row)
{
    const int n_sys = A.n_samples * A.n_replicas;
    const int sg = w / A.a.n_rg, rg = w - sg * A.a.n_rg;
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        const int r_local = lane / A.spw, sl = lane - r_local * A.spw;
        const int sample = sg * A.spw + sl, rep = rg * A.rpw + r_local;
        unsigned long long* cu = A.ma.cntU + (long long)w * 32 + lane;
        unsigned long long* cmv = A.ma.cntM + (long long)w * 32 + lane;
        if (sample < A.n_samples && rep < A.n_replicas) {
            const int t = sample * A.n_replicas + rep;
            const long long E = 2 * (long long)__ldcg(cu) - 3 * A.N;
            row[t] = E;
            row[n_sys + t] = 4 * (long long)__ldcg(cmv);
            if (A.min_E && E < A.min_E[t]) A.min_E[t] = E;
        }
        *cu = 0ull; *cmv = 0ull;
        if (A.n_replicas == 2) {                    // the pair shares the word (rpw == 2, n_rg == 1)
            unsigned long long* cx = A.ma.cntX + (long long)sg * 32 + lane;
            if (lane < A.spw && sample < A.n_samples) row[2 * n_sys + sample] = A.N - 2 * (long long)__ldcg(cx);
            *cx = 0ull;
        }
    }
}

// grid = n_words * cs CTAs in clusters of cs; block = a multiple of 32, at most 512
template <int RPW>
__global__ void __launch_bounds__(512)
small_step_kernel(SmallArgs A, PhiloxKeys ks, RefreshThr thr)
{
    typedef typename BondT<RPW>::type JT;
    __shared__ unsigned int s_cnt[32];
    const int w = blockIdx.x / A.cs, rank = blockIdx.x - w * A.cs;
    const int tid = rank * (int)blockDim.x + (int)threadIdx.x, nthr = A.cs * (int)blockDim.x;
    const int L = A.a.L, Lh = A.a.Lh, nq = Lh >> 2;
    const long long half = A.a.half;
    const int items = L * L * nq;                  // quad-rows per parity
    const bool pair = (RPW == 2) && A.n_replicas == 2;

    if (A.do_refresh) {
        unsigned calls = 0;
        for (int u = tid; u < 2 * (int)half; u += nthr) {
            const int p = (u >= (int)half) ? 1 : 0;
            calls += small_refresh_word<RPW>(A, ks, thr, w, p, u - p * (int)half);
        }
        calls = __reduce_add_sync(0xFFFFFFFFu, calls);
        if ((threadIdx.x & 31) == 0 && calls) atomicAdd(A.n_calls, (unsigned long long)calls);
        cluster_sync_all();
    }
    long long r = A.row0;
    for (int t = 1; t <= A.n_sweeps; ++t) {
        for (int p = 0; p < 2; ++p) {
            for (int it = tid; it < items; it += nthr) small_update_item<RPW>(A.a, w, p, it);
            cluster_sync_all();
        }
        if (A.measure_every > 0 && t % A.measure_every == 0) {
            // every thread counts its share of the lattice (L1 holds nothing stale: other CTAs' data were only
            // ever read through ld.global.cg, and a cluster barrier with acquire semantics came in between)
            const uint32_t items_p = (uint32_t)(half / 4), n_items = 2u * items_p;
            const uint32_t* s0 = A.a.spin + (long long)w * 2 * half;
            const uint32_t* d0 = A.a.m0 + (long long)w * 2 * half;
            const uint32_t* d1 = A.a.m1 + (long long)w * 2 * half;
            const JT* Jb = reinterpret_cast<const JT*>(A.a.J) + (long long)(w / A.a.n_rg) * 6 * half;
            VCount<kMeasurePlanes> accU, accM, accX; accU.clear(); accM.clear(); accX.clear();
            for (uint32_t it = (uint32_t)tid; it < n_items; it += (uint32_t)nthr) {
                ItemSums S;
                if (pair) measure_item<4, RPW, true>(S, it, items_p, (uint32_t)nq, (uint32_t)L, (uint32_t)Lh, half, s0, d0, d1, Jb);
                else      measure_item<4, RPW, false>(S, it, items_p, (uint32_t)nq, (uint32_t)L, (uint32_t)Lh, half, s0, d0, d1, Jb);
                accU.add(S.u); accM.add(S.m);
                if (pair) accX.add(S.x);
            }
            block_warp_lane_counts<kMeasurePlanes, 512>(accU.c, s_cnt, A.ma.cntU + (long long)w * 32);
            block_warp_lane_counts<kMeasurePlanes, 512>(accM.c, s_cnt, A.ma.cntM + (long long)w * 32);
            if (pair) block_warp_lane_counts<kMeasurePlanes, 512>(accX.c, s_cnt, A.ma.cntX + (long long)(w / A.a.n_rg) * 32);
            __threadfence();
            cluster_sync_all();
            if (rank == 0) {
                long long* row = (r < A.rows_cap) ? A.rows + r * A.row_len : A.scratch_row;
                small_finalize_lattice(A, w, row);
            }
            ++r;
            // the counters are zero again before anybody adds to them: two cluster barriers (the next sweep) lie between
        }
    }
}

}  // namespace micsa
