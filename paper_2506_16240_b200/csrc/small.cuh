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
// The lattice is held ON CHIP for the whole launch: every CTA of the cluster loads a slab of L/cs planes (spins,
// daemon planes, bonds; both parities) into its shared memory, the opposite-parity planes just across a slab
// boundary are read from the neighbouring CTA's shared memory (distributed shared memory, ld.shared::cluster), and
// the slabs go back to global memory once at the end; the update is the same 20-operation Boolean
// core as the large-lattice kernels (creutz_word20, sweep.cuh), the refresh the same lazy
// bit-plane compare (refresh_chunk, refresh.cuh), the counting the same carry-save trees
// (measure_item, measure.cuh).
#pragma once
#include "measure.cuh"
#include "refresh.cuh"
#include "sweep.cuh"

namespace micsa {

constexpr int kSmallChain = 8;   // schedule steps one launch can walk through

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
    // The launch walks through n_chain schedule steps.  Step j first takes its daemon levels from the planes
    // ch_m0[j] / ch_m1[j] (a refresh generated beforehand by refresh_kernel; nullptr, step 0 only: the levels the
    // state holds, refreshed here if do_refresh), then does ch_sweeps[j] sweeps and measures after every
    // ch_every[j]-th of them (0 = never).
    int n_chain;
    const uint32_t* ch_m0[kSmallChain]; const uint32_t* ch_m1[kSmallChain];
    int ch_sweeps[kSmallChain], ch_every[kSmallChain];
    int n_samples, n_replicas, rpw, spw;
    long long N;
};

__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
// shared::cta address -> the same offset in the shared memory of CTA `rank` of this cluster
__device__ __forceinline__ uint32_t dsmem_addr(uint32_t local, uint32_t rank) {
    uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local), "r"(rank));
    return r;
}
__device__ __forceinline__ uint4 ld_cluster4(uint32_t a) {
    uint4 v; asm volatile("ld.shared::cluster.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ uint4 lds4(uint32_t a) {
    uint4 v; asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ uint32_t lds1(uint32_t a) {
    uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts4(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.u32 [%0], {%1,%2,%3,%4};" :: "r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}

// Shared-memory image of the ZP planes a CTA owns (both parities): byte offsets from the start of dynamic smem.
// PW = words per parity plane (L * Lh).  The z-bond arrays carry one more plane in front (plane z0 - 1, periodic):
// the bond towards -z of a site in the CTA's first plane is owned by the plane below, and bonds never change.
template <int RPW> struct SlabLayout {
    typedef typename BondT<RPW>::type JT;
    uint32_t ZP, PW, ZPW, ZPJ;
    __host__ __device__ SlabLayout(int zp, int pw) : ZP((uint32_t)zp), PW((uint32_t)pw), ZPW((uint32_t)zp * pw * 4u), ZPJ((uint32_t)zp * pw * (uint32_t)sizeof(JT)) {}
    __host__ __device__ uint32_t spin(int p) const { return (uint32_t)p * ZPW; }
    __host__ __device__ uint32_t m0(int p) const { return 2u * ZPW + (uint32_t)p * ZPW; }
    __host__ __device__ uint32_t m1(int p) const { return 4u * ZPW + (uint32_t)p * ZPW; }
    __host__ __device__ uint32_t jx(int p) const { return 6u * ZPW + (uint32_t)p * ZPJ; }
    __host__ __device__ uint32_t jy(int p) const { return 6u * ZPW + (2u + (uint32_t)p) * ZPJ; }
    __host__ __device__ uint32_t jz(int p) const { return 6u * ZPW + 4u * ZPJ + (uint32_t)p * (ZP + 1u) * PW * (uint32_t)sizeof(JT); }   // plane -1 first
    __host__ __device__ uint32_t total() const { return 6u * ZPW + 4u * ZPJ + 2u * (ZP + 1u) * PW * (uint32_t)sizeof(JT); }
};

template <int RPW> __device__ __forceinline__ void lds_bonds4(uint32_t addr, uint32_t (&o)[4]);
template <> __device__ __forceinline__ void lds_bonds4<2>(uint32_t addr, uint32_t (&o)[4]) {
    uint2 t; asm volatile("ld.shared.v2.u32 {%0,%1}, [%2];" : "=r"(t.x), "=r"(t.y) : "r"(addr));
    Bond4<2>::expand(t, o);
}
template <> __device__ __forceinline__ void lds_bonds4<1>(uint32_t addr, uint32_t (&o)[4]) {
    const uint4 t = lds4(addr); Bond4<1>::expand(t, o);
}
template <int RPW> __device__ __forceinline__ uint32_t lds_bond1(uint32_t addr);
template <> __device__ __forceinline__ uint32_t lds_bond1<2>(uint32_t addr) {
    uint32_t v; asm volatile("{ .reg .u16 t; ld.shared.u16 t, [%1]; cvt.u32.u16 %0, t; }" : "=r"(v) : "r"(addr));
    return __byte_perm(v, 0u, 0x1010);
}
template <> __device__ __forceinline__ uint32_t lds_bond1<1>(uint32_t addr) { return lds1(addr); }

// one item = the quad xq of row y of the CTA's plane zl (lattice plane z0 + zl), parity p; everything in shared
// memory, the opposite-parity planes z +- 1 possibly in the neighbouring CTA's (distributed shared memory)
template <int RPW>
__device__ __forceinline__ void slab_update_item(const SlabLayout<RPW>& S, uint32_t sm, int L, int Lh, int z0, int rank, int cs,
                                                 int p, int it)
{
    typedef typename BondT<RPW>::type JT;
    constexpr uint32_t JS = sizeof(JT);
    const int nq = Lh >> 2, q = 1 - p, ZP = (int)S.ZP;
    const int xq = it % nq, r2 = it / nq, y = r2 % L, zl = r2 / L;
    const int z = z0 + zl;
    const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const int xh0 = 4 * xq;
    const uint32_t row = (uint32_t)(zl * L + y) * Lh, h = row + xh0;
    const uint32_t h_yp = (uint32_t)(zl * L + yp) * Lh + xh0, h_ym = (uint32_t)(zl * L + ym) * Lh + xh0;
    const int c = (y + z + p) & 1;
    const uint32_t cm = 0u - (uint32_t)c;
    const int xe = c ? ((xh0 + 4 == Lh) ? 0 : xh0 + 4) : ((xh0 == 0) ? Lh - 1 : xh0 - 1);

    const uint32_t a_s = sm + S.spin(p) + h * 4u, a_0 = sm + S.m0(p) + h * 4u, a_1 = sm + S.m1(p) + h * 4u;
    const uint4 s4 = lds4(a_s), d04 = lds4(a_0), d14 = lds4(a_1);
    const uint32_t sq = sm + S.spin(q);
    const uint4 A4 = lds4(sq + h * 4u), yp4 = lds4(sq + h_yp * 4u), ym4 = lds4(sq + h_ym * 4u);
    const uint32_t e = lds1(sq + (row + xe) * 4u);
    // planes z + 1 and z - 1 of the opposite parity: in this CTA, or in the next / previous one of the cluster
    const uint32_t in_plane = ((uint32_t)y * Lh + xh0) * 4u;
    uint4 zp4, zm4;
    if (zl + 1 < ZP) zp4 = lds4(sq + ((uint32_t)(zl + 1) * S.PW) * 4u + in_plane);
    else             zp4 = ld_cluster4(dsmem_addr(sq + in_plane, (uint32_t)((rank + 1 == cs) ? 0 : rank + 1)));
    if (zl > 0)      zm4 = lds4(sq + ((uint32_t)(zl - 1) * S.PW) * 4u + in_plane);
    else             zm4 = ld_cluster4(dsmem_addr(sq + ((uint32_t)(ZP - 1) * S.PW) * 4u + in_plane, (uint32_t)((rank == 0) ? cs - 1 : rank - 1)));
    uint32_t jxo[4], jyo[4], jzo[4], Bx[4], jym[4], jzm[4];
    lds_bonds4<RPW>(sm + S.jx(p) + h * JS, jxo);
    lds_bonds4<RPW>(sm + S.jy(p) + h * JS, jyo);
    lds_bonds4<RPW>(sm + S.jz(p) + (S.PW + h) * JS, jzo);           // the z arrays start at plane -1
    lds_bonds4<RPW>(sm + S.jx(q) + h * JS, Bx);
    lds_bonds4<RPW>(sm + S.jy(q) + h_ym * JS, jym);
    lds_bonds4<RPW>(sm + S.jz(q) + h * JS, jzm);                    // plane zl - 1
    const uint32_t eJ = lds_bond1<RPW>(sm + S.jx(q) + (row + xe) * JS);
    const uint32_t aw[4] = { A4.x, A4.y, A4.z, A4.w };
    uint32_t sv[4] = { s4.x, s4.y, s4.z, s4.w }, v0[4] = { d04.x, d04.y, d04.z, d04.w }, v1[4] = { d14.x, d14.y, d14.z, d14.w };
    const uint32_t ypv[4] = { yp4.x, yp4.y, yp4.z, yp4.w }, ymv[4] = { ym4.x, ym4.y, ym4.z, ym4.w };
    const uint32_t zpv[4] = { zp4.x, zp4.y, zp4.z, zp4.w }, zmv[4] = { zm4.x, zm4.y, zm4.z, zm4.w };
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        // c = 1: x = 2xh+1, the -x neighbour has the same xh, the +x one xh+1;  c = 0: x = 2xh, +x same xh, -x at xh-1
        const uint32_t up = (k < 3) ? aw[k + 1] : e, dn = (k > 0) ? aw[k - 1] : e;
        const uint32_t bdn = (k > 0) ? Bx[k - 1] : eJ;
        const uint32_t nxp = lop3<kSel>(cm, up, aw[k]);
        const uint32_t nxm = lop3<kSel>(cm, aw[k], dn);
        const uint32_t jxm = lop3<kSel>(cm, Bx[k], bdn);
        const uint32_t g = sv[k];
        creutz_word20(bond_flag(g, nxp, jxo[k]), bond_flag(g, nxm, jxm),
                      bond_flag(g, ypv[k], jyo[k]), bond_flag(g, ymv[k], jym[k]),
                      bond_flag(g, zpv[k], jzo[k]), bond_flag(g, zmv[k], jzm[k]),
                      sv[k], v0[k], v1[k]);
    }
    sts4(a_s, sv[0], sv[1], sv[2], sv[3]);
    sts4(a_0, v0[0], v0[1], v0[2], v0[3]);
    sts4(a_1, v1[0], v1[1], v1[2], v1[3]);
}

// counting of one item (quad of row y, plane zl, parity p): unsatisfied own +x, +y, +z bonds, levels, replica differences
template <int RPW, bool PAIR>
__device__ __forceinline__ void slab_measure_item(const SlabLayout<RPW>& S, uint32_t sm, int L, int Lh, int z0, int rank, int cs,
                                                  int p, int it, ItemSums& r)
{
    typedef typename BondT<RPW>::type JT;
    constexpr uint32_t JS = sizeof(JT);
    const int nq = Lh >> 2, q = 1 - p, ZP = (int)S.ZP;
    const int xq = it % nq, r2 = it / nq, y = r2 % L, zl = r2 / L;
    const int z = z0 + zl;
    const int yp = (y + 1 == L) ? 0 : y + 1;
    const int xh0 = 4 * xq;
    const uint32_t row = (uint32_t)(zl * L + y) * Lh, h = row + xh0;
    const int c = (y + z + p) & 1;                      // c = 1: the +x neighbour is word xh+1, else the same xh
    const uint32_t sq = sm + S.spin(q);
    const uint4 s4 = lds4(sm + S.spin(p) + h * 4u), A4 = lds4(sq + h * 4u);
    const uint32_t e = lds1(sq + (row + ((xh0 + 4 == Lh) ? 0 : xh0 + 4)) * 4u);
    const uint4 ny4 = lds4(sq + ((uint32_t)(zl * L + yp) * Lh + xh0) * 4u);
    const uint32_t in_plane = ((uint32_t)y * Lh + xh0) * 4u;
    uint4 nz4;
    if (zl + 1 < ZP) nz4 = lds4(sq + ((uint32_t)(zl + 1) * S.PW) * 4u + in_plane);
    else             nz4 = ld_cluster4(dsmem_addr(sq + in_plane, (uint32_t)((rank + 1 == cs) ? 0 : rank + 1)));
    uint32_t jx[4], jy[4], jz[4];
    lds_bonds4<RPW>(sm + S.jx(p) + h * JS, jx);
    lds_bonds4<RPW>(sm + S.jy(p) + h * JS, jy);
    lds_bonds4<RPW>(sm + S.jz(p) + (S.PW + h) * JS, jz);
    const uint4 b04 = lds4(sm + S.m0(p) + h * 4u), b14 = lds4(sm + S.m1(p) + h * 4u);
    const uint32_t sv[4] = { s4.x, s4.y, s4.z, s4.w }, aw[4] = { A4.x, A4.y, A4.z, A4.w };
    const uint32_t ny[4] = { ny4.x, ny4.y, ny4.z, ny4.w }, nz[4] = { nz4.x, nz4.y, nz4.z, nz4.w };
    uint32_t us[4], uc[4], xs[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t up = (k < 3) ? aw[k + 1] : e;
        const uint32_t nx = c ? up : aw[k];
        full_add(sv[k] ^ nx ^ jx[k], sv[k] ^ ny[k] ^ jy[k], sv[k] ^ nz[k] ^ jz[k], us[k], uc[k]);
        xs[k] = PAIR ? ((sv[k] ^ (sv[k] >> 16)) & 0xFFFFu) : 0u;
    }
    const uint32_t m_lo[4] = { b04.x, b04.y, b04.z, b04.w }, m_hi[4] = { b14.x, b14.y, b14.z, b14.w };
    csa_4x1_4x2(us, uc, r.u);
    csa_4x1_4x2(m_lo, m_hi, r.m);
    if (PAIR) {
        uint32_t a2, b2, b3;
        full_add(xs[0], xs[1], xs[2], a2, b2);
        half_add(a2, xs[3], r.x[0], b3);
        r.x[1] = b2 ^ b3; r.x[2] = b2 & b3;
    } else { r.x[0] = r.x[1] = r.x[2] = 0u; }
}

// Eq. (11) for one word of the CTA's slab: the lazy bit-plane compare of refresh.cuh, all chunks in this thread
template <int RPW>
__device__ __forceinline__ unsigned slab_refresh_word(const SmallArgs& A, const PhiloxKeys& ks, const RefreshThr& thr,
                                                      const SlabLayout<RPW>& S, unsigned char* smem, int w, int z0, int p, int word)
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
    const int rowi = word / g.Lh, xh = word - rowi * g.Lh, zl = rowi / g.L, y = rowi - zl * g.L;
    wd.i = canonical_site(g.L, p, z0 + zl, y, xh);
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
    reinterpret_cast<uint32_t*>(smem + S.m0(p))[word] = (ge0 ^ ge1 ^ ge2) & vm;
    reinterpret_cast<uint32_t*>(smem + S.m1(p))[word] = ge1 & vm;
    return calls;
}

__device__ __forceinline__ uint32_t ld_cluster1(uint32_t a) {
    uint32_t v; asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(a));
    return v;
}

// Counts of one lattice -> its entries of a measurement row.  The lattice belongs to one cluster, so its counts never
// leave the chip: every CTA leaves the lane totals of its slab in its shared memory (s_tot[3][32]: unsatisfied bonds,
// levels, replica differences), and after a cluster barrier the first 32 threads of CTA 0 add them up through
// distributed shared memory and write the row -- no global atomics, no fence, no counters to read back and re-zero
// (the first version went through the global counters of the general path: 5.5 us per row instead of 3).
// run_min: the finalising thread's running minimum of E over the rows of this launch (folded into min_E at the end of
// the launch: a read-modify-write of global memory per row sat on the critical path between two cluster barriers).
__device__ __forceinline__ void small_finalize_lattice(const SmallArgs& A, int w, long long* row, const unsigned int* s_tot, int cs,
                                                       long long& run_min)
{
    const int n_sys = A.n_samples * A.n_replicas;
    const int sg = w / A.a.n_rg, rg = w - sg * A.a.n_rg;
    if (threadIdx.x < 32) {
        const int lane = threadIdx.x;
        unsigned long long U = 0, M = 0, X = 0;
        const uint32_t base = smem_u32(s_tot + lane);
        for (int q = 0; q < cs; ++q) {
            const uint32_t a = dsmem_addr(base, (uint32_t)q);
            U += ld_cluster1(a); M += ld_cluster1(a + 32u * 4u); X += ld_cluster1(a + 64u * 4u);
        }
        const int r_local = lane / A.spw, sl = lane - r_local * A.spw;
        const int sample = sg * A.spw + sl, rep = rg * A.rpw + r_local;
        if (sample < A.n_samples && rep < A.n_replicas) {
            const int t = sample * A.n_replicas + rep;
            const long long E = 2 * (long long)U - 3 * A.N;
            row[t] = E;
            row[n_sys + t] = 4 * (long long)M;
            run_min = E < run_min ? E : run_min;
        }
        if (A.n_replicas == 2 && lane < A.spw && sample < A.n_samples)     // the pair shares the word (rpw == 2, n_rg == 1)
            row[2 * n_sys + sample] = A.N - 2 * (long long)X;
    }
}

// grid = n_words * cs CTAs in clusters of cs (cs divides L); block = a multiple of 32, at most 512;
// dynamic shared memory = SlabLayout(L / cs, L * Lh).total()
template <int RPW>
__global__ void __launch_bounds__(512)
small_step_kernel(SmallArgs A, PhiloxKeys ks, RefreshThr thr)
{
    typedef typename BondT<RPW>::type JT;
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ unsigned int s_tot[3 * 32];                            // lane totals of this CTA's slab: U | M | X
    const int w = blockIdx.x / A.cs, rank = blockIdx.x - w * A.cs, cs = A.cs;
    const int L = A.a.L, Lh = A.a.Lh, nq = Lh >> 2;
    const int ZP = L / cs, z0 = rank * ZP, PW = L * Lh;
    const SlabLayout<RPW> S(ZP, PW);
    const uint32_t sm = smem_u32(smem);
    const long long half = A.a.half;
    const int tid = threadIdx.x, nthr = blockDim.x;
    const bool pair = (RPW == 2) && A.n_replicas == 2;
    const int slab_words = ZP * PW;                                   // words per parity of this CTA
    const JT* Jb = reinterpret_cast<const JT*>(A.a.J) + (long long)(w / A.a.n_rg) * 6 * half;

    // ---- global -> shared: the CTA's planes of every array (both parities); 128-bit copies
    for (int p = 0; p < 2; ++p) {
        const long long go = ((long long)w * 2 + p) * half + (long long)z0 * PW;
        const uint4* gs = reinterpret_cast<const uint4*>(A.a.spin + go);
        uint4* ss = reinterpret_cast<uint4*>(smem + S.spin(p));
        for (int i = tid; i < slab_words / 4; i += nthr) ss[i] = gs[i];
        // bonds: PW * sizeof(JT) bytes per plane, a multiple of 16 (Lh % 4 == 0 and L even)
        const int jq = (int)((size_t)slab_words * sizeof(JT) / 16), pq = (int)((size_t)PW * sizeof(JT) / 16);
        const uint4* gx = reinterpret_cast<const uint4*>(Jb + (0 * 2 + p) * half + (long long)z0 * PW);
        const uint4* gy = reinterpret_cast<const uint4*>(Jb + (1 * 2 + p) * half + (long long)z0 * PW);
        const uint4* gz = reinterpret_cast<const uint4*>(Jb + (2 * 2 + p) * half + (long long)z0 * PW);
        const uint4* gzm = reinterpret_cast<const uint4*>(Jb + (2 * 2 + p) * half + (long long)((z0 == 0) ? L - 1 : z0 - 1) * PW);
        uint4* sx = reinterpret_cast<uint4*>(smem + S.jx(p));
        uint4* sy = reinterpret_cast<uint4*>(smem + S.jy(p));
        uint4* sz = reinterpret_cast<uint4*>(smem + S.jz(p));
        for (int i = tid; i < jq; i += nthr) { sx[i] = gx[i]; sy[i] = gy[i]; sz[pq + i] = gz[i]; }
        for (int i = tid; i < pq; i += nthr) sz[i] = gzm[i];
    }
    const int items = ZP * L * nq;                                    // quad rows per parity of this CTA
    long long r = A.row0;
    long long run_min = 0x7FFFFFFFFFFFFFFFll;                         // rank 0, threads 0..31: minimum of E of "their" system
    const bool few = 2 * items <= 2 * nthr;                           // at most two items per thread: counts < 32, five planes
#pragma unroll 1
    for (int j = 0; j < A.n_chain; ++j) {
        // ---- this step's daemon levels: global -> shared.  Nobody reads the CTA's daemon planes any more: the last
        // half-sweep and the last measurement of the previous step ended with a cluster barrier.
        {
            const uint32_t* src0 = A.ch_m0[j] ? A.ch_m0[j] : A.a.m0;
            const uint32_t* src1 = A.ch_m1[j] ? A.ch_m1[j] : A.a.m1;
            for (int p = 0; p < 2; ++p) {
                const long long go = ((long long)w * 2 + p) * half + (long long)z0 * PW;
                const uint4* g0 = reinterpret_cast<const uint4*>(src0 + go);
                const uint4* g1 = reinterpret_cast<const uint4*>(src1 + go);
                uint4* s0 = reinterpret_cast<uint4*>(smem + S.m0(p));
                uint4* s1 = reinterpret_cast<uint4*>(smem + S.m1(p));
                for (int i = tid; i < slab_words / 4; i += nthr) { s0[i] = g0[i]; s1[i] = g1[i]; }
            }
        }
        __syncthreads();
        if (j == 0 && A.do_refresh) {
            unsigned calls = 0;
            for (int u = tid; u < 2 * slab_words; u += nthr) {
                const int p = (u >= slab_words) ? 1 : 0;
                calls += slab_refresh_word<RPW>(A, ks, thr, S, smem, w, z0, p, u - p * slab_words);
            }
            calls = __reduce_add_sync(0xFFFFFFFFu, calls);
            if ((threadIdx.x & 31) == 0 && calls) atomicAdd(A.n_calls, (unsigned long long)calls);
        }
        cluster_sync_all();                                           // every CTA's slab is in place
        const int n_sweeps = A.ch_sweeps[j], every = A.ch_every[j];
        for (int t = 1; t <= n_sweeps; ++t) {
            for (int p = 0; p < 2; ++p) {
                for (int it = tid; it < items; it += nthr) slab_update_item<RPW>(S, sm, L, Lh, z0, rank, cs, p, it);
                cluster_sync_all();
            }
            if (every > 0 && t % every == 0) {
                VCount<kMeasurePlanes> accU, accM, accX; accU.clear(); accM.clear(); accX.clear();
                for (int u = tid; u < 2 * items; u += nthr) {
                    const int p = (u >= items) ? 1 : 0;
                    ItemSums Sm;
                    if (pair) slab_measure_item<RPW, true>(S, sm, L, Lh, z0, rank, cs, p, u - p * items, Sm);
                    else      slab_measure_item<RPW, false>(S, sm, L, Lh, z0, rank, cs, p, u - p * items, Sm);
                    accU.add(Sm.u); accM.add(Sm.m);
                    if (pair) accX.add(Sm.x);
                }
                unsigned int mU, mM, mX = 0u;
                if (few) {                                            // block-uniform
                    typedef const uint32_t (&P5)[5];
                    mU = warp_lane_count<5>(reinterpret_cast<P5>(accU.c)); mM = warp_lane_count<5>(reinterpret_cast<P5>(accM.c));
                    if (pair) mX = warp_lane_count<5>(reinterpret_cast<P5>(accX.c));
                } else {
                    mU = warp_lane_count<kMeasurePlanes>(accU.c); mM = warp_lane_count<kMeasurePlanes>(accM.c);
                    if (pair) mX = warp_lane_count<kMeasurePlanes>(accX.c);
                }
                if (tid < 96) s_tot[tid] = 0u;                        // nobody reads the previous row's totals any more:
                __syncthreads();                                      // at least one sweep (two cluster barriers) lies between
                const int lane = tid & 31;
                if (mU) atomicAdd(&s_tot[lane], mU);
                if (mM) atomicAdd(&s_tot[32 + lane], mM);
                if (mX) atomicAdd(&s_tot[64 + lane], mX);
                cluster_sync_all();                                   // every CTA's totals are in place and visible
                if (rank == 0) {
                    long long* row = (r < A.rows_cap) ? A.rows + r * A.row_len : A.scratch_row;
                    small_finalize_lattice(A, w, row, s_tot, cs, run_min);
                }
                ++r;
            }
        }
    }
    // ---- the launch's minimum energies (same thread -> system map as small_finalize_lattice)
    if (rank == 0 && tid < 32 && A.min_E && run_min != 0x7FFFFFFFFFFFFFFFll) {
        const int sg = w / A.a.n_rg, rg = w - sg * A.a.n_rg;
        const int r_local = tid / A.spw, sl = tid - r_local * A.spw;
        const int sample = sg * A.spw + sl, rep = rg * A.rpw + r_local;
        if (sample < A.n_samples && rep < A.n_replicas) {
            const int t = sample * A.n_replicas + rep;
            if (run_min < A.min_E[t]) A.min_E[t] = run_min;
        }
    }
    // ---- shared -> global: spins and daemon planes
    for (int p = 0; p < 2; ++p) {
        const long long go = ((long long)w * 2 + p) * half + (long long)z0 * PW;
        uint4* gs = reinterpret_cast<uint4*>(A.a.spin + go);
        uint4* g0 = reinterpret_cast<uint4*>(A.a.m0 + go);
        uint4* g1 = reinterpret_cast<uint4*>(A.a.m1 + go);
        const uint4* ss = reinterpret_cast<const uint4*>(smem + S.spin(p));
        const uint4* s0 = reinterpret_cast<const uint4*>(smem + S.m0(p));
        const uint4* s1 = reinterpret_cast<const uint4*>(smem + S.m1(p));
        for (int i = tid; i < slab_words / 4; i += nthr) { gs[i] = ss[i]; g0[i] = s0[i]; g1[i] = s1[i]; }
    }
    cluster_sync_all();          // no CTA leaves while a neighbour may still read its shared memory
}

}  // namespace micsa
