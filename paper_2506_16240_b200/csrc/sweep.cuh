// sweep.cuh -- the microcanonical half-sweep.
//
// Elementary move, PAPER.md:119-124 (Eq. 8) and :150 (Eq. 10), for every site
// of one parity and all 32 systems of a word at once, Boolean operations only
// (PAPER.md:152).  With U = number of unsatisfied bonds among the six of the
// site, dH = 12 - 4U and n = 4m, so n - dH = 4(m + U - 3): the flip is legal
// iff 3 <= m + U <= 6 and then m <- m + U - 3.
#pragma once
#include "layout.cuh"
#include "measure.cuh"

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
    int w0;                 // first word lattice of this launch (pipelined kernel: blockIdx.z + w0)
    uint32_t inv_nxv;       // fastdiv_magic(Lh / 4) (pipelined kernels)
    uint32_t inv_pp;        // fastdiv_magic((L / YC) * (Lh / 4)): items per plane of the launched pipelined kernel
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


// ---------------------------------------------------------------------------
// Row-marching half-sweep for L % 8 == 0 (all BASELINE configs).
//
// One thread owns 4 consecutive words (16 B) of a row and marches over YC
// consecutive rows y0..y0+YC-1 of plane z (grid.y) of word lattice w (grid.z):
//  * the three opposite-parity rows y-1, y, y+1 slide through registers, so each
//    step loads one new row instead of three;
//  * all array bases are block-uniform and the per-thread offsets are 32-bit byte
//    offsets advanced by a constant, which removes the 64-bit index arithmetic
//    that dominated the first version (ncu: 104 instructions per site word);
//  * y0 is even, so the x-shift flag c = (y+z+p)&1 equals (iy&1) ^ f with
//    f = (z+p)&1 uniform over the block: the block branches once on f and c is
//    a compile-time constant in the unrolled body -- no per-word selects.
// Lanes run along (row chunk, x): a warp reads whole 128-byte lines.
// ---------------------------------------------------------------------------
template <typename T>
__device__ __forceinline__ T ld_off(const void* base, uint32_t byte_off) {
    return *reinterpret_cast<const T*>(static_cast<const char*>(base) + byte_off);
}
template <typename T>
__device__ __forceinline__ void st_off(void* base, uint32_t byte_off, T v) {
    *reinterpret_cast<T*>(static_cast<char*>(base) + byte_off) = v;
}

template <int RPW> struct Bond4;                      // 4 consecutive bond words
template <> struct Bond4<2> {
    typedef uint2 raw; typedef uint16_t elem;
    static __device__ __forceinline__ void expand(const raw& r, uint32_t (&o)[4]) {
        o[0] = __byte_perm(r.x, 0u, 0x1010); o[1] = __byte_perm(r.x, 0u, 0x3232);
        o[2] = __byte_perm(r.y, 0u, 0x1010); o[3] = __byte_perm(r.y, 0u, 0x3232);
    }
    static __device__ __forceinline__ uint32_t expand1(elem e) { return __byte_perm((uint32_t)e, 0u, 0x1010); }
};
template <> struct Bond4<1> {
    typedef uint4 raw; typedef uint32_t elem;
    static __device__ __forceinline__ void expand(const raw& r, uint32_t (&o)[4]) {
        o[0] = r.x; o[1] = r.y; o[2] = r.z; o[3] = r.w;
    }
    static __device__ __forceinline__ uint32_t expand1(elem e) { return e; }
};

struct RowPtrs {            // block-uniform bases of plane z (and z+-1) of lattice w
    uint32_t* sp; uint32_t* m0; uint32_t* m1;          // own parity, plane z
    const uint32_t* sq; const uint32_t* sq_zp; const uint32_t* sq_zm;   // opposite parity
    const void* jx; const void* jy; const void* jz;    // own bonds, plane z
    const void* jxq; const void* jyq; const void* jzq_zm;   // neighbours' bonds
};

template <int RPW, int YC, int F>
__device__ __forceinline__ void march_rows(const RowPtrs& P, int L, int Lh, int y0, int xh0)
{
    typedef Bond4<RPW> B4;
    constexpr uint32_t JS = sizeof(typename B4::elem);          // bytes per bond word
    const uint32_t rowB = (uint32_t)Lh * 4u;                    // bytes per spin row
    const uint32_t x4 = (uint32_t)xh0 * 4u;
    const int ym0 = (y0 == 0) ? L - 1 : y0 - 1;
    // byte offsets inside a plane (spin-word units * 4)
    uint32_t o = (uint32_t)y0 * rowB + x4;
    uint32_t o_prev = (uint32_t)ym0 * rowB + x4;
    const uint32_t xe_up = ((xh0 + 4 == Lh) ? 0u : (uint32_t)(xh0 + 4)) * 4u;     // xh+1 of the last word
    const uint32_t xe_dn = ((xh0 == 0) ? (uint32_t)(Lh - 1) : (uint32_t)(xh0 - 1)) * 4u;

    uint4 Aprev = ld_off<uint4>(P.sq, o_prev);
    uint4 Acur  = ld_off<uint4>(P.sq, o);
#pragma unroll
    for (int iy = 0; iy < YC; ++iy) {
        const int c = (iy & 1) ^ F;                    // compile-time after unrolling
        const int y = y0 + iy;
        const uint32_t o_next = (y + 1 == L) ? x4 : o + rowB;
        const uint32_t rowstart = o - x4;
        const uint4 Anext = ld_off<uint4>(P.sq, o_next);
        uint4 s  = ld_off<uint4>(P.sp, o);
        uint4 d0 = ld_off<uint4>(P.m0, o);
        uint4 d1 = ld_off<uint4>(P.m1, o);
        const uint4 nzp = ld_off<uint4>(P.sq_zp, o);
        const uint4 nzm = ld_off<uint4>(P.sq_zm, o);
        const uint32_t oj = o / 4u * JS, ojm = o_prev / 4u * JS;
        uint32_t jxo[4], jyo[4], jzo[4], jxm[4], jym[4], jzm[4];
        B4::expand(ld_off<typename B4::raw>(P.jx, oj), jxo);
        B4::expand(ld_off<typename B4::raw>(P.jy, oj), jyo);
        B4::expand(ld_off<typename B4::raw>(P.jz, oj), jzo);
        B4::expand(ld_off<typename B4::raw>(P.jyq, ojm), jym);
        B4::expand(ld_off<typename B4::raw>(P.jzq_zm, oj), jzm);
        uint32_t Bx[4];
        B4::expand(ld_off<typename B4::raw>(P.jxq, oj), Bx);
        const uint32_t a[4] = { Acur.x, Acur.y, Acur.z, Acur.w };
        uint32_t nxp[4], nxm[4];
        if (c) {        // x = 2xh+1: -x neighbour at xh (bond owned by it), +x neighbour at xh+1
            const uint32_t e = ld_off<uint32_t>(P.sq, rowstart + xe_up);
            nxp[0] = a[1]; nxp[1] = a[2]; nxp[2] = a[3]; nxp[3] = e;
            nxm[0] = a[0]; nxm[1] = a[1]; nxm[2] = a[2]; nxm[3] = a[3];
            jxm[0] = Bx[0]; jxm[1] = Bx[1]; jxm[2] = Bx[2]; jxm[3] = Bx[3];
        } else {        // x = 2xh: +x neighbour at xh, -x neighbour at xh-1 (bond owned by it)
            const uint32_t e = ld_off<uint32_t>(P.sq, rowstart + xe_dn);
            const uint32_t eJ = B4::expand1(ld_off<typename B4::elem>(P.jxq, (rowstart + xe_dn) / 4u * JS));
            nxp[0] = a[0]; nxp[1] = a[1]; nxp[2] = a[2]; nxp[3] = a[3];
            nxm[0] = e; nxm[1] = a[0]; nxm[2] = a[1]; nxm[3] = a[2];
            jxm[0] = eJ; jxm[1] = Bx[0]; jxm[2] = Bx[1]; jxm[3] = Bx[2];
        }
        uint32_t sv[4] = { s.x, s.y, s.z, s.w };
        uint32_t v0[4] = { d0.x, d0.y, d0.z, d0.w };
        uint32_t v1[4] = { d1.x, d1.y, d1.z, d1.w };
        const uint32_t yp[4] = { Anext.x, Anext.y, Anext.z, Anext.w };
        const uint32_t ym[4] = { Aprev.x, Aprev.y, Aprev.z, Aprev.w };
        const uint32_t zp[4] = { nzp.x, nzp.y, nzp.z, nzp.w };
        const uint32_t zm[4] = { nzm.x, nzm.y, nzm.z, nzm.w };
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t g = sv[k];
            creutz_word(g ^ nxp[k] ^ jxo[k], g ^ nxm[k] ^ jxm[k],
                        g ^ yp[k] ^ jyo[k],  g ^ ym[k] ^ jym[k],
                        g ^ zp[k] ^ jzo[k],  g ^ zm[k] ^ jzm[k],
                        sv[k], v0[k], v1[k]);
        }
        st_off<uint4>(P.sp, o, make_uint4(sv[0], sv[1], sv[2], sv[3]));
        st_off<uint4>(P.m0, o, make_uint4(v0[0], v0[1], v0[2], v0[3]));
        st_off<uint4>(P.m1, o, make_uint4(v1[0], v1[1], v1[2], v1[3]));
        Aprev = Acur; Acur = Anext;
        o_prev = o; o = o_next;
    }
}

// grid = (ceil((L/YC)*(Lh/4) / block), L, n_words)
template <int RPW, int YC>
__global__ void __launch_bounds__(128)
half_sweep_rows_kernel(SweepArgs a, int p)
{
    typedef typename Bond4<RPW>::elem JT;
    const int L = a.L, Lh = a.Lh;
    const int nxv = Lh >> 2;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (L / YC) * nxv) return;
    const int chunk = t / nxv, xv = t - chunk * nxv;
    const int z = blockIdx.y, w = blockIdx.z, q = 1 - p;
    const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    const long long half = a.half;
    const long long plane = (long long)L * Lh;
    const int sg = w / a.n_rg;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;

    RowPtrs P;
    P.sp = a.spin + ((long long)w * 2 + p) * half + z * plane;
    P.m0 = a.m0 + ((long long)w * 2 + p) * half + z * plane;
    P.m1 = a.m1 + ((long long)w * 2 + p) * half + z * plane;
    const uint32_t* sqb = a.spin + ((long long)w * 2 + q) * half;
    P.sq = sqb + z * plane; P.sq_zp = sqb + zp * plane; P.sq_zm = sqb + zm * plane;
    P.jx = Jb + (0 * 2 + p) * half + z * plane;
    P.jy = Jb + (1 * 2 + p) * half + z * plane;
    P.jz = Jb + (2 * 2 + p) * half + z * plane;
    P.jxq = Jb + (0 * 2 + q) * half + z * plane;
    P.jyq = Jb + (1 * 2 + q) * half + z * plane;
    P.jzq_zm = Jb + (2 * 2 + q) * half + zm * plane;

    if ((z + p) & 1) march_rows<RPW, YC, 1>(P, L, Lh, chunk * YC, xv * 4);
    else             march_rows<RPW, YC, 0>(P, L, Lh, chunk * YC, xv * 4);
}


// ---------------------------------------------------------------------------
// Pipelined row-marching half-sweep (L % 8 == 0): the same thread -> data map
// as half_sweep_rows_kernel, with
//  * the loads of row iy+1 issued BEFORE the update of row iy (explicit
//    software pipeline; stores and loads go through different pointers, which
//    the compiler cannot prove apart, so it never hoists them by itself).  All
//    warps of the single resident wave start together; without the pipeline
//    they alternate between "everybody waits for loads" and "everybody
//    computes" and neither the memory system nor the integer pipe is kept busy;
//  * a shorter Boolean update (creutz_word20): the daemon's low bit and the
//    constant +1 join the population count as the 7th and 8th input, so that
//    V = m + U + 1 has "accept" in bit 2 alone and the new level in bits 1:0.
// ---------------------------------------------------------------------------

// V = m + U + 1 in [1, 10]; accept iff 3 <= m + U <= 6 iff 4 <= V <= 7 iff bit 2
// of V is set and bit 3 is not -- and bit 3 set implies bit 2 clear here, so
// accept = V2; new level m + U - 3 = V - 4 = bits 1:0 of V.
// Every line below is one three-input logic operation, written as the LOP3 it is meant to be (layout.cuh, lop3).
__device__ __forceinline__ void creutz_word20(uint32_t u1, uint32_t u2, uint32_t u3,
                                              uint32_t u4, uint32_t u5, uint32_t u6,
                                              uint32_t& sigma, uint32_t& m0, uint32_t& m1) {
    const uint32_t sa = lop3<kXor3>(u1, u2, u3), ca = lop3<kMaj3>(u1, u2, u3);
    const uint32_t sb = lop3<kXor3>(u4, u5, u6), cb = lop3<kMaj3>(u4, u5, u6);
    const uint32_t t0 = lop3<kXor3>(sa, sb, m0), cd = lop3<kMaj3>(sa, sb, m0);   // weight 1 without the +1
    // + 1: V0 = ~t0 and a carry t0 into weight 2
    const uint32_t s1 = lop3<kXor3>(ca, cb, cd), c1a = lop3<kMaj3>(ca, cb, cd);
    const uint32_t V1 = lop3<kXor3>(s1, t0, m1), c1b = lop3<kMaj3>(s1, t0, m1);
    const uint32_t acc = c1a ^ c1b;                                              // V2 (V3 = c1a & c1b excludes it)
    sigma = lop3<kXor3>(sigma, c1a, c1b);
    m0 = lop3<kSelNot>(acc, t0, m0);
    m1 = lop3<kSel>(acc, V1, m1);
}

struct PipeBase {           // block-uniform bases of lattice w: plane 0 of each parity array
    uint32_t* sp; uint32_t* m0; uint32_t* m1;          // own parity
    const uint32_t* sq;                                // opposite parity
    uint32_t* m0q; uint32_t* m1q;                      // opposite parity's daemon planes (walkers only)
    const void* jx; const void* jy; const void* jz;    // own bonds
    const void* jxq; const void* jyq; const void* jzq; // the -d neighbours' bonds (opposite parity arrays)
};

template <int RPW>
struct RowRegs {                 // everything one row step reads
    typedef Bond4<RPW> B4;
    uint4 An, s, d0, d1, zp, zm;
    typename B4::raw jx, jy, jz, jyq, jzq, jxq;
    uint32_t e;
    typename B4::elem eJ;
    uint4 w0, w1;                // walkers: the exchange partners' planes, same quad ...
    uint32_t we0, we1;           // ... and the word just outside it (X), or
    uint32_t po;                 // the partner quad's byte offset (Y, Z)
};

// o, o_prev, o_next: byte offsets (inside a parity array of spin words) of
// the thread's 4 words in rows y, y-1, y+1 of plane z; dzp, dzm: byte distance
// to the same row of planes z+1, z-1 (mod 2^32, periodic); rowstart = o - x4.
// Where the x-neighbour words just outside a thread's 4 words come from: the
// lane that owns the adjacent quad of the same row holds them in registers, so
// they are fetched with a shuffle; only lanes whose neighbour sits in another
// warp (or is not running) load them.  A lone 4-byte load costs a whole 32-byte
// sector of L2 bandwidth, which is what bounds this kernel.
struct XNb {
    unsigned mask;          // lanes taking part (all of them run the same row step)
    int lane_up, lane_dn;   // lanes owning quads xv+1 and xv-1 (periodic) of the same row
    bool in_up, in_dn;      // ... and whether they can be reached by a shuffle
    int walk_z;             // walkers along Y (0) or Z (1) when the launch's DIR is +-2
};

template <int RPW, int C, int DIR = 0>
__device__ __forceinline__ void load_row(RowRegs<RPW>& r, const PipeBase& P, uint32_t o, uint32_t o_prev,
                                         uint32_t o_next, uint32_t x4, uint32_t xe_up, uint32_t xe_dn,
                                         uint32_t dzp, uint32_t dzm, const XNb& nb)
{
    typedef Bond4<RPW> B4;
    constexpr uint32_t JS = sizeof(typename B4::elem);
    const uint32_t rowstart = o - x4;
    const uint32_t oj = o / 4u * JS, ojm = o_prev / 4u * JS;
    r.An = ld_off<uint4>(P.sq, o_next);
    r.s  = ld_off<uint4>(P.sp, o);
    r.d0 = ld_off<uint4>(P.m0, o);
    r.d1 = ld_off<uint4>(P.m1, o);
    r.zp = ld_off<uint4>(P.sq, o + dzp);
    r.zm = ld_off<uint4>(P.sq, o + dzm);
    r.jx = ld_off<typename B4::raw>(P.jx, oj);
    r.jy = ld_off<typename B4::raw>(P.jy, oj);
    r.jz = ld_off<typename B4::raw>(P.jz, oj);
    r.jyq = ld_off<typename B4::raw>(P.jyq, ojm);
    r.jzq = ld_off<typename B4::raw>(P.jzq, (o + dzm) / 4u * JS);
    r.jxq = ld_off<typename B4::raw>(P.jxq, oj);
    if (DIR == 2 || DIR == -2) { // walkers along Y or Z: the partner is the same quad of the next / previous row or plane
        r.po = nb.walk_z ? o + (DIR > 0 ? dzp : dzm) : (DIR > 0 ? o_next : o_prev);
        r.w0 = ld_off<uint4>(P.m0q, r.po);
        r.w1 = ld_off<uint4>(P.m1q, r.po);
    } else if (DIR != 0) {       // walkers along X: the planes of the sites these sites exchange with (see exchange_walkers)
        r.w0 = ld_off<uint4>(P.m0q, o);
        r.w1 = ld_off<uint4>(P.m1q, o);
        if (DIR > 0 && C)  { r.we0 = ld_off<uint32_t>(P.m0q, rowstart + xe_up); r.we1 = ld_off<uint32_t>(P.m1q, rowstart + xe_up); }
        if (DIR < 0 && !C) { r.we0 = ld_off<uint32_t>(P.m0q, rowstart + xe_dn); r.we1 = ld_off<uint32_t>(P.m1q, rowstart + xe_dn); }
    }
    r.e = 0; r.eJ = 0;
    if (C) {
        if (!nb.in_up) r.e = ld_off<uint32_t>(P.sq, rowstart + xe_up);
    } else if (!nb.in_dn) {
        r.e = ld_off<uint32_t>(P.sq, rowstart + xe_dn);
        r.eJ = ld_off<typename B4::elem>(P.jxq, (rowstart + xe_dn) / 4u * JS);
    }
}

template <int RPW> __device__ __forceinline__ uint32_t last_bond_word(const typename Bond4<RPW>::raw& j);
template <> __device__ __forceinline__ uint32_t last_bond_word<2>(const uint2& j) { return j.y >> 16; }
template <> __device__ __forceinline__ uint32_t last_bond_word<1>(const uint4& j) { return j.w; }

// ---- measurement fused into the last sweep of a group ----
// After a sweep every bond has exactly one odd end, and the odd half-sweep has
// all six bonds of each odd site in registers: the unsatisfied bonds after its
// update, summed over the odd sites, are U_tot of Eq. (1).  Daemon levels and
// replica differences of a site are final once its own half-sweep of the last
// sweep has passed.  So the even launch of the last sweep adds the levels and
// differences of the even sites (MEAS = 1), the odd launch those of the odd
// sites plus all unsatisfied bonds (MEAS = 2) and its last CTA writes the row;
// the state is not read again.
template <int YC> struct MeasAcc {            // per-thread vertical counters over YC rows x 4 words
    static constexpr int PU = (YC <= 4) ? 7 : 8;     // <= 24 * YC unsatisfied bonds per lane
    static constexpr int PM = (YC <= 4) ? 6 : 7;     // <= 12 * YC level units
    static constexpr int PX = (YC <= 4) ? 5 : 6;     // <=  4 * YC differing sites
    VCount<PU> u; VCount<PM> m; VCount<PX> x;
    __device__ __forceinline__ void clear() { u.clear(); m.clear(); x.clear(); }
};

// lane-wise sum of 6 flags for each of 4 words -> 5 planes (<= 24)
__device__ __forceinline__ void count6x4(const uint32_t (&f)[6][4], uint32_t (&o)[5]) {
    uint32_t sa[4], ca[4], sb[4], cb[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        full_add(f[0][k], f[1][k], f[2][k], sa[k], ca[k]);
        full_add(f[3][k], f[4][k], f[5][k], sb[k], cb[k]);
    }
    uint32_t p0, p1, p2, q0, q1, q2, q3;                     // weight 1: sa, sb
    full_add(sa[0], sa[1], sa[2], p0, q0);
    full_add(sa[3], sb[0], sb[1], p1, q1);
    full_add(sb[2], sb[3], p0, p2, q2);
    half_add(p1, p2, o[0], q3);
    uint32_t r0, r1, r2, r3, r4, t0, t1, t2, t3, t4, t5;     // weight 2: ca, cb, q
    full_add(ca[0], ca[1], ca[2], r0, t0);
    full_add(ca[3], cb[0], cb[1], r1, t1);
    full_add(cb[2], cb[3], q0, r2, t2);
    full_add(q1, q2, q3, r3, t3);
    full_add(r0, r1, r2, r4, t4);
    half_add(r4, r3, o[1], t5);
    uint32_t v0, v1, x0, x1, x2;                             // weight 4: t
    full_add(t0, t1, t2, v0, x0);
    full_add(t3, t4, t5, v1, x1);
    half_add(v0, v1, o[2], x2);
    full_add(x0, x1, x2, o[3], o[4]);                        // weight 8, 16
}

// Walkers: the wandering half-cycle that closes a timestep
// exchanges every walker of the source parity with its +X neighbour's.  It is
// done by the ODD half-sweep of that timestep, the last one to touch daemon
// values: an odd site x sends its just-updated level to its partner -- the even
// site x-1 when the even sites are the sources (t even, DIR = -1), x+1 when the
// odd sites are (t odd, DIR = +1) -- and takes the partner's level (final since
// the even half-sweep) in return.  In the x-compressed arrays the partner of
// word xh is word xh of the other parity's planes, or xh+1 (DIR > 0, rows with
// C = 1) / xh-1 (DIR < 0, rows with C = 0): the same edge word as the spin
// neighbour's.  Along Y and Z (DIR = +-2, axis in XNb::walk_z) the partner is the
// same quad of the next / previous row or plane.  Every word is written by
// exactly one thread, and a row's partner words are loaded one row step ahead
// of the exchange that overwrites a DIFFERENT row's (or plane's) words.
template <int RPW, int C, int DIR>
__device__ __forceinline__ void exchange_walkers(const RowRegs<RPW>& r, const PipeBase& P, uint32_t o,
                                                 uint32_t rowstart, uint32_t xe_up, uint32_t xe_dn,
                                                 uint32_t (&v0)[4], uint32_t (&v1)[4], const XNb& nb)
{
    const uint32_t a0[4] = { r.w0.x, r.w0.y, r.w0.z, r.w0.w }, a1[4] = { r.w1.x, r.w1.y, r.w1.z, r.w1.w };
    if (DIR == 2 || DIR == -2) {                          // Y / Z: the same quad of the neighbouring row / plane
        st_off<uint4>(P.m0q, r.po, make_uint4(v0[0], v0[1], v0[2], v0[3]));
        st_off<uint4>(P.m1q, r.po, make_uint4(v1[0], v1[1], v1[2], v1[3]));
#pragma unroll
        for (int k = 0; k < 4; ++k) { v0[k] = a0[k]; v1[k] = a1[k]; }
    } else if ((DIR > 0 && !C) || (DIR < 0 && C)) {       // X, partner words = the same quad
        st_off<uint4>(P.m0q, o, make_uint4(v0[0], v0[1], v0[2], v0[3]));
        st_off<uint4>(P.m1q, o, make_uint4(v1[0], v1[1], v1[2], v1[3]));
#pragma unroll
        for (int k = 0; k < 4; ++k) { v0[k] = a0[k]; v1[k] = a1[k]; }
    } else if (DIR > 0) {                                 // partner words xh0+1 .. xh0+4 (periodic)
        // word xh0 of the partner planes belongs to the left neighbour's exchange: take its last new level by
        // shuffle and write one aligned quad; lanes whose neighbour is in another warp fall back to 32-bit stores
        const uint32_t l0 = __shfl_sync(nb.mask, v0[3], nb.lane_dn), l1 = __shfl_sync(nb.mask, v1[3], nb.lane_dn);
        if (nb.in_dn) {
            st_off<uint4>(P.m0q, o, make_uint4(l0, v0[0], v0[1], v0[2]));
            st_off<uint4>(P.m1q, o, make_uint4(l1, v1[0], v1[1], v1[2]));
        } else {
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                st_off<uint32_t>(P.m0q, o + 4u * (k + 1), v0[k]);
                st_off<uint32_t>(P.m1q, o + 4u * (k + 1), v1[k]);
            }
        }
        if (!nb.in_up) {                                  // nobody will fetch my last level: store it myself
            st_off<uint32_t>(P.m0q, rowstart + xe_up, v0[3]);
            st_off<uint32_t>(P.m1q, rowstart + xe_up, v1[3]);
        }
        v0[0] = a0[1]; v0[1] = a0[2]; v0[2] = a0[3]; v0[3] = r.we0;
        v1[0] = a1[1]; v1[1] = a1[2]; v1[2] = a1[3]; v1[3] = r.we1;
    } else {                                              // partner words xh0-1 .. xh0+2 (periodic)
        const uint32_t r0 = __shfl_sync(nb.mask, v0[0], nb.lane_up), r1 = __shfl_sync(nb.mask, v1[0], nb.lane_up);
        if (nb.in_up) {
            st_off<uint4>(P.m0q, o, make_uint4(v0[1], v0[2], v0[3], r0));
            st_off<uint4>(P.m1q, o, make_uint4(v1[1], v1[2], v1[3], r1));
        } else {
#pragma unroll
            for (int k = 1; k < 4; ++k) {
                st_off<uint32_t>(P.m0q, o + 4u * (k - 1), v0[k]);
                st_off<uint32_t>(P.m1q, o + 4u * (k - 1), v1[k]);
            }
        }
        if (!nb.in_dn) {
            st_off<uint32_t>(P.m0q, rowstart + xe_dn, v0[0]);
            st_off<uint32_t>(P.m1q, rowstart + xe_dn, v1[0]);
        }
        v0[3] = a0[2]; v0[2] = a0[1]; v0[1] = a0[0]; v0[0] = r.we0;
        v1[3] = a1[2]; v1[2] = a1[1]; v1[1] = a1[0]; v1[0] = r.we1;
    }
}

template <int RPW, int C, int MEAS, int YC, int DIR = 0>
__device__ __forceinline__ void update_row(const RowRegs<RPW>& r, const uint4& Aprev, const uint4& Acur,
                                           const PipeBase& P, uint32_t o, const XNb& nb,
                                           MeasAcc<YC>* acc, bool pair,
                                           uint32_t x4 = 0, uint32_t xe_up = 0, uint32_t xe_dn = 0)
{
    typedef Bond4<RPW> B4;
    uint32_t jxo[4], jyo[4], jzo[4], jxm[4], jym[4], jzm[4], Bx[4];
    B4::expand(r.jx, jxo); B4::expand(r.jy, jyo); B4::expand(r.jz, jzo);
    B4::expand(r.jyq, jym); B4::expand(r.jzq, jzm); B4::expand(r.jxq, Bx);
    const uint32_t a[4] = { Acur.x, Acur.y, Acur.z, Acur.w };
    uint32_t nxp[4], nxm[4];
    if (C) {        // x = 2xh+1: -x neighbour at xh (bond owned by it), +x neighbour at xh+1
        uint32_t e = __shfl_sync(nb.mask, Acur.x, nb.lane_up);
        if (!nb.in_up) e = r.e;
        nxp[0] = a[1]; nxp[1] = a[2]; nxp[2] = a[3]; nxp[3] = e;
        nxm[0] = a[0]; nxm[1] = a[1]; nxm[2] = a[2]; nxm[3] = a[3];
        jxm[0] = Bx[0]; jxm[1] = Bx[1]; jxm[2] = Bx[2]; jxm[3] = Bx[3];
    } else {        // x = 2xh: +x neighbour at xh, -x neighbour at xh-1 (bond owned by it)
        uint32_t e = __shfl_sync(nb.mask, Acur.w, nb.lane_dn);
        uint32_t eJ = __shfl_sync(nb.mask, last_bond_word<RPW>(r.jxq), nb.lane_dn);
        if (!nb.in_dn) { e = r.e; eJ = (uint32_t)r.eJ; }
        nxp[0] = a[0]; nxp[1] = a[1]; nxp[2] = a[2]; nxp[3] = a[3];
        nxm[0] = e; nxm[1] = a[0]; nxm[2] = a[1]; nxm[3] = a[2];
        jxm[0] = B4::expand1((typename B4::elem)eJ); jxm[1] = Bx[0]; jxm[2] = Bx[1]; jxm[3] = Bx[2];
    }
    uint32_t sv[4] = { r.s.x, r.s.y, r.s.z, r.s.w };
    uint32_t v0[4] = { r.d0.x, r.d0.y, r.d0.z, r.d0.w };
    uint32_t v1[4] = { r.d1.x, r.d1.y, r.d1.z, r.d1.w };
    const uint32_t yp[4] = { r.An.x, r.An.y, r.An.z, r.An.w };
    const uint32_t ym[4] = { Aprev.x, Aprev.y, Aprev.z, Aprev.w };
    const uint32_t zp[4] = { r.zp.x, r.zp.y, r.zp.z, r.zp.w };
    const uint32_t zm[4] = { r.zm.x, r.zm.y, r.zm.z, r.zm.w };
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const uint32_t g = sv[k];
        creutz_word20(bond_flag(g, nxp[k], jxo[k]), bond_flag(g, nxm[k], jxm[k]),
                      bond_flag(g, yp[k], jyo[k]),  bond_flag(g, ym[k], jym[k]),
                      bond_flag(g, zp[k], jzo[k]),  bond_flag(g, zm[k], jzm[k]),
                      sv[k], v0[k], v1[k]);
    }
    st_off<uint4>(P.sp, o, make_uint4(sv[0], sv[1], sv[2], sv[3]));
    if (DIR == 0) {
        st_off<uint4>(P.m0, o, make_uint4(v0[0], v0[1], v0[2], v0[3]));
        st_off<uint4>(P.m1, o, make_uint4(v1[0], v1[1], v1[2], v1[3]));
    }
    if (MEAS) {
        uint32_t pm[4];
        csa_4x1_4x2(v0, v1, pm);                              // levels after the update
        acc->m.add(pm);
        if (RPW == 2 && pair) {                               // lanes where the two replicas of a sample differ
            uint32_t xs[4], a2, b2, b3, px[3];
#pragma unroll
            for (int k = 0; k < 4; ++k) xs[k] = (sv[k] ^ (sv[k] >> 16)) & 0xFFFFu;
            full_add(xs[0], xs[1], xs[2], a2, b2);
            half_add(a2, xs[3], px[0], b3);
            px[1] = b2 ^ b3; px[2] = b2 & b3;
            acc->x.add(px);
        }
        if (MEAS == 2) {                                      // bonds of these sites that are unsatisfied NOW
            uint32_t f[6][4], pu[5];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
                const uint32_t g = sv[k];
                f[0][k] = g ^ nxp[k] ^ jxo[k]; f[1][k] = g ^ nxm[k] ^ jxm[k];
                f[2][k] = g ^ yp[k] ^ jyo[k];  f[3][k] = g ^ ym[k] ^ jym[k];
                f[4][k] = g ^ zp[k] ^ jzo[k];  f[5][k] = g ^ zm[k] ^ jzm[k];
            }
            count6x4(f, pu);
            acc->u.add(pu);
        }
    }
    if (DIR != 0) {              // walkers: hand the new levels to the partner sites, keep theirs
        exchange_walkers<RPW, C, DIR>(r, P, o, o - x4, xe_up, xe_dn, v0, v1, nb);
        st_off<uint4>(P.m0, o, make_uint4(v0[0], v0[1], v0[2], v0[3]));
        st_off<uint4>(P.m1, o, make_uint4(v1[0], v1[1], v1[2], v1[3]));
    }
}

// rows y0 .. y0+YC-1 of plane z (y0 % YC == 0, YC even, L % YC == 0), words xh0 .. xh0+3
template <int RPW, int YC, int F, int MEAS = 0, int DIR = 0>
__device__ __forceinline__ void march_rows_pipe(const PipeBase& P, int L, int Lh, int z, int y0, int xh0,
                                                const XNb& nb, MeasAcc<YC>* acc = nullptr, bool pair = false)
{
    const uint32_t rowB = (uint32_t)Lh * 4u;
    const uint32_t planeB = (uint32_t)L * rowB;
    const uint32_t x4 = (uint32_t)xh0 * 4u;
    const uint32_t zB = (uint32_t)z * planeB;
    const uint32_t dzp = (z + 1 == L) ? 0u - zB : planeB;
    const uint32_t dzm = (z == 0) ? (uint32_t)(L - 1) * planeB : 0u - planeB;
    const int ym0 = (y0 == 0) ? L - 1 : y0 - 1;
    const uint32_t xe_up = ((xh0 + 4 == Lh) ? 0u : (uint32_t)(xh0 + 4)) * 4u;
    const uint32_t xe_dn = ((xh0 == 0) ? (uint32_t)(Lh - 1) : (uint32_t)(xh0 - 1)) * 4u;
    const uint32_t row0 = zB + x4;                       // row 0 of the plane, this thread's words
    uint32_t o = row0 + (uint32_t)y0 * rowB;
    uint32_t o_prev = row0 + (uint32_t)ym0 * rowB;

    uint4 Aprev = ld_off<uint4>(P.sq, o_prev);
    uint4 Acur  = ld_off<uint4>(P.sq, o);
    RowRegs<RPW> cur, nxt;
    {
        const uint32_t o_next = (y0 + 1 == L) ? row0 : o + rowB;
        load_row<RPW, F, DIR>(cur, P, o, o_prev, o_next, x4, xe_up, xe_dn, dzp, dzm, nb);
    }
#pragma unroll
    for (int iy = 0; iy < YC; ++iy) {
        const int y = y0 + iy;
        const uint32_t o_next = (y + 1 == L) ? row0 : o + rowB;
        if (iy + 1 < YC) {                          // y + 1 < L inside a chunk
            const uint32_t o_next2 = (y + 2 == L) ? row0 : o_next + rowB;
            if ((iy & 1) ^ F) load_row<RPW, 0, DIR>(nxt, P, o_next, o, o_next2, x4, xe_up, xe_dn, dzp, dzm, nb);
            else              load_row<RPW, 1, DIR>(nxt, P, o_next, o, o_next2, x4, xe_up, xe_dn, dzp, dzm, nb);
        }
        if ((iy & 1) ^ F) update_row<RPW, 1, MEAS, YC, DIR>(cur, Aprev, Acur, P, o, nb, acc, pair, x4, xe_up, xe_dn);
        else              update_row<RPW, 0, MEAS, YC, DIR>(cur, Aprev, Acur, P, o, nb, acc, pair, x4, xe_up, xe_dn);
        Aprev = Acur; Acur = cur.An;
        if (iy + 1 < YC) cur = nxt;
        o_prev = o; o = o_next;
    }
}

// x-neighbour lanes of the thread whose item index inside its warp-aligned
// index space is `idx` (consecutive idx = consecutive quads of a row, rows of
// nxv quads one after the other); mask = lanes running this step.
__device__ __forceinline__ XNb x_neighbours(int idx, int xv, int nxv, unsigned mask, bool use_shuffle)
{
    XNb nb;
    nb.mask = mask;
    const int up = (xv == nxv - 1) ? idx - (nxv - 1) : idx + 1;
    const int dn = (xv == 0) ? idx + (nxv - 1) : idx - 1;
    nb.lane_up = up & 31; nb.lane_dn = dn & 31;
    nb.in_up = use_shuffle && (up >> 5) == (idx >> 5) && ((mask >> nb.lane_up) & 1u);
    nb.in_dn = use_shuffle && (dn >> 5) == (idx >> 5) && ((mask >> nb.lane_dn) & 1u);
    nb.walk_z = 0;
    return nb;
}

template <int RPW>
__device__ __forceinline__ PipeBase pipe_base(const SweepArgs& a, int w, int p)
{
    typedef typename Bond4<RPW>::elem JT;
    const int q = 1 - p;
    const long long half = a.half;
    const int sg = w / a.n_rg;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;
    PipeBase P;
    P.sp = a.spin + ((long long)w * 2 + p) * half;
    P.m0 = a.m0 + ((long long)w * 2 + p) * half;
    P.m1 = a.m1 + ((long long)w * 2 + p) * half;
    P.m0q = a.m0 + ((long long)w * 2 + q) * half;
    P.m1q = a.m1 + ((long long)w * 2 + q) * half;
    P.sq = a.spin + ((long long)w * 2 + q) * half;
    P.jx = Jb + (0 * 2 + p) * half; P.jy = Jb + (1 * 2 + p) * half; P.jz = Jb + (2 * 2 + p) * half;
    P.jxq = Jb + (0 * 2 + q) * half; P.jyq = Jb + (1 * 2 + q) * half; P.jzq = Jb + (2 * 2 + q) * half;
    return P;
}

// thread -> (plane z, item t inside the plane, index idx whose low 5 bits are the lane and in which neighbouring
// items of a row are neighbours).  ZW = 4: see below.  ZW = 1: the planes of one parity class of z (blockIdx.y) follow
// each other in one index space, so that the last warp of a plane is filled up from the next plane of the class --
// a plane of L = 80 has 200 items, 1.56 blocks of 128.  (z + p) & 1, which selects the code path, is the same for
// every thread of the grid row.
template <int ZW>
__device__ __forceinline__ bool pipe_item(const SweepArgs& a, int per_plane, int& z, int& t, int& idx) {
    if (ZW == 1) {
        const uint32_t flat = blockIdx.x * blockDim.x + threadIdx.x;
        uint32_t rem;
        const uint32_t q = fastdivmod(flat, (uint32_t)per_plane, a.inv_pp, rem);
        idx = (int)flat; t = (int)rem; z = (int)(2u * q + blockIdx.y);
        return z < a.L;
    }
    t = (int)(blockIdx.x * 32 + (threadIdx.x & 31)); idx = t;
    z = (int)(blockIdx.y * ZW + (threadIdx.x >> 5));
    return t < per_plane;
}

// ZW = 1: grid = (ceil((L/2)*(L/YC)*(Lh/4) / 128), 2, n_words): blockIdx.y = parity class of the planes (pipe_item).
// ZW = 4: grid = (ceil((L/YC)*(Lh/4) / 32), L/4, n_words), warp k of a CTA works on plane
//         4*blockIdx.y + k with the same (row chunk, quad) items as its sibling warps: the
//         +-z neighbour rows of a warp are the own-plane rows of the next / previous warp and
//         are found in the SM's L1 (hit or hit-on-miss) instead of crossing the L2 -> SM path,
//         which is what bounds this kernel.
// DIR = +-1: this (odd) launch also performs the wandering half-cycle that closes the timestep
// (exchange_walkers).
template <int RPW, int YC, int ZW, int DIR = 0>
__global__ void __launch_bounds__(128)
half_sweep_pipe_kernel(SweepArgs a, int p, int walk_z)
{
    const int L = a.L, Lh = a.Lh;
    const int nxv = Lh >> 2;
    int z, t, idx;
    const bool active = pipe_item<ZW>(a, (L / YC) * nxv, z, t, idx);
    const unsigned mask = __ballot_sync(0xFFFFFFFFu, active);
    if (!active) return;
    const int chunk = (int)fastdiv((uint32_t)t, a.inv_nxv), xv = t - chunk * nxv;
    const int w = blockIdx.z + a.w0;
    const PipeBase P = pipe_base<RPW>(a, w, p);
    XNb nb = x_neighbours(idx, xv, nxv, mask, true);              // (z + p) & 1 is warp-uniform: one code path per warp
    nb.walk_z = walk_z;
    // programmatic dependent launch: this grid may have been scheduled while the
    // previous half-sweep was still draining; its results are needed from here on,
    // and the next grid may be scheduled as soon as every CTA of this one got here
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if ((z + p) & 1) march_rows_pipe<RPW, YC, 1, 0, DIR>(P, L, Lh, z, chunk * YC, xv * 4, nb);
    else             march_rows_pipe<RPW, YC, 0, 0, DIR>(P, L, Lh, z, chunk * YC, xv * 4, nb);
}

// The two launches of the LAST sweep of a measured group: same update, plus the
// counting described above MeasAcc.  MEAS = 1: even launch (levels, replica
// differences); MEAS = 2: odd launch (also unsatisfied bonds) whose last CTA turns
// the counts into the measurement row (finalize_rows) and re-zeroes them.
// Same grids as half_sweep_pipe_kernel<RPW, 4, ZW>; every thread stays for the
// block-wide reduction (warp_sum_lane_counts: one shuffle butterfly per counter and block).
template <int RPW, int ZW, int MEAS, int DIR = 0>
__global__ void __launch_bounds__(128, 4)
half_sweep_pipe_meas_kernel(SweepArgs a, int p, MeasureArgs ma)
{
    constexpr int YC = 4;
    __shared__ uint32_t s_pl[MeasAcc<YC>::PU + MeasAcc<YC>::PM + MeasAcc<YC>::PX][128];
    const int L = a.L, Lh = a.Lh;
    const int nxv = Lh >> 2;
    int z, t, idx;
    const bool active = pipe_item<ZW>(a, (L / YC) * nxv, z, t, idx);
    const unsigned mask = __ballot_sync(0xFFFFFFFFu, active);
    const int w = blockIdx.z;
    const bool pair = (RPW == 2) && ma.n_replicas == 2;
    MeasAcc<YC> acc; acc.clear();
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    if (active) {
        const int chunk = (int)fastdiv((uint32_t)t, a.inv_nxv), xv = t - chunk * nxv;
        const PipeBase P = pipe_base<RPW>(a, w, p);
        const XNb nb = x_neighbours(idx, xv, nxv, mask, true);
        if ((z + p) & 1) march_rows_pipe<RPW, YC, 1, MEAS, DIR>(P, L, Lh, z, chunk * YC, xv * 4, nb, &acc, pair);
        else             march_rows_pipe<RPW, YC, 0, MEAS, DIR>(P, L, Lh, z, chunk * YC, xv * 4, nb, &acc, pair);
    }
    // planes -> shared memory; warp 0 sums the unsatisfied bonds, warp 1 the levels, warp 2 the replica differences
    typedef MeasAcc<YC> Acc;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (MEAS == 2) {
#pragma unroll
        for (int k = 0; k < Acc::PU; ++k) s_pl[k][tid] = acc.u.c[k];
    }
#pragma unroll
    for (int k = 0; k < Acc::PM; ++k) s_pl[Acc::PU + k][tid] = acc.m.c[k];
    if (pair) {
#pragma unroll
        for (int k = 0; k < Acc::PX; ++k) s_pl[Acc::PU + Acc::PM + k][tid] = acc.x.c[k];
    }
    __syncthreads();
    if (MEAS == 2 && warp == 0) warp_sum_lane_counts<Acc::PU>(s_pl, lane, ma.cntU + (long long)w * 32);
    if (warp == 1) warp_sum_lane_counts<Acc::PM>(s_pl + Acc::PU, lane, ma.cntM + (long long)w * 32);
    if (pair && warp == 2) warp_sum_lane_counts<Acc::PX>(s_pl + Acc::PU + Acc::PM, lane, ma.cntX + (long long)(w / a.n_rg) * 32);
}

// counts -> measurement row, after the odd measuring launch (one block; a ticket in that launch would cost every one
// of its blocks a __threadfence behind its row stores)
__global__ void __launch_bounds__(128)
finalize_kernel(FinalizeArgs fa)
{
    asm volatile("griddepcontrol.wait;" ::: "memory");
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    finalize_rows(fa);
}

}  // namespace micsa
