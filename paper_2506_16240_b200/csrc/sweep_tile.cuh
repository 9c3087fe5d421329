// sweep_tile.cuh -- tiled half-sweep for L % 8 == 0 (all BASELINE configs).
//
// Same elementary move as sweep.cuh (PAPER.md:119-124 Eq. 8, :150 Eq. 10,
// checkerboard order PAPER.md:198); what changes is how the data reaches the
// registers.
//
// A CTA owns a tile of TY rows (y) x TZ planes (z) x the full x extent of the
// parity-p arrays of word lattice w (layout.cuh).  Per half-sweep every datum
// of the tile is used by exactly one thread EXCEPT the opposite-parity spins
// (each is a neighbour of up to six updated sites) and the x-bond of the
// opposite-parity row (shifted by one word for half of the rows):
//  * those two are staged in shared memory by the TMA engine (cp.async.bulk,
//    one mbarrier): the tile's rows plus the one-row halo in +-y and +-z, so
//    every opposite-parity word crosses L2->SM once per tile (1.75x with the
//    8x4 tile) instead of once per neighbour, and the +-1 word shifts along x
//    and the periodic wrap become shared-memory indexing;
//  * own spin, the two daemon planes and the five remaining bond vectors are
//    single-use: each thread loads them straight into registers with one
//    128-bit (spins, daemons) or 64/128-bit (bonds) access, all issued before
//    the first wait, so a CTA has its whole working set in flight at once.
// One thread updates 4 consecutive words = 128 spin-flip attempts.
#pragma once
#include "sweep.cuh"

namespace micsa {

__device__ __forceinline__ uint32_t smem_addr(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(bar), "r"(bytes) : "memory");
}
// global -> shared bulk copy (TMA, 1D); bytes % 16 == 0, both addresses 16-byte aligned
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}" :: "r"(bar), "r"(parity) : "memory");
}

template <int RPW, int TY, int TZ>
struct TileSmem {
    typedef typename Bond4<RPW>::elem JT;
    static constexpr int kOppRows = (TZ + 2) * (TY + 2);        // corners unused
    static __host__ __device__ size_t bytes(int Lh) {
        return 16 + (size_t)kOppRows * Lh * 4 + (size_t)TY * TZ * Lh * sizeof(JT);
    }
};

// grid = ((L/TY)*(L/TZ), n_words); block = min(TY*TZ*Lh/4, cap) rounded to 32
template <int RPW, int TY, int TZ>
__global__ void __launch_bounds__(640, 2)
half_sweep_tile_kernel(SweepArgs a, int p)
{
    typedef Bond4<RPW> B4;
    typedef typename B4::elem JT;
    typedef typename B4::raw JRaw;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int L = a.L, Lh = a.Lh, q = 1 - p;
    const int nq = Lh >> 2;
    const int n_ty = L / TY;
    const int tz = blockIdx.x / n_ty, ty = blockIdx.x - tz * n_ty;
    const int y0 = ty * TY, z0 = tz * TZ, w = blockIdx.y;
    const long long half = a.half;
    const uint32_t rowB = (uint32_t)Lh * 4u;                   // bytes per spin row

    uint32_t* oppS = reinterpret_cast<uint32_t*>(smem_raw + 16);
    JT* jxqS = reinterpret_cast<JT*>(smem_raw + 16 + (size_t)TileSmem<RPW, TY, TZ>::kOppRows * rowB);
    const uint32_t bar = smem_addr(smem_raw);

    const uint32_t* sqb = a.spin + ((long long)w * 2 + q) * half;
    const int sg = w / a.n_rg;
    const JT* Jb = reinterpret_cast<const JT*>(a.J) + (long long)sg * 6 * half;
    const JT* Jxq = Jb + (0 * 2 + q) * half;

    if (threadIdx.x == 0) { mbar_init(bar, 1); mbar_fence_init(); }
    __syncthreads();
    if (threadIdx.x < 32) {
        // copies: per tile plane 3 (interior rows, row y0-1, row y0+TY), the two halo
        // planes (interior rows only), and the x-bond rows of the tile planes
        constexpr int kCopies = 3 * TZ + 2 + TZ;
        if (threadIdx.x == 0) {
            const uint32_t total = (uint32_t)(TZ * (TY + 2) + 2 * TY) * rowB
                                 + (uint32_t)(TZ * TY) * (uint32_t)Lh * (uint32_t)sizeof(JT);
            mbar_expect_tx(bar, total);
        }
        __syncwarp();
        const int ym = (y0 == 0) ? L - 1 : y0 - 1;
        const int yp = (y0 + TY == L) ? 0 : y0 + TY;
        for (int c = threadIdx.x; c < kCopies; c += 32) {
            if (c < 3 * TZ) {
                const int lz = c / 3, kind = c - 3 * lz;
                const int z = z0 + lz;
                const int yy = kind == 0 ? y0 : (kind == 1 ? ym : yp);
                const int ly = kind == 0 ? 0 : (kind == 1 ? -1 : TY);
                const uint32_t n = kind == 0 ? (uint32_t)TY * rowB : rowB;
                bulk_g2s(smem_addr(oppS + ((lz + 1) * (TY + 2) + ly + 1) * Lh),
                         sqb + ((long long)z * L + yy) * Lh, n, bar);
            } else if (c < 3 * TZ + 2) {
                const int up = c - 3 * TZ;                     // 0: plane z0-1, 1: plane z0+TZ
                const int z = up ? ((z0 + TZ == L) ? 0 : z0 + TZ) : ((z0 == 0) ? L - 1 : z0 - 1);
                const int lz = up ? TZ : -1;
                bulk_g2s(smem_addr(oppS + ((lz + 1) * (TY + 2) + 1) * Lh),
                         sqb + ((long long)z * L + y0) * Lh, (uint32_t)TY * rowB, bar);
            } else {
                const int lz = c - (3 * TZ + 2);
                bulk_g2s(smem_addr(jxqS + lz * TY * Lh),
                         Jxq + ((long long)(z0 + lz) * L + y0) * Lh,
                         (uint32_t)(TY * Lh) * (uint32_t)sizeof(JT), bar);
            }
        }
    }

    uint32_t* spb = a.spin + ((long long)w * 2 + p) * half;
    uint32_t* m0b = a.m0 + ((long long)w * 2 + p) * half;
    uint32_t* m1b = a.m1 + ((long long)w * 2 + p) * half;
    const JT* Jxp = Jb + (0 * 2 + p) * half;
    const JT* Jyp = Jb + (1 * 2 + p) * half;
    const JT* Jzp = Jb + (2 * 2 + p) * half;
    const JT* Jyq = Jb + (1 * 2 + q) * half;
    const JT* Jzq = Jb + (2 * 2 + q) * half;

    const int items = TY * TZ * nq;
    bool waited = false;
    for (int it = threadIdx.x; it < items; it += blockDim.x) {
        const int r = it / nq, xq = it - r * nq;
        const int lz = r / TY, ly = r - lz * TY;
        const int y = y0 + ly, z = z0 + lz;
        const int xh0 = xq * 4;
        const int ym = (y == 0) ? L - 1 : y - 1;
        const int zm = (z == 0) ? L - 1 : z - 1;
        const long long h = ((long long)z * L + y) * Lh + xh0;
        const long long h_ym = ((long long)z * L + ym) * Lh + xh0;
        const long long h_zm = ((long long)zm * L + y) * Lh + xh0;

        // single-use data: straight to registers
        const uint4 s4 = *reinterpret_cast<const uint4*>(spb + h);
        const uint4 d04 = *reinterpret_cast<const uint4*>(m0b + h);
        const uint4 d14 = *reinterpret_cast<const uint4*>(m1b + h);
        const JRaw rjx = *reinterpret_cast<const JRaw*>(Jxp + h);
        const JRaw rjy = *reinterpret_cast<const JRaw*>(Jyp + h);
        const JRaw rjz = *reinterpret_cast<const JRaw*>(Jzp + h);
        const JRaw rjym = *reinterpret_cast<const JRaw*>(Jyq + h_ym);
        const JRaw rjzm = *reinterpret_cast<const JRaw*>(Jzq + h_zm);

        if (!waited) { mbar_wait(bar, 0); waited = true; }

        // c = 1: x = 2xh+1, -x neighbour at xh (it owns the bond), +x neighbour at xh+1
        // c = 0: x = 2xh,   +x neighbour at xh, -x neighbour at xh-1 (it owns the bond)
        const int c = (y + z + p) & 1;
        const uint32_t cm = c ? 0xFFFFFFFFu : 0u;
        const uint32_t* rowS = oppS + ((lz + 1) * (TY + 2) + ly + 1) * Lh;
        const JT* jrowS = jxqS + (lz * TY + ly) * Lh;
        const int xe = c ? ((xh0 + 4 == Lh) ? 0 : xh0 + 4) : ((xh0 == 0) ? Lh - 1 : xh0 - 1);
        const uint4 A4 = *reinterpret_cast<const uint4*>(rowS + xh0);
        const uint32_t e = rowS[xe];
        const uint32_t eJ = B4::expand1(jrowS[xe]);
        const uint4 yp4 = *reinterpret_cast<const uint4*>(rowS + Lh + xh0);
        const uint4 ym4 = *reinterpret_cast<const uint4*>(rowS - Lh + xh0);
        const uint4 zp4 = *reinterpret_cast<const uint4*>(rowS + (TY + 2) * Lh + xh0);
        const uint4 zm4 = *reinterpret_cast<const uint4*>(rowS - (TY + 2) * Lh + xh0);
        const JRaw rBx = *reinterpret_cast<const JRaw*>(jrowS + xh0);

        uint32_t jxo[4], jyo[4], jzo[4], jym[4], jzm[4], Bx[4];
        B4::expand(rjx, jxo); B4::expand(rjy, jyo); B4::expand(rjz, jzo);
        B4::expand(rjym, jym); B4::expand(rjzm, jzm); B4::expand(rBx, Bx);
        const uint32_t av[4] = { A4.x, A4.y, A4.z, A4.w };
        const uint32_t yp[4] = { yp4.x, yp4.y, yp4.z, yp4.w };
        const uint32_t ymv[4] = { ym4.x, ym4.y, ym4.z, ym4.w };
        const uint32_t zp[4] = { zp4.x, zp4.y, zp4.z, zp4.w };
        const uint32_t zmv[4] = { zm4.x, zm4.y, zm4.z, zm4.w };
        uint32_t sv[4] = { s4.x, s4.y, s4.z, s4.w };
        uint32_t v0[4] = { d04.x, d04.y, d04.z, d04.w };
        uint32_t v1[4] = { d14.x, d14.y, d14.z, d14.w };
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const uint32_t up   = (k < 3) ? av[k + 1] : e;
            const uint32_t down = (k > 0) ? av[k - 1] : e;
            const uint32_t Bdn  = (k > 0) ? Bx[k - 1] : eJ;
            const uint32_t n_xp = (cm & up) | (~cm & av[k]);
            const uint32_t n_xm = (cm & av[k]) | (~cm & down);
            const uint32_t j_xm = (cm & Bx[k]) | (~cm & Bdn);
            const uint32_t g = sv[k];
            creutz_word(g ^ n_xp ^ jxo[k], g ^ n_xm ^ j_xm,
                        g ^ yp[k] ^ jyo[k], g ^ ymv[k] ^ jym[k],
                        g ^ zp[k] ^ jzo[k], g ^ zmv[k] ^ jzm[k],
                        sv[k], v0[k], v1[k]);
        }
        *reinterpret_cast<uint4*>(spb + h) = make_uint4(sv[0], sv[1], sv[2], sv[3]);
        *reinterpret_cast<uint4*>(m0b + h) = make_uint4(v0[0], v0[1], v0[2], v0[3]);
        *reinterpret_cast<uint4*>(m1b + h) = make_uint4(v1[0], v1[1], v1[2], v1[3]);
    }
}

}  // namespace micsa
