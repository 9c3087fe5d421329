// philox.cuh -- Philox4x32-10 counter-based generator (Salmon, Moraes, Dror,
// Shaw 2011; the same generator as cuRAND's PHILOX4_32_10).  DESIGN.md R8.
// Written for the GPU: the ten round keys depend only on the seed, so the host
// computes them once and every thread reads them from kernel parameters.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace micsa {

struct PhiloxKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

inline PhiloxKeys philox_make_keys(uint64_t seed) {
    PhiloxKeys ks;
    uint32_t a = (uint32_t)(seed & 0xFFFFFFFFull), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        ks.k0[r] = a; ks.k1[r] = b;
        a += 0x9E3779B9u;          // Weyl increments of the key schedule
        b += 0xBB67AE85u;
    }
    return ks;
}

__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2,
                                                uint32_t c3, const PhiloxKeys& ks) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        // one 32x32 -> 64 multiply (IMAD.WIDE) per product instead of IMAD + IMAD.HI
        const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
        const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
        const uint32_t lo0 = (uint32_t)p0, hi0 = (uint32_t)(p0 >> 32);
        const uint32_t lo1 = (uint32_t)p1, hi1 = (uint32_t)(p1 >> 32);
        c0 = hi1 ^ c1 ^ ks.k0[r];
        c1 = lo1;
        c2 = hi0 ^ c3 ^ ks.k1[r];
        c3 = lo0;
    }
    return make_uint4(c0, c1, c2, c3);
}

// domain tags carried in the top byte of counter word c2
enum : uint32_t { kTagRefresh = 0u, kTagSpinInit = 1u << 24, kTagBondInit = 2u << 24, kTagMetropolis = 3u << 24 };

}  // namespace micsa
