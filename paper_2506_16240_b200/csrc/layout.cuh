// layout.cuh -- private bit-sliced device layout of the MicSA state.
//
// PAPER.md:146 ("different bits in a memory word represent different physical
// spins"; daemon level in two bit-planes) leaves open what shares a word; here
// a 32-bit word holds the same lattice site of 32 different SYSTEMS
// (DESIGN.md "Data layout"):
//
//   word lattice  w = sg * n_rg + rg        sg = sample group, rg = replica group
//   lane          l = r_local * spw + s_local
//   rpw = replicas per word (2 if n_replicas is even, else 1), spw = 32 / rpw
//   sample = sg*spw + s_local, replica = rg*rpw + r_local
//
// so the rpw replicas in a word share ONE bond word of spw bits (PAPER.md:240:
// replicas evolve under the same couplings), stored as uint16 (rpw=2) or
// uint32 (rpw=1) and replicated across the replica fields in registers.
//
// Every plane is split by site parity and compressed in x (PAPER.md:84
// checkerboard): index of site (x,y,z) inside its parity array is
//   h = (z*L + y)*Lh + (x >> 1),   Lh = L/2,   parity p = (x+y+z)&1,
//   x = 2*(x>>1) + ((y+z+p)&1).
// Arrays:  spin/m0/m1 : uint32 [n_words][2 parities][half]   half = L*L*Lh
//          bonds      : JT     [n_sg][3 dirs][2 parities][half]  (owner's parity)
// Encodings (R1): spin bit 1 <=> s = -1; bond bit 1 <=> J = -1;
// then "bond unsatisfied" = sigma_x ^ sigma_y ^ j.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace micsa {

struct Geom {
    int L, Lh;
    int n_samples, n_replicas, sample_offset;
    int rpw, spw;
    int n_sg, n_rg, n_words;
    long long half;        // sites per parity = L*L*Lh
    long long N;           // L^3
    int n_sys, n_pairs;    // n_pairs = n_samples * n_replicas(n_replicas-1)/2
};

struct State {
    uint32_t* spin;        // [n_words][2][half]
    uint32_t* m0;          // daemon level bit 0
    uint32_t* m1;          // daemon level bit 1
    void*     J;           // uint16 or uint32 [n_sg][3][2][half]
};

// ---- small fixed-size vectors of 32-bit words with the widest legal access
template <int V> struct Vec { uint32_t v[V]; };

template <int V> __device__ __forceinline__ Vec<V> ldg_vec(const uint32_t* p);
template <> __device__ __forceinline__ Vec<1> ldg_vec<1>(const uint32_t* p) {
    Vec<1> r; r.v[0] = *p; return r;
}
template <> __device__ __forceinline__ Vec<2> ldg_vec<2>(const uint32_t* p) {
    uint2 t = *reinterpret_cast<const uint2*>(p);
    Vec<2> r; r.v[0] = t.x; r.v[1] = t.y; return r;
}
template <> __device__ __forceinline__ Vec<4> ldg_vec<4>(const uint32_t* p) {
    uint4 t = *reinterpret_cast<const uint4*>(p);
    Vec<4> r; r.v[0] = t.x; r.v[1] = t.y; r.v[2] = t.z; r.v[3] = t.w; return r;
}
template <int V> __device__ __forceinline__ void stg_vec(uint32_t* p, const Vec<V>& a);
template <> __device__ __forceinline__ void stg_vec<1>(uint32_t* p, const Vec<1>& a) { *p = a.v[0]; }
template <> __device__ __forceinline__ void stg_vec<2>(uint32_t* p, const Vec<2>& a) {
    *reinterpret_cast<uint2*>(p) = make_uint2(a.v[0], a.v[1]);
}
template <> __device__ __forceinline__ void stg_vec<4>(uint32_t* p, const Vec<4>& a) {
    *reinterpret_cast<uint4*>(p) = make_uint4(a.v[0], a.v[1], a.v[2], a.v[3]);
}

// ---- bond words: load V consecutive bond words and replicate each across the
// rpw replica fields of a 32-bit spin word.
template <int RPW> struct BondT;
template <> struct BondT<1> { typedef uint32_t type; };
template <> struct BondT<2> { typedef uint16_t type; };

template <int RPW> __device__ __forceinline__ uint32_t bond_expand(typename BondT<RPW>::type j);
template <> __device__ __forceinline__ uint32_t bond_expand<1>(uint32_t j) { return j; }
template <> __device__ __forceinline__ uint32_t bond_expand<2>(uint16_t j) {
    return __byte_perm((uint32_t)j, 0u, 0x1010);
}

template <int V, int RPW> __device__ __forceinline__ Vec<V> ldg_bonds(const typename BondT<RPW>::type* p);
template <> __device__ __forceinline__ Vec<1> ldg_bonds<1, 1>(const uint32_t* p) { return ldg_vec<1>(p); }
template <> __device__ __forceinline__ Vec<2> ldg_bonds<2, 1>(const uint32_t* p) { return ldg_vec<2>(p); }
template <> __device__ __forceinline__ Vec<4> ldg_bonds<4, 1>(const uint32_t* p) { return ldg_vec<4>(p); }
template <> __device__ __forceinline__ Vec<1> ldg_bonds<1, 2>(const uint16_t* p) {
    Vec<1> r; r.v[0] = bond_expand<2>(*p); return r;
}
template <> __device__ __forceinline__ Vec<2> ldg_bonds<2, 2>(const uint16_t* p) {
    uint32_t t = *reinterpret_cast<const uint32_t*>(p);
    Vec<2> r; r.v[0] = __byte_perm(t, 0u, 0x1010); r.v[1] = __byte_perm(t, 0u, 0x3232); return r;
}
template <> __device__ __forceinline__ Vec<4> ldg_bonds<4, 2>(const uint16_t* p) {
    uint2 t = *reinterpret_cast<const uint2*>(p);
    Vec<4> r;
    r.v[0] = __byte_perm(t.x, 0u, 0x1010); r.v[1] = __byte_perm(t.x, 0u, 0x3232);
    r.v[2] = __byte_perm(t.y, 0u, 0x1010); r.v[3] = __byte_perm(t.y, 0u, 0x3232);
    return r;
}

// One three-input logic operation, written as the LOP3 it is meant to be.  Left as C++ (in the update) the
// compiler re-associates the XOR chains (it forms neighbour ^ bond first and then needs two or three operations for
// every sum and carry of the first adder level) and the 20 operations per word become 43.
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
    uint32_t d;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return d;
}
constexpr int kXor3 = 0x96, kMaj3 = 0xE8, kSel = 0xCA /* a ? b : c */, kSelNot = 0x3A /* a ? ~b : c */;

// unsatisfied-bond flag of one neighbour: own spin ^ neighbour spin ^ bond
__device__ __forceinline__ uint32_t bond_flag(uint32_t g, uint32_t n, uint32_t j) { return lop3<kXor3>(g, n, j); }

// n / d by one multiply: m = ceil(2^32 / d) (host, d >= 2), q = umulhi(n, m) is exact whenever n * d <= 2^32
// (the error of n * m / 2^32 against n / d is below n * d / (d * 2^32) <= 1 / d).  Every use here divides an index
// inside one lattice plane (< L * L/2 < 2^20) by a row length (< 2^10).  d = 1: m = 0 and the quotient is n.
inline uint32_t fastdiv_magic(uint32_t d) { return d >= 2 ? (uint32_t)(((1ull << 32) + d - 1) / d) : 0u; }
__device__ __forceinline__ uint32_t fastdiv(uint32_t n, uint32_t m) { return m ? __umulhi(n, m) : n; }

// n / d and n % d for ANY n < 2^32 with the same magic number: umulhi(n, m) overshoots n / d by less than n / 2^32 < 1,
// so it is the quotient or one more -- one multiply and a correction.
__device__ __forceinline__ uint32_t fastdivmod(uint32_t n, uint32_t d, uint32_t m, uint32_t& rem) {
    if (m == 0u) { rem = 0u; return n; }
    uint32_t q = __umulhi(n, m);
    uint32_t r = n - q * d;
    if ((int32_t)r < 0) { q -= 1u; r += d; }
    rem = r;
    return q;
}

// canonical site index i = x + L*(y + L*z) of element xh of row (y,z), parity p
__device__ __forceinline__ uint32_t canonical_site(int L, int p, int z, int y, int xh) {
    const int x = 2 * xh + ((y + z + p) & 1);
    return (uint32_t)x + (uint32_t)L * ((uint32_t)y + (uint32_t)L * (uint32_t)z);
}

}  // namespace micsa
