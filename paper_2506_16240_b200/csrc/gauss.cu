// gauss.cu -- continuous daemons / walkers with real-valued couplings
// (SURVEY.md 8(f) rank 4): PAPER.md:136-140 (Sec. 2.4, Eq. 9) and :436-454
// (Appendix C: Gaussian couplings, "continuous walker variables", the
// uncapped elementary move of Sec. 2.3).  Float64 path, one thread per
// (site, system); no bit-slicing -- the daemons are real numbers.
//
// Arithmetic contract (R18-R21), chosen so that the accept decision
// n - dH >= 0 is taken on the same float64 number by any plain restatement of the move:
//   h  = ((((J(+x) s(+x) + J(-x) s(-x)) + J(+y) s(+y)) + J(-y) s(-y)) + J(+z) s(+z)) + J(-z) s(-z)
//   dH = (2 s) * h;  n' = n - dH;  flip iff n' >= 0
// every operation a separately rounded IEEE float64 operation (__dmul_rn /
// __dadd_rn / __dsub_rn: no fused multiply-add).  Refresh: n = -T log(u),
// u = (x + 1/2) 2^-32 with x = word 0 of Philox4x32-10 at counter
// (i, global sample, (5 << 24) | replica, step).
//
// Device layout: every array split by site parity and compressed in x like the
// bit-sliced path (layout.cuh): index h = (z L + y) L/2 + (x >> 1) inside the
// parity array, so all accesses of a warp are unit-stride:
//   spin : int8   [n_sys][2][half]      n : double [n_sys][2][half]
//   J    : double [n_samples][3][2][half]   (owner's parity)
#include "../../include/micsa.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <new>

#include "philox.cuh"

void micsa_internal_set_error(const char* fmt, const char* detail);      // micsa.cu

using namespace micsa;

struct micsa_gauss_ctx {
    int L, Lh, n_samples, n_replicas, n_sys, n_pairs, sample_offset;
    long long N, half;
    int8_t* spin; double* n; double* J;
    double* part; unsigned long long* qcnt;     // measurement scratch
    void* stage; size_t stage_bytes;            // canonical-layout staging (grow-only)
    double* host_row;                           // pinned: E, E_daemon per system
    PhiloxKeys ks;
    cudaStream_t stream;
    int walkers; long long t;
    int n_part;
    uint64_t attempts, rns;
    int sticky;
};

namespace {

#define GCK(ctx, call)                                                                     \
    do {                                                                                   \
        cudaError_t e_ = (call);                                                           \
        if (e_ != cudaSuccess) {                                                           \
            micsa_internal_set_error("CUDA error: %s", cudaGetErrorString(e_));            \
            if (ctx) (ctx)->sticky = MICSA_ERR_CUDA;                                       \
            return MICSA_ERR_CUDA;                                                         \
        }                                                                                  \
    } while (0)

int gcheck(micsa_gauss_ctx* c) {
    if (!c) { micsa_internal_set_error("null context", ""); return MICSA_ERR_INVALID; }
    if (c->sticky) { micsa_internal_set_error("context is in a sticky CUDA error state", ""); return c->sticky; }
    return MICSA_OK;
}

struct GGeom { int L, Lh; long long half; uint32_t inv_Lh, inv_L; };   // inv_d = ceil(2^32 / d), 0 for d = 1

// n / d and n % d for any n < 2^32 by one multiply and a correction: q' = umulhi(n, ceil(2^32 / d)) overshoots n / d
// by less than n / 2^32 < 1, so it is the quotient or one more (a 32-bit division costs ~36 instructions, and the
// refresh and wandering kernels of this file are bound by instruction issue)
inline uint32_t gdiv_magic(uint32_t d) { return d >= 2 ? (uint32_t)(((1ull << 32) + d - 1) / d) : 0u; }
__device__ __forceinline__ uint32_t gdivmod(uint32_t n, uint32_t d, uint32_t inv, uint32_t& rem) {
    if (inv == 0u) { rem = 0u; return n; }
    uint32_t q = __umulhi(n, inv);
    uint32_t r = n - q * d;
    if ((int32_t)r < 0) { q -= 1u; r += d; }
    rem = r;
    return q;
}

// thread -> site of parity p: t = (z L + y) Lh + xh (32-bit arithmetic: half = L^3 / 2 < 2^30)
__device__ __forceinline__ bool site_of(const GGeom& g, long long t, int p, int& xh, int& y, int& z, int& c) {
    if (t >= g.half) return false;
    uint32_t rx, ry;
    const uint32_t r = gdivmod((uint32_t)t, (uint32_t)g.Lh, g.inv_Lh, rx);
    z = (int)gdivmod(r, (uint32_t)g.L, g.inv_L, ry);
    xh = (int)rx; y = (int)ry;
    c = (y + z + p) & 1;
    return true;
}

// grid = (ceil(half / 256), n_sys)
__global__ void __launch_bounds__(256)
gauss_half_sweep_kernel(int8_t* __restrict__ spin, double* __restrict__ nd, const double* __restrict__ J,
                        GGeom g, int n_replicas, int p)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    int xh, y, z, c;
    if (!site_of(g, t, p, xh, y, z, c)) return;
    const int sys = blockIdx.y, sample = sys / n_replicas, q = 1 - p;
    const int L = g.L, Lh = g.Lh;
    const long long half = g.half;
    int8_t* sp = spin + ((long long)sys * 2 + p) * half;
    const int8_t* sq = spin + ((long long)sys * 2 + q) * half;
    double* np_ = nd + ((long long)sys * 2 + p) * half;
    const double* Jb = J + (long long)sample * 6 * half;
    const uint32_t row = (uint32_t)(z * L + y) * (uint32_t)Lh;
    const int yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const int zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    // x = 2 xh + c: the +x neighbour sits at xh + c, the -x neighbour at xh + c - 1 of the other parity's row
    const int xp = (xh + c == Lh) ? 0 : xh + c;
    const int xm = (xh + c - 1 < 0) ? Lh - 1 : xh + c - 1;
    const uint32_t h_xp = row + (uint32_t)xp, h_xm = row + (uint32_t)xm;
    const uint32_t h_yp = (uint32_t)(z * L + yp) * (uint32_t)Lh + (uint32_t)xh, h_ym = (uint32_t)(z * L + ym) * (uint32_t)Lh + (uint32_t)xh;
    const uint32_t h_zp = (uint32_t)(zp * L + y) * (uint32_t)Lh + (uint32_t)xh, h_zm = (uint32_t)(zm * L + y) * (uint32_t)Lh + (uint32_t)xh;
    const double s0 = (double)sp[t];
    double h = __dmul_rn(Jb[(0 * 2 + p) * half + t], (double)sq[h_xp]);
    h = __dadd_rn(h, __dmul_rn(Jb[(0 * 2 + q) * half + h_xm], (double)sq[h_xm]));
    h = __dadd_rn(h, __dmul_rn(Jb[(1 * 2 + p) * half + t], (double)sq[h_yp]));
    h = __dadd_rn(h, __dmul_rn(Jb[(1 * 2 + q) * half + h_ym], (double)sq[h_ym]));
    h = __dadd_rn(h, __dmul_rn(Jb[(2 * 2 + p) * half + t], (double)sq[h_zp]));
    h = __dadd_rn(h, __dmul_rn(Jb[(2 * 2 + q) * half + h_zm], (double)sq[h_zm]));
    const double dH = __dmul_rn(__dmul_rn(2.0, s0), h);          // Eq. (1): change of H_EA if this spin flips
    const double nn = __dsub_rn(np_[t], dH);                    // Eq. (8)
    if (nn >= 0.0) { sp[t] = (int8_t)(-(int)sp[t]); np_[t] = nn; }
}

// V consecutive sites of a row per thread (V = 2 or 4, Lh % V == 0): the same move, the index arithmetic paid once
// per V attempts and the daemon energies / couplings moved with 128-bit accesses.
template <int V> __device__ __forceinline__ void ld_f64(const double* p, double (&o)[V]) {
    if (V == 1) { o[0] = p[0]; return; }
#pragma unroll
    for (int k = 0; k < V; k += 2) { const double2 t = *reinterpret_cast<const double2*>(p + k); o[k] = t.x; o[k + 1] = t.y; }
}
template <int V> __device__ __forceinline__ void ld_s8(const int8_t* p, double (&o)[V]) {
    if (V == 4) { const char4 t = *reinterpret_cast<const char4*>(p); o[0] = (double)t.x; o[1] = (double)t.y; o[2] = (double)t.z; o[3] = (double)t.w; }
    else if (V == 2) { const char2 t = *reinterpret_cast<const char2*>(p); o[0] = (double)t.x; o[1] = (double)t.y; }
    else o[0] = (double)p[0];
}

// grid = (ceil(half / V / 256), n_sys)
template <int V>
__global__ void __launch_bounds__(256)
gauss_half_sweep_vec_kernel(int8_t* __restrict__ spin, double* __restrict__ nd, const double* __restrict__ J,
                            GGeom g, int n_replicas, int p)
{
    const uint32_t L = (uint32_t)g.L, Lh = (uint32_t)g.Lh, Lv = Lh / V;
    const uint32_t tv = blockIdx.x * blockDim.x + threadIdx.x;
    if ((long long)tv * V >= g.half) return;
    const uint32_t r = tv / Lv, xv = tv - r * Lv, z = r / L, y = r - z * L;
    const uint32_t c = (y + z + (uint32_t)p) & 1u, xh0 = xv * V;
    const int sys = blockIdx.y, sample = sys / n_replicas, q = 1 - p;
    const long long half = g.half;
    int8_t* sp = spin + ((long long)sys * 2 + p) * half;
    const int8_t* sq = spin + ((long long)sys * 2 + q) * half;
    double* np_ = nd + ((long long)sys * 2 + p) * half;
    const double* Jb = J + (long long)sample * 6 * half;
    const uint32_t yp = (y + 1 == L) ? 0 : y + 1, ym = (y == 0) ? L - 1 : y - 1;
    const uint32_t zp = (z + 1 == L) ? 0 : z + 1, zm = (z == 0) ? L - 1 : z - 1;
    const uint32_t row = (z * L + y) * Lh, h = row + xh0;
    const uint32_t h_yp = (z * L + yp) * Lh + xh0, h_ym = (z * L + ym) * Lh + xh0;
    const uint32_t h_zp = (zp * L + y) * Lh + xh0, h_zm = (zm * L + y) * Lh + xh0;
    // x = 2 xh + c: the site just outside the V words that is an x-neighbour: xh0 + V (c = 1) or xh0 - 1 (c = 0)
    const uint32_t xe = c ? ((xh0 + V == Lh) ? 0 : xh0 + V) : ((xh0 == 0) ? Lh - 1 : xh0 - 1);
    double nn[V], s0[V], A[V], syp[V], sym[V], szp[V], szm[V], jx[V], jy[V], jz[V], jxq[V], jym[V], jzm[V];
    ld_f64<V>(np_ + h, nn);
    ld_s8<V>(sp + h, s0); ld_s8<V>(sq + h, A);
    ld_s8<V>(sq + h_yp, syp); ld_s8<V>(sq + h_ym, sym); ld_s8<V>(sq + h_zp, szp); ld_s8<V>(sq + h_zm, szm);
    const double E = (double)sq[row + xe];
    ld_f64<V>(Jb + (0 * 2 + p) * half + h, jx); ld_f64<V>(Jb + (1 * 2 + p) * half + h, jy); ld_f64<V>(Jb + (2 * 2 + p) * half + h, jz);
    ld_f64<V>(Jb + (0 * 2 + q) * half + h, jxq);
    const double eJ = Jb[(0 * 2 + q) * half + row + xe];            // bond of site xh0 - 1 towards +x (used when c = 0)
    ld_f64<V>(Jb + (1 * 2 + q) * half + h_ym, jym); ld_f64<V>(Jb + (2 * 2 + q) * half + h_zm, jzm);
    int8_t snew[V];
#pragma unroll
    for (int k = 0; k < V; ++k) {
        const double s_xp = c ? ((k + 1 < V) ? A[(k + 1 < V) ? k + 1 : k] : E) : A[k];
        const double s_xm = c ? A[k] : ((k > 0) ? A[(k > 0) ? k - 1 : 0] : E);
        const double j_xm = c ? jxq[k] : ((k > 0) ? jxq[(k > 0) ? k - 1 : 0] : eJ);
        double hh = __dmul_rn(jx[k], s_xp);
        hh = __dadd_rn(hh, __dmul_rn(j_xm, s_xm));
        hh = __dadd_rn(hh, __dmul_rn(jy[k], syp[k]));
        hh = __dadd_rn(hh, __dmul_rn(jym[k], sym[k]));
        hh = __dadd_rn(hh, __dmul_rn(jz[k], szp[k]));
        hh = __dadd_rn(hh, __dmul_rn(jzm[k], szm[k]));
        const double dH = __dmul_rn(__dmul_rn(2.0, s0[k]), hh);      // Eq. (1): change of H_EA if this spin flips
        const double nk = __dsub_rn(nn[k], dH);                     // Eq. (8)
        const bool acc = nk >= 0.0;
        nn[k] = acc ? nk : nn[k];
        snew[k] = (int8_t)(acc ? -(int)s0[k] : (int)s0[k]);
    }
    if (V == 1) { np_[h] = nn[0]; sp[h] = snew[0]; }
    else {
#pragma unroll
        for (int k = 0; k < V; k += 2) *reinterpret_cast<double2*>(np_ + h + k) = make_double2(nn[k], nn[(k + 1 < V) ? k + 1 : k]);
        if (V == 4) *reinterpret_cast<char4*>(sp + h) = make_char4(snew[0], snew[1], snew[(V > 2) ? 2 : 0], snew[(V > 3) ? 3 : 0]);
        else        *reinterpret_cast<char2*>(sp + h) = make_char2(snew[0], snew[(V > 1) ? 1 : 0]);
    }
}

__global__ void __launch_bounds__(256)
gauss_refresh_kernel(double* __restrict__ nd, GGeom g, int n_replicas, int sample_offset, PhiloxKeys ks,
                     uint32_t step, double T)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.z;
    int xh, y, z, c;
    if (!site_of(g, t, p, xh, y, z, c)) return;
    const int sys = blockIdx.y, sample = sys / n_replicas, rep = sys - sample * n_replicas;
    const uint32_t i = (uint32_t)(2 * xh + c) + (uint32_t)g.L * ((uint32_t)y + (uint32_t)g.L * (uint32_t)z);
    const uint4 o = philox4x32_10(i, (uint32_t)(sample_offset + sample), (5u << 24) | (uint32_t)rep, step, ks);
    const double u = __dmul_rn(__dadd_rn((double)o.x, 0.5), 1.0 / 4294967296.0);
    nd[((long long)sys * 2 + p) * g.half + t] = __dmul_rn(-T, log(u));       // Eq. (9)
}

__global__ void __launch_bounds__(256)
gauss_init_spins_kernel(int8_t* __restrict__ spin, GGeom g, int n_replicas, int sample_offset, PhiloxKeys ks)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.z;
    int xh, y, z, c;
    if (!site_of(g, t, p, xh, y, z, c)) return;
    const int sys = blockIdx.y, sample = sys / n_replicas, rep = sys - sample * n_replicas;
    const uint32_t i = (uint32_t)(2 * xh + c) + (uint32_t)g.L * ((uint32_t)y + (uint32_t)g.L * (uint32_t)z);
    const uint32_t gs = (uint32_t)(sample_offset + sample);
    // the spin start of the bit-sliced path: counter (i, gs >> 7, (1 << 24) | replica, 0),
    // bit gs & 31 of output word (gs >> 5) & 3, bit 1 <=> s = -1
    const uint4 o = philox4x32_10(i, gs >> 7, (1u << 24) | (uint32_t)rep, 0u, ks);
    const uint32_t wsel = (gs >> 5) & 3u;
    const uint32_t word = wsel == 0 ? o.x : wsel == 1 ? o.y : wsel == 2 ? o.z : o.w;
    spin[((long long)sys * 2 + p) * g.half + t] = ((word >> (gs & 31u)) & 1u) ? (int8_t)-1 : (int8_t)1;
}

// canonical <-> device layout.  kind 0: spins (int8), 1: daemons (double), 2: bonds (double, blockIdx.y = sample*3+d)
template <typename T, bool TO_DEVICE>
__global__ void __launch_bounds__(256)
gauss_relayout_kernel(T* __restrict__ dev, T* __restrict__ canon, GGeom g)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int p = blockIdx.z;
    int xh, y, z, c;
    if (!site_of(g, t, p, xh, y, z, c)) return;
    const long long N = 2 * g.half;
    const long long i = (long long)(2 * xh + c) + (long long)g.L * ((long long)y + (long long)g.L * z);
    const long long d = ((long long)blockIdx.y * 2 + p) * g.half + t, cidx = (long long)blockIdx.y * N + i;
    if (TO_DEVICE) dev[d] = canon[cidx]; else canon[cidx] = dev[d];
}

__global__ void __launch_bounds__(256)
gauss_validate_spins_kernel(const int8_t* __restrict__ s, long long n, int* bad)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        if (s[i] != 1 && s[i] != -1) *bad = 1;
}

__global__ void __launch_bounds__(256)
gauss_validate_real_kernel(const double* __restrict__ v, long long n, int nonneg, int* bad)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        if (!isfinite(v[i]) || (nonneg && v[i] < 0.0)) *bad = 1;
}

// walkers on the sites of parity p exchange with their neighbour at +sign along axis.
// A pass over all daemon energies (16 B read + 16 B written per thread-site): kWanderSites sites per thread, every
// load issued before the first store, so that enough bytes are in flight to cover the HBM latency (one site per
// thread: 85 us at 64^3 x 64 systems, 3.2 TB/s).  Every pair is touched by exactly one thread.
constexpr int kWanderSites = 4;
__global__ void __launch_bounds__(256)
gauss_wander_kernel(double* __restrict__ nd, GGeom g, int axis, int sign, int p)
{
    const int sys = blockIdx.y, L = g.L, Lh = g.Lh;
    double* const pa = nd + ((long long)sys * 2 + p) * g.half;
    double* const pb = nd + ((long long)sys * 2 + (1 - p)) * g.half;
    long long ia[kWanderSites], ib[kWanderSites];
    double va[kWanderSites], vb[kWanderSites];
#pragma unroll
    for (int k = 0; k < kWanderSites; ++k) {
        const long long t = ((long long)blockIdx.x * kWanderSites + k) * blockDim.x + threadIdx.x;
        int xh, y, z, c;
        ia[k] = -1;
        if (!site_of(g, t, p, xh, y, z, c)) continue;
        int xo = xh, yo = y, zo = z;
        if (axis == 0) { const int d = (sign > 0) ? xh + c : xh + c - 1; xo = (d == Lh) ? 0 : (d < 0 ? Lh - 1 : d); }
        else if (axis == 1) yo = (y + sign + L) % L;
        else zo = (z + sign + L) % L;
        ia[k] = t; ib[k] = ((long long)zo * L + yo) * Lh + xo;
        va[k] = pa[ia[k]]; vb[k] = pb[ib[k]];
    }
#pragma unroll
    for (int k = 0; k < kWanderSites; ++k)
        if (ia[k] >= 0) { pa[ia[k]] = vb[k]; pb[ib[k]] = va[k]; }
}

// E = -sum J s s over the bonds owned by the block's sites, E_daemon = sum n: fixed-shape tree per block, the
// partial sums are added in block order by gauss_finish_kernel (deterministic).  grid = (n_part, n_sys)
__global__ void __launch_bounds__(256)
gauss_measure_kernel(const int8_t* __restrict__ spin, const double* __restrict__ nd, const double* __restrict__ J,
                     GGeom g, int n_replicas, double* __restrict__ part)
{
    __shared__ double sE[256], sD[256];
    const int sys = blockIdx.y, sample = sys / n_replicas;
    const int L = g.L, Lh = g.Lh;
    const long long half = g.half;
    const double* Jb = J + (long long)sample * 6 * half;
    double e = 0.0, d = 0.0;
    for (long long u = (long long)blockIdx.x * blockDim.x + threadIdx.x; u < 2 * half; u += (long long)gridDim.x * blockDim.x) {
        const int p = (u >= half) ? 1 : 0, q = 1 - p;
        const long long t = u - (long long)p * half;
        int xh, y, z, c;
        site_of(g, t, p, xh, y, z, c);
        const int8_t* sq = spin + ((long long)sys * 2 + q) * half;
        const int yp = (y + 1 == L) ? 0 : y + 1, zp = (z + 1 == L) ? 0 : z + 1;
        const int xp = (xh + c == Lh) ? 0 : xh + c;
        const double s0 = (double)spin[((long long)sys * 2 + p) * half + t];
        const double sx = (double)sq[((long long)z * L + y) * Lh + xp];
        const double sy = (double)sq[((long long)z * L + yp) * Lh + xh];
        const double sz = (double)sq[((long long)zp * L + y) * Lh + xh];
        e -= s0 * (Jb[(0 * 2 + p) * half + t] * sx + Jb[(1 * 2 + p) * half + t] * sy + Jb[(2 * 2 + p) * half + t] * sz);
        d += nd[((long long)sys * 2 + p) * half + t];
    }
    sE[threadIdx.x] = e; sD[threadIdx.x] = d;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) { sE[threadIdx.x] += sE[threadIdx.x + o]; sD[threadIdx.x] += sD[threadIdx.x + o]; }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        part[((long long)sys * gridDim.x + blockIdx.x) * 2 + 0] = sE[0];
        part[((long long)sys * gridDim.x + blockIdx.x) * 2 + 1] = sD[0];
    }
}

__global__ void gauss_finish_kernel(const double* __restrict__ part, int n_part, int n_sys, double* __restrict__ out)
{
    const int sys = blockIdx.x * blockDim.x + threadIdx.x;
    if (sys >= n_sys) return;
    double e = 0.0, d = 0.0;
    for (int b = 0; b < n_part; ++b) { e += part[((long long)sys * n_part + b) * 2]; d += part[((long long)sys * n_part + b) * 2 + 1]; }
    out[sys] = e; out[n_sys + sys] = d;
}

// differing spins of replicas (a, b) of a sample: grid = (nblk, n_pairs_total); pair index -> (sample, a, b) on the host
__global__ void __launch_bounds__(256)
gauss_overlap_kernel(const int8_t* __restrict__ spin, long long n, const int* __restrict__ pa, const int* __restrict__ pb,
                     unsigned long long* __restrict__ cnt)
{
    const int8_t* A = spin + (long long)pa[blockIdx.y] * n;
    const int8_t* B = spin + (long long)pb[blockIdx.y] * n;
    unsigned int diff = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        diff += (A[i] != B[i]) ? 1u : 0u;
    diff = __reduce_add_sync(0xFFFFFFFFu, diff);
    if ((threadIdx.x & 31) == 0 && diff) atomicAdd(&cnt[blockIdx.y], (unsigned long long)diff);
}

GGeom ggeom(const micsa_gauss_ctx* c) {
    GGeom g; g.L = c->L; g.Lh = c->Lh; g.half = c->half;
    g.inv_Lh = gdiv_magic((uint32_t)c->Lh); g.inv_L = gdiv_magic((uint32_t)c->L);
    return g;
}
unsigned gblocks(const micsa_gauss_ctx* c) { return (unsigned)((c->half + 255) / 256); }

int greserve(micsa_gauss_ctx* c, size_t bytes) {
    if (bytes > c->stage_bytes) {
        GCK(c, cudaStreamSynchronize(c->stream));
        if (c->stage) cudaFree(c->stage);
        c->stage = nullptr; c->stage_bytes = 0;
        if (cudaMalloc(&c->stage, bytes) != cudaSuccess) {
            cudaGetLastError(); micsa_internal_set_error("out of device memory (staging)", ""); return MICSA_ERR_NOMEM;
        }
        c->stage_bytes = bytes;
    }
    return MICSA_OK;
}

int glaunch_half_sweep(micsa_gauss_ctx* c, int parity) {
    const int V = (c->Lh % 4 == 0) ? 4 : (c->Lh % 2 == 0) ? 2 : 1;
    const dim3 grid((unsigned)((c->half / V + 255) / 256), (unsigned)c->n_sys);
    if (V == 4)      gauss_half_sweep_vec_kernel<4><<<grid, 256, 0, c->stream>>>(c->spin, c->n, c->J, ggeom(c), c->n_replicas, parity);
    else if (V == 2) gauss_half_sweep_vec_kernel<2><<<grid, 256, 0, c->stream>>>(c->spin, c->n, c->J, ggeom(c), c->n_replicas, parity);
    else             gauss_half_sweep_kernel<<<grid, 256, 0, c->stream>>>(c->spin, c->n, c->J, ggeom(c), c->n_replicas, parity);
    GCK(c, cudaGetLastError());
    c->attempts += (uint64_t)c->half * (uint64_t)c->n_sys;
    return MICSA_OK;
}

int glaunch_wander(micsa_gauss_ctx* c, int axis, int sign, int parity) {
    gauss_wander_kernel<<<dim3((gblocks(c) + kWanderSites - 1) / kWanderSites, (unsigned)c->n_sys), 256, 0, c->stream>>>(c->n, ggeom(c), axis, sign, parity);
    GCK(c, cudaGetLastError());
    return MICSA_OK;
}

void gfree(micsa_gauss_ctx* c) {
    if (c->spin) cudaFree(c->spin);
    if (c->n) cudaFree(c->n);
    if (c->J) cudaFree(c->J);
    if (c->part) cudaFree(c->part);
    if (c->qcnt) cudaFree(c->qcnt);
    if (c->stage) cudaFree(c->stage);
    if (c->host_row) cudaFreeHost(c->host_row);
    delete c;
}

}  // namespace

extern "C" {

micsa_gauss_ctx* micsa_gauss_create(int L, int n_samples, int n_replicas, uint64_t seed, int sample_offset,
                                    void* cuda_stream)
{
    if (L < 2 || (L & 1)) { micsa_internal_set_error("L must be even and >= 2", ""); return nullptr; }
    if (n_samples < 1 || n_replicas < 1 || (long long)n_samples * n_replicas > 65535) {
        micsa_internal_set_error("n_samples, n_replicas >= 1 and n_samples * n_replicas <= 65535", ""); return nullptr;
    }
    const long long N = (long long)L * L * L;
    if (N > 0x7FFFFFFFll || sample_offset < 0) { micsa_internal_set_error("L^3 must be below 2^31 and sample_offset >= 0", ""); return nullptr; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError(); micsa_internal_set_error("no usable CUDA device (this library has no CPU fallback)", ""); return nullptr;
    }
    micsa_gauss_ctx* c = new (std::nothrow) micsa_gauss_ctx();
    if (!c) { micsa_internal_set_error("out of host memory", ""); return nullptr; }
    c->L = L; c->Lh = L / 2; c->n_samples = n_samples; c->n_replicas = n_replicas; c->n_sys = n_samples * n_replicas;
    c->n_pairs = n_samples * (n_replicas * (n_replicas - 1) / 2); c->sample_offset = sample_offset;
    c->N = N; c->half = N / 2;
    c->ks = philox_make_keys(seed); c->stream = (cudaStream_t)cuda_stream;
    c->walkers = 0; c->t = 0; c->attempts = c->rns = 0; c->sticky = 0;
    c->stage = nullptr; c->stage_bytes = 0;
    c->n_part = (int)std::min<long long>(64, (N + 4095) / 4096);
    const size_t sys_sites = (size_t)c->n_sys * (size_t)N;
    if (cudaMalloc((void**)&c->spin, sys_sites) != cudaSuccess ||
        cudaMalloc((void**)&c->n, sys_sites * 8) != cudaSuccess ||
        cudaMalloc((void**)&c->J, (size_t)n_samples * 3 * (size_t)N * 8) != cudaSuccess ||
        cudaMalloc((void**)&c->part, (size_t)c->n_sys * c->n_part * 2 * 8 + (size_t)c->n_sys * 2 * 8) != cudaSuccess ||
        cudaMalloc((void**)&c->qcnt, (size_t)std::max(c->n_pairs, 1) * (8 + 8)) != cudaSuccess ||
        cudaHostAlloc((void**)&c->host_row, (size_t)c->n_sys * 2 * 8, cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError(); micsa_internal_set_error("out of device memory", ""); gfree(c); return nullptr;
    }
    cudaMemsetAsync(c->n, 0, sys_sites * 8, c->stream);
    cudaMemsetAsync(c->J, 0, (size_t)n_samples * 3 * (size_t)N * 8, c->stream);
    gauss_init_spins_kernel<<<dim3(gblocks(c), (unsigned)c->n_sys, 2), 256, 0, c->stream>>>(
        c->spin, ggeom(c), n_replicas, sample_offset, c->ks);
    if (cudaGetLastError() != cudaSuccess || cudaStreamSynchronize(c->stream) != cudaSuccess) {
        micsa_internal_set_error("CUDA error while initialising the state", ""); gfree(c); return nullptr;
    }
    return c;
}

int micsa_gauss_destroy(micsa_gauss_ctx* c) {
    if (!c) return MICSA_OK;
    cudaStreamSynchronize(c->stream);
    gfree(c);
    return MICSA_OK;
}

int micsa_gauss_set_couplings(micsa_gauss_ctx* c, const double* J) {
    int rc = gcheck(c); if (rc) return rc;
    if (!J) { micsa_internal_set_error("null pointer", ""); return MICSA_ERR_INVALID; }
    const size_t count = (size_t)c->n_samples * 3 * (size_t)c->N;
    rc = greserve(c, count * 8 + 256); if (rc) return rc;
    int* bad = (int*)((char*)c->stage + count * 8);
    GCK(c, cudaMemcpyAsync(c->stage, J, count * 8, cudaMemcpyHostToDevice, c->stream));
    GCK(c, cudaMemsetAsync(bad, 0, sizeof(int), c->stream));
    gauss_validate_real_kernel<<<256, 256, 0, c->stream>>>((const double*)c->stage, (long long)count, 0, bad);
    int h_bad = 0;
    GCK(c, cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    GCK(c, cudaStreamSynchronize(c->stream));
    if (h_bad) { micsa_internal_set_error("couplings must be finite", ""); return MICSA_ERR_INVALID; }
    gauss_relayout_kernel<double, true><<<dim3(gblocks(c), (unsigned)(c->n_samples * 3), 2), 256, 0, c->stream>>>(
        c->J, (double*)c->stage, ggeom(c));
    GCK(c, cudaGetLastError());
    GCK(c, cudaStreamSynchronize(c->stream));
    return MICSA_OK;
}

int micsa_gauss_set_state(micsa_gauss_ctx* c, const int8_t* s, const double* n) {
    int rc = gcheck(c); if (rc) return rc;
    const size_t count = (size_t)c->n_sys * (size_t)c->N;
    rc = greserve(c, count * 8 + 256); if (rc) return rc;
    int* bad = (int*)((char*)c->stage + count * 8);
    for (int kind = 0; kind < 2; ++kind) {
        const void* src = kind == 0 ? (const void*)s : (const void*)n;
        if (!src) continue;
        const size_t bytes = count * (kind == 0 ? 1 : 8);
        GCK(c, cudaMemcpyAsync(c->stage, src, bytes, cudaMemcpyHostToDevice, c->stream));
        GCK(c, cudaMemsetAsync(bad, 0, sizeof(int), c->stream));
        if (kind == 0) gauss_validate_spins_kernel<<<256, 256, 0, c->stream>>>((const int8_t*)c->stage, (long long)count, bad);
        else           gauss_validate_real_kernel<<<256, 256, 0, c->stream>>>((const double*)c->stage, (long long)count, 1, bad);
        int h_bad = 0;
        GCK(c, cudaMemcpyAsync(&h_bad, bad, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        GCK(c, cudaStreamSynchronize(c->stream));
        if (h_bad) {
            micsa_internal_set_error(kind == 0 ? "spin values must be -1 or +1" : "daemon energies must be finite and >= 0", "");
            return MICSA_ERR_INVALID;
        }
        const dim3 grid(gblocks(c), (unsigned)c->n_sys, 2);
        if (kind == 0) gauss_relayout_kernel<int8_t, true><<<grid, 256, 0, c->stream>>>(c->spin, (int8_t*)c->stage, ggeom(c));
        else           gauss_relayout_kernel<double, true><<<grid, 256, 0, c->stream>>>(c->n, (double*)c->stage, ggeom(c));
        GCK(c, cudaGetLastError());
        GCK(c, cudaStreamSynchronize(c->stream));
    }
    return MICSA_OK;
}

int micsa_gauss_get_state(micsa_gauss_ctx* c, int8_t* s, double* n, double* J) {
    int rc = gcheck(c); if (rc) return rc;
    const size_t count = (size_t)c->n_sys * (size_t)c->N, jcount = (size_t)c->n_samples * 3 * (size_t)c->N;
    rc = greserve(c, std::max(count, jcount) * 8 + 256); if (rc) return rc;
    const dim3 grid(gblocks(c), (unsigned)c->n_sys, 2);
    if (s) {
        gauss_relayout_kernel<int8_t, false><<<grid, 256, 0, c->stream>>>(c->spin, (int8_t*)c->stage, ggeom(c));
        GCK(c, cudaGetLastError());
        GCK(c, cudaMemcpyAsync(s, c->stage, count, cudaMemcpyDeviceToHost, c->stream));
        GCK(c, cudaStreamSynchronize(c->stream));
    }
    if (n) {
        gauss_relayout_kernel<double, false><<<grid, 256, 0, c->stream>>>(c->n, (double*)c->stage, ggeom(c));
        GCK(c, cudaGetLastError());
        GCK(c, cudaMemcpyAsync(n, c->stage, count * 8, cudaMemcpyDeviceToHost, c->stream));
        GCK(c, cudaStreamSynchronize(c->stream));
    }
    if (J) {
        gauss_relayout_kernel<double, false><<<dim3(gblocks(c), (unsigned)(c->n_samples * 3), 2), 256, 0, c->stream>>>(
            c->J, (double*)c->stage, ggeom(c));
        GCK(c, cudaGetLastError());
        GCK(c, cudaMemcpyAsync(J, c->stage, jcount * 8, cudaMemcpyDeviceToHost, c->stream));
        GCK(c, cudaStreamSynchronize(c->stream));
    }
    return MICSA_OK;
}

int micsa_gauss_refresh(micsa_gauss_ctx* c, double T, uint32_t step) {
    int rc = gcheck(c); if (rc) return rc;
    if (!(T > 0.0) || !std::isfinite(T)) { micsa_internal_set_error("temperature must be finite and > 0", ""); return MICSA_ERR_INVALID; }
    gauss_refresh_kernel<<<dim3(gblocks(c), (unsigned)c->n_sys, 2), 256, 0, c->stream>>>(
        c->n, ggeom(c), c->n_replicas, c->sample_offset, c->ks, step, T);
    GCK(c, cudaGetLastError());
    c->rns += (uint64_t)c->N * (uint64_t)c->n_sys;
    return MICSA_OK;
}

int micsa_gauss_half_sweep(micsa_gauss_ctx* c, int parity) {
    int rc = gcheck(c); if (rc) return rc;
    if (parity != 0 && parity != 1) { micsa_internal_set_error("parity must be 0 or 1", ""); return MICSA_ERR_INVALID; }
    return glaunch_half_sweep(c, parity);
}

int micsa_gauss_sweep(micsa_gauss_ctx* c, int n) {
    int rc = gcheck(c); if (rc) return rc;
    if (n < 0) { micsa_internal_set_error("n must be >= 0", ""); return MICSA_ERR_INVALID; }
    for (int k = 0; k < n; ++k) {
        rc = glaunch_half_sweep(c, 0); if (rc) return rc;
        rc = glaunch_half_sweep(c, 1); if (rc) return rc;
        if (c->walkers) { rc = glaunch_wander(c, 0, +1, (int)(c->t & 1)); if (rc) return rc; }
        c->t += 1;
    }
    return MICSA_OK;
}

int micsa_gauss_wander(micsa_gauss_ctx* c, int axis, int sign, int parity) {
    int rc = gcheck(c); if (rc) return rc;
    if (axis < 0 || axis > 2 || (sign != 1 && sign != -1) || (parity != 0 && parity != 1)) {
        micsa_internal_set_error("axis must be 0..2, sign +1 or -1, parity 0 or 1", ""); return MICSA_ERR_INVALID;
    }
    return glaunch_wander(c, axis, sign, parity);
}

int micsa_gauss_set_walkers(micsa_gauss_ctx* c, int mode, int64_t t) {
    int rc = gcheck(c); if (rc) return rc;
    if ((mode != 0 && mode != 1) || t < 0) { micsa_internal_set_error("mode must be 0 or 1 and t >= 0", ""); return MICSA_ERR_INVALID; }
    c->walkers = mode; c->t = t;
    return MICSA_OK;
}

int micsa_gauss_measure(micsa_gauss_ctx* c, double* E, double* Ed, int64_t* Q) {
    int rc = gcheck(c); if (rc) return rc;
    if (Q && c->n_replicas < 2) { micsa_internal_set_error("q_overlap needs n_replicas >= 2", ""); return MICSA_ERR_INVALID; }
    double* out = c->part + (size_t)c->n_sys * c->n_part * 2;
    gauss_measure_kernel<<<dim3((unsigned)c->n_part, (unsigned)c->n_sys), 256, 0, c->stream>>>(
        c->spin, c->n, c->J, ggeom(c), c->n_replicas, c->part);
    gauss_finish_kernel<<<(c->n_sys + 127) / 128, 128, 0, c->stream>>>(c->part, c->n_part, c->n_sys, out);
    GCK(c, cudaGetLastError());
    GCK(c, cudaMemcpyAsync(c->host_row, out, (size_t)c->n_sys * 2 * 8, cudaMemcpyDeviceToHost, c->stream));
    unsigned long long* hq = nullptr;
    if (Q) {
        int* pa = (int*)(c->qcnt + c->n_pairs);
        int* pb = pa + c->n_pairs;
        hq = new (std::nothrow) unsigned long long[(size_t)c->n_pairs * 2];
        if (!hq) { micsa_internal_set_error("out of host memory", ""); return MICSA_ERR_NOMEM; }
        int* ha = (int*)hq; int* hb = ha + c->n_pairs;
        int k = 0;
        for (int sample = 0; sample < c->n_samples; ++sample)
            for (int a = 0; a < c->n_replicas; ++a)
                for (int b = a + 1; b < c->n_replicas; ++b) { ha[k] = sample * c->n_replicas + a; hb[k] = sample * c->n_replicas + b; ++k; }
        cudaError_t e = cudaMemcpyAsync(pa, ha, (size_t)c->n_pairs * 2 * sizeof(int), cudaMemcpyHostToDevice, c->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync(c->qcnt, 0, (size_t)c->n_pairs * 8, c->stream);
        if (e == cudaSuccess) {
            const unsigned nb = (unsigned)std::min<long long>(64, (c->N + 4095) / 4096);
            gauss_overlap_kernel<<<dim3(nb, (unsigned)c->n_pairs), 256, 0, c->stream>>>(c->spin, c->N, pa, pb, c->qcnt);
            e = cudaGetLastError();
        }
        if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);      // ha / hb consumed
        if (e == cudaSuccess) e = cudaMemcpyAsync(hq, c->qcnt, (size_t)c->n_pairs * 8, cudaMemcpyDeviceToHost, c->stream);
        if (e != cudaSuccess) { delete[] hq; GCK(c, e); }
    }
    cudaError_t e = cudaStreamSynchronize(c->stream);
    if (e != cudaSuccess) { delete[] hq; GCK(c, e); }
    if (E)  for (int i = 0; i < c->n_sys; ++i) E[i] = c->host_row[i];
    if (Ed) for (int i = 0; i < c->n_sys; ++i) Ed[i] = c->host_row[c->n_sys + i];
    if (Q) for (int i = 0; i < c->n_pairs; ++i) Q[i] = (int64_t)c->N - 2 * (int64_t)hq[i];
    delete[] hq;
    return MICSA_OK;
}

int micsa_gauss_counters(micsa_gauss_ctx* c, uint64_t* attempts, uint64_t* rns) {
    if (!c) { micsa_internal_set_error("null context", ""); return MICSA_ERR_INVALID; }
    if (attempts) *attempts = c->attempts;
    if (rns) *rns = c->rns;
    return MICSA_OK;
}

int micsa_gauss_synchronize(micsa_gauss_ctx* c) {
    int rc = gcheck(c); if (rc) return rc;
    GCK(c, cudaStreamSynchronize(c->stream));
    return MICSA_OK;
}

}  // extern "C"
