// micsa.cu -- context management and the C ABI of include/micsa.h.
// Every step of the path runs in the kernels of sweep.cuh / refresh.cuh /
// measure.cuh; this file only validates arguments, sizes grids and queues
// launches on the context's stream.  There is no CPU fallback.
#include "../../include/micsa.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <mutex>
#include <new>
#include <vector>

#include "layout.cuh"
#include "measure.cuh"
#include "c4.cuh"
#include "metropolis.cuh"
#include "pack.cuh"
#include "philox.cuh"
#include "refresh.cuh"
#include "small.cuh"
#include "sweep.cuh"
#include "wander.cuh"

using namespace micsa;

namespace {

thread_local char g_err[256] = "";

void set_err(const char* fmt, const char* detail = "") {
    snprintf(g_err, sizeof g_err, fmt, detail);
}

}  // namespace

// ---- scratch of micsa_measure_noalloc (include/micsa.h): counters + ticket of the measurement kernels ----
// Lives in the module image: every GPU that loads the library holds these 128.25 KiB until exit, and every
// context on a device shares them.  In HOST code the name below is a host-side stand-in, not a device address;
// noalloc_scratch() asks the runtime for the address on the current device (cudaGetSymbolAddress) once per
// device and that pointer is what the kernels get.
constexpr size_t kNoAllocCounters = MICSA_NOALLOC_MAX_COUNTERS;     // 64-bit lane counters (cntU | cntM | cntX)
constexpr size_t kNoAllocTicket = 32;                               // one 256-byte line for the ticket word
static __device__ __align__(256) unsigned long long g_noalloc_scratch[kNoAllocCounters + kNoAllocTicket];

namespace {

// device address of g_noalloc_scratch on the CURRENT device; queried once per device ordinal
cudaError_t noalloc_scratch(unsigned long long** out) {
    constexpr int kMaxDev = 64;
    static std::mutex mu;
    static unsigned long long* cache[kMaxDev] = {};
    *out = nullptr;
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    std::lock_guard<std::mutex> lock(mu);
    if (dev >= 0 && dev < kMaxDev && cache[dev]) { *out = cache[dev]; return cudaSuccess; }
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < kMaxDev) cache[dev] = (unsigned long long*)p;
    *out = (unsigned long long*)p;
    return cudaSuccess;
}

}  // namespace

// for the other translation units of the library (gauss.cu): the same thread-local message
void micsa_internal_set_error(const char* fmt, const char* detail) { snprintf(g_err, sizeof g_err, fmt, detail); }

namespace {

constexpr size_t kAlign = 256;
size_t align_up(size_t x) { return (x + kAlign - 1) / kAlign * kAlign; }

struct Plan {                 // byte offsets inside the workspace
    size_t spin, m0, m1, m0s, m1s, J, cnt, ticket, row, minE, bad, calls, total;
    size_t plane_bytes, J_bytes, cnt_words, row_len;
};

bool make_geom(int L, int n_samples, int n_replicas, int sample_offset, Geom& g) {
    if (L < 2 || (L & 1)) { set_err("L must be even and >= 2"); return false; }
    if (n_samples < 1 || n_replicas < 1) { set_err("n_samples and n_replicas must be >= 1"); return false; }
    if (sample_offset < 0 || (sample_offset & 15)) { set_err("sample_offset must be a non-negative multiple of 16"); return false; }
    const long long N = (long long)L * L * L;
    if (N > 0x7FFFFFFFll) { set_err("L^3 must be below 2^31 (32-bit site index and byte offsets inside a parity array)"); return false; }
    if ((long long)n_samples * n_replicas > (1ll << 24) || n_replicas >= (1 << 20)) {
        set_err("too many systems"); return false;
    }
    if ((long long)n_replicas * (n_replicas - 1) / 2 > 65535) {      // gridDim.z of the replica-pair counting kernel
        set_err("too many replica pairs per sample (n_replicas <= 362)"); return false;
    }
    if ((long long)sample_offset + n_samples > 0x7FFFFFFFll) { set_err("sample index overflow"); return false; }
    g.L = L; g.Lh = L / 2;
    g.n_samples = n_samples; g.n_replicas = n_replicas; g.sample_offset = sample_offset;
    g.rpw = (n_replicas % 2 == 0) ? 2 : 1;
    g.spw = 32 / g.rpw;
    g.n_sg = (n_samples + g.spw - 1) / g.spw;
    g.n_rg = n_replicas / g.rpw;
    if ((long long)g.n_sg * g.n_rg * 2 > 65535 || (long long)g.n_sg * 6 > 65535) {
        set_err("too many word lattices for one grid"); return false;
    }
    g.n_words = g.n_sg * g.n_rg;
    g.half = (long long)L * L * g.Lh;
    g.N = N;
    g.n_sys = n_samples * n_replicas;
    g.n_pairs = n_samples * (n_replicas * (n_replicas - 1) / 2);
    return true;
}

Plan make_plan(const Geom& g) {
    Plan p;
    p.plane_bytes = (size_t)g.n_words * 2 * g.half * sizeof(uint32_t);
    p.J_bytes = (size_t)g.n_sg * 6 * g.half * (g.rpw == 2 ? 2 : 4);
    const int pps = g.n_replicas * (g.n_replicas - 1) / 2;
    p.cnt_words = (size_t)g.n_words * 32 * 2 + (size_t)g.n_sg * pps * 32;
    p.row_len = (size_t)2 * g.n_sys + g.n_pairs;
    size_t o = 0;
    p.spin = o; o += align_up(p.plane_bytes);
    p.m0 = o;   o += align_up(p.plane_bytes);
    p.m1 = o;   o += align_up(p.plane_bytes);
    p.m0s = o;  o += align_up(p.plane_bytes);      // staging planes of a prefetched refresh
    p.m1s = o;  o += align_up(p.plane_bytes);
    p.J = o;    o += align_up(p.J_bytes);
    p.cnt = o;  o += align_up(p.cnt_words * 8);
    p.ticket = o; o += align_up(sizeof(unsigned int));
    p.row = o;  o += align_up(p.row_len * 8);
    p.minE = o; o += align_up((size_t)g.n_sys * 8);
    p.bad = o;  o += align_up(sizeof(int));
    p.calls = o; o += align_up(sizeof(unsigned long long));
    p.total = o;
    return p;
}

int vec_width(int Lh) { return (Lh % 4 == 0) ? 4 : (Lh % 2 == 0) ? 2 : 1; }

}  // namespace

struct micsa_ctx {
    Geom g;
    Plan plan;
    State st;
    PhiloxKeys ks;
    uint64_t seed;
    cudaStream_t stream;
    char* ws;
    bool owns_ws;
    unsigned long long* cnt;
    unsigned int* ticket;
    long long* row;
    long long* minE;
    int* bad;
    uint32_t* m0s; uint32_t* m1s;             // staging planes (swapped with st.m0/m1 when consumed)
    cudaStream_t side;                        // generates prefetched refreshes under the sweeps
    bool side_below;                          // the context's stream has a higher priority than the side stream
    unsigned long long* noalloc;              // device address of g_noalloc_scratch on this context's device (or null)
    char* chain_buf;                          // refreshed planes of chained small-lattice steps (micsa_anneal), or null
    cudaEvent_t ev_main, ev_side;
    bool pending; double pending_T; uint32_t pending_step;
    bool measure_queued;                      // micsa_measure_begin without its _end yet
    void* stage_dev; size_t stage_bytes;      // canonical-layout staging of set_* / get_state (grow-only)
    void* trace_dev; size_t trace_bytes;      // measurement rows of micsa_anneal (grow-only)
    void* c4_dev; size_t c4_bytes;            // overlap field + counters of micsa_measure_c4 (grow-only)
    unsigned long long* c4_host; size_t c4_host_bytes;   // pinned read-back of the C4 counters
    long long* host_row;        // pinned host staging for one measurement row
    unsigned long long* calls;  // Philox calls made by the refresh kernels (device counter)
    int V;
    int sweep_kernel;          // L % 8 == 0: 1 = row-marching, 2 = pipelined row-marching
    int sms;                   // multiprocessors of the device (grid sizing)
    int gamma;                 // daemon families per spin; family 0 lives in st.m0/m1
    int sel;                   // family that set_daemons / get_state address
    std::vector<uint32_t*> xm0, xm1;   // families 1 .. gamma-1 (library-owned)
    std::vector<uint32_t*> xm0s, xm1s; // their staging planes for a prefetched refresh (allocated at the first one)
    int l2_groups;             // run multi-sweep calls lattice group by lattice group when the state exceeds L2
    bool small_attr_set;       // small lattices: kernel attributes (shared memory size, cluster size) set
    int small_items;           // small lattices: quad rows per CTA aimed at (0 = default)
    int small_path;            // small lattices: whole groups of sweeps (+ refresh, + rows) in one cluster launch
    int fuse_walk;             // walkers: exchange inside the odd half-sweep instead of a separate kernel
    int walkers;               // 0 = daemons stay on their site, 1 = one forward-X walker per spin
    long long t;               // time index (timesteps = sweeps done since create / micsa_set_time)
    int fuse_measure;          // count the observables inside the last sweep of a measured group
    int pipe_planes;           // planes per CTA of the pipelined kernel (1 or 4)
    int use_pdl;               // programmatic dependent launch for the pipelined kernel
    int pipe_rows;             // rows per thread of the pipelined kernel (4 or 8)
    uint64_t attempts, rns, launches;
    cudaError_t launch_err;    // first failed cudaLaunchKernelEx since the last post_launch()
    int sticky;
};

namespace {

#define CK(ctx, call)                                                          \
    do {                                                                       \
        cudaError_t e_ = (call);                                               \
        if (e_ != cudaSuccess) {                                               \
            set_err("CUDA error: %s", cudaGetErrorString(e_));                 \
            if (ctx) (ctx)->sticky = MICSA_ERR_CUDA;                           \
            return MICSA_ERR_CUDA;                                             \
        }                                                                      \
    } while (0)

int check_ctx(micsa_ctx* c) {
    if (!c) { set_err("null context"); return MICSA_ERR_INVALID; }
    if (c->sticky) { set_err("context is in a sticky CUDA error state"); return c->sticky; }
    return MICSA_OK;
}

SiteGrid site_grid(const Geom& g) {
    SiteGrid s; s.L = g.L; s.Lh = g.Lh; s.n_rg = g.n_rg; s.n_samples = g.n_samples;
    s.sample_offset = g.sample_offset; s.half = g.half; s.inv_Lh = fastdiv_magic((uint32_t)g.Lh);
    return s;
}

dim3 site_blocks(const Geom& g, int nz) {
    return dim3((unsigned)((g.L * g.Lh + 127) / 128), (unsigned)g.L, (unsigned)nz);
}

int post_launch(micsa_ctx* c, int n = 1) {
    c->launches += (uint64_t)n;
    if (c->launch_err != cudaSuccess) { const cudaError_t e = c->launch_err; c->launch_err = cudaSuccess; cudaGetLastError(); CK(c, e); }
    CK(c, cudaGetLastError());
    return MICSA_OK;
}

// ---- launches -----------------------------------------------------------
template <int V, int RPW>
void launch_half_sweep_t(micsa_ctx* c, int parity) {
    SweepArgs a;
    a.spin = c->st.spin; a.m0 = c->st.m0; a.m1 = c->st.m1; a.J = c->st.J;
    a.L = c->g.L; a.Lh = c->g.Lh; a.n_rg = c->g.n_rg; a.half = c->g.half; a.w0 = 0; a.inv_nxv = fastdiv_magic((uint32_t)c->g.Lh / 4u); a.inv_pp = 0u;
    const int per_plane = c->g.L * (c->g.Lh / V);
    dim3 grid((unsigned)((per_plane + 127) / 128), (unsigned)c->g.L, (unsigned)c->g.n_words);
    half_sweep_kernel<V, RPW><<<grid, 128, 0, c->stream>>>(a, parity);
}

constexpr int kRowsPerThread = 4;

template <int RPW>
void launch_half_sweep_rows(micsa_ctx* c, int parity) {
    SweepArgs a;
    a.spin = c->st.spin; a.m0 = c->st.m0; a.m1 = c->st.m1; a.J = c->st.J;
    a.L = c->g.L; a.Lh = c->g.Lh; a.n_rg = c->g.n_rg; a.half = c->g.half; a.w0 = 0; a.inv_nxv = fastdiv_magic((uint32_t)c->g.Lh / 4u); a.inv_pp = 0u;
    const int per_plane = (c->g.L / kRowsPerThread) * (c->g.Lh / 4);
    dim3 grid((unsigned)((per_plane + 127) / 128), (unsigned)c->g.L, (unsigned)c->g.n_words);
    half_sweep_rows_kernel<RPW, kRowsPerThread><<<grid, 128, 0, c->stream>>>(a, parity);
}

// dir != 0 (odd launches of walker timesteps): the launch also does the wandering exchange
// a failed launch is remembered on the context and reported by the next post_launch()
#define LK(call) do { const cudaError_t e_ = (call); if (e_ != cudaSuccess && c->launch_err == cudaSuccess) c->launch_err = e_; } while (0)

template <int RPW>
void launch_half_sweep_pipe(micsa_ctx* c, int parity, int dir = 0, int w0 = 0, int nw = -1) {
    SweepArgs a;
    a.spin = c->st.spin; a.m0 = c->st.m0; a.m1 = c->st.m1; a.J = c->st.J;
    a.L = c->g.L; a.Lh = c->g.Lh; a.n_rg = c->g.n_rg; a.half = c->g.half; a.w0 = w0; a.inv_nxv = fastdiv_magic((uint32_t)c->g.Lh / 4u); a.inv_pp = 0u;
    const unsigned gz = (unsigned)(nw < 0 ? c->g.n_words : nw);
    const int yc = c->pipe_rows;
    const int per_plane = (c->g.L / yc) * (c->g.Lh / 4);
    const int zw = c->pipe_planes;
    // zw == 1: the planes of one parity class of z in one index space (sweep.cuh, pipe_item)
    dim3 grid = (zw == 4) ? dim3((unsigned)((per_plane + 31) / 32), (unsigned)(c->g.L / 4), gz)
                          : dim3((unsigned)(((long long)(c->g.L / 2) * per_plane + 127) / 128), 2u, gz);
    a.inv_pp = fastdiv_magic((uint32_t)per_plane);
    // programmatic dependent launch (the kernel waits with griddepcontrol.wait before
    // its first load): launch latency and ramp overlap the previous grid's tail
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = c->use_pdl ? 1 : 0;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (dir != 0) {                                  // 4 rows per thread only (grid was sized for yc; redo it)
        const int pp4 = (c->g.L / 4) * (c->g.Lh / 4);
        cfg.gridDim = (zw == 4) ? dim3((unsigned)((pp4 + 31) / 32), (unsigned)(c->g.L / 4), gz)
                                : dim3((unsigned)(((long long)(c->g.L / 2) * pp4 + 127) / 128), 2u, gz);
        a.inv_pp = fastdiv_magic((uint32_t)pp4);
        // dir = +-1: along X; +-2: along Y; +-3: along Z (Y and Z share the DIR = +-2 kernels)
        const int axis = (dir > 0 ? dir : -dir) - 1, walk_z = (axis == 2) ? 1 : 0;
        if (axis == 0) {
            if (zw == 4) {
                if (dir > 0) LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 4, +1>, a, parity, 0));
                else         LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 4, -1>, a, parity, 0));
            } else {
                if (dir > 0) LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 1, +1>, a, parity, 0));
                else         LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 1, -1>, a, parity, 0));
            }
        } else {
            if (zw == 4) {
                if (dir > 0) LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 4, +2>, a, parity, walk_z));
                else         LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 4, -2>, a, parity, walk_z));
            } else {
                if (dir > 0) LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 1, +2>, a, parity, walk_z));
                else         LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 1, -2>, a, parity, walk_z));
            }
        }
    } else if (zw == 4) {
        if (yc == 8) LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 8, 4>, a, parity, 0));
        else         LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 4>, a, parity, 0));
    } else {
        if (yc == 8) LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 8, 1>, a, parity, 0));
        else         LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_kernel<RPW, 4, 1>, a, parity, 0));
    }
}

int launch_half_sweep(micsa_ctx* c, int parity) {
    const int key = c->V * 10 + c->g.rpw;
    switch (key) {
        case 41: if (c->sweep_kernel == 2) launch_half_sweep_pipe<1>(c, parity);      // L % 8 == 0
                 else launch_half_sweep_rows<1>(c, parity);
                 break;
        case 42: if (c->sweep_kernel == 2) launch_half_sweep_pipe<2>(c, parity);
                 else launch_half_sweep_rows<2>(c, parity);
                 break;
        case 21: launch_half_sweep_t<2, 1>(c, parity); break;
        case 22: launch_half_sweep_t<2, 2>(c, parity); break;
        case 11: launch_half_sweep_t<1, 1>(c, parity); break;
        default: launch_half_sweep_t<1, 2>(c, parity); break;
    }
    c->attempts += (uint64_t)(c->g.N / 2) * (uint64_t)c->g.n_sys;
    return post_launch(c);
}

int launch_wander(micsa_ctx* c, int axis, int sign, int parity) {
    WanderArgs a;
    a.m0 = c->st.m0; a.m1 = c->st.m1; a.L = c->g.L; a.Lh = c->g.Lh; a.half = c->g.half;
    wander_kernel<<<site_blocks(c->g, c->g.n_words), 128, 0, c->stream>>>(a, axis, sign, parity);
    return post_launch(c);
}

int launch_plain_sweeps(micsa_ctx* c, int n);

// n timesteps (PAPER.md:208-217 step 3 with gamma = 1): a sweep, then -- for
// walkers -- the half of the wandering cycle given by the parity of the time
// index, then t += 1.  Without walkers: n sweeps back to back.
// the wandering can ride on the odd half-sweep (sweep.cuh exchange_walkers) with the pipelined kernel
bool fused_walk(const micsa_ctx* c) { return c->walkers && c->fuse_walk && c->V == 4 && c->sweep_kernel == 2; }

int launch_sweeps(micsa_ctx* c, int n) {
    if (n <= 0) return MICSA_OK;
    if (c->gamma > 1) {                         // a timestep = gamma sweeps, the alpha-th with family alpha
        static const int kAxis[6] = { 0, 1, 2, 0, 1, 2 }, kSign[6] = { +1, +1, +1, -1, -1, -1 };   // Eq. (13)
        uint32_t* const h0 = c->st.m0; uint32_t* const h1 = c->st.m1;
        int rc = MICSA_OK;
        for (int k = 0; k < n && rc == MICSA_OK; ++k) {
            for (int alpha = 0; alpha < c->gamma && rc == MICSA_OK; ++alpha) {
                c->st.m0 = alpha == 0 ? h0 : c->xm0[alpha - 1];
                c->st.m1 = alpha == 0 ? h1 : c->xm1[alpha - 1];
                if (fused_walk(c)) {
                    // the family's own odd half-sweep does its exchange: sources (parity t & 1) swap with their
                    // +sign*axis neighbour, i.e. an odd site with +sign*axis if t is odd, else with -sign*axis
                    rc = launch_half_sweep(c, 0); if (rc) break;
                    const int dir = ((c->t & 1) ? kSign[alpha] : -kSign[alpha]) * (kAxis[alpha] + 1);
                    if (c->g.rpw == 2) launch_half_sweep_pipe<2>(c, 1, dir); else launch_half_sweep_pipe<1>(c, 1, dir);
                    c->attempts += (uint64_t)(c->g.N / 2) * (uint64_t)c->g.n_sys;
                    rc = post_launch(c);
                } else {
                    rc = launch_plain_sweeps(c, 1);
                }
            }
            if (c->walkers && !fused_walk(c)) {     // PAPER.md:204 Eq. (13): family alpha -> its wandering direction
                for (int alpha = 0; alpha < c->gamma && rc == MICSA_OK; ++alpha) {
                    c->st.m0 = alpha == 0 ? h0 : c->xm0[alpha - 1];
                    c->st.m1 = alpha == 0 ? h1 : c->xm1[alpha - 1];
                    rc = launch_wander(c, kAxis[alpha], kSign[alpha], (int)(c->t & 1));
                }
            }
            c->t += 1;
        }
        c->st.m0 = h0; c->st.m1 = h1;
        return rc;
    }
    if (!c->walkers) { c->t += n; return launch_plain_sweeps(c, n); }
    for (int k = 0; k < n; ++k) {
        if (fused_walk(c)) {
            // sources of parity t & 1 exchange with their +X neighbour: seen from the odd sites the
            // partner is x+1 when they are the sources (t odd), x-1 when the even sites are (t even)
            int rc = launch_half_sweep(c, 0); if (rc) return rc;
            const int dir = (c->t & 1) ? +1 : -1;
            if (c->g.rpw == 2) launch_half_sweep_pipe<2>(c, 1, dir); else launch_half_sweep_pipe<1>(c, 1, dir);
            c->attempts += (uint64_t)(c->g.N / 2) * (uint64_t)c->g.n_sys;
            rc = post_launch(c); if (rc) return rc;
        } else {
            int rc = launch_plain_sweeps(c, 1); if (rc) return rc;
            rc = launch_wander(c, 0, +1, (int)(c->t & 1)); if (rc) return rc;
        }
        c->t += 1;
    }
    return MICSA_OK;
}

// n full sweeps (even, odd, even, ...)
int launch_plain_sweeps(micsa_ctx* c, int n) {
    if (n <= 0) return MICSA_OK;
    const Geom& g = c->g;
    // State larger than L2 (config 5: 201 MB): lattices never interact, so run all n sweeps on a group of
    // lattices that fits in L2 before touching the next group -- each group is read from HBM once per call
    // instead of once per half-sweep.
    if (n >= 2 && c->l2_groups && c->V == 4 && c->sweep_kernel == 2 && g.n_words > 1) {
        const double per_lattice = (double)g.N * (12.0 + 3.0 * (g.rpw == 2 ? 2 : 4) / g.n_rg);
        const int fit = (int)std::max(1.0, 96e6 / per_lattice);
        if (fit < g.n_words) {
            const int n_groups = (g.n_words + fit - 1) / fit, per = (g.n_words + n_groups - 1) / n_groups;
            for (int w0 = 0; w0 < g.n_words; w0 += per) {
                const int nw = std::min(per, g.n_words - w0);
                for (int t = 0; t < n; ++t)
                    for (int parity = 0; parity < 2; ++parity) {
                        if (g.rpw == 2) launch_half_sweep_pipe<2>(c, parity, 0, w0, nw);
                        else            launch_half_sweep_pipe<1>(c, parity, 0, w0, nw);
                        const int rc = post_launch(c); if (rc) return rc;
                    }
            }
            c->attempts += (uint64_t)n * (uint64_t)g.N * (uint64_t)g.n_sys;
            return MICSA_OK;
        }
    }
    for (int t = 0; t < n; ++t) {
        int rc = launch_half_sweep(c, 0); if (rc) return rc;
        rc = launch_half_sweep(c, 1); if (rc) return rc;
    }
    return MICSA_OK;
}

// raw generator output for the pins of tests/ (R8, pin P6)
__global__ void debug_philox_kernel(const uint4* ctr, uint4* out, int n, PhiloxKeys ks) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = philox4x32_10(ctr[i].x, ctr[i].y, ctr[i].z, ctr[i].w, ks);
}

int thresholds_host(double T, uint64_t thr[3]) {
    if (!(T > 0.0) || !std::isfinite(T)) return MICSA_ERR_INVALID;
    // DESIGN.md R7: cumulative Eq. (11) in float64, this operation order
    const double x = std::exp(-4.0 / T);
    const double x2 = x * x;
    const double x3 = x2 * x;
    const double Z = ((1.0 + x) + x2) + x3;
    const double cdf[3] = { 1.0 / Z, (1.0 + x) / Z, ((1.0 + x) + x2) / Z };
    for (int k = 0; k < 3; ++k) {
        double t = std::floor(std::ldexp(cdf[k], 32));
        if (t > 4294967296.0) t = 4294967296.0;
        thr[k] = (uint64_t)t;
    }
    return MICSA_OK;
}

int metropolis_thresholds_host(double T, uint64_t thr[3]) {
    if (!(T > 0.0) || !std::isfinite(T)) return MICSA_ERR_INVALID;
    // Boltzmann factors of dH = 4, 8, 12 in float64, this operation order (metropolis.cuh)
    const double x = std::exp(-4.0 / T);
    const double x2 = x * x;
    const double x3 = x2 * x;
    const double p[3] = { x, x2, x3 };
    for (int k = 0; k < 3; ++k) {
        double t = std::floor(std::ldexp(p[k], 32));
        if (t > 4294967296.0) t = 4294967296.0;
        thr[k] = (uint64_t)t;
    }
    return MICSA_OK;
}

RefreshThr make_thr(const uint64_t thr[3]) {
    RefreshThr rt;
    for (int k = 0; k < 3; ++k) {
        rt.never[k] = (thr[k] >> 32) ? 1u : 0u;
        for (int p = 0; p < 32; ++p) rt.tb[k][p] = ((thr[k] >> (31 - p)) & 1u) ? 0xFFFFFFFFu : 0u;
    }
    return rt;
}

int launch_metropolis_half_sweep(micsa_ctx* c, const RefreshThr& rt, uint32_t tau, int parity) {
    const Geom& g = c->g;
    MetropolisArgs a;
    a.spin = c->st.spin; a.J = c->st.J; a.L = g.L; a.Lh = g.Lh; a.n_rg = g.n_rg;
    a.n_samples = g.n_samples; a.sample_offset = g.sample_offset; a.half = g.half; a.inv_Lh = fastdiv_magic((uint32_t)g.Lh);
    dim3 grid = site_blocks(g, g.n_words);
    grid.x = (grid.x + kMetroSub - 1) / kMetroSub;           // kMetroSub groups of 128 words per block
    if (g.rpw == 2) metropolis_half_sweep_kernel<2><<<grid, 128, 0, c->stream>>>(a, parity, c->ks, tau, rt, c->calls);
    else            metropolis_half_sweep_kernel<1><<<grid, 128, 0, c->stream>>>(a, parity, c->ks, tau, rt, c->calls);
    c->attempts += (uint64_t)(g.N / 2) * (uint64_t)g.n_sys;
    c->rns += (uint64_t)(g.N / 2) * (uint64_t)g.n_sys;
    return post_launch(c);
}

int launch_refresh_into(micsa_ctx* c, double T, uint32_t step, uint32_t* m0, uint32_t* m1,
                        cudaStream_t stream, int alpha = 0) {
    uint64_t thr[3];
    if (thresholds_host(T, thr) != MICSA_OK || thr[0] == 0) {
        set_err("temperature must be finite and > 0"); return MICSA_ERR_INVALID;
    }
    RefreshThr rt;
    for (int k = 0; k < 3; ++k) {
        rt.never[k] = (thr[k] >> 32) ? 1u : 0u;           // 2^32: level k+1 has probability < 2^-32
        for (int p = 0; p < 32; ++p) rt.tb[k][p] = ((thr[k] >> (31 - p)) & 1u) ? 0xFFFFFFFFu : 0u;
    }
    const SiteGrid sg = site_grid(c->g);
    dim3 grid = site_blocks(c->g, c->g.n_words * 2);
    grid.x = (grid.x + kRefreshSub - 1) / kRefreshSub;       // kRefreshSub groups of 128 words per block
    if (c->g.rpw == 2)
        refresh_kernel<2><<<grid, 128, 0, stream>>>(m0, m1, sg, c->ks, step, rt, c->calls, (uint32_t)alpha << 20);
    else
        refresh_kernel<1><<<grid, 128, 0, stream>>>(m0, m1, sg, c->ks, step, rt, c->calls, (uint32_t)alpha << 20);
    return post_launch(c);
}

// Refresh (T, step) on the context's stream.  If exactly this refresh was
// prefetched, its planes are already (being) generated on the side stream:
// wait for them and swap the plane pointers -- the old levels are thrown away
// anyway.
uint32_t* family_m0(micsa_ctx* c, int alpha) { return alpha == 0 ? c->st.m0 : c->xm0[alpha - 1]; }
uint32_t* family_m1(micsa_ctx* c, int alpha) { return alpha == 0 ? c->st.m1 : c->xm1[alpha - 1]; }

int launch_refresh(micsa_ctx* c, double T, uint32_t step) {
    const uint64_t drawn = (uint64_t)c->gamma * (uint64_t)c->g.N * (uint64_t)c->g.n_sys;
    if (c->pending && c->pending_step == step && memcmp(&c->pending_T, &T, sizeof T) == 0) {
        CK(c, cudaStreamWaitEvent(c->stream, c->ev_side, 0));
        std::swap(c->st.m0, c->m0s);
        std::swap(c->st.m1, c->m1s);
        for (int alpha = 1; alpha < c->gamma; ++alpha) {
            std::swap(c->xm0[alpha - 1], c->xm0s[alpha - 1]);
            std::swap(c->xm1[alpha - 1], c->xm1s[alpha - 1]);
        }
        c->pending = false;
    } else {                                    // every family in place, its index in the counter
        for (int alpha = 0; alpha < c->gamma; ++alpha) {
            const int rc = launch_refresh_into(c, T, step, family_m0(c, alpha), family_m1(c, alpha), c->stream, alpha);
            if (rc) return rc;
        }
    }
    c->rns += drawn;
    return MICSA_OK;
}

// Queue the generation of refresh (T, step) into the staging planes (of every
// family) on the side stream; it starts once the main stream has reached this
// point (everything that still reads the staging planes' previous role has
// finished).
int launch_prefetch(micsa_ctx* c, double T, uint32_t step) {
    uint64_t thr[3];
    if (thresholds_host(T, thr) != MICSA_OK || thr[0] == 0) {
        set_err("temperature must be finite and > 0"); return MICSA_ERR_INVALID;
    }
    while ((int)c->xm0s.size() < c->gamma - 1) {
        void* a = nullptr; void* b = nullptr;
        if (cudaMalloc(&a, c->plan.plane_bytes) != cudaSuccess || cudaMalloc(&b, c->plan.plane_bytes) != cudaSuccess) {
            cudaGetLastError(); if (a) cudaFree(a); set_err("out of device memory (daemon family staging)"); return MICSA_ERR_NOMEM;
        }
        c->xm0s.push_back((uint32_t*)a); c->xm1s.push_back((uint32_t*)b);
    }
    CK(c, cudaEventRecord(c->ev_main, c->stream));
    CK(c, cudaStreamWaitEvent(c->side, c->ev_main, 0));
    for (int alpha = 0; alpha < c->gamma; ++alpha) {
        const int rc = launch_refresh_into(c, T, step, alpha == 0 ? c->m0s : c->xm0s[alpha - 1],
                                           alpha == 0 ? c->m1s : c->xm1s[alpha - 1], c->side, alpha);
        if (rc) return rc;
    }
    CK(c, cudaEventRecord(c->ev_side, c->side));
    c->pending = true; c->pending_T = T; c->pending_step = step;
    return MICSA_OK;
}

unsigned count_blocks(const micsa_ctx* c, long long nvec, long long other) {
    long long nb = (nvec + kCountBlock * 16 - 1) / (kCountBlock * 16);
    const long long cap = std::max<long long>(1, ((long long)c->sms * 8) / std::max<long long>(1, other));
    nb = std::min(nb, cap);
    const long long need = (nvec + (long long)kCountBlock * 4096 - 1) / ((long long)kCountBlock * 4096);
    nb = std::max<long long>(std::max<long long>(nb, need), 1);
    return (unsigned)nb;
}

template <int V, int RPW>
void launch_measure_t(micsa_ctx* c, const MeasureArgs& a, const FinalizeArgs& f) {
    const Geom& g = c->g;
    const int pps = g.n_replicas * (g.n_replicas - 1) / 2;
    const bool pair_in_word = (g.n_replicas == 2);          // then RPW == 2
    if (pps > 0 && !pair_in_word) {
        count_xor_kernel<V, RPW><<<dim3(count_blocks(c, 2 * g.half / V, (long long)g.n_sg * pps),
                                        (unsigned)g.n_sg, (unsigned)pps),
                                   kCountBlock, 0, c->stream>>>(a);
        c->launches += 1;
    }
    // two resident blocks per SM over all word lattices, never more than
    // kMeasureMaxItems items per thread (10-plane per-thread counters)
    const long long n_items = 2 * g.half / V;
    long long nb = (n_items + (long long)kMeasureBlock * 4 - 1) / ((long long)kMeasureBlock * 4);
    nb = std::min(nb, std::max<long long>(1, ((long long)c->sms * 2) / g.n_words));
    const long long need = (n_items + (long long)kMeasureBlock * kMeasureMaxItems - 1) / ((long long)kMeasureBlock * kMeasureMaxItems);
    nb = std::max<long long>(std::max<long long>(nb, need), 1);
    const dim3 grid((unsigned)nb, (unsigned)g.n_words);
    if (RPW == 2 && pair_in_word) measure_kernel<V, RPW, true><<<grid, kMeasureBlock, 0, c->stream>>>(a, f);
    else                          measure_kernel<V, RPW, false><<<grid, kMeasureBlock, 0, c->stream>>>(a, f);
}

// one measurement: exact sums into the device row `row`, optional min fold.
// The counters are zero on entry (create, and the finalising block re-zeroes).
void make_measure_args(micsa_ctx* c, long long* row, bool fold_min, MeasureArgs& a, FinalizeArgs& f) {
    const Geom& g = c->g;
    a.spin = c->st.spin; a.m0 = c->st.m0; a.m1 = c->st.m1; a.J = c->st.J;
    a.L = g.L; a.Lh = g.Lh; a.n_rg = g.n_rg; a.n_replicas = g.n_replicas; a.n_samples = g.n_samples;
    a.half = g.half;
    a.cntU = c->cnt; a.cntM = c->cnt + (size_t)g.n_words * 32; a.cntX = c->cnt + (size_t)g.n_words * 64;
    f.cntU = a.cntU; f.cntM = a.cntM; f.cntX = a.cntX;
    f.cnt_words = (long long)c->plan.cnt_words; f.ticket = c->ticket;
    f.row = row; f.min_E = fold_min ? c->minE : nullptr;
    f.n_samples = g.n_samples; f.n_replicas = g.n_replicas; f.n_rg = g.n_rg;
    f.rpw = g.rpw; f.spw = g.spw; f.pairs_per_sample = g.n_replicas * (g.n_replicas - 1) / 2;
    f.N = g.N;
}

int launch_measure(micsa_ctx* c, long long* row, bool fold_min) {
    const Geom& g = c->g;
    if (g.n_replicas * (g.n_replicas - 1) / 2 > 65535) { set_err("too many replica pairs"); return MICSA_ERR_INVALID; }
    MeasureArgs a; FinalizeArgs f;
    make_measure_args(c, row, fold_min, a, f);
    for (int alpha = 1; alpha < c->gamma; ++alpha) {        // E_daemon sums over the families
        const long long n = 2 * g.half;
        long long nbl = std::min<long long>((n + kCountBlock * 64 - 1) / (kCountBlock * 64), std::max(1, 4 * c->sms / g.n_words));
        // 16-plane per-thread counters, up to 3 per word: at most 16384 words per thread
        nbl = std::max<long long>(nbl, (n + (long long)kCountBlock * 16384 - 1) / ((long long)kCountBlock * 16384));
        const unsigned nb = (unsigned)std::max<long long>(1, nbl);
        count_levels_kernel<<<dim3(nb, (unsigned)g.n_words), kCountBlock, 0, c->stream>>>(c->xm0[alpha - 1], c->xm1[alpha - 1], n, a.cntM);
        c->launches += 1;
    }
    switch (c->V * 10 + g.rpw) {
        case 41: launch_measure_t<4, 1>(c, a, f); break;
        case 42: launch_measure_t<4, 2>(c, a, f); break;
        case 21: launch_measure_t<2, 1>(c, a, f); break;
        case 22: launch_measure_t<2, 2>(c, a, f); break;
        case 11: launch_measure_t<1, 1>(c, a, f); break;
        default: launch_measure_t<1, 2>(c, a, f); break;
    }
    return post_launch(c);
}

// The last sweep of a measured group with the counting fused into its two launches
// (sweep.cuh, MeasAcc): the state is not read again for the observables.
template <int RPW>
int launch_measuring_sweep(micsa_ctx* c, long long* row, bool fold_min) {
    const Geom& g = c->g;
    SweepArgs a;
    a.spin = c->st.spin; a.m0 = c->st.m0; a.m1 = c->st.m1; a.J = c->st.J;
    a.L = g.L; a.Lh = g.Lh; a.n_rg = g.n_rg; a.half = g.half; a.w0 = 0; a.inv_nxv = fastdiv_magic((uint32_t)g.Lh / 4u); a.inv_pp = 0u;
    MeasureArgs ma; FinalizeArgs fa;
    make_measure_args(c, row, fold_min, ma, fa);
    const int per_plane = (g.L / 4) * (g.Lh / 4);
    const int zw = c->pipe_planes;
    dim3 grid = (zw == 4) ? dim3((unsigned)((per_plane + 31) / 32), (unsigned)(g.L / 4), (unsigned)g.n_words)
                          : dim3((unsigned)(((long long)(g.L / 2) * per_plane + 127) / 128), 2u, (unsigned)g.n_words);
    a.inv_pp = fastdiv_magic((uint32_t)per_plane);
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(128); cfg.dynamicSmemBytes = 0; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = c->use_pdl ? 1 : 0;
    cfg.attrs = attr; cfg.numAttrs = 1;
    if (zw == 4) {
        LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_meas_kernel<RPW, 4, 1>, a, 0, ma));
        LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_meas_kernel<RPW, 4, 2>, a, 1, ma));
    } else {
        LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_meas_kernel<RPW, 1, 1>, a, 0, ma));
        LK(cudaLaunchKernelEx(&cfg, half_sweep_pipe_meas_kernel<RPW, 1, 2>, a, 1, ma));
    }
    cfg.gridDim = dim3(1);
    LK(cudaLaunchKernelEx(&cfg, finalize_kernel, fa));
    c->attempts += (uint64_t)g.N * (uint64_t)g.n_sys;
    return post_launch(c, 3);
}

// ---- small lattices: one cluster per word lattice walks through refresh + sweeps + rows (small.cuh) ----
// cluster size (CTAs per word lattice, each holding L/cs planes in shared memory), threads per CTA, shared bytes
struct SmallShape { bool ok; int cs, block; size_t smem; };

SmallShape small_shape(const micsa_ctx* c) {
    const Geom& g = c->g;
    SmallShape sh; sh.ok = false; sh.cs = 1; sh.block = 32; sh.smem = 0;
    if (c->V != 4 || g.L > 64) return sh;
    const int target = c->small_items > 0 ? c->small_items : 128;      // quad rows per CTA and parity aimed at (measured: DESIGN.md 6.8)
    for (int cs = 1; cs <= 16; cs *= 2) {
        if (g.L % cs) break;
        const size_t smem = (g.rpw == 2) ? SlabLayout<2>(g.L / cs, g.L * g.Lh).total() : SlabLayout<1>(g.L / cs, g.L * g.Lh).total();
        const int items = (g.L / cs) * g.L * (g.Lh / 4);
        const bool last = (cs == 16) || (g.L % (2 * cs)) != 0;
        if (smem <= 200 * 1024 && (items <= target || (last && items <= 1024))) {
            sh.ok = true; sh.cs = cs; sh.smem = smem;
            sh.block = items >= 512 ? 512 : std::max(256, (items + 31) / 32 * 32);    // refresh and counting use every thread
            return sh;
        }
    }
    return sh;
}

bool small_eligible(const micsa_ctx* c) {
    const Geom& g = c->g;
    return c->small_path && g.n_replicas <= 2 && c->gamma == 1 && !c->walkers && small_shape(c).ok;
}

// One link of a chain of schedule steps walked by a single launch (small.cuh): the planes holding the step's
// refreshed daemon levels (nullptr: the state's own), its sweeps and its measurement interval.
struct SmallLink { const uint32_t* m0; const uint32_t* m1; int n_sweeps, measure_every; };

int launch_small_chain(micsa_ctx* c, bool do_refresh, double T, uint32_t step, const SmallLink* links, int n_links,
                       long long* rows, long long row0, long long rows_cap, bool fold_min) {
    const Geom& g = c->g;
    SmallArgs A;
    A.a.spin = c->st.spin; A.a.m0 = c->st.m0; A.a.m1 = c->st.m1; A.a.J = c->st.J;
    A.a.L = g.L; A.a.Lh = g.Lh; A.a.n_rg = g.n_rg; A.a.half = g.half; A.a.w0 = 0; A.a.inv_nxv = fastdiv_magic((uint32_t)g.Lh / 4u); A.a.inv_pp = 0u;
    A.sg = site_grid(g);
    MeasureArgs ma; FinalizeArgs fa;
    make_measure_args(c, c->row, fold_min, ma, fa);
    A.ma = ma;
    A.rows = rows; A.scratch_row = c->row; A.min_E = fold_min ? c->minE : nullptr;
    A.row_len = (long long)c->plan.row_len; A.row0 = row0; A.rows_cap = rows_cap;
    A.n_calls = c->calls;
    A.n_words = g.n_words;
    A.do_refresh = do_refresh ? 1 : 0; A.step = step; A.alpha_bits = 0u;
    A.n_chain = n_links;
    long long total_sweeps = 0;
    for (int j = 0; j < kSmallChain; ++j) {
        const bool in = j < n_links;
        A.ch_m0[j] = in ? links[j].m0 : nullptr; A.ch_m1[j] = in ? links[j].m1 : nullptr;
        A.ch_sweeps[j] = in ? links[j].n_sweeps : 0; A.ch_every[j] = in ? links[j].measure_every : 0;
        total_sweeps += A.ch_sweeps[j];
    }
    A.n_samples = g.n_samples; A.n_replicas = g.n_replicas; A.rpw = g.rpw; A.spw = g.spw; A.N = g.N;
    RefreshThr rt = {};
    if (do_refresh) {
        uint64_t thr[3];
        if (thresholds_host(T, thr) != MICSA_OK || thr[0] == 0) { set_err("temperature must be finite and > 0"); return MICSA_ERR_INVALID; }
        rt = make_thr(thr);
    }
    const SmallShape sh = small_shape(c);
    A.cs = sh.cs;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)(g.n_words * sh.cs)); cfg.blockDim = dim3((unsigned)sh.block);
    cfg.dynamicSmemBytes = sh.smem; cfg.stream = c->stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)sh.cs; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    // Function attributes belong to the (device, kernel), not to the context: another context with a smaller slab
    // must not lower what this one needs (a launch above the attribute fails with "invalid argument").  So every
    // context raises them, once, to values no shape exceeds: the device's opt-in shared-memory maximum and the
    // non-portable cluster size.
    if (!c->small_attr_set) {
        int dev = 0, optin = 0;
        CK(c, cudaGetDevice(&dev));
        CK(c, cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
        cudaFuncAttributes fa;                     // the kernel's static shared memory counts against the maximum
        if (g.rpw == 2) {
            CK(c, cudaFuncGetAttributes(&fa, small_step_kernel<2>));
            CK(c, cudaFuncSetAttribute(small_step_kernel<2>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
            CK(c, cudaFuncSetAttribute(small_step_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes));
        } else {
            CK(c, cudaFuncGetAttributes(&fa, small_step_kernel<1>));
            CK(c, cudaFuncSetAttribute(small_step_kernel<1>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
            CK(c, cudaFuncSetAttribute(small_step_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, optin - (int)fa.sharedSizeBytes));
        }
        c->small_attr_set = true;
    }
    if (g.rpw == 2) CK(c, cudaLaunchKernelEx(&cfg, small_step_kernel<2>, A, c->ks, rt));
    else            CK(c, cudaLaunchKernelEx(&cfg, small_step_kernel<1>, A, c->ks, rt));
    c->attempts += (uint64_t)total_sweeps * (uint64_t)g.N * (uint64_t)g.n_sys;
    c->t += total_sweeps;
    return post_launch(c);
}

// do_refresh: Eq. (11) at (T, step) first; then n_sweeps sweeps; a measurement row after every measure_every-th
// sweep (0 = none) into rows[row0 ...] (row index >= rows_cap: into the context's scratch row)
int launch_small_step(micsa_ctx* c, bool do_refresh, double T, uint32_t step, int n_sweeps, int measure_every,
                      long long* rows, long long row0, long long rows_cap, bool fold_min) {
    const SmallLink one = { nullptr, nullptr, n_sweeps, measure_every };
    return launch_small_chain(c, do_refresh, T, step, &one, 1, rows, row0, rows_cap, fold_min);
}

// Staging planes of the chained small-lattice steps of micsa_anneal: two sets of kSmallChain plane pairs (one being
// read by the running launch, one being generated on the side stream), allocated at the first chained call.
int chain_reserve(micsa_ctx* c) {
    if (c->chain_buf) return MICSA_OK;
    const size_t need = (size_t)2 * kSmallChain * 2 * c->plan.plane_bytes;
    if (cudaMalloc((void**)&c->chain_buf, need) != cudaSuccess) {
        cudaGetLastError(); c->chain_buf = nullptr; set_err("out of device memory (chained refresh planes)"); return MICSA_ERR_NOMEM;
    }
    return MICSA_OK;
}
uint32_t* chain_plane(micsa_ctx* c, int set, int j, int which) {
    return (uint32_t*)(c->chain_buf + ((size_t)(set * kSmallChain + j) * 2 + which) * c->plan.plane_bytes);
}

// n sweeps, then one measurement into `row`
int launch_sweeps_measured(micsa_ctx* c, int n, long long* row, bool fold_min) {
    const Geom& g = c->g;
    if (n >= 1 && small_eligible(c)) return launch_small_step(c, false, 0.0, 0u, n, n, row, 0, 1, fold_min);
    const bool fused = n >= 1 && c->fuse_measure && c->V == 4 && c->sweep_kernel == 2 && g.n_replicas <= 2 && c->gamma == 1;
    if (!fused) {
        const int rc = launch_sweeps(c, n); if (rc) return rc;
        return launch_measure(c, row, fold_min);
    }
    int rc = launch_sweeps(c, n - 1); if (rc) return rc;
    // The wandering only permutes the walkers: E, E_daemon and q of the timestep are counted before it, and it follows
    // as a launch of its own -- counting AND exchanging in the odd launch spilled 700-840 bytes per thread and made a
    // walker step 1 % slower than this (322 against 319 us at config 4).
    rc = (g.rpw == 2) ? launch_measuring_sweep<2>(c, row, fold_min) : launch_measuring_sweep<1>(c, row, fold_min);
    if (rc) return rc;
    if (c->walkers) { rc = launch_wander(c, 0, +1, (int)(c->t & 1)); if (rc) return rc; }
    c->t += 1;
    return MICSA_OK;
}

// host <-> device staging for the canonical layouts
struct Staging {
    void* dev = nullptr;
    ~Staging() { if (dev) cudaFree(dev); }
};

// Device staging for the canonical (one byte per spin / bond / daemon) boundary layouts: owned by the
// context and grow-only, so that the set / get calls do not pay a cudaMalloc + cudaFree each time.
int stage_reserve(micsa_ctx* c, size_t bytes, void** out) {
    if (bytes > c->stage_bytes) {
        CK(c, cudaStreamSynchronize(c->stream));
        if (c->stage_dev) cudaFree(c->stage_dev);
        c->stage_dev = nullptr; c->stage_bytes = 0;
        if (cudaMalloc(&c->stage_dev, bytes) != cudaSuccess) {
            cudaGetLastError(); set_err("out of device memory (staging)"); return MICSA_ERR_NOMEM;
        }
        c->stage_bytes = bytes;
    }
    *out = c->stage_dev;
    return MICSA_OK;
}

int set_sys(micsa_ctx* c, const int8_t* src, int kind) {
    int rc = check_ctx(c); if (rc) return rc;
    if (!src) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    const Geom& g = c->g;
    const size_t bytes = (size_t)g.n_sys * (size_t)g.N;
    struct { void* dev; } st = { nullptr };
    rc = stage_reserve(c, bytes, &st.dev); if (rc) return rc;
    CK(c, cudaMemcpyAsync(st.dev, src, bytes, cudaMemcpyHostToDevice, c->stream));
    CK(c, cudaMemsetAsync(c->bad, 0, sizeof(int), c->stream));
    validate_kernel<<<c->sms * 4, 256, 0, c->stream>>>((const int8_t*)st.dev, (long long)bytes, kind, c->bad);
    rc = post_launch(c); if (rc) return rc;
    int bad = 0;
    CK(c, cudaMemcpyAsync(&bad, c->bad, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    if (bad) { set_err(kind == 0 ? "spin values must be -1 or +1" : "daemon levels must be 0..3"); return MICSA_ERR_INVALID; }
    const SiteGrid sg = site_grid(g);
    const dim3 grid = site_blocks(g, g.n_words * 2);
    uint32_t* d0 = kind == 0 ? c->st.spin : family_m0(c, c->sel);
    uint32_t* d1 = family_m1(c, c->sel);
    if (g.rpw == 2) pack_sys_kernel<2><<<grid, 128, 0, c->stream>>>((const int8_t*)st.dev, d0, d1, sg, g.n_replicas, kind);
    else            pack_sys_kernel<1><<<grid, 128, 0, c->stream>>>((const int8_t*)st.dev, d0, d1, sg, g.n_replicas, kind);
    rc = post_launch(c); if (rc) return rc;
    CK(c, cudaStreamSynchronize(c->stream));
    return MICSA_OK;
}

void destroy_side(micsa_ctx* c) {
    if (c->side) { cudaStreamSynchronize(c->side); cudaStreamDestroy(c->side); c->side = nullptr; }
    if (c->ev_main) { cudaEventDestroy(c->ev_main); c->ev_main = nullptr; }
    if (c->ev_side) { cudaEventDestroy(c->ev_side); c->ev_side = nullptr; }
}

int init_state(micsa_ctx* c) {
    const Geom& g = c->g;
    const SiteGrid sg = site_grid(g);
    CK(c, cudaMemsetAsync(c->calls, 0, sizeof(unsigned long long), c->stream));
    CK(c, cudaMemsetAsync(c->cnt, 0, c->plan.cnt_words * 8, c->stream));
    CK(c, cudaMemsetAsync(c->ticket, 0, sizeof(unsigned int), c->stream));
    CK(c, cudaMemsetAsync(c->st.m0, 0, c->plan.plane_bytes, c->stream));
    CK(c, cudaMemsetAsync(c->st.m1, 0, c->plan.plane_bytes, c->stream));
    if (g.rpw == 2) {
        init_spins_kernel<2><<<site_blocks(g, g.n_words * 2), 128, 0, c->stream>>>(c->st.spin, sg, c->ks);
        init_bonds_kernel<2><<<site_blocks(g, g.n_sg * 6), 128, 0, c->stream>>>((uint16_t*)c->st.J, sg, c->ks);
    } else {
        init_spins_kernel<1><<<site_blocks(g, g.n_words * 2), 128, 0, c->stream>>>(c->st.spin, sg, c->ks);
        init_bonds_kernel<1><<<site_blocks(g, g.n_sg * 6), 128, 0, c->stream>>>((uint32_t*)c->st.J, sg, c->ks);
    }
    int rc = post_launch(c, 2); if (rc) return rc;
    CK(c, cudaStreamSynchronize(c->stream));
    return MICSA_OK;
}

}  // namespace

// =========================================================================
extern "C" {

const char* micsa_last_error(void) { return g_err; }

size_t micsa_workspace_bytes(int L, int n_samples, int n_replicas) {
    Geom g;
    if (!make_geom(L, n_samples, n_replicas, 0, g)) return 0;
    return make_plan(g).total;
}

micsa_ctx* micsa_create_ex(int L, int n_samples, int n_replicas, uint64_t seed,
                           int sample_offset, void* dev_workspace, size_t workspace_bytes,
                           void* cuda_stream)
{
    g_err[0] = 0;
    Geom g;
    if (!make_geom(L, n_samples, n_replicas, sample_offset, g)) return nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        set_err("no usable CUDA device (this library has no CPU fallback)");
        return nullptr;
    }
    micsa_ctx* c = new (std::nothrow) micsa_ctx();
    if (!c) { set_err("out of host memory"); return nullptr; }
    c->g = g;
    c->plan = make_plan(g);
    c->seed = seed;
    c->ks = philox_make_keys(seed);
    c->stream = (cudaStream_t)cuda_stream;
    c->V = vec_width(g.Lh);
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess ||
            cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) {
            cudaGetLastError(); set_err("could not query the device"); delete c; return nullptr;
        }
        c->sms = sms;
    }
    c->sweep_kernel = 2;
    c->pipe_rows = 4;
    c->use_pdl = 1;
    c->pipe_planes = ((g.L / 4) * (g.Lh / 4) >= 512) ? 4 : 1;   // big lattices, measured: DESIGN.md 6.1
    c->fuse_measure = 1;
    c->walkers = 0; c->t = 0; c->fuse_walk = 1; c->l2_groups = 1; c->small_path = 1; c->small_items = 0; c->small_attr_set = false; c->gamma = 1; c->sel = 0;
    c->attempts = c->rns = c->launches = 0;
    c->sticky = 0; c->launch_err = cudaSuccess;
    if (dev_workspace) {
        if (workspace_bytes < c->plan.total || ((uintptr_t)dev_workspace % kAlign)) {
            set_err("workspace too small or not 256-byte aligned"); delete c; return nullptr;
        }
        c->ws = (char*)dev_workspace; c->owns_ws = false;
    } else {
        void* p = nullptr;
        if (cudaMalloc(&p, c->plan.total) != cudaSuccess) {
            cudaGetLastError(); set_err("out of device memory"); delete c; return nullptr;
        }
        c->ws = (char*)p; c->owns_ws = true;
    }
    c->st.spin = (uint32_t*)(c->ws + c->plan.spin);
    c->st.m0 = (uint32_t*)(c->ws + c->plan.m0);
    c->st.m1 = (uint32_t*)(c->ws + c->plan.m1);
    c->st.J = (void*)(c->ws + c->plan.J);
    c->m0s = (uint32_t*)(c->ws + c->plan.m0s);
    c->m1s = (uint32_t*)(c->ws + c->plan.m1s);
    c->pending = false; c->pending_T = 0.0; c->pending_step = 0;
    c->measure_queued = false;
    c->cnt = (unsigned long long*)(c->ws + c->plan.cnt);
    c->ticket = (unsigned int*)(c->ws + c->plan.ticket);
    c->row = (long long*)(c->ws + c->plan.row);
    c->minE = (long long*)(c->ws + c->plan.minE);
    c->bad = (int*)(c->ws + c->plan.bad);
    c->calls = (unsigned long long*)(c->ws + c->plan.calls);
    c->trace_dev = nullptr; c->trace_bytes = 0;
    c->stage_dev = nullptr; c->stage_bytes = 0;
    c->c4_dev = nullptr; c->c4_bytes = 0; c->c4_host = nullptr; c->c4_host_bytes = 0;
    c->host_row = nullptr; c->side = nullptr; c->ev_main = nullptr; c->ev_side = nullptr;
    c->noalloc = nullptr; c->chain_buf = nullptr;
    if (cudaStreamCreateWithFlags(&c->side, cudaStreamNonBlocking) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_main, cudaEventDisableTiming) != cudaSuccess ||
        cudaEventCreateWithFlags(&c->ev_side, cudaEventDisableTiming) != cudaSuccess) {
        cudaGetLastError(); set_err("could not create the side stream");
        destroy_side(c); if (c->owns_ws) cudaFree(c->ws); delete c; return nullptr;
    }
    {   // The side stream has the lowest priority there is.  Only a context stream ABOVE it keeps the sweeps ahead
        // of the refresh generated beside them; at equal priority the two grids take turns block by block and a
        // step of config 4 costs 366 us instead of 243, so micsa_anneal then generates its refreshes in line (251 us).
        int p_main = 0, p_side = 0;
        c->side_below = cudaStreamGetPriority(c->stream, &p_main) == cudaSuccess &&
                        cudaStreamGetPriority(c->side, &p_side) == cudaSuccess && p_main < p_side;
        cudaGetLastError();
    }
    // set-up for micsa_measure_noalloc: the static scratch array's address on this device (no allocation; a failure
    // is not fatal here, the call itself reports it)
    if (noalloc_scratch(&c->noalloc) != cudaSuccess) { cudaGetLastError(); c->noalloc = nullptr; }
    if (cudaHostAlloc((void**)&c->host_row, c->plan.row_len * 8, cudaHostAllocDefault) != cudaSuccess) {
        cudaGetLastError(); set_err("out of pinned host memory");
        destroy_side(c); if (c->owns_ws) cudaFree(c->ws); delete c; return nullptr;
    }
    if (init_state(c) != MICSA_OK) {
        cudaFreeHost(c->host_row); destroy_side(c); if (c->owns_ws) cudaFree(c->ws); delete c; return nullptr;
    }
    return c;
}

micsa_ctx* micsa_create(int L, int n_samples, int n_replicas, uint64_t seed) {
    return micsa_create_ex(L, n_samples, n_replicas, seed, 0, nullptr, 0, nullptr);
}

int micsa_destroy(micsa_ctx* c) {
    if (!c) return MICSA_OK;
    cudaStreamSynchronize(c->stream);
    destroy_side(c);
    if (c->trace_dev) cudaFree(c->trace_dev);
    if (c->stage_dev) cudaFree(c->stage_dev);
    if (c->chain_buf) cudaFree(c->chain_buf);
    if (c->c4_dev) cudaFree(c->c4_dev);
    if (c->c4_host) cudaFreeHost(c->c4_host);
    for (uint32_t* p : c->xm0) cudaFree(p);
    for (uint32_t* p : c->xm1) cudaFree(p);
    for (uint32_t* p : c->xm0s) cudaFree(p);
    for (uint32_t* p : c->xm1s) cudaFree(p);
    if (c->owns_ws) cudaFree(c->ws);
    cudaFreeHost(c->host_row);
    delete c;
    return MICSA_OK;
}

int micsa_synchronize(micsa_ctx* c) {
    int rc = check_ctx(c); if (rc) return rc;
    CK(c, cudaStreamSynchronize(c->stream));
    CK(c, cudaStreamSynchronize(c->side));
    return MICSA_OK;
}

int micsa_set_spins(micsa_ctx* c, const int8_t* s) { return set_sys(c, s, 0); }
int micsa_set_daemons(micsa_ctx* c, const uint8_t* m) { return set_sys(c, (const int8_t*)m, 1); }
int micsa_set_demons(micsa_ctx* c, const uint8_t* m) { return micsa_set_daemons(c, m); }

int micsa_set_couplings(micsa_ctx* c, const int8_t* J) {
    int rc = check_ctx(c); if (rc) return rc;
    if (!J) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    const Geom& g = c->g;
    const size_t bytes = (size_t)g.n_samples * 3 * (size_t)g.N;
    struct { void* dev; } st = { nullptr };
    rc = stage_reserve(c, bytes, &st.dev); if (rc) return rc;
    CK(c, cudaMemcpyAsync(st.dev, J, bytes, cudaMemcpyHostToDevice, c->stream));
    CK(c, cudaMemsetAsync(c->bad, 0, sizeof(int), c->stream));
    validate_kernel<<<c->sms * 4, 256, 0, c->stream>>>((const int8_t*)st.dev, (long long)bytes, 0, c->bad);
    rc = post_launch(c); if (rc) return rc;
    int bad = 0;
    CK(c, cudaMemcpyAsync(&bad, c->bad, sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    if (bad) { set_err("couplings must be -1 or +1"); return MICSA_ERR_INVALID; }
    const SiteGrid sg = site_grid(g);
    const dim3 grid = site_blocks(g, g.n_sg * 6);
    if (g.rpw == 2) pack_bonds_kernel<2><<<grid, 128, 0, c->stream>>>((const int8_t*)st.dev, (uint16_t*)c->st.J, sg);
    else            pack_bonds_kernel<1><<<grid, 128, 0, c->stream>>>((const int8_t*)st.dev, (uint32_t*)c->st.J, sg);
    rc = post_launch(c); if (rc) return rc;
    CK(c, cudaStreamSynchronize(c->stream));
    return MICSA_OK;
}

int micsa_get_state(micsa_ctx* c, int8_t* s, uint8_t* m, int8_t* J) {
    int rc = check_ctx(c); if (rc) return rc;
    const Geom& g = c->g;
    const SiteGrid sg = site_grid(g);
    const size_t sys_bytes = (size_t)g.n_sys * (size_t)g.N;
    const size_t J_bytes = (size_t)g.n_samples * 3 * (size_t)g.N;
    struct { void* dev; } st = { nullptr };
    rc = stage_reserve(c, std::max(sys_bytes, J_bytes), &st.dev); if (rc) return rc;
    for (int kind = 0; kind < 2; ++kind) {
        void* dst = kind == 0 ? (void*)s : (void*)m;
        if (!dst) continue;
        const dim3 grid = site_blocks(g, g.n_words * 2);
        const uint32_t* d0 = kind == 0 ? c->st.spin : family_m0(c, c->sel);
        const uint32_t* d1 = family_m1(c, c->sel);
        if (g.rpw == 2) unpack_sys_kernel<2><<<grid, 128, 0, c->stream>>>((int8_t*)st.dev, d0, d1, sg, g.n_replicas, kind);
        else            unpack_sys_kernel<1><<<grid, 128, 0, c->stream>>>((int8_t*)st.dev, d0, d1, sg, g.n_replicas, kind);
        rc = post_launch(c); if (rc) return rc;
        CK(c, cudaMemcpyAsync(dst, st.dev, sys_bytes, cudaMemcpyDeviceToHost, c->stream));
        CK(c, cudaStreamSynchronize(c->stream));
    }
    if (J) {
        const dim3 grid = site_blocks(g, g.n_sg * 6);
        if (g.rpw == 2) unpack_bonds_kernel<2><<<grid, 128, 0, c->stream>>>((int8_t*)st.dev, (const uint16_t*)c->st.J, sg);
        else            unpack_bonds_kernel<1><<<grid, 128, 0, c->stream>>>((int8_t*)st.dev, (const uint32_t*)c->st.J, sg);
        rc = post_launch(c); if (rc) return rc;
        CK(c, cudaMemcpyAsync(J, st.dev, J_bytes, cudaMemcpyDeviceToHost, c->stream));
        CK(c, cudaStreamSynchronize(c->stream));
    }
    return MICSA_OK;
}

int micsa_half_sweep(micsa_ctx* c, int parity) {
    int rc = check_ctx(c); if (rc) return rc;
    if (parity != 0 && parity != 1) { set_err("parity must be 0 or 1"); return MICSA_ERR_INVALID; }
    return launch_half_sweep(c, parity);
}

int micsa_sweep(micsa_ctx* c, int n) {
    int rc = check_ctx(c); if (rc) return rc;
    if (n < 0) { set_err("n must be >= 0"); return MICSA_ERR_INVALID; }
    if (n >= 1 && small_eligible(c)) return launch_small_step(c, false, 0.0, 0u, n, 0, c->row, 0, 0, false);
    return launch_sweeps(c, n);
}

int micsa_wander(micsa_ctx* c, int axis, int sign, int parity) {
    int rc = check_ctx(c); if (rc) return rc;
    if (axis < 0 || axis > 2 || (sign != 1 && sign != -1) || (parity != 0 && parity != 1)) {
        set_err("axis must be 0..2, sign +1 or -1, parity 0 or 1"); return MICSA_ERR_INVALID;
    }
    uint32_t* const h0 = c->st.m0; uint32_t* const h1 = c->st.m1;      // the selected family
    c->st.m0 = family_m0(c, c->sel); c->st.m1 = family_m1(c, c->sel);
    rc = launch_wander(c, axis, sign, parity);
    c->st.m0 = h0; c->st.m1 = h1;
    return rc;
}

int micsa_set_gamma(micsa_ctx* c, int gamma) {
    int rc = check_ctx(c); if (rc) return rc;
    if (gamma < 1 || gamma > 6) { set_err("gamma must be 1..6"); return MICSA_ERR_INVALID; }
    CK(c, cudaStreamSynchronize(c->stream));
    CK(c, cudaStreamSynchronize(c->side));
    while ((int)c->xm0.size() > gamma - 1) {
        cudaFree(c->xm0.back()); cudaFree(c->xm1.back()); c->xm0.pop_back(); c->xm1.pop_back();
    }
    while ((int)c->xm0s.size() > gamma - 1) {
        cudaFree(c->xm0s.back()); cudaFree(c->xm1s.back()); c->xm0s.pop_back(); c->xm1s.pop_back();
    }
    while ((int)c->xm0.size() < gamma - 1) {       // new families start at level 0, like family 0 at create
        void* a = nullptr; void* b = nullptr;
        if (cudaMalloc(&a, c->plan.plane_bytes) != cudaSuccess || cudaMalloc(&b, c->plan.plane_bytes) != cudaSuccess) {
            cudaGetLastError(); if (a) cudaFree(a); set_err("out of device memory (daemon families)"); return MICSA_ERR_NOMEM;
        }
        CK(c, cudaMemsetAsync(a, 0, c->plan.plane_bytes, c->stream));
        CK(c, cudaMemsetAsync(b, 0, c->plan.plane_bytes, c->stream));
        c->xm0.push_back((uint32_t*)a); c->xm1.push_back((uint32_t*)b);
    }
    c->gamma = gamma; c->sel = std::min(c->sel, gamma - 1);
    c->pending = false;                           // a prefetched refresh was generated for the old number of families
    return MICSA_OK;
}

int micsa_select_daemon_set(micsa_ctx* c, int alpha) {
    int rc = check_ctx(c); if (rc) return rc;
    if (alpha < 0 || alpha >= c->gamma) { set_err("alpha must be 0 .. gamma-1"); return MICSA_ERR_INVALID; }
    c->sel = alpha;
    return MICSA_OK;
}

int micsa_set_walkers(micsa_ctx* c, int mode) {
    int rc = check_ctx(c); if (rc) return rc;

    if (mode != 0 && mode != 1) { set_err("walkers mode must be 0 (daemons) or 1 (one forward-X walker per spin)"); return MICSA_ERR_INVALID; }
    c->walkers = mode;
    return MICSA_OK;
}

int micsa_set_time(micsa_ctx* c, int64_t t) {
    int rc = check_ctx(c); if (rc) return rc;
    if (t < 0) { set_err("t must be >= 0"); return MICSA_ERR_INVALID; }
    c->t = t;
    return MICSA_OK;
}

int micsa_get_time(micsa_ctx* c, int64_t* t) {
    if (!c || !t) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    *t = c->t;
    return MICSA_OK;
}

int micsa_metropolis_sweep(micsa_ctx* c, double T, uint32_t tau0, int n) {
    int rc = check_ctx(c); if (rc) return rc;
    uint64_t thr[3];
    if (n < 0 || metropolis_thresholds_host(T, thr) != MICSA_OK) { set_err("n must be >= 0 and T finite and > 0"); return MICSA_ERR_INVALID; }
    const RefreshThr rt = make_thr(thr);
    for (int t = 0; t < n; ++t)
        for (int parity = 0; parity < 2; ++parity) {
            rc = launch_metropolis_half_sweep(c, rt, tau0 + (uint32_t)t, parity); if (rc) return rc;
        }
    return MICSA_OK;
}

int micsa_metropolis_half_sweep(micsa_ctx* c, double T, uint32_t tau, int parity) {
    int rc = check_ctx(c); if (rc) return rc;
    uint64_t thr[3];
    if ((parity != 0 && parity != 1) || metropolis_thresholds_host(T, thr) != MICSA_OK) {
        set_err("parity must be 0 or 1 and T finite and > 0"); return MICSA_ERR_INVALID;
    }
    return launch_metropolis_half_sweep(c, make_thr(thr), tau, parity);
}

int micsa_debug_metropolis_thresholds(double T, uint64_t thr[3]) {
    if (!thr) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    if (metropolis_thresholds_host(T, thr) != MICSA_OK) { set_err("temperature must be finite and > 0"); return MICSA_ERR_INVALID; }
    return MICSA_OK;
}

int micsa_effective_temperature(double e_daemon_per_variable, double* T) {
    // invert Eq. (12): <H_aux>/(gamma N) = 4x/(1-x) - 16x^4/(1-x^4), x = exp(-4/T), is
    // increasing in T from 0 (T -> 0) to 6 (T -> infinity, uniform levels): bisection on x in float64
    if (!T) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    if (!(e_daemon_per_variable > 0.0) || !(e_daemon_per_variable < 6.0)) {
        set_err("the daemon energy per auxiliary variable must lie strictly between 0 and 6"); return MICSA_ERR_INVALID;
    }
    auto f = [](double x) {           // regular at x -> 1: 4(x + 2x^2 + 3x^3)/(1 + x + x^2 + x^3)
        return 4.0 * (x + 2.0 * x * x + 3.0 * x * x * x) / (1.0 + x + x * x + x * x * x);
    };
    double lo = 0.0, hi = 1.0;
    for (int it = 0; it < 200; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (f(mid) < e_daemon_per_variable) lo = mid; else hi = mid;
    }
    const double x = 0.5 * (lo + hi);
    *T = -4.0 / std::log(x);
    return MICSA_OK;
}

int micsa_debug_philox(uint64_t seed, const uint32_t* counters, int n, uint32_t* out) {
    if (!counters || !out || n < 0) { set_err("null pointer or negative count"); return MICSA_ERR_INVALID; }
    if (n == 0) return MICSA_OK;
    void* dev = nullptr;
    const size_t bytes = (size_t)n * 16;
    if (cudaMalloc(&dev, 2 * bytes) != cudaSuccess) { cudaGetLastError(); set_err("no usable CUDA device or out of memory"); return MICSA_ERR_CUDA; }
    cudaError_t e = cudaMemcpy(dev, counters, bytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) {
        debug_philox_kernel<<<(n + 127) / 128, 128>>>((const uint4*)dev, (uint4*)((char*)dev + bytes), n, philox_make_keys(seed));
        e = cudaGetLastError();
    }
    if (e == cudaSuccess) e = cudaMemcpy(out, (char*)dev + bytes, bytes, cudaMemcpyDeviceToHost);
    cudaFree(dev);
    if (e != cudaSuccess) { set_err("CUDA error: %s", cudaGetErrorString(e)); return MICSA_ERR_CUDA; }
    return MICSA_OK;
}

int micsa_debug_thresholds(double T, uint64_t thr[3]) {
    if (!thr) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    if (thresholds_host(T, thr) != MICSA_OK) { set_err("temperature must be finite and > 0"); return MICSA_ERR_INVALID; }
    return MICSA_OK;
}

int micsa_refresh_demons(micsa_ctx* c, double T, uint32_t step) {
    int rc = check_ctx(c); if (rc) return rc;
    return launch_refresh(c, T, step);
}

int micsa_prefetch_refresh(micsa_ctx* c, double T, uint32_t step) {
    int rc = check_ctx(c); if (rc) return rc;
    return launch_prefetch(c, T, step);
}

int micsa_measure_begin(micsa_ctx* c) {
    int rc = check_ctx(c); if (rc) return rc;
    rc = launch_measure(c, c->row, false); if (rc) return rc;
    CK(c, cudaMemcpyAsync(c->host_row, c->row, c->plan.row_len * 8, cudaMemcpyDeviceToHost, c->stream));
    c->measure_queued = true;
    return MICSA_OK;
}

int micsa_sweep_measure(micsa_ctx* c, int n) {
    int rc = check_ctx(c); if (rc) return rc;
    if (n < 0) { set_err("n must be >= 0"); return MICSA_ERR_INVALID; }
    rc = launch_sweeps_measured(c, n, c->row, false); if (rc) return rc;
    CK(c, cudaMemcpyAsync(c->host_row, c->row, c->plan.row_len * 8, cudaMemcpyDeviceToHost, c->stream));
    c->measure_queued = true;
    return MICSA_OK;
}

int micsa_measure_end(micsa_ctx* c, int64_t* E, int64_t* Ed, int64_t* Q) {
    int rc = check_ctx(c); if (rc) return rc;
    const Geom& g = c->g;
    if (Q && g.n_replicas < 2) { set_err("q_overlap needs n_replicas >= 2"); return MICSA_ERR_INVALID; }
    if (!c->measure_queued) { set_err("micsa_measure_end without micsa_measure_begin"); return MICSA_ERR_INVALID; }
    CK(c, cudaStreamSynchronize(c->stream));
    c->measure_queued = false;
    if (E)  memcpy(E, c->host_row, (size_t)g.n_sys * 8);
    if (Ed) memcpy(Ed, c->host_row + g.n_sys, (size_t)g.n_sys * 8);
    if (Q)  memcpy(Q, c->host_row + 2 * g.n_sys, (size_t)g.n_pairs * 8);
    return MICSA_OK;
}

int micsa_measure_i64(micsa_ctx* c, int64_t* E, int64_t* Ed, int64_t* Q) {
    int rc = check_ctx(c); if (rc) return rc;
    if (Q && c->g.n_replicas < 2) { set_err("q_overlap needs n_replicas >= 2"); return MICSA_ERR_INVALID; }
    rc = micsa_measure_begin(c); if (rc) return rc;
    return micsa_measure_end(c, E, Ed, Q);
}

// The measurement with its counters and ticket in the library's static scratch array instead of the context's
// workspace, the row written to the caller's DEVICE buffer: no allocation, no host synchronisation, no copy.
int micsa_measure_noalloc(micsa_ctx* c, int64_t* d_row) {
    int rc = check_ctx(c); if (rc) return rc;
    if (!d_row) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    if (!c->noalloc) { set_err("the address of the static scratch array could not be obtained on this device"); return MICSA_ERR_CUDA; }
    const size_t need = c->plan.cnt_words;
    if (need > kNoAllocCounters) {
        char msg[160];
        snprintf(msg, sizeof msg, "this context needs %zu lane counters, the static scratch of micsa_measure_noalloc holds %zu "
                 "(MICSA_NOALLOC_MAX_COUNTERS)", need, kNoAllocCounters);
        set_err("%s", msg); return MICSA_ERR_INVALID;
    }
    cudaPointerAttributes pa;
    if (cudaPointerGetAttributes(&pa, d_row) != cudaSuccess ||
        (pa.type != cudaMemoryTypeDevice && pa.type != cudaMemoryTypeManaged)) {
        cudaGetLastError(); set_err("d_row must be device (or managed) memory"); return MICSA_ERR_INVALID;
    }
    // the array keeps whatever the last call (of any context on this device) left: counters and ticket start at zero
    CK(c, cudaMemsetAsync(c->noalloc, 0, need * sizeof(unsigned long long), c->stream));
    CK(c, cudaMemsetAsync(c->noalloc + kNoAllocCounters, 0, kNoAllocTicket * sizeof(unsigned long long), c->stream));
    // the same launches as micsa_measure_begin, with the scratch pointers exchanged for the duration of the call
    unsigned long long* const cnt0 = c->cnt; unsigned int* const ticket0 = c->ticket;
    c->cnt = c->noalloc; c->ticket = reinterpret_cast<unsigned int*>(c->noalloc + kNoAllocCounters);
    rc = launch_measure(c, reinterpret_cast<long long*>(d_row), false);
    c->cnt = cnt0; c->ticket = ticket0;
    return rc;
}

int micsa_measure_c4(micsa_ctx* c, int64_t* S) {
    int rc = check_ctx(c); if (rc) return rc;
    const Geom& g = c->g;
    if (!S) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    if (g.n_replicas < 2) { set_err("micsa_measure_c4 needs n_replicas >= 2"); return MICSA_ERR_INVALID; }
    const int R = g.L / 2 + 1;
    const int pps = g.n_replicas * (g.n_replicas - 1) / 2;
    const size_t x_bytes = align_up((size_t)g.n_sg * (size_t)g.N * sizeof(uint32_t));
    const size_t pair_words = (size_t)g.n_sg * 3 * R * 32, cnt_words = pair_words * pps;
    // context-owned, grow-only: no cudaMalloc / cudaFree per measurement
    if (x_bytes + cnt_words * 8 > c->c4_bytes) {
        CK(c, cudaStreamSynchronize(c->stream));
        if (c->c4_dev) cudaFree(c->c4_dev);
        c->c4_dev = nullptr; c->c4_bytes = 0;
        if (cudaMalloc(&c->c4_dev, x_bytes + cnt_words * 8) != cudaSuccess) {
            cudaGetLastError(); set_err("out of device memory (c4)"); return MICSA_ERR_NOMEM;
        }
        c->c4_bytes = x_bytes + cnt_words * 8;
    }
    if (cnt_words * 8 > c->c4_host_bytes) {
        if (c->c4_host) cudaFreeHost(c->c4_host);
        c->c4_host = nullptr; c->c4_host_bytes = 0;
        if (cudaHostAlloc((void**)&c->c4_host, cnt_words * 8, cudaHostAllocDefault) != cudaSuccess) {
            cudaGetLastError(); set_err("out of pinned host memory (c4)"); return MICSA_ERR_NOMEM;
        }
        c->c4_host_bytes = cnt_words * 8;
    }
    uint32_t* X = (uint32_t*)c->c4_dev;
    unsigned long long* cnt = (unsigned long long*)((char*)c->c4_dev + x_bytes);
    CK(c, cudaMemsetAsync(cnt, 0, cnt_words * 8, c->stream));
    // every thread counts at most 65535 sites (16-plane counters)
    long long nb = std::max<long long>(1, std::min<long long>((g.N + kCountBlock * 64 - 1) / (kCountBlock * 64), 64));
    nb = std::max<long long>(nb, (g.N + (long long)kCountBlock * 60000 - 1) / ((long long)kCountBlock * 60000));
    const uint32_t mask = (g.rpw == 2) ? 0xFFFFu : 0xFFFFFFFFu;
    int k = 0;
    for (int ra = 0; ra < g.n_replicas; ++ra)
        for (int rb = ra + 1; rb < g.n_replicas; ++rb, ++k) {        // pairs a < b, lexicographic (Eq. 16 sums all of them)
            overlap_field_kernel<<<site_blocks(g, g.n_sg * 2), 128, 0, c->stream>>>(
                c->st.spin, X, g.L, g.Lh, g.half, g.n_rg, ra / g.rpw, 16 * (ra % g.rpw), rb / g.rpw, 16 * (rb % g.rpw), mask);
            c4_count_kernel<<<dim3((unsigned)nb, (unsigned)R, (unsigned)(3 * g.n_sg)), kCountBlock, 0, c->stream>>>(
                X, cnt + (size_t)k * pair_words, g.L);
            rc = post_launch(c, 2); if (rc) return rc;
        }
    const unsigned long long* host = c->c4_host;
    CK(c, cudaMemcpyAsync(c->c4_host, cnt, cnt_words * 8, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    for (int sample = 0; sample < g.n_samples; ++sample) {
        const int sg = sample / g.spw, sl = sample - sg * g.spw;
        for (int pk = 0; pk < pps; ++pk)
            for (int d = 0; d < 3; ++d)
                for (int r = 0; r < R; ++r)
                    S[(((size_t)sample * pps + pk) * 3 + d) * R + r] =
                        (int64_t)g.N - 2 * (int64_t)host[(size_t)pk * pair_words + (((size_t)sg * 3 + d) * R + r) * 32 + sl];
    }
    return MICSA_OK;
}

int micsa_xi(const double* C4, int n_r, double c_min, double I[3], double* xi12, double* xi23_over_xi12) {
    // Eq. (17)-(18), reading R22 of DESIGN.md: trapezoidal rule on r = 0, 1, ..., cut before the
    // first value at or below c_min, no tail
    if (!C4 || n_r < 2) { set_err("C4 must hold at least r = 0 and r = 1"); return MICSA_ERR_INVALID; }
    int n = n_r;
    for (int r = 0; r < n_r; ++r)
        if (!(C4[r] > c_min)) { n = r; break; }
    if (n < 2) { set_err("C4 is at or below the cut-off from r = 1 on"); return MICSA_ERR_INVALID; }
    double In[3] = { 0.0, 0.0, 0.0 };
    for (int k = 0; k < 3; ++k)
        for (int r = 0; r + 1 < n; ++r) {
            const double f0 = std::pow((double)r, k + 1) * C4[r], f1 = std::pow((double)(r + 1), k + 1) * C4[r + 1];
            In[k] += 0.5 * (f0 + f1);
        }
    if (I) { I[0] = In[0]; I[1] = In[1]; I[2] = In[2]; }
    if (xi12) *xi12 = In[1] / In[0];
    if (xi23_over_xi12) *xi23_over_xi12 = (In[2] / In[1]) / (In[1] / In[0]);
    return MICSA_OK;
}

int micsa_measure(micsa_ctx* c, double* e, double* ed, double* q) {
    int rc = check_ctx(c); if (rc) return rc;
    const Geom& g = c->g;
    if (q && g.n_replicas < 2) { set_err("q_overlap needs n_replicas >= 2"); return MICSA_ERR_INVALID; }
    std::vector<int64_t> E(g.n_sys), Ed(g.n_sys), Q(std::max(g.n_pairs, 1));
    rc = micsa_measure_i64(c, E.data(), Ed.data(), g.n_pairs ? Q.data() : nullptr);
    if (rc) return rc;
    const double N = (double)g.N;
    if (e)  for (int i = 0; i < g.n_sys; ++i) e[i] = (double)E[i] / N;
    if (ed) for (int i = 0; i < g.n_sys; ++i) ed[i] = (double)Ed[i] / N;
    if (q)  for (int i = 0; i < g.n_pairs; ++i) q[i] = (double)Q[i] / N;
    return MICSA_OK;
}

int micsa_anneal(micsa_ctx* c, const micsa_step* sched, int n_steps, uint32_t step0,
                 double* min_energy, micsa_trace* trace)
{
    int rc = check_ctx(c); if (rc) return rc;
    if (n_steps < 0 || (n_steps > 0 && !sched)) { set_err("bad schedule"); return MICSA_ERR_INVALID; }
    const Geom& g = c->g;
    long long rows = 0;
    for (int k = 0; k < n_steps; ++k) {
        uint64_t thr[3];
        if (thresholds_host(sched[k].T, thr) != MICSA_OK) { set_err("temperature must be finite and > 0"); return MICSA_ERR_INVALID; }
        if (sched[k].n_sweeps < 0 || sched[k].measure_every < 0) { set_err("negative sweep count"); return MICSA_ERR_INVALID; }
        if (sched[k].measure_every > 0) rows += sched[k].n_sweeps / sched[k].measure_every;
    }
    if (trace && trace->capacity < 0) { set_err("negative trace capacity"); return MICSA_ERR_INVALID; }
    const long long keep = trace ? std::min<long long>(rows, trace->capacity) : 0;
    const size_t row_len = c->plan.row_len;
    // the trace rows live in a context-owned device buffer that only grows: no cudaMalloc / cudaFree
    // (and their implicit synchronisation) per call
    struct { void* dev; } dev_rows = { c->trace_dev };
    if ((size_t)keep * row_len * 8 > c->trace_bytes) {
        CK(c, cudaStreamSynchronize(c->stream));
        if (c->trace_dev) cudaFree(c->trace_dev);
        c->trace_dev = nullptr; c->trace_bytes = 0;
        const size_t want = std::max<size_t>((size_t)keep * row_len * 8, 4096);
        if (cudaMalloc(&c->trace_dev, want) != cudaSuccess) {
            cudaGetLastError(); set_err("out of device memory (trace)"); return MICSA_ERR_NOMEM;
        }
        c->trace_bytes = want;
        dev_rows.dev = c->trace_dev;
    }
    fill_i64_kernel<<<(g.n_sys + 127) / 128, 128, 0, c->stream>>>(c->minE, std::numeric_limits<long long>::max(), g.n_sys);
    rc = post_launch(c); if (rc) return rc;

    std::vector<int64_t> row_sweep;
    std::vector<double> row_T;
    long long r = 0, t = 0;
    bool chain_ready = false; int chain_first = 0, chain_n = 0, chain_set = 0;   // refreshes generated ahead (small lattices)
    for (int k = 0; k < n_steps; ++k) {
        if (small_eligible(c) && sched[k].n_sweeps > 0) {     // small lattice: whole steps in one cluster launch
            // The clusters of a small lattice leave most SMs idle: when that is so, up to kSmallChain steps go into
            // ONE launch (the lattice stays in shared memory across them) and their refreshes are generated by the
            // stand-alone kernel into staging planes -- the first batch's on this stream, every later batch's on the
            // side stream beside the launch before it.
            auto chain_len = [&](int from) {
                int n = 0;
                while (from + n < n_steps && n < kSmallChain && sched[from + n].n_sweeps > 0) ++n;
                return n;
            };
            if (c->g.n_words * small_shape(c).cs * 2 <= c->sms) {
                rc = chain_reserve(c); if (rc) return rc;
                const int n = chain_len(k);
                if (!(chain_ready && chain_first == k && chain_n == n)) {          // nothing generated ahead: do it in line
                    chain_set = 0;
                    for (int j = 0; j < n; ++j) {
                        rc = launch_refresh_into(c, sched[k + j].T, step0 + (uint32_t)(k + j), chain_plane(c, chain_set, j, 0),
                                                 chain_plane(c, chain_set, j, 1), c->stream);
                        if (rc) return rc;
                    }
                } else {
                    CK(c, cudaStreamWaitEvent(c->stream, c->ev_side, 0));
                }
                chain_ready = false;
                const int n2 = chain_len(k + n);
                if (n2 > 0) {                              // the next batch, under this one; the set it overwrites was
                    CK(c, cudaEventRecord(c->ev_main, c->stream));      // read by the launch before this one
                    CK(c, cudaStreamWaitEvent(c->side, c->ev_main, 0));
                    for (int j = 0; j < n2; ++j) {
                        rc = launch_refresh_into(c, sched[k + n + j].T, step0 + (uint32_t)(k + n + j),
                                                 chain_plane(c, chain_set ^ 1, j, 0), chain_plane(c, chain_set ^ 1, j, 1), c->side);
                        if (rc) return rc;
                    }
                    CK(c, cudaEventRecord(c->ev_side, c->side));
                }
                SmallLink links[kSmallChain];
                for (int j = 0; j < n; ++j)
                    links[j] = { chain_plane(c, chain_set, j, 0), chain_plane(c, chain_set, j, 1), sched[k + j].n_sweeps,
                                 sched[k + j].measure_every };
                rc = launch_small_chain(c, false, 0.0, 0u, links, n, (long long*)dev_rows.dev, r, keep, true);
                if (rc) return rc;
                c->rns += (uint64_t)n * (uint64_t)g.N * (uint64_t)g.n_sys;
                for (int j = 0; j < n; ++j) {
                    const int me = sched[k + j].measure_every, n_rows = me > 0 ? sched[k + j].n_sweeps / me : 0;
                    for (int i = 1; i <= n_rows; ++i)
                        if (r + i - 1 < keep) { row_sweep.push_back(t + (long long)i * me); row_T.push_back(sched[k + j].T); }
                    r += n_rows; t += sched[k + j].n_sweeps;
                }
                if (n2 > 0) { chain_ready = true; chain_first = k + n; chain_n = n2; chain_set ^= 1; }
                k += n - 1;
                continue;
            }
            // many lattices (no idle SMs to generate beside): one step per launch, refreshed inside the kernel
            const int me = sched[k].measure_every, n_rows = me > 0 ? sched[k].n_sweeps / me : 0;
            const bool prefetched = c->pending && c->pending_step == step0 + (uint32_t)k &&
                                    memcmp(&c->pending_T, &sched[k].T, sizeof(double)) == 0;
            if (prefetched) { rc = launch_refresh(c, sched[k].T, step0 + (uint32_t)k); if (rc) return rc; }
            else c->rns += (uint64_t)g.N * (uint64_t)g.n_sys;
            rc = launch_small_step(c, !prefetched, sched[k].T, step0 + (uint32_t)k, sched[k].n_sweeps, me,
                                   (long long*)dev_rows.dev, r, keep, true);
            if (rc) return rc;
            for (int i = 1; i <= n_rows; ++i)
                if (r + i - 1 < keep) { row_sweep.push_back(t + (long long)i * me); row_T.push_back(sched[k].T); }
            r += n_rows; t += sched[k].n_sweeps;
            continue;
        }
        rc = launch_refresh(c, sched[k].T, step0 + (uint32_t)k); if (rc) return rc;
        if (k + 1 < n_steps && sched[k].n_sweeps > 0 && c->side_below) {       // generated under this step's sweeps
            rc = launch_prefetch(c, sched[k + 1].T, step0 + (uint32_t)k + 1u); if (rc) return rc;
        }
        // sweeps in groups that end at a measurement (or at the end of the step)
        const int me = sched[k].measure_every;
        for (int j = 0; j < sched[k].n_sweeps; ) {
            const int group = (me > 0) ? std::min(me - j % me, sched[k].n_sweeps - j) : sched[k].n_sweeps - j;
            j += group; t += group;
            if (me > 0 && j % me == 0) {
                long long* dst = (r < keep) ? (long long*)dev_rows.dev + (size_t)r * row_len : c->row;
                rc = launch_sweeps_measured(c, group, dst, true); if (rc) return rc;
                if (r < keep) { row_sweep.push_back(t); row_T.push_back(sched[k].T); }
                ++r;
            } else {
                rc = launch_sweeps(c, group); if (rc) return rc;
            }
        }
    }
    std::vector<long long> host((size_t)keep * row_len);
    std::vector<long long> minE(g.n_sys);
    if (keep > 0)
        CK(c, cudaMemcpyAsync(host.data(), dev_rows.dev, host.size() * 8, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaMemcpyAsync(minE.data(), c->minE, (size_t)g.n_sys * 8, cudaMemcpyDeviceToHost, c->stream));
    CK(c, cudaStreamSynchronize(c->stream));
    if (min_energy)
        for (int i = 0; i < g.n_sys; ++i)
            min_energy[i] = (rows > 0) ? (double)minE[i] / (double)g.N : std::numeric_limits<double>::infinity();
    if (trace) {
        trace->n_rows = rows;
        for (long long i = 0; i < keep; ++i) {
            const long long* src = host.data() + (size_t)i * row_len;
            if (trace->sweep) trace->sweep[i] = row_sweep[i];
            if (trace->T) trace->T[i] = row_T[i];
            if (trace->E) memcpy(trace->E + (size_t)i * g.n_sys, src, (size_t)g.n_sys * 8);
            if (trace->E_daemon) memcpy(trace->E_daemon + (size_t)i * g.n_sys, src + g.n_sys, (size_t)g.n_sys * 8);
            if (trace->Q && g.n_pairs) memcpy(trace->Q + (size_t)i * g.n_pairs, src + 2 * g.n_sys, (size_t)g.n_pairs * 8);
        }
    }
    return MICSA_OK;
}

int micsa_counters(micsa_ctx* c, uint64_t* attempts, uint64_t* rns, uint64_t* philox_calls) {
    if (!c) { set_err("null context"); return MICSA_ERR_INVALID; }
    if (attempts) *attempts = c->attempts;
    if (rns) *rns = c->rns;
    if (philox_calls) {
        // lazy refresh: the number of calls is data dependent and counted on the device
        if (c->sticky) { set_err("context is in a sticky CUDA error state"); return c->sticky; }
        unsigned long long n = 0;
        CK(c, cudaStreamSynchronize(c->side));
        CK(c, cudaMemcpyAsync(&n, c->calls, sizeof n, cudaMemcpyDeviceToHost, c->stream));
        CK(c, cudaStreamSynchronize(c->stream));
        *philox_calls = (uint64_t)n;
    }
    return MICSA_OK;
}

int micsa_set_tuning(micsa_ctx* c, int key, int value) {
    int rc = check_ctx(c); if (rc) return rc;
    switch (key) {
        case MICSA_TUNE_SWEEP_KERNEL:
            if (value != 1 && value != 2) { set_err("sweep kernel must be 1 or 2"); return MICSA_ERR_INVALID; }
            c->sweep_kernel = value; return MICSA_OK;
        case MICSA_TUNE_PIPE_PLANES:
            if (value != 1 && value != 4) { set_err("pipe_planes must be 1 or 4"); return MICSA_ERR_INVALID; }
            c->pipe_planes = value; return MICSA_OK;
        case MICSA_TUNE_L2_GROUPS:
            if (value != 0 && value != 1) { set_err("l2_groups must be 0 or 1"); return MICSA_ERR_INVALID; }
            c->l2_groups = value; return MICSA_OK;
        case MICSA_TUNE_SMALL_ITEMS:
            if (value < 0 || value > 1024) { set_err("small_items must be 0 (default) .. 1024"); return MICSA_ERR_INVALID; }
            c->small_items = value; c->small_attr_set = false; return MICSA_OK;
        case MICSA_TUNE_SMALL_PATH:
            if (value != 0 && value != 1) { set_err("small_path must be 0 or 1"); return MICSA_ERR_INVALID; }
            c->small_path = value; return MICSA_OK;
        case MICSA_TUNE_FUSE_WALK:
            if (value != 0 && value != 1) { set_err("fuse_walk must be 0 or 1"); return MICSA_ERR_INVALID; }
            c->fuse_walk = value; return MICSA_OK;
        case MICSA_TUNE_FUSE_MEASURE:
            if (value != 0 && value != 1) { set_err("fuse_measure must be 0 or 1"); return MICSA_ERR_INVALID; }
            c->fuse_measure = value; return MICSA_OK;
        case MICSA_TUNE_PDL:
            if (value != 0 && value != 1) { set_err("pdl must be 0 or 1"); return MICSA_ERR_INVALID; }
            c->use_pdl = value; return MICSA_OK;
        case MICSA_TUNE_PIPE_ROWS:
            if (value != 4 && value != 8) { set_err("pipe_rows must be 4 or 8"); return MICSA_ERR_INVALID; }
            c->pipe_rows = value; return MICSA_OK;
        default:
            set_err("unknown tuning key"); return MICSA_ERR_INVALID;
    }
}

int micsa_layout_info(micsa_ctx* c, uint64_t info[5]) {
    if (!c || !info) { set_err("null pointer"); return MICSA_ERR_INVALID; }
    const Geom& g = c->g;
    const uint64_t sites = (uint64_t)g.N;
    const uint64_t spin_b = sites * g.n_words * 4, dem_b = 2 * spin_b;
    const uint64_t J_b = 3 * sites * g.n_sg * (g.rpw == 2 ? 2 : 4);
    info[0] = spin_b + dem_b + J_b;
    info[1] = 2 * (spin_b + dem_b) + J_b;     // state read once + written once, bonds read once
    info[2] = (uint64_t)g.n_words;
    info[3] = (uint64_t)(32 / g.rpw);
    info[4] = c->launches;
    return MICSA_OK;
}

}  // extern "C"
