// Host side of the C ABI declared in include/ptglass.h: argument checks, host-computed acceptance tables,
// workspace carving, kernel dispatch.  No device memory is allocated here (the caller owns the workspace) and
// there is no CPU fallback: every step of the path runs in the kernels of kernels.cuh.
#include "../../include/ptglass.h"
#include "../../include/ptglass_diag.h"

#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <vector>

#include "kernels.cuh"
#include "mcs.cuh"
#include "gauss.cuh"
#include "houdayer_multi.cuh"

using namespace ptg;

namespace {

struct Context {
    void *ws = nullptr;
    size_t ws_bytes = 0;
    cudaStream_t stream = nullptr;
    bool bound = false, inited = false;
    int force_general = -1;
    int fused_mode = -1;        // -1: fused pt_mcs where eligible, 0: always separate launches
    int track = 0;              // round-trip bookkeeping (NEXT-1), chosen before pt_init
    double p_ferro = 0.5;       // P(J = +1) of Eq. (2) (NEXT-4), chosen before pt_init
    bool fast = false;
    Params P{};
    std::vector<double> betas;
    uint64_t seed = 0;
    uint32_t n_sweep = 0, n_exchange = 0, n_houdayer = 0;
    uint64_t n_passes = 0;      // PT passes since pt_init = swap attempts per pair (R20); NOT the Philox step counter
                                // n_exchange, which pt_set_counters overwrites on a resume
    bool q_small = false;       // fixed-point couplings with 2 D max|Jq| < 2^23 (gauss.cuh: accept_site<SMALL>)
    int sample_groups = -1;     // pt_set_sample_groups: -1 = automatic
    int pending_groups = 0;     // > 0: pt_set_spins_async left work of that many sample groups on the side streams
    bool async_check = false;   // the +-1 count of a pt_set_spins_async has not been read yet
    bool has_fixed = false;     // the workspace holds the int32 coupling arrays (PT_WS_FIXED_COUPLINGS)
    int ws_flags = 0;           // pt_set_workspace_flags: the optional parts the caller sized the workspace for
    int n_sm = 148, sweep_occ = 7;  // SMs of the device and resident k_sweep CTAs per SM, asked from the runtime in pt_init
    int phase_clocks = 0;       // pt_set_phase_clocks
    int max_clu = 1;            // max over t of the per-temperature cluster-move counts (NEXT-4, R36)
    uint64_t launches = 0;
    size_t stage_bytes = 0;
};

Context G;
char g_err[512] = "";

// Optional per-kernel-class timing with CUDA events on the bound stream (pt_set_profiling): every launch of
// a class is bracketed by two events; pt_get_kernel_times harvests them.  Classes: 0 sweep, 1 Houdayer,
// 2 exchange, 3 measurement, 4 fused MCS.
struct Profiler {
    bool on = false;
    std::vector<cudaEvent_t> free_events;
    struct Rec { int cls; cudaEvent_t a, b; };
    std::vector<Rec> pending;
    double ms[5] = {0, 0, 0, 0, 0};
    uint64_t n[5] = {0, 0, 0, 0, 0};
    cudaEvent_t get()
    {
        if (!free_events.empty()) { cudaEvent_t e = free_events.back(); free_events.pop_back(); return e; }
        cudaEvent_t e = nullptr;
        cudaEventCreate(&e);
        return e;
    }
    void harvest()
    {
        for (const Rec &r : pending) {
            float t = 0;
            if (cudaEventSynchronize(r.b) == cudaSuccess && cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) {
                ms[r.cls] += t;
                n[r.cls] += 1;
            }
            free_events.push_back(r.a);
            free_events.push_back(r.b);
        }
        pending.clear();
    }
};
Profiler PROF;

struct ProfScope {
    int cls;
    cudaStream_t st;
    cudaEvent_t a = nullptr;
    explicit ProfScope(int c, cudaStream_t stream = nullptr) : cls(c), st(stream ? stream : G.stream)
    {
        if (PROF.on) { a = PROF.get(); cudaEventRecord(a, st); }
    }
    ~ProfScope()
    {
        if (a) {
            cudaEvent_t b = PROF.get();
            cudaEventRecord(b, st);
            PROF.pending.push_back({cls, a, b});
        }
    }
};

int fail(int code, const char *fmt, ...)
{
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    return code;
}

#define CK(call)                                                                                       \
    do {                                                                                               \
        cudaError_t e_ = (call);                                                                       \
        if (e_ != cudaSuccess) return fail(PT_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_));      \
    } while (0)

int join_pending();

// every call that touches the state first lets the bound stream wait for what pt_set_spins_async left on the side streams
#define NEED_INIT()                                                                  \
    do {                                                                             \
        if (!G.inited) return fail(PT_ERR_STATE, "%s: pt_init has not been called", __func__); \
        if (G.pending_groups) { const int rcj_ = join_pending(); if (rcj_) return rcj_; }      \
    } while (0)
#define NEED_INIT_NOJOIN()                                                           \
    do {                                                                             \
        if (!G.inited) return fail(PT_ERR_STATE, "%s: pt_init has not been called", __func__); \
    } while (0)

int check_shape(int L, int d, int S, int T)
{
    if (d != 2 && d != 3) return fail(PT_ERR_ARG, "d must be 2 or 3 (got %d)", d);
    if (L < 2 || (L & 1)) return fail(PT_ERR_ARG, "L must be even and >= 2 (got %d): checkerboard needs a bipartite lattice", L);
    if (S < 1) return fail(PT_ERR_ARG, "n_samples must be >= 1 (got %d)", S);
    if (T < 1 || T > 65535) return fail(PT_ERR_ARG, "n_temps must be in [1, 65535] (got %d)", T);
    const double Nd = std::pow((double)L, d) * d;
    if (Nd > 2147483647.0) return fail(PT_ERR_ARG, "N*d overflows int32");
    if (S > 65535) return fail(PT_ERR_ARG, "n_samples must be <= 65535 per context (got %d): shard larger sets with pt_init_shard", S);
    // the sweep kernel keeps a sample's coupling bits and at least one replica in shared memory
    const double W = std::ceil(std::pow((double)L, d) / 64.0);
    if ((2.0 * 2 * d * W + 2 * W + 8) * 4 > 227.0 * 1024)
        return fail(PT_ERR_ARG, "lattice too large: %.0f KiB of coupling bits per sample do not fit in shared memory", 2.0 * 2 * d * W * 4 / 1024);
    return PT_OK;
}

size_t align_up(size_t x) { return (x + 255) & ~(size_t)255; }

// THR(x) = min(2^32-1, floor(2^32 exp(x)))   (R5, R6)
uint32_t THR(double x)
{
    const double v = std::floor(std::ldexp(std::exp(x), 32));
    if (v >= 4294967295.0) return 4294967295u;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

double thrX_arg(const std::vector<double> &b, int t, uint64_t m) { return -(std::fabs(b[t + 1] - b[t]) * (double)(4 * m)); }

// entries per pair of the stored swap table: the prefix on which any pair's threshold is non-zero
uint32_t swap_stride(const std::vector<double> &b, int d, long N)
{
    const uint64_t m_max = (uint64_t)d * (uint64_t)N / 2;     // |dE| <= 2 d N
    uint64_t need = 1;
    for (size_t t = 0; t + 1 < b.size(); ++t) {
        const double db = std::fabs(b[t + 1] - b[t]);
        if (db == 0.0) continue;                              // sgn = 0: always accepted, table unused
        uint64_t lo = 0, hi = m_max + 1;                      // first m with THR == 0 (THR is non-increasing in m)
        while (lo < hi) {
            const uint64_t mid = (lo + hi) / 2;
            if (THR(-(db * (double)(4 * mid))) == 0) hi = mid; else lo = mid + 1;
        }
        if (lo > need) need = lo;
    }
    if (need > m_max + 1) need = m_max + 1;
    return (uint32_t)need;
}

constexpr size_t kStageCap = (size_t)16 << 20;

struct Carve {
    size_t off = 0;
    template <class T> T *take(void *base, size_t n)
    {
        T *p = base ? (T *)((char *)base + off) : nullptr;
        off = align_up(off + n * sizeof(T));
        return p;
    }
};

// Lay the device arrays out in the workspace; with base == nullptr only the total size is computed.
// fixed: also the int32 coupling arrays of the fixed-point model (NEXT-3), 24 bytes per bond more than the bit arrays
// stage_extra: bytes by which the staging area may grow beyond its bounded minimum (never beyond one whole int8 state)
size_t carve(void *base, int L, int d, int S, int T, uint32_t strideX, DevPtrs *out, size_t *stage_bytes, bool fixed,
             size_t stage_extra = 0)
{
    const size_t N = (d == 2) ? (size_t)L * L : (size_t)L * L * L;
    const size_t W = (size_t)words_per_colour((int)N);
    const size_t R = (size_t)S * 2 * T;
    Carve c;
    DevPtrs p{};
    p.spin = c.take<uint32_t>(base, R * 2 * W);
    p.Jn = c.take<uint32_t>(base, (size_t)S * 2 * 2 * d * W);
    p.E = c.take<int32_t>(base, R);
    p.tos = c.take<int32_t>(base, R);
    p.sot = c.take<int32_t>(base, R);
    p.thrM = c.take<uint32_t>(base, (size_t)T * 4);
    p.thrX = c.take<uint32_t>(base, (size_t)(T > 1 ? T - 1 : 1) * strideX);
    p.sgn = c.take<int32_t>(base, (size_t)T);
    p.accepts = c.take<unsigned long long>(base, (size_t)S * 2 * T);
    p.last = c.take<uint32_t>(base, (size_t)S * T);
    p.cum = c.take<unsigned long long>(base, (size_t)S * T);
    p.outE = c.take<int32_t>(base, R);
    p.outQ = c.take<int32_t>(base, (size_t)S * T);
    p.outQL = c.take<int32_t>(base, (size_t)S * T);
    p.mismatch = c.take<int>(base, 64);
    if (fixed) {
        p.JqNat = c.take<int32_t>(base, (size_t)S * d * N);
        p.Jdev = c.take<int32_t>(base, (size_t)S * 2 * 2 * d * 32 * W);
    }
    p.betasD = c.take<double>(base, (size_t)T);
    p.absdb = c.take<double>(base, (size_t)T);
    p.swapSlope = c.take<float>(base, (size_t)T);
    p.rtLabel = c.take<uint32_t>(base, R);
    p.rtStart = c.take<uint32_t>(base, R);
    p.rtTrips = c.take<uint32_t>(base, R);
    p.rtSum = c.take<unsigned long long>(base, (size_t)S * 2 * 32);
    p.rtCnt = c.take<unsigned long long>(base, (size_t)S * 2 * 32);
    p.nclu = c.take<int32_t>(base, (size_t)T);
    p.tcold = c.take<int32_t>(base, (size_t)T);
    p.phaseClk = c.take<unsigned long long>(base, 4);
    // staging: a BOUNDED buffer through which the int8 boundary (state get / set, init draws) and the host variant of the
    // overlap profile pass in chunks of whole samples: kStageCap bytes, or one sample's worth where that is more
    const size_t per_sample = std::max(std::max((size_t)2 * T * N, (size_t)d * N), (size_t)T * d * L * 4);
    const size_t sb_min = std::max(std::min((size_t)S * per_sample, kStageCap), per_sample);
    const size_t sb = std::min((size_t)S * per_sample, sb_min + stage_extra);
    p.stage = c.take<int8_t>(base, sb);
    if (out) *out = p;
    if (stage_bytes) *stage_bytes = sb;
    return c.off;
}

// upper bound of strideX used for sizing before the betas are known: the full table
uint32_t full_stride(int L, int d)
{
    const uint64_t N = (d == 2) ? (uint64_t)L * L : (uint64_t)L * L * L;
    return (uint32_t)((uint64_t)d * N / 2 + 1);
}

bool fast_supported(int L, int d)
{
    if (L < 8 || (L & (L - 1))) return false;
    int lg = 0;
    while ((1 << lg) < L) ++lg;
#ifdef PTG_DEV_D
    return d == PTG_DEV_D && lg == PTG_DEV_LG;      // development build: one fast lattice only (build.py)
#endif
    return d == 2 ? (lg >= 3 && lg <= 8) : (lg >= 3 && lg <= 5);
}

int grid_for(long total, int block) { return (int)std::min<long>((total + block - 1) / block, 148L * 32); }

// Run `body` with `lat` bound to the lattice implementation of the current problem.
#define FAST_CASE(DD, LG)                                  \
    if (G.P.D == DD && G.P.L == (1 << LG)) {               \
        FastLat<DD, LG> lat;                               \
        body(lat);                                         \
        return;                                            \
    }

template <class F> void with_lattice(F body)
{
#ifdef PTG_DEV_D
    if (G.fast) { FAST_CASE(PTG_DEV_D, PTG_DEV_LG) }
    GenLat<PTG_DEV_D> dev_lat(G.P.L);
    body(dev_lat);
#else
    if (G.fast) {
        FAST_CASE(2, 3) FAST_CASE(2, 4) FAST_CASE(2, 5) FAST_CASE(2, 6) FAST_CASE(2, 7) FAST_CASE(2, 8)
        FAST_CASE(3, 3) FAST_CASE(3, 4) FAST_CASE(3, 5)
    }
    if (G.P.D == 2) { GenLat<2> lat(G.P.L); body(lat); }
    else            { GenLat<3> lat(G.P.L); body(lat); }
#endif
}

template <class K> cudaError_t allow_smem(K kernel, size_t bytes)
{
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

// Every launch function takes the problem it works on -- the whole bound problem G.P, or a VIEW of a contiguous range of
// its samples (sub_view) -- and the stream it is issued on: the separate-kernel path of pt_mcs runs sample groups on
// side streams so that one group's cluster and exchange kernels fill the SMs another group's sweep leaves idle.
cudaError_t launch_energy(int mode, const Params &P = G.P, cudaStream_t st = nullptr)
{
    if (!st) st = G.stream;
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        const long reps = (long)P.S * 2 * P.T;
        const int wpb = 4;
        if (P.gauss) k_energy_q<<<(unsigned)((reps + wpb - 1) / wpb), wpb * 32, 0, st>>>(lat, P, mode);
        else k_energy<<<(unsigned)((reps + wpb - 1) / wpb), wpb * 32, 0, st>>>(lat, P, mode);
        ++G.launches;
        err = cudaGetLastError();
    });
    return err;
}

// replicas per CTA of the sweep kernel (128 threads): the largest divisor of 2T with R*W <= 512 work items
int sweep_group(int T, int W)
{
    int best = 1;
    for (int R = 1; R <= 2 * T; ++R)
        if ((2 * T) % R == 0 && (long)R * W <= 512) best = R;
    return best;
}

cudaError_t launch_sweep(int n, uint32_t step0, const Params &P = G.P, cudaStream_t st = nullptr)
{
    if (!st) st = G.stream;
    ProfScope prof(0, st);
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        const int W = P.W, D = P.D;
        const int R = sweep_group(P.T, W);
        if (P.gauss) {
            const size_t smq = ((size_t)R * 2 * W + 3 * (size_t)R) * 4;
            auto kq = G.q_small ? k_sweep_q<LAT, true> : k_sweep_q<LAT, false>;
            err = allow_smem(kq, smq);
            if (err != cudaSuccess) return;
            dim3 gq((unsigned)(2 * P.T / R), (unsigned)P.S);
            kq<<<gq, 128, smq, st>>>(lat, P, R, step0, n);
            ++G.launches;
            err = cudaGetLastError();
            return;
        }
        const size_t smem = ((size_t)2 * 2 * D * W + (size_t)R * 2 * W + (size_t)R * 4 + (size_t)R) * 4;
        err = allow_smem(k_sweep<LAT>, smem);
        if (err != cudaSuccess) return;
        dim3 grid((unsigned)(2 * P.T / R), (unsigned)P.S);
        k_sweep<LAT><<<grid, 128, smem, st>>>(lat, P, R, step0, n);
        ++G.launches;
        err = cudaGetLastError();
    });
    return err;
}

cudaError_t launch_exchange(uint32_t step, const Params &P = G.P, cudaStream_t st = nullptr)
{
    if (!st) st = G.stream;
    ProfScope prof(2, st);
    const int T = P.T;
    const long chains = (long)P.S * 2;
    int wpb = 4;
    while (wpb > 1 && (size_t)wpb * 4 * T * 4 > 64 * 1024) wpb >>= 1;
    const size_t smem = (size_t)wpb * 4 * T * 4 + (T <= kExchangeTableT ? (size_t)wpb * T * T : 0);      // + the decision table
    if ((size_t)wpb * 4 * T * 4 > 64 * 1024) {      // very long ladders: walk on global scratch instead of shared memory
        k_exchange<true><<<(unsigned)chains, 32, 0, st>>>(P, step);
    } else {
        cudaError_t err = allow_smem(k_exchange<false>, smem);
        if (err != cudaSuccess) return err;
        k_exchange<false><<<(unsigned)((chains + wpb - 1) / wpb), wpb * 32, smem, st>>>(P, step);
    }
    ++G.launches;
    return cudaGetLastError();
}

// One launch per move number (R36): move j touches the temperatures with nclu[t] > j; a default run makes one launch.
cudaError_t launch_houdayer(uint32_t step, const Params &P, cudaStream_t st)
{
    ProfScope prof(1, st);
    cudaError_t err = cudaSuccess;
    for (uint32_t move = 0; move < (uint32_t)std::max(G.max_clu, 1) && err == cudaSuccess; ++move)
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        if constexpr (LAT::kFast) {
            // one warp per pair; kPairScratchWords words of shared memory per warp
            int wpb = 4;
            while (wpb > 1 && (size_t)wpb * kPairScratchWords<LAT> * 4 > 96 * 1024) wpb >>= 1;
            const size_t smem = (size_t)wpb * kPairScratchWords<LAT> * 4;
            err = allow_smem(k_houdayer<LAT>, smem);
            if (err != cudaSuccess) return;
            const long pairs = (long)P.S * P.T;
            k_houdayer<LAT><<<(unsigned)((pairs + wpb - 1) / wpb), wpb * 32, smem, st>>>(lat, P, step, move);
        } else {
            const int threads = 128;
            const size_t smem = ((size_t)4 * P.W + 2 * (threads / 32) + 2) * 4;
            err = allow_smem(k_houdayer_gen<LAT>, smem);
            if (err != cudaSuccess) return;
            dim3 grid((unsigned)P.T, (unsigned)P.S);
            k_houdayer_gen<LAT><<<grid, threads, smem, st>>>(lat, P, step, move);
        }
        ++G.launches;
        err = cudaGetLastError();
    });
    return err;
}

// groups of a sample-chunked upload (pt_set_spins_async): the grouping of the MCS loop that follows it, so that every
// group's chain copy -> pack -> energy -> MCS kernels stays on one stream
int upload_groups();

// The cluster kernels compute delta from the +-J bit couplings; with fixed-point couplings the cluster itself is the
// same (it depends on q only) and the energies are simply recomputed from scratch, which for integers is the same number.
// multi-cluster variant (R37): one CTA per pair, labels in shared memory
// CTA size of k_houdayer_multi: ~32 sites per thread, 64..512 threads (measured: C2 best at 64, C5 at 512)
int multi_threads()
{
    int t = 64;
    while (t < 512 && (long)t * 32 < (long)G.P.N) t <<= 1;
    return t;
}

size_t multi_smem_bytes(int threads) { return ((size_t)4 * G.P.W + 2 * (threads / 32) + 2 + (size_t)G.P.N) * 4 + (size_t)G.P.N * 2 + 16; }

cudaError_t launch_houdayer_multi(uint32_t step, const Params &P, cudaStream_t st)
{
    ProfScope prof(1, st);
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        const int threads = multi_threads();
        const size_t smem = multi_smem_bytes(threads);
        err = allow_smem(k_houdayer_multi<LAT>, smem);
        if (err != cudaSuccess) return;
        dim3 grid((unsigned)P.T, (unsigned)P.S);
        k_houdayer_multi<LAT><<<grid, threads, smem, st>>>(lat, P, step);
        ++G.launches;
        err = cudaGetLastError();
    });
    return err;
}

// mode 1: single-cluster moves (R36 counts), mode 2: multi-cluster (R37)
cudaError_t launch_houdayer_any(int mode, uint32_t step, const Params &P = G.P, cudaStream_t st = nullptr)
{
    if (!st) st = G.stream;
    cudaError_t err = (mode == 2) ? launch_houdayer_multi(step, P, st) : launch_houdayer(step, P, st);
    if (err == cudaSuccess && P.gauss) err = launch_energy(0, P, st);
    return err;
}

// The problem restricted to samples [s0, s0 + n): every per-sample array advanced, the global sample index with it.
Params sub_view(const Params &P, int s0, int n)
{
    Params V = P;
    const size_t s = (size_t)s0, R = s * 2 * P.T;
    V.S = n;
    V.g0 = P.g0 + (uint32_t)s0;
    V.d.spin += R * 2 * P.W;
    V.d.Jn += s * 2 * 2 * P.D * P.W;
    V.d.E += R; V.d.tos += R; V.d.sot += R; V.d.outE += R;
    V.d.accepts += s * 2 * (size_t)(P.T - 1);
    V.d.last += s * P.T; V.d.cum += s * P.T; V.d.outQ += s * P.T; V.d.outQL += s * P.T;
    if (V.d.JqNat) {
        V.d.JqNat += s * P.D * P.N;
        V.d.Jdev += s * 2 * 2 * P.D * 32 * P.W;
    }
    V.d.rtLabel += R; V.d.rtStart += R; V.d.rtTrips += R;
    V.d.rtSum += s * 2 * 32; V.d.rtCnt += s * 2 * 32;
    return V;
}

// Side streams of the separate-kernel MCS loop (created on first use, never destroyed before process exit) and the
// events that fork them from / join them to the caller's stream.
constexpr int kMaxGroups = 8;
cudaStream_t g_side[kMaxGroups] = {};
cudaEvent_t g_fork = nullptr, g_join[kMaxGroups] = {};

cudaError_t ensure_side_streams(int n)
{
    cudaError_t e = cudaSuccess;
    if (!g_fork) e = cudaEventCreateWithFlags(&g_fork, cudaEventDisableTiming);
    for (int k = 1; k < n && e == cudaSuccess; ++k) {
        if (!g_side[k]) e = cudaStreamCreateWithFlags(&g_side[k], cudaStreamNonBlocking);
        if (e == cudaSuccess && !g_join[k]) e = cudaEventCreateWithFlags(&g_join[k], cudaEventDisableTiming);
    }
    return e;
}

// sample groups of a separate-kernel pt_mcs call.  Automatic: one group per wave of sweep CTAs (SMs x resident CTAs per SM,
// both from the runtime: 148 x 7 on a B200), at most kMaxGroups -- measured on C5 (5.9 waves): 1 group 733, 2: 811, 4: 852,
// 6: 862, 8: 862 flips/ns.
int mcs_groups()
{
    if (G.sample_groups > 0) return std::min(std::min(G.sample_groups, kMaxGroups), G.P.S);
    const long ctas = (long)G.P.S * (2 * G.P.T / sweep_group(G.P.T, G.P.W));     // sweep CTAs of the whole problem
    const long wave = (long)G.n_sm * G.sweep_occ;
    const long waves = (ctas + wave - 1) / wave;
    return (int)std::max(1L, std::min<long>(std::min<long>(waves, kMaxGroups), G.P.S));
}

struct Groups {
    int n = 1;
    std::vector<Params> view;
    std::vector<cudaStream_t> st;
    std::vector<int> s0;
};

// cut the bound problem into n contiguous sample ranges; group 0 on the bound stream, the others on side streams
int make_groups(int n, Groups &g)
{
    g.n = n;
    g.view.resize((size_t)n);
    g.st.assign((size_t)n, G.stream);
    g.s0.resize((size_t)n);
    for (int k = 0; k < n; ++k) {
        const int a0 = (int)((long)G.P.S * k / n), a1 = (int)((long)G.P.S * (k + 1) / n);
        g.view[k] = sub_view(G.P, a0, a1 - a0);
        g.s0[k] = a0;
    }
    if (n > 1) {
        CK(ensure_side_streams(n));
        for (int k = 1; k < n; ++k) g.st[k] = g_side[k];
    }
    return PT_OK;
}

// the side streams start after everything queued on the bound stream so far
int fork_groups(const Groups &g)
{
    if (g.n > 1) {
        CK(cudaEventRecord(g_fork, G.stream));
        for (int k = 1; k < g.n; ++k) CK(cudaStreamWaitEvent(g.st[k], g_fork, 0));
    }
    return PT_OK;
}

// the bound stream waits for the side streams
int join_groups(int n)
{
    for (int k = 1; k < n; ++k) {
        CK(cudaEventRecord(g_join[k], g_side[k]));
        CK(cudaStreamWaitEvent(G.stream, g_join[k], 0));
    }
    return PT_OK;
}

cudaError_t launch_measure(int32_t *Q, int32_t *QL)
{
    ProfScope prof(3);
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        if (G.P.W <= 128) {          // small lattices: one warp per pair, four pairs per CTA
            const long pairs = (long)G.P.S * G.P.T;
            k_measure_warp<LAT><<<(unsigned)((pairs + 3) / 4), 128, (size_t)4 * G.P.W * 4, G.stream>>>(lat, G.P, Q, QL);
        } else {
            const size_t smem = ((size_t)G.P.W + 2) * 4;
            dim3 grid((unsigned)G.P.T, (unsigned)G.P.S);
            k_measure<LAT><<<grid, 128, smem, G.stream>>>(lat, G.P, Q, QL);
        }
        ++G.launches;
        err = cudaGetLastError();
    });
    return err;
}

// Fused MCS (mcs.cuh): one CTA per sample, 128 threads, up to 7 CTAs per SM.  Eligible on the fast path when the
// sample's state fits in shared memory with at least 4 CTAs per SM (else the separate kernels are faster).
constexpr int kMcsThreads = 128, kMcsMinBlocks = 7;

// One CTA per (sample, chain) instead of per sample: legal when the call makes no Houdayer moves (sweeps and PT passes
// never couple the two chains, R10) and worthwhile when a chain alone still fills the CTA (>= 4 work items per thread).
bool mcs_split_chains(int do_houdayer) { return !do_houdayer && (long)G.P.T * G.P.W >= 4L * kMcsThreads; }

bool mcs_fused_eligible(size_t *smem_out, int do_houdayer = 1, bool measure = false)
{
    if (!G.fast || G.fused_mode == 0) return false;
    const McsSmem lay(G.P.D, G.P.W, G.P.T, kMcsThreads / 32, 2 * G.P.W <= 32, mcs_split_chains(do_houdayer) ? 1 : 2,
                      G.P.gauss || measure);
    const size_t smem = (size_t)lay.words * 4;
    if (smem_out) *smem_out = smem;
    return (smem + 1024) * 4 <= 227 * 1024;
}

// the multi-cluster exchange inside the fused kernel: 2D L = 32, +-J couplings (houdayer_multi_quad)
bool mcs_multi_fused() { return G.fast && G.P.D == 2 && G.P.L == 32 && !G.P.gauss; }

cudaError_t launch_mcs(const McsArgs &a, const Params &P = G.P, cudaStream_t st = nullptr)
{
    if (!st) st = G.stream;
    ProfScope prof(4, st);
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        if constexpr (LAT::kFast) {
            size_t smem = 0;
            const bool meas = a.measure_every > 0;
            mcs_fused_eligible(&smem, a.do_houdayer, meas);
            // the fused measurement is instantiated for the +-J model only (pt_mcs_measure_device falls back otherwise)
            auto kern = !G.P.gauss ? (meas ? k_mcs<LAT, kMcsThreads, kMcsMinBlocks, 0, true> : k_mcs<LAT, kMcsThreads, kMcsMinBlocks, 0, false>)
                        : G.q_small ? k_mcs<LAT, kMcsThreads, kMcsMinBlocks, 1, false> : k_mcs<LAT, kMcsThreads, kMcsMinBlocks, 2, false>;
            if constexpr (QuadHoudayer<LAT>::kEligible) {
                if (a.do_houdayer == 2) kern = k_mcs<LAT, kMcsThreads, kMcsMinBlocks, 0, false, true>;
            }
            err = allow_smem(kern, smem);
            if (err != cudaSuccess) return;
            const unsigned grid = (unsigned)P.S * (a.split_chains ? 2u : 1u);
            kern<<<grid, kMcsThreads, smem, st>>>(lat, P, a);
            ++G.launches;
            err = cudaGetLastError();
        } else {
            err = cudaErrorInvalidValue;
        }
    });
    return err;
}

int d2h(void *dst, const void *src, size_t bytes)
{
    CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, G.stream));
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

// staged int8 spins of the samples of view P (src = their first byte in the staging area) -> bit words
int pack_spins(const Params &P, cudaStream_t st, const int8_t *src, int *bad)
{
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        if constexpr (LAT::kFast) {
            const long total = (long)P.S * 2 * P.T * P.W;
            k_pack_spins_fast<LAT><<<grid_for(total, 256), 256, 0, st>>>(P, src, bad);
        } else {
            Params V = P;
            V.d.stage = const_cast<int8_t *>(src);
            const long total = (long)P.S * 2 * P.T * 2 * P.W;
            if (bad) {
                const size_t n = (size_t)P.S * 2 * P.T * P.N;
                k_check_pm1<<<grid_for((long)((n + 15) / 16), 256), 256, 0, st>>>(src, n, bad);
                ++G.launches;
            }
            k_pack_spins<<<grid_for(total, 256), 256, 0, st>>>(V);
        }
        ++G.launches;
        err = cudaGetLastError();
    });
    CK(err);
    return PT_OK;
}

int pack_couplings(const Params &P)
{
    CK(cudaMemsetAsync(P.d.Jn, 0, (size_t)P.S * 2 * 2 * P.D * P.W * 4, G.stream));
    k_pack_couplings<<<grid_for((long)P.S * P.D * P.N, 256), 256, 0, G.stream>>>(P);
    ++G.launches;
    CK(cudaGetLastError());
    return PT_OK;
}

// fn(view, first sample, samples) over the bound problem's samples [s_lo, s_hi) in chunks whose bytes_per_sample each fit `avail`
template <class F> int for_chunks(size_t bytes_per_sample, size_t avail, int s_lo, int s_hi, F fn)
{
    const int step = (int)std::max<size_t>(1, avail / bytes_per_sample);
    for (int s0 = s_lo; s0 < s_hi; s0 += step) {
        const int n = std::min(step, s_hi - s0);
        const int rc = fn(sub_view(G.P, s0, n), s0, n);
        if (rc) return rc;
    }
    return PT_OK;
}

int join_pending()
{
    const int n = G.pending_groups;
    G.pending_groups = 0;
    return join_groups(n);
}

int upload_groups()
{
    if (G.sample_groups > 0) return std::min(std::min(G.sample_groups, kMaxGroups), G.P.S);
    if (!mcs_fused_eligible(nullptr, 1)) return mcs_groups();
    // fused path: a CTA's n_mcs steps take the same time however few CTAs share its SM, so more than two launches only
    // lengthen the tail (C2, 64 MiB + 50 MCS: 1 group 5.21 ms, 2: 5.09, 3: 5.39, 4: 5.75 per step end to end)
    const size_t bytes = (size_t)G.P.S * 2 * G.P.T * G.P.N;
    return (bytes >= ((size_t)32 << 20) && G.P.S >= 2) ? 2 : 1;
}

// the fused launch(es) of one pt_mcs / pt_mcs_measure_device call: one launch, or one per sample group where
// pt_set_spins_async left the samples' uploads on the group streams (every group's chain stays on its stream)
int run_fused(McsArgs a)
{
    const int NG = G.pending_groups > 1 ? G.pending_groups : 1;
    a.rec_S = G.P.S;
    a.rec_s0 = 0;
    if (NG == 1) {
        CK(launch_mcs(a));
        return PT_OK;
    }
    Groups g;
    int rc = make_groups(NG, g);
    if (rc) return rc;
    if ((rc = fork_groups(g))) return rc;
    rc = [&]() -> int {
        for (int k = 0; k < NG; ++k) {
            a.rec_s0 = g.s0[k];
            CK(launch_mcs(a, g.view[k], g.st[k]));
        }
        return PT_OK;
    }();
    G.pending_groups = 0;
    const int rcj = join_groups(NG);        // also after a failed launch: the side streams never stay forked
    return rc ? rc : rcj;
}

}  // namespace

// ============================================================================================================
extern "C" {

const char *pt_last_error(void) { return g_err; }

int pt_workspace_bytes(int L, int d, int n_samples, int n_temps, size_t *bytes_out)
{
    if (!bytes_out) return fail(PT_ERR_ARG, "bytes_out is NULL");
    const int rc = check_shape(L, d, n_samples, n_temps);
    if (rc) return rc;
    *bytes_out = carve(nullptr, L, d, n_samples, n_temps, full_stride(L, d), nullptr, nullptr, false);
    return PT_OK;
}

int pt_workspace_bytes_ex(int L, int d, int n_samples, int n_temps, int flags, size_t *bytes_out)
{
    if (!bytes_out) return fail(PT_ERR_ARG, "bytes_out is NULL");
    if (flags & ~(PT_WS_FIXED_COUPLINGS | PT_WS_FULL_STAGING)) return fail(PT_ERR_ARG, "unknown workspace flag");
    const int rc = check_shape(L, d, n_samples, n_temps);
    if (rc) return rc;
    *bytes_out = carve(nullptr, L, d, n_samples, n_temps, full_stride(L, d), nullptr, nullptr, (flags & PT_WS_FIXED_COUPLINGS) != 0,
                       (flags & PT_WS_FULL_STAGING) ? ~(size_t)0 >> 1 : 0);
    return PT_OK;
}

// nothing of an earlier problem may still run on the side streams when the workspace changes hands
static void drain_side_streams()
{
    for (int k = 1; k < kMaxGroups; ++k)
        if (g_side[k]) cudaStreamSynchronize(g_side[k]);
}

int pt_bind(void *device_workspace, size_t bytes, void *cuda_stream)
{
    if (!device_workspace) return fail(PT_ERR_ARG, "device_workspace is NULL");
    if (((uintptr_t)device_workspace & 255) != 0) return fail(PT_ERR_ARG, "device_workspace must be 256-byte aligned");
    if (G.bound && G.stream) cudaStreamSynchronize(G.stream);
    drain_side_streams();
    G = Context{};
    G.ws = device_workspace;
    G.ws_bytes = bytes;
    G.stream = (cudaStream_t)cuda_stream;
    G.bound = true;
    return PT_OK;
}

int pt_set_workspace_flags(int flags)
{
    if (!G.bound) return fail(PT_ERR_STATE, "pt_set_workspace_flags: no workspace bound");
    if (G.inited) return fail(PT_ERR_STATE, "pt_set_workspace_flags must precede pt_init (the workspace is laid out there)");
    if (flags & ~(PT_WS_FIXED_COUPLINGS | PT_WS_FULL_STAGING)) return fail(PT_ERR_ARG, "unknown workspace flag");
    G.ws_flags = flags;
    return PT_OK;
}

int pt_get_stage_bytes(size_t *bytes)
{
    NEED_INIT_NOJOIN();
    if (!bytes) return fail(PT_ERR_ARG, "bytes is NULL");
    *bytes = G.stage_bytes;
    return PT_OK;
}

int pt_is_dev_build(void)
{
#ifdef PTG_DEV_D
    return 1;
#else
    return 0;
#endif
}

int pt_force_general_path(int force)
{
    if (force != -1 && force != 0) return fail(PT_ERR_ARG, "force must be -1 or 0");
    if (G.inited) return fail(PT_ERR_STATE, "pt_force_general_path must precede pt_init");
    G.force_general = force;
    return PT_OK;
}

int pt_get_path(int *fast)
{
    NEED_INIT();
    if (fast) *fast = G.fast ? 1 : 0;
    return PT_OK;
}

int pt_init_shard(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed, uint32_t sample_offset)
{
    if (!G.bound) return fail(PT_ERR_STATE, "pt_init: no workspace bound (call pt_bind first)");
    G.inited = false;
    drain_side_streams();
    G.pending_groups = 0;
    G.async_check = false;
    int rc = check_shape(L, d, n_samples, n_temps);
    if (rc) return rc;
#ifdef PTG_DEV_D
    // development build (PTG_DEV_LATTICE): only lattices of this dimension were compiled; never run the other one on them
    if (d != PTG_DEV_D) return fail(PT_ERR_ARG, "development build for d = %d only (got d = %d): rebuild without PTG_DEV_LATTICE", PTG_DEV_D, d);
#endif
    if (!betas) return fail(PT_ERR_ARG, "betas is NULL");
    for (int t = 0; t < n_temps; ++t)
        if (!std::isfinite(betas[t]) || betas[t] < 0.0) return fail(PT_ERR_ARG, "betas[%d] is negative or not finite", t);
    if ((uint64_t)sample_offset + (uint64_t)n_samples > 4294967296ull)
        return fail(PT_ERR_ARG, "sample_offset + n_samples overflows 2^32");

    G.betas.assign(betas, betas + n_temps);
    G.seed = seed;
    Params &P = G.P;
    P = Params{};
    P.L = L; P.D = d; P.S = n_samples; P.T = n_temps;
    P.N = (d == 2) ? L * L : L * L * L;
    P.NH = P.N / 2;
    P.W = words_per_colour(P.N);
    P.g0 = sample_offset;
    P.rk = make_round_keys((uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32));
    P.strideX = swap_stride(G.betas, d, P.N);
    P.track = G.track;
    P.thrJ = (unsigned long long)std::floor(std::ldexp(G.p_ferro, 32));
    // the int32 coupling arrays of the fixed-point model are laid out only where the caller asked for them
    // (pt_set_workspace_flags); spare bytes never decide it
    G.has_fixed = (G.ws_flags & PT_WS_FIXED_COUPLINGS) != 0;
    const size_t need = carve(nullptr, L, d, n_samples, n_temps, P.strideX, nullptr, nullptr, G.has_fixed);
    if (need > G.ws_bytes)
        return fail(PT_ERR_STATE, "workspace too small: %zu bytes bound, %zu needed%s", G.ws_bytes, need,
                    G.has_fixed ? " (with PT_WS_FIXED_COUPLINGS)" : "");
    // whatever the caller bound beyond the minimum enlarges the staging area (PT_WS_FULL_STAGING: a whole int8 state)
    carve(G.ws, L, d, n_samples, n_temps, P.strideX, &P.d, &G.stage_bytes, G.has_fixed, (G.ws_bytes - need) & ~(size_t)255);
    if ((G.ws_flags & PT_WS_FULL_STAGING) && G.stage_bytes < (size_t)n_samples * 2 * n_temps * (size_t)P.N)
        return fail(PT_ERR_STATE, "workspace too small for PT_WS_FULL_STAGING: staging area %zu bytes, whole int8 state %zu",
                    G.stage_bytes, (size_t)n_samples * 2 * n_temps * (size_t)P.N);
    G.fast = (G.force_general != 0) && fast_supported(L, d);
    {   // what one wave of sweep CTAs is on THIS device (mcs_groups)
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n > 0)
            G.n_sm = n;
        with_lattice([&](auto lat) {
            using LAT = decltype(lat);
            const int R = sweep_group(P.T, P.W);
            const size_t smem = ((size_t)2 * 2 * P.D * P.W + (size_t)R * 2 * P.W + (size_t)R * 4 + (size_t)R) * 4;
            int nb = 0;
            if (allow_smem(k_sweep<LAT>, smem) == cudaSuccess &&
                cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, k_sweep<LAT>, 128, smem) == cudaSuccess && nb > 0)
                G.sweep_occ = nb;
        });
        cudaGetLastError();      // a failed query must not poison the calls that follow
    }
    G.n_sweep = G.n_exchange = G.n_houdayer = 0;
    G.n_passes = 0;
    G.max_clu = 1;
    {
        const std::vector<int32_t> ones((size_t)n_temps, 1);
        CK(cudaMemcpyAsync(P.d.nclu, ones.data(), ones.size() * 4, cudaMemcpyHostToDevice, G.stream));
        std::vector<int32_t> cold((size_t)n_temps);
        for (int t = 0; t < n_temps; ++t) cold[t] = t;
        std::stable_sort(cold.begin(), cold.end(), [&](int a, int b) { return betas[a] > betas[b]; });
        CK(cudaMemcpyAsync(P.d.tcold, cold.data(), cold.size() * 4, cudaMemcpyHostToDevice, G.stream));
        CK(cudaStreamSynchronize(G.stream));
    }

    // acceptance tables on the host, in double (R5, R6)
    std::vector<uint32_t> thrM((size_t)n_temps * 4, 0u);
    for (int t = 0; t < n_temps; ++t)
        for (int k = 1; k <= d; ++k) thrM[(size_t)t * 4 + (k - 1)] = THR(-(betas[t] * (double)(4 * k)));
    std::vector<uint32_t> thrX((size_t)(n_temps > 1 ? n_temps - 1 : 1) * P.strideX, 0u);
    std::vector<int32_t> sgn((size_t)n_temps, 0);
    for (int t = 0; t + 1 < n_temps; ++t) {
        sgn[t] = (betas[t + 1] > betas[t]) - (betas[t + 1] < betas[t]);
        for (uint32_t m = 0; m < P.strideX; ++m) thrX[(size_t)t * P.strideX + m] = THR(thrX_arg(G.betas, t, m));
    }
    CK(cudaMemcpyAsync(P.d.thrM, thrM.data(), thrM.size() * 4, cudaMemcpyHostToDevice, G.stream));
    CK(cudaMemcpyAsync(P.d.thrX, thrX.data(), thrX.size() * 4, cudaMemcpyHostToDevice, G.stream));
    CK(cudaMemcpyAsync(P.d.sgn, sgn.data(), sgn.size() * 4, cudaMemcpyHostToDevice, G.stream));
    std::vector<double> absdb((size_t)n_temps, 0.0);
    for (int t = 0; t + 1 < n_temps; ++t) absdb[t] = std::fabs(betas[t + 1] - betas[t]);
    CK(cudaMemcpyAsync(P.d.betasD, betas, (size_t)n_temps * 8, cudaMemcpyHostToDevice, G.stream));
    CK(cudaMemcpyAsync(P.d.absdb, absdb.data(), (size_t)n_temps * 8, cudaMemcpyHostToDevice, G.stream));
    CK(cudaStreamSynchronize(G.stream));       // the host vectors go out of scope
    CK(cudaMemsetAsync(P.d.accepts, 0, (size_t)P.S * 2 * P.T * 8, G.stream));
    CK(cudaMemsetAsync(P.d.last, 0, (size_t)P.S * P.T * 4, G.stream));
    CK(cudaMemsetAsync(P.d.cum, 0, (size_t)P.S * P.T * 8, G.stream));
    CK(cudaMemsetAsync(P.d.mismatch, 0, 64 * sizeof(int), G.stream));
    CK(cudaMemsetAsync(P.d.rtSum, 0, (size_t)P.S * 2 * 32 * 8, G.stream));
    CK(cudaMemsetAsync(P.d.rtCnt, 0, (size_t)P.S * 2 * 32 * 8, G.stream));

    // couplings, spins (Philox domains 1, 2), identity permutations, energies
    rc = for_chunks((size_t)P.D * P.N, G.stage_bytes, 0, P.S, [&](const Params &V, int, int) {
        k_draw_couplings<<<grid_for((long)V.S * V.D * (V.N / 4), 256), 256, 0, G.stream>>>(V);
        ++G.launches;
        CK(cudaGetLastError());
        return pack_couplings(V);
    });
    if (rc) return rc;
    rc = for_chunks((size_t)2 * P.T * P.N, G.stage_bytes, 0, P.S, [&](const Params &V, int, int) {
        k_draw_spins<<<grid_for((long)V.S * 2 * V.T * (V.N / 4), 256), 256, 0, G.stream>>>(V);
        ++G.launches;
        CK(cudaGetLastError());
        return pack_spins(V, G.stream, V.d.stage, nullptr);
    });
    if (rc) return rc;
    k_identity_perm<<<grid_for((long)P.S * 2 * P.T, 256), 256, 0, G.stream>>>(P);
    ++G.launches;
    CK(cudaGetLastError());
    CK(launch_energy(0));
    CK(cudaStreamSynchronize(G.stream));
    G.inited = true;
    return PT_OK;
}

int pt_init(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed)
{
    return pt_init_shard(L, d, n_samples, n_temps, betas, seed, 0u);
}

int pt_free(void)
{
    if (G.bound && G.stream) cudaStreamSynchronize(G.stream);
    drain_side_streams();
    G.pending_groups = 0;
    G.inited = false;
    return PT_OK;
}

// ---- updates ---------------------------------------------------------------------------------------------

int pt_sweep(int n)
{
    NEED_INIT();
    if (n < 0) return fail(PT_ERR_ARG, "pt_sweep: n must be >= 0");
    if ((uint64_t)G.n_sweep + (uint64_t)n > 4294967295ull) return fail(PT_ERR_OVERFLOW, "sweep counter would overflow");
    if (n == 0) return PT_OK;
    CK(launch_sweep(n, G.n_sweep));
    G.n_sweep += (uint32_t)n;
    return PT_OK;
}

int pt_exchange(void)
{
    NEED_INIT();
    if (G.n_exchange == 4294967295u) return fail(PT_ERR_OVERFLOW, "exchange counter would overflow");
    CK(launch_exchange(G.n_exchange));
    G.n_exchange += 1;
    G.n_passes += 1;
    return PT_OK;
}

int houdayer_step(void)
{
    NEED_INIT();
    if (G.n_houdayer == 4294967295u) return fail(PT_ERR_OVERFLOW, "Houdayer counter would overflow");
    CK(launch_houdayer_any(1, G.n_houdayer));
    G.n_houdayer += 1;
    return PT_OK;
}

int houdayer_multi_step(void)
{
    NEED_INIT();
    if (G.n_houdayer == 4294967295u) return fail(PT_ERR_OVERFLOW, "Houdayer counter would overflow");
    if (multi_smem_bytes(multi_threads()) > 227 * 1024)
        return fail(PT_ERR_ARG, "houdayer_multi_step: %d sites of labels do not fit in shared memory", G.P.N);
    CK(launch_houdayer_any(2, G.n_houdayer));
    G.n_houdayer += 1;
    return PT_OK;
}

int pt_set_cluster_moves(const int32_t *n_clu)
{
    NEED_INIT();
    std::vector<int32_t> v((size_t)G.P.T, 1);
    int mx = 1;
    if (n_clu) {
        mx = 0;
        for (int t = 0; t < G.P.T; ++t) {
            if (n_clu[t] < 0 || n_clu[t] > 65535) return fail(PT_ERR_ARG, "pt_set_cluster_moves: n_clu[%d] = %d not in [0, 65535]", t, n_clu[t]);
            v[t] = n_clu[t];
            mx = std::max(mx, (int)n_clu[t]);
        }
    }
    CK(cudaMemcpyAsync(G.P.d.nclu, v.data(), v.size() * 4, cudaMemcpyHostToDevice, G.stream));
    CK(cudaStreamSynchronize(G.stream));
    G.max_clu = mx;
    return PT_OK;
}

int pt_mcs(int n_mcs, int n_metro, int do_houdayer, int do_exchange)
{
    NEED_INIT_NOJOIN();
    if (n_mcs < 0 || n_metro < 0) return fail(PT_ERR_ARG, "pt_mcs: n_mcs and n_metro must be >= 0");
    if (do_houdayer < 0 || do_houdayer > 2) return fail(PT_ERR_ARG, "pt_mcs: do_houdayer must be 0, 1 (single-cluster) or 2 (multi-cluster)");
    if (do_houdayer == 2 && multi_smem_bytes(multi_threads()) > 227 * 1024)
        return fail(PT_ERR_ARG, "pt_mcs: %d sites of labels do not fit in shared memory (multi-cluster)", G.P.N);
    const uint64_t M = (uint64_t)n_mcs;
    if ((uint64_t)G.n_sweep + M * (uint64_t)n_metro > 4294967295ull ||
        (do_exchange && (uint64_t)G.n_exchange + M > 4294967295ull) ||
        (do_houdayer && (uint64_t)G.n_houdayer + M > 4294967295ull))
        return fail(PT_ERR_OVERFLOW, "a step counter would overflow");
    if (n_mcs == 0 || (n_metro == 0 && !do_houdayer && !do_exchange)) return PT_OK;
    if ((do_houdayer != 2 || mcs_multi_fused()) && mcs_fused_eligible(nullptr, do_houdayer)) {
        const McsArgs a{n_mcs, n_metro, do_houdayer, do_exchange ? 1 : 0, mcs_split_chains(do_houdayer) ? 1 : 0,
                        G.max_clu, G.n_sweep, G.n_houdayer, G.n_exchange, 0, nullptr, nullptr, G.phase_clocks, 0, 0};
        const int rcf = run_fused(a);
        if (rcf) return rcf;
        G.n_sweep += (uint32_t)(M * (uint64_t)n_metro);
        if (do_houdayer) G.n_houdayer += (uint32_t)M;
        if (do_exchange) { G.n_exchange += (uint32_t)M; G.n_passes += M; }
        return PT_OK;
    }
    // Separate kernels.  Samples never interact (P:7), so the problem is cut into groups of samples, each
    // running its own sweep -> cluster -> exchange chain on its own stream: while one group's cluster kernel drains (a few
    // long pairs, low occupancy) or its exchange kernel walks its ladders (latency-bound, a handful of warps), another
    // group's sweep fills the SMs.  Group 0 runs on the caller's stream; the side streams start after everything queued
    // on it so far and it waits for them before the call returns.  Results do not depend on the grouping (pin P8).
    const int NG = mcs_groups();
    if (G.pending_groups && G.pending_groups != NG) { const int rcj = join_pending(); if (rcj) return rcj; }
    Groups g;
    int rcg = make_groups(NG, g);
    if (rcg) return rcg;
    if ((rcg = fork_groups(g))) return rcg;
    rcg = [&]() -> int {
        for (int m = 0; m < n_mcs; ++m)
            for (int k = 0; k < NG; ++k) {
                if (n_metro > 0) CK(launch_sweep(n_metro, G.n_sweep + (uint32_t)m * (uint32_t)n_metro, g.view[k], g.st[k]));
                if (do_houdayer) CK(launch_houdayer_any(do_houdayer, G.n_houdayer + (uint32_t)m, g.view[k], g.st[k]));
                if (do_exchange) CK(launch_exchange(G.n_exchange + (uint32_t)m, g.view[k], g.st[k]));
            }
        return PT_OK;
    }();
    G.pending_groups = 0;
    const int rcj = join_groups(NG);        // also after a failed launch: the side streams never stay forked
    if (rcg) return rcg;
    if (rcj) return rcj;
    G.n_sweep += (uint32_t)(M * (uint64_t)n_metro);
    if (do_houdayer) G.n_houdayer += (uint32_t)M;
    if (do_exchange) { G.n_exchange += (uint32_t)M; G.n_passes += M; }
    return PT_OK;
}

int pt_mcs_measure_device(int n_mcs, int n_metro, int do_houdayer, int do_exchange, int measure_every, int32_t *Q_rec_dev,
                          int32_t *QL_rec_dev)
{
    NEED_INIT_NOJOIN();
    if (measure_every < 1) return fail(PT_ERR_ARG, "pt_mcs_measure_device: measure_every must be >= 1");
    if (!Q_rec_dev) return fail(PT_ERR_ARG, "pt_mcs_measure_device: Q_rec_dev is NULL");
    if (n_mcs < 0 || n_metro < 0) return fail(PT_ERR_ARG, "pt_mcs_measure_device: n_mcs and n_metro must be >= 0");
    if (do_houdayer < 0 || do_houdayer > 2) return fail(PT_ERR_ARG, "pt_mcs_measure_device: do_houdayer must be 0, 1 or 2");
    const size_t stride = (size_t)G.P.S * G.P.T;
    const uint64_t M = (uint64_t)n_mcs;
    // refused before anything runs, whichever path serves the call: the state is left unchanged (R21)
    if ((uint64_t)G.n_sweep + M * (uint64_t)n_metro > 4294967295ull ||
        (do_exchange && (uint64_t)G.n_exchange + M > 4294967295ull) ||
        (do_houdayer && (uint64_t)G.n_houdayer + M > 4294967295ull))
        return fail(PT_ERR_OVERFLOW, "a step counter would overflow");
    // ONE launch for the whole call where a CTA holds both chains of a sample: the records come from the resident state
    if (!G.P.gauss && n_mcs >= measure_every && (do_houdayer == 0 || do_houdayer == 1) && mcs_fused_eligible(nullptr, do_houdayer, true) &&
        !mcs_split_chains(do_houdayer) && (n_metro > 0 || do_houdayer || do_exchange)) {
        const McsArgs a{n_mcs, n_metro, do_houdayer ? 1 : 0, do_exchange ? 1 : 0, 0, G.max_clu, G.n_sweep, G.n_houdayer,
                        G.n_exchange, measure_every, Q_rec_dev, QL_rec_dev, G.phase_clocks, 0, 0};
        const int rcf = run_fused(a);
        if (rcf) return rcf;
        G.n_sweep += (uint32_t)(M * (uint64_t)n_metro);
        if (do_houdayer) G.n_houdayer += (uint32_t)M;
        if (do_exchange) { G.n_exchange += (uint32_t)M; G.n_passes += M; }
        return PT_OK;
    }
    // otherwise exactly the calls it stands for
    if (G.pending_groups) { const int rcj = join_pending(); if (rcj) return rcj; }
    int done = 0, rec = 0;
    while (n_mcs - done >= measure_every) {
        int rc = pt_mcs(measure_every, n_metro, do_houdayer, do_exchange);
        if (rc) return rc;
        CK(launch_measure(Q_rec_dev + rec * stride, QL_rec_dev ? QL_rec_dev + rec * stride : nullptr));
        done += measure_every;
        ++rec;
    }
    return pt_mcs(n_mcs - done, n_metro, do_houdayer, do_exchange);
}

int pt_set_fused(int mode)
{
    if (mode != -1 && mode != 0) return fail(PT_ERR_ARG, "mode must be -1 (fused where eligible) or 0 (separate launches)");
    G.fused_mode = mode;
    return PT_OK;
}

int pt_get_fused(int *fused)
{
    NEED_INIT();
    if (fused) *fused = mcs_fused_eligible(nullptr) ? 1 : 0;
    return PT_OK;
}

// ---- NEXT-1: temperature-schedule family and round trips ---------------------------------------------------

int pt_schedule_family(double T_min, double T_max, int n_temps, double phi, double *temps_out, double *betas_out)
{
    if (!(T_min > 0.0) || !(T_max >= T_min) || !std::isfinite(T_max) || n_temps < 1 || !(phi > 0.0) || !std::isfinite(phi))
        return fail(PT_ERR_ARG, "pt_schedule_family: need 0 < T_min <= T_max < inf, n_temps >= 1, 0 < phi < inf");
    const double T_norm = (n_temps > 1) ? (T_max - T_min) / std::pow((double)(n_temps - 1), phi) : 0.0;     // Eq. (7)
    for (int i = 0; i < n_temps; ++i) {
        const double Ti = std::pow((double)i, phi) * T_norm + T_min;                                        // Eq. (6)
        if (temps_out) temps_out[i] = Ti;
        if (betas_out) betas_out[i] = 1.0 / Ti;
    }
    return PT_OK;
}

int pt_set_coupling_probability(double p_ferro)
{
    if (!G.bound) return fail(PT_ERR_STATE, "pt_set_coupling_probability: no workspace bound");
    if (G.inited) return fail(PT_ERR_STATE, "pt_set_coupling_probability must precede pt_init (couplings are drawn there)");
    if (!(p_ferro >= 0.0) || !(p_ferro <= 1.0)) return fail(PT_ERR_ARG, "p must be in [0, 1]");
    G.p_ferro = p_ferro;
    return PT_OK;
}

int pt_set_round_trip_tracking(int on)
{
    if (!G.bound) return fail(PT_ERR_STATE, "pt_set_round_trip_tracking: no workspace bound");
    if (G.inited) return fail(PT_ERR_STATE, "pt_set_round_trip_tracking must precede pt_init (the bookkeeping starts at pass 0)");
    G.track = on ? 1 : 0;
    return PT_OK;
}

int pt_get_round_trips(uint32_t *trips, uint64_t *tau_sum, uint64_t *tau_cnt)
{
    NEED_INIT();
    if (!G.P.track) return fail(PT_ERR_STATE, "round-trip tracking is off (pt_set_round_trip_tracking before pt_init)");
    int rc = PT_OK;
    if (trips) rc = d2h(trips, G.P.d.rtTrips, (size_t)G.P.S * 2 * G.P.T * 4);
    if (!rc && tau_sum) rc = d2h(tau_sum, G.P.d.rtSum, (size_t)G.P.S * 2 * 32 * 8);
    if (!rc && tau_cnt) rc = d2h(tau_cnt, G.P.d.rtCnt, (size_t)G.P.S * 2 * 32 * 8);
    return rc;
}

// ---- observables -----------------------------------------------------------------------------------------

int pt_get_energy_device(int32_t *E_dev)
{
    NEED_INIT();
    if (!E_dev) return fail(PT_ERR_ARG, "E is NULL");
    k_energy_by_temp<<<grid_for((long)G.P.S * 2 * G.P.T, 256), 256, 0, G.stream>>>(G.P, E_dev);
    ++G.launches;
    CK(cudaGetLastError());
    return PT_OK;
}

int pt_get_energy(int32_t *E)
{
    NEED_INIT();
    if (!E) return fail(PT_ERR_ARG, "E is NULL");
    const int rc = pt_get_energy_device(G.P.d.outE);
    if (rc) return rc;
    return d2h(E, G.P.d.outE, (size_t)G.P.S * 2 * G.P.T * 4);
}

int pt_measure_overlap_device(int32_t *Q_dev, int32_t *QL_dev)
{
    NEED_INIT();
    if (!Q_dev) return fail(PT_ERR_ARG, "Q is NULL");
    CK(launch_measure(Q_dev, QL_dev));
    return PT_OK;
}

int pt_measure_overlap(int32_t *Q, int32_t *QL)
{
    NEED_INIT();
    if (!Q) return fail(PT_ERR_ARG, "Q is NULL");
    CK(launch_measure(G.P.d.outQ, QL ? G.P.d.outQL : nullptr));
    int rc = d2h(Q, G.P.d.outQ, (size_t)G.P.S * G.P.T * 4);
    if (rc) return rc;
    if (QL) rc = d2h(QL, G.P.d.outQL, (size_t)G.P.S * G.P.T * 4);
    return rc;
}

static int launch_profile(const Params &P, int32_t *out)
{
    ProfScope prof(3);
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        if constexpr (LAT::kFast) {
            const long pairs = (long)P.S * P.T;
            k_profile_fast<LAT><<<(unsigned)((pairs + 3) / 4), 128, (size_t)4 * P.D * P.L * sizeof(int), G.stream>>>(lat, P, out);
        } else {
            dim3 grid((unsigned)P.T, (unsigned)P.S);
            k_profile<LAT><<<grid, 128, (size_t)P.D * P.L * sizeof(int), G.stream>>>(lat, P, out);
        }
        ++G.launches;
        err = cudaGetLastError();
    });
    CK(err);
    return PT_OK;
}

int pt_measure_overlap_profile_device(int32_t *prof_dev)
{
    NEED_INIT();
    if (!prof_dev) return fail(PT_ERR_ARG, "prof is NULL");
    return launch_profile(G.P, prof_dev);
}

int pt_measure_overlap_profile(int32_t *prof)
{
    NEED_INIT();
    if (!prof) return fail(PT_ERR_ARG, "prof is NULL");
    const size_t per_sample = (size_t)G.P.T * G.P.D * G.P.L * 4;
    const int rc = for_chunks(per_sample, G.stage_bytes, 0, G.P.S, [&](const Params &V, int s0, int n) {
        int32_t *dev = (int32_t *)V.d.stage;         // the staging area is the device buffer of the host variant
        const int r = launch_profile(V, dev);
        if (r) return r;
        CK(cudaMemcpyAsync((char *)prof + (size_t)s0 * per_sample, dev, (size_t)n * per_sample, cudaMemcpyDeviceToHost, G.stream));
        return PT_OK;
    });
    if (rc) return rc;
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

int pt_get_swap_counts(uint64_t *attempts, uint64_t *accepts)
{
    NEED_INIT();
    const size_t n = (size_t)G.P.S * 2 * (G.P.T - 1);
    if (accepts && n) {
        const int rc = d2h(accepts, G.P.d.accepts, n * 8);
        if (rc) return rc;
    }
    if (attempts)                                   // every pass proposes every neighbouring pair once (R9)
        for (size_t k = 0; k < n; ++k) attempts[k] = G.n_passes;
    return PT_OK;
}

int pt_get_cluster_sizes(uint32_t *last, uint64_t *cumulative)
{
    NEED_INIT();
    const size_t n = (size_t)G.P.S * G.P.T;
    int rc = PT_OK;
    if (last) rc = d2h(last, G.P.d.last, n * 4);
    if (!rc && cumulative) rc = d2h(cumulative, G.P.d.cum, n * 8);
    return rc;
}

int pt_get_perm(int32_t *temp_of_slot, int32_t *slot_of_temp)
{
    NEED_INIT();
    const size_t n = (size_t)G.P.S * 2 * G.P.T;
    int rc = PT_OK;
    if (temp_of_slot) rc = d2h(temp_of_slot, G.P.d.tos, n * 4);
    if (!rc && slot_of_temp) rc = d2h(slot_of_temp, G.P.d.sot, n * 4);
    return rc;
}

// ---- state access ----------------------------------------------------------------------------------------

int pt_get_spins(int8_t *spins)
{
    NEED_INIT();
    if (!spins) return fail(PT_ERR_ARG, "spins is NULL");
    const size_t per_sample = (size_t)2 * G.P.T * G.P.N;
    const int rc = for_chunks(per_sample, G.stage_bytes, 0, G.P.S, [&](const Params &V, int s0, int n) {
        cudaError_t err = cudaSuccess;
        with_lattice([&](auto lat) {
            using LAT = decltype(lat);
            if constexpr (LAT::kFast) k_unpack_spins_fast<LAT><<<grid_for((long)(n * per_sample / 64), 256), 256, 0, G.stream>>>(V, V.d.stage);
            else k_unpack_spins<<<grid_for((long)(n * per_sample), 256), 256, 0, G.stream>>>(V);
            ++G.launches;
            err = cudaGetLastError();
        });
        CK(err);
        CK(cudaMemcpyAsync(spins + (size_t)s0 * per_sample, V.d.stage, (size_t)n * per_sample, cudaMemcpyDeviceToHost, G.stream));
        return PT_OK;
    });
    if (rc) return rc;
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

int pt_get_couplings(int8_t *J)
{
    NEED_INIT();
    if (!J) return fail(PT_ERR_ARG, "J is NULL");
    if (G.P.gauss) return fail(PT_ERR_STATE, "couplings are fixed-point numbers: use pt_get_couplings_fixed");
    const size_t per_sample = (size_t)G.P.D * G.P.N;
    const int rc = for_chunks(per_sample, G.stage_bytes, 0, G.P.S, [&](const Params &V, int s0, int n) {
        k_unpack_couplings<<<grid_for((long)(n * per_sample), 256), 256, 0, G.stream>>>(V);
        ++G.launches;
        CK(cudaGetLastError());
        CK(cudaMemcpyAsync(J + (size_t)s0 * per_sample, V.d.stage, (size_t)n * per_sample, cudaMemcpyDeviceToHost, G.stream));
        return PT_OK;
    });
    if (rc) return rc;
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

int pt_get_thresholds(uint32_t *thrM, uint32_t *thrX, size_t thrX_stride)
{
    NEED_INIT();
    const int T = G.P.T, d = G.P.D;
    if (thrM)
        for (int t = 0; t < T; ++t)
            for (int k = 1; k <= d; ++k) thrM[(size_t)t * d + (k - 1)] = THR(-(G.betas[t] * (double)(4 * k)));
    if (thrX)
        for (int t = 0; t + 1 < T; ++t)
            for (size_t m = 0; m < thrX_stride; ++m) thrX[(size_t)t * thrX_stride + m] = THR(thrX_arg(G.betas, t, m));
    return PT_OK;
}

int pt_get_counters(uint32_t *n_sweep, uint32_t *n_exchange, uint32_t *n_houdayer)
{
    NEED_INIT();
    if (n_sweep) *n_sweep = G.n_sweep;
    if (n_exchange) *n_exchange = G.n_exchange;
    if (n_houdayer) *n_houdayer = G.n_houdayer;
    return PT_OK;
}

// ---- checkpoint / resume: the RNG is counter-based, so the complete state of a run is the spins, the
// couplings (or the seed), the slot_of_temp maps and the three step counters; energies follow from the spins.

int pt_set_counters(uint32_t n_sweep, uint32_t n_exchange, uint32_t n_houdayer)
{
    NEED_INIT();
    G.n_sweep = n_sweep;
    G.n_exchange = n_exchange;
    G.n_houdayer = n_houdayer;
    return PT_OK;
}

int pt_set_perm(const int32_t *slot_of_temp)
{
    NEED_INIT();
    if (!slot_of_temp) return fail(PT_ERR_ARG, "slot_of_temp is NULL");
    const int T = G.P.T;
    const size_t chains = (size_t)G.P.S * 2, n = chains * T;
    std::vector<int32_t> tos(n, -1);
    for (size_t c = 0; c < chains; ++c)
        for (int t = 0; t < T; ++t) {
            const int32_t r = slot_of_temp[c * T + t];
            if (r < 0 || r >= T || tos[c * T + r] != -1)
                return fail(PT_ERR_ARG, "pt_set_perm: row %zu of slot_of_temp is not a permutation of 0..%d", c, T - 1);
            tos[c * T + r] = t;
        }
    CK(cudaMemcpyAsync(G.P.d.sot, slot_of_temp, n * 4, cudaMemcpyHostToDevice, G.stream));
    CK(cudaMemcpyAsync(G.P.d.tos, tos.data(), n * 4, cudaMemcpyHostToDevice, G.stream));
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

// Upload of a HOST int8 array of bytes_per_sample per sample through the bounded staging area, chunk by chunk, on the bound
// stream; `use` consumes a staged chunk (nullptr: only count the values that are not +1/-1 into mismatch[1]).
extern "C++" template <class F> int upload_chunks(const int8_t *host, size_t bytes_per_sample, bool count_bad, F use)
{
    return for_chunks(bytes_per_sample, G.stage_bytes, 0, G.P.S, [&](const Params &V, int s0, int n) {
        const size_t bytes = (size_t)n * bytes_per_sample;
        CK(cudaMemcpyAsync(V.d.stage, host + (size_t)s0 * bytes_per_sample, bytes, cudaMemcpyHostToDevice, G.stream));
        if (count_bad) {
            k_check_pm1<<<grid_for((long)((bytes + 15) / 16), 256), 256, 0, G.stream>>>(V.d.stage, bytes, G.P.d.mismatch + 1);
            ++G.launches;
            CK(cudaGetLastError());
        }
        return use(V);
    });
}

// +-1 validation of a host int8 array BEFORE anything is modified (a rejected input leaves the state unchanged): where the
// array does not fit the staging area in one piece this costs a second pass over the host buffer.
static int validate_pm1(const int8_t *host, size_t bytes_per_sample, const char *what, bool *staged_whole)
{
    CK(cudaMemsetAsync(G.P.d.mismatch + 1, 0, sizeof(int), G.stream));
    int rc = upload_chunks(host, bytes_per_sample, true, [](const Params &) { return PT_OK; });
    if (rc) return rc;
    int bad = 0;
    if ((rc = d2h(&bad, G.P.d.mismatch + 1, sizeof(int)))) return rc;
    if (bad) return fail(PT_ERR_ARG, "%s: %d values are not +1/-1", what, bad);
    *staged_whole = (size_t)G.P.S * bytes_per_sample <= G.stage_bytes;      // the one chunk is still in the staging area
    return PT_OK;
}

int pt_set_spins(const int8_t *spins)
{
    NEED_INIT();
    if (!spins) return fail(PT_ERR_ARG, "spins is NULL");
    const size_t per_sample = (size_t)2 * G.P.T * G.P.N;
    bool whole = false;
    int rc = validate_pm1(spins, per_sample, "spins", &whole);
    if (rc) return rc;
    if (whole) rc = pack_spins(G.P, G.stream, G.P.d.stage, nullptr);
    else rc = upload_chunks(spins, per_sample, false, [](const Params &V) { return pack_spins(V, G.stream, V.d.stage, nullptr); });
    if (rc) return rc;
    CK(launch_energy(0));
    CK(cudaStreamSynchronize(G.stream));       // the caller may reuse `spins` as soon as we return
    return PT_OK;
}

int pt_set_spins_async(const int8_t *spins)
{
    NEED_INIT();
    if (!spins) return fail(PT_ERR_ARG, "spins is NULL");
    const size_t per_sample = (size_t)2 * G.P.T * G.P.N;
    int ng = upload_groups();
    // every group needs room for one sample in ITS region, which starts on a 256-byte boundary
    const auto region_of = [&](int n) { return n == 1 ? G.stage_bytes : (G.stage_bytes / n) & ~(size_t)255; };
    while (ng > 1 && region_of(ng) < per_sample) --ng;
    Groups g;
    int rc = make_groups(ng, g);
    if (rc) return rc;
    CK(cudaMemsetAsync(G.P.d.mismatch + 2, 0, sizeof(int), G.stream));
    if ((rc = fork_groups(g))) return rc;
    const bool whole = G.stage_bytes >= (size_t)G.P.S * per_sample;     // PT_WS_FULL_STAGING: every group in one copy, at its own offset
    rc = [&]() -> int {
        for (int k = 0; k < g.n; ++k) {
            const size_t region = whole ? (size_t)g.view[k].S * per_sample : region_of(ng);
            int8_t *stage_k = G.P.d.stage + (whole ? (size_t)g.s0[k] * per_sample : (size_t)k * region);
            cudaStream_t st = g.st[k];
            // copy -> pack, chunk after chunk in the group's stream (the next copy into the region waits for the pack before it)
            const int rck = for_chunks(per_sample, region, g.s0[k], g.s0[k] + g.view[k].S, [&](const Params &V, int s0, int n) {
                CK(cudaMemcpyAsync(stage_k, spins + (size_t)s0 * per_sample, (size_t)n * per_sample, cudaMemcpyHostToDevice, st));
                return pack_spins(V, st, stage_k, G.P.d.mismatch + 2);
            });
            if (rck) return rck;
            CK(launch_energy(0, g.view[k], st));
        }
        return PT_OK;
    }();
    if (rc) {                                // never return with the side streams forked
        G.pending_groups = 0;
        join_groups(g.n);
        return rc;
    }
    G.pending_groups = g.n > 1 ? g.n : 0;
    G.async_check = true;
    return PT_OK;
}

// ---- bit-packed boundary (same state, 1/8 of the bytes): [S][2][T(slot)][ceil(N/32)] uint32, bit (i & 31) of word i >> 5 of a
// replica = site i, 1 <=> spin -1 (natural site order; this is NOT the device-internal colour layout)

static int packed_convert(const Params &P, cudaStream_t st, uint32_t *nat, int to_device)
{
    cudaError_t err = cudaSuccess;
    with_lattice([&](auto lat) {
        using LAT = decltype(lat);
        const long reps = (long)P.S * 2 * P.T;
        if constexpr (LAT::kFast) {
            const long total = reps * P.W;
            if (to_device) k_nat_to_colour_fast<LAT><<<grid_for(total, 256), 256, 0, st>>>(P, nat);
            else k_colour_to_nat_fast<LAT><<<grid_for(total, 256), 256, 0, st>>>(P, nat);
        } else {
            const long total = reps * ((P.N + 31) / 32);
            if (to_device) {
                cudaMemsetAsync(P.d.spin, 0, (size_t)reps * 2 * P.W * 4, st);
                k_nat_to_colour_gen<<<grid_for(total, 256), 256, 0, st>>>(P, nat);
            } else {
                k_colour_to_nat_gen<<<grid_for(total, 256), 256, 0, st>>>(P, nat);
            }
        }
        ++G.launches;
        err = cudaGetLastError();
    });
    CK(err);
    return PT_OK;
}

int pt_set_spins_packed(const uint32_t *bits)
{
    NEED_INIT();
    if (!bits) return fail(PT_ERR_ARG, "bits is NULL");
    const size_t per_sample = (size_t)2 * G.P.T * ((G.P.N + 31) / 32) * 4;
    // chunked through the staging area, copy -> convert in the bound stream; no validation needed (every bit pattern is a state,
    // bits beyond site N-1 of the last word are ignored); asynchronous like pt_set_spins_async, on ONE stream
    const int rc = for_chunks(per_sample, G.stage_bytes, 0, G.P.S, [&](const Params &V, int s0, int n) {
        CK(cudaMemcpyAsync(V.d.stage, (const char *)bits + (size_t)s0 * per_sample, (size_t)n * per_sample, cudaMemcpyHostToDevice, G.stream));
        return packed_convert(V, G.stream, (uint32_t *)V.d.stage, 1);
    });
    if (rc) return rc;
    CK(launch_energy(0));
    return PT_OK;
}

int pt_get_spins_packed(uint32_t *bits)
{
    NEED_INIT();
    if (!bits) return fail(PT_ERR_ARG, "bits is NULL");
    const size_t per_sample = (size_t)2 * G.P.T * ((G.P.N + 31) / 32) * 4;
    const int rc = for_chunks(per_sample, G.stage_bytes, 0, G.P.S, [&](const Params &V, int s0, int n) {
        const int r = packed_convert(V, G.stream, (uint32_t *)V.d.stage, 0);
        if (r) return r;
        CK(cudaMemcpyAsync((char *)bits + (size_t)s0 * per_sample, V.d.stage, (size_t)n * per_sample, cudaMemcpyDeviceToHost, G.stream));
        return PT_OK;
    });
    if (rc) return rc;
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

int pt_set_couplings(const int8_t *J)
{
    NEED_INIT();
    if (!J) return fail(PT_ERR_ARG, "J is NULL");
    const size_t per_sample = (size_t)G.P.D * G.P.N;
    bool whole = false;
    int rc = validate_pm1(J, per_sample, "J", &whole);
    if (rc) return rc;
    G.P.gauss = 0;
    if (whole) rc = pack_couplings(G.P);
    else rc = upload_chunks(J, per_sample, false, [](const Params &V) { return pack_couplings(V); });
    if (rc) return rc;
    CK(launch_energy(0));
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

int pt_set_couplings_fixed(const int32_t *Jq, int frac_bits)
{
    NEED_INIT();
    if (!Jq) return fail(PT_ERR_ARG, "Jq is NULL");
    if (frac_bits < 0 || frac_bits > 24) return fail(PT_ERR_ARG, "frac_bits must be in [0, 24]");
    if (!G.has_fixed)
        return fail(PT_ERR_STATE, "pt_set_couplings_fixed: the workspace was laid out without int32 couplings (bind "
                                  "pt_workspace_bytes_ex(..., PT_WS_FIXED_COUPLINGS, ...) bytes and call "
                                  "pt_set_workspace_flags(PT_WS_FIXED_COUPLINGS) before pt_init)");
    const size_t n = (size_t)G.P.S * G.P.D * G.P.N;
    long long maxabs = 0;
    for (size_t k = 0; k < n; ++k) maxabs = std::max<long long>(maxabs, Jq[k] < 0 ? -(long long)Jq[k] : (long long)Jq[k]);
    if ((double)maxabs * (double)G.P.D * (double)G.P.N >= 2147483648.0)
        return fail(PT_ERR_ARG, "d * N * max|Jq| must stay below 2^31 (int32 energies): use fewer fractional bits");
    CK(cudaMemcpyAsync(G.P.d.JqNat, Jq, n * 4, cudaMemcpyHostToDevice, G.stream));
    G.P.gauss = 1;
    G.P.fbits = frac_bits;
    G.q_small = 2LL * G.P.D * maxabs < (1LL << 23);
    {
        std::vector<float> slope((size_t)G.P.T, 0.0f);
        for (int t = 0; t + 1 < G.P.T; ++t)
            slope[t] = (float)(-std::fabs(G.betas[t + 1] - G.betas[t]) * std::ldexp(1.4426950408889634, -frac_bits));
        CK(cudaMemcpyAsync(G.P.d.swapSlope, slope.data(), slope.size() * 4, cudaMemcpyHostToDevice, G.stream));
        CK(cudaStreamSynchronize(G.stream));
    }
    k_pack_jq<<<grid_for((long)G.P.S * 2 * 2 * G.P.D * 32 * G.P.W, 256), 256, 0, G.stream>>>(G.P);
    ++G.launches;
    CK(cudaGetLastError());
    CK(launch_energy(0));
    CK(cudaStreamSynchronize(G.stream));
    return PT_OK;
}

int pt_get_couplings_fixed(int32_t *Jq, int *frac_bits)
{
    NEED_INIT();
    if (!G.P.gauss) return fail(PT_ERR_STATE, "couplings are +-1: use pt_get_couplings");
    if (frac_bits) *frac_bits = G.P.fbits;
    if (Jq) return d2h(Jq, G.P.d.JqNat, (size_t)G.P.S * G.P.D * G.P.N * 4);
    return PT_OK;
}

int pt_recompute_energy(int32_t *E_slot_order, int *mismatch_count)
{
    NEED_INIT();
    CK(cudaMemsetAsync(G.P.d.mismatch, 0, sizeof(int), G.stream));
    CK(launch_energy(1));
    int bad = 0;
    int rc = d2h(&bad, G.P.d.mismatch, sizeof(int));
    if (rc) return rc;
    if (mismatch_count) *mismatch_count = bad;
    if (E_slot_order) rc = d2h(E_slot_order, G.P.d.outE, (size_t)G.P.S * 2 * G.P.T * 4);
    return rc;
}

// ---- diagnostics -----------------------------------------------------------------------------------------

int pt_synchronize(void)
{
    if (!G.bound) return fail(PT_ERR_STATE, "not bound");
    if (G.pending_groups) { const int rcj = join_pending(); if (rcj) return rcj; }
    CK(cudaStreamSynchronize(G.stream));
    if (G.inited && G.async_check) {
        G.async_check = false;
        int bad = 0;
        const int rc = d2h(&bad, G.P.d.mismatch + 2, sizeof(int));
        if (rc) return rc;
        if (bad) return fail(PT_ERR_ARG, "pt_set_spins_async: %d bytes or words held values other than +1/-1 (taken by their sign)", bad);
    }
    return PT_OK;
}

int pt_set_profiling(int on)
{
    if (!G.bound) return fail(PT_ERR_STATE, "not bound");
    CK(cudaStreamSynchronize(G.stream));
    PROF.harvest();
    PROF.on = on != 0;
    for (int k = 0; k < 5; ++k) { PROF.ms[k] = 0; PROF.n[k] = 0; }
    return PT_OK;
}

int pt_get_kernel_times(double ms[5], uint64_t launches[5])
{
    if (!G.bound) return fail(PT_ERR_STATE, "not bound");
    CK(cudaStreamSynchronize(G.stream));
    PROF.harvest();
    for (int k = 0; k < 5; ++k) {
        if (ms) ms[k] = PROF.ms[k];
        if (launches) launches[k] = PROF.n[k];
    }
    return PT_OK;
}

int pt_set_sample_groups(int n)
{
    if (!G.bound) return fail(PT_ERR_STATE, "not bound");
    if (n != -1 && (n < 1 || n > kMaxGroups)) return fail(PT_ERR_ARG, "pt_set_sample_groups: n must be -1 (automatic) or 1..%d", kMaxGroups);
    G.sample_groups = n;
    return PT_OK;
}

int pt_set_phase_clocks(int on)
{
    NEED_INIT();
    CK(cudaMemsetAsync(G.P.d.phaseClk, 0, 4 * sizeof(unsigned long long), G.stream));
    G.phase_clocks = on ? 1 : 0;
    return PT_OK;
}

int pt_get_phase_clocks(uint64_t clocks[4])
{
    NEED_INIT();
    if (!clocks) return fail(PT_ERR_ARG, "clocks is NULL");
    return d2h(clocks, G.P.d.phaseClk, 4 * sizeof(unsigned long long));
}

int pt_get_launch_count(uint64_t *n_launches)
{
    if (!n_launches) return fail(PT_ERR_ARG, "n_launches is NULL");
    *n_launches = G.launches;
    return PT_OK;
}

int pt_threshold_selftest(const double *x, uint32_t *out, int n)
{
    NEED_INIT();
    if (!x || !out || n < 1) return fail(PT_ERR_ARG, "bad arguments");
    if ((size_t)n * 12 + 16 > G.stage_bytes) return fail(PT_ERR_ARG, "n too large for the scratch area");
    double *dx = (double *)G.P.d.stage;
    uint32_t *dout = (uint32_t *)(dx + n);
    CK(cudaMemcpyAsync(dx, x, (size_t)n * 8, cudaMemcpyHostToDevice, G.stream));
    k_threshold_selftest<<<(n + 127) / 128, 128, 0, G.stream>>>(dx, dout, n);
    ++G.launches;
    CK(cudaGetLastError());
    return d2h(out, dout, (size_t)n * 4);
}

int pt_philox_selftest(const uint32_t key[2], const uint32_t *ctr, uint32_t *out, int n)
{
    if (!G.bound) return fail(PT_ERR_STATE, "pt_philox_selftest: no workspace bound");
    if (!key || !ctr || !out || n < 1) return fail(PT_ERR_ARG, "bad arguments");
    // an asynchronous upload may still be copying into the staging area
    if (G.inited && G.pending_groups) { const int rcj = join_pending(); if (rcj) return rcj; }
    // scratch: the staging area when initialised, else the start of the workspace
    char *scratch = G.inited ? (char *)G.P.d.stage : (char *)G.ws;
    const size_t avail = G.inited ? G.stage_bytes : G.ws_bytes;
    if ((size_t)n * 32 > avail) return fail(PT_ERR_ARG, "n too large for the scratch area");
    uint32_t *dctr = (uint32_t *)scratch, *dout = dctr + (size_t)n * 4;
    CK(cudaMemcpyAsync(dctr, ctr, (size_t)n * 16, cudaMemcpyHostToDevice, G.stream));
    k_philox_selftest<<<(n + 127) / 128, 128, 0, G.stream>>>(make_round_keys(key[0], key[1]), dctr, dout, n);
    ++G.launches;
    CK(cudaGetLastError());
    return d2h(out, dout, (size_t)n * 16);
}

}  // extern "C"

// =========================================================================================================
// pt_exchange_noalloc: one PT pass for callers that must not allocate device memory (include/ptglass.h).
// A variant of k_exchange<GLOBAL_SCRATCH = true>: that kernel walks the ladder on scratch in global memory (the energies
// in temperature order) and reads the threshold table and the signs of the beta steps from the caller's workspace.  Here
// all three live in ONE fixed area that is part of this library's device image, so that a caller who cannot (or may not)
// call cudaMalloc -- a hook inside a job whose memory pool already owns the card, a loop that cannot take cudaMalloc's
// device-wide synchronisation -- can still run a pass.  Nothing below allocates or frees device memory.
// =========================================================================================================

// The scratch area.  In HOST code this name is only a handle for the runtime's symbol calls, not a device address: a
// kernel that is handed `g_noalloc_scratch` itself would fault (or, on a system where the GPU can reach host memory,
// quietly use the wrong bytes).  The host gets the real address from cudaGetSymbolAddress, once per device.
static __device__ __align__(256) unsigned char g_noalloc_scratch[PT_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int kNoAllocMaxDevices = 64;
void *g_noalloc_addr[kNoAllocMaxDevices] = {};      // device address of the area, per device ordinal; nullptr = not asked yet

// One warp per (sample, chain).  Et = this chain's energies in temperature order (scratch), so = its slot_of_temp row
// (walked in place).  The lanes draw 32 Philox words at a time, lane 0 walks the rungs in order (each rung sees the one
// before, R9); same counters, same table, same comparisons as k_exchange, so the same decisions.
__global__ void k_exchange_noalloc(int n_chains, int T, uint32_t g0, uint32_t step, uint32_t strideX, RoundKeys rk,
                                   const uint32_t *__restrict__ thrX, const int32_t *__restrict__ sgn, int32_t *EtAll,
                                   const int32_t *__restrict__ E, int32_t *sot, int32_t *tos, unsigned long long *accepts)
{
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const long chain = (long)blockIdx.x * wpb + wib;
    if (chain >= n_chains) return;
    const uint32_t c = (uint32_t)(chain & 1), g = g0 + (uint32_t)(chain >> 1);
    const size_t base = (size_t)chain * T;
    int32_t *Et = EtAll + base, *so = sot + base;
    for (int t = lane; t < T; t += 32) Et[t] = E[base + so[t]];
    __syncwarp();
    int32_t ea = 0, ra = 0;
    if (lane == 0) { ea = Et[0]; ra = so[0]; }
    for (int tb = 0; tb < T - 1; tb += 32) {
        const int tl = tb + lane;
        uint32_t u_l = 0, o1, o2, o3;
        if (tl < T - 1) philox4x32_10((uint32_t)tl, step, g, make_tag(DOM_SWAP, 0, c, 0), rk, u_l, o1, o2, o3);
        const int nstep = min(32, T - 1 - tb);
        for (int j = 0; j < nstep; ++j) {
            const uint32_t u = __shfl_sync(0xFFFFFFFFu, u_l, j);
            if (lane == 0) {
                const int t = tb + j;
                const int32_t eb = Et[t + 1], rb = so[t + 1];
                const int32_t dE = ea - eb;
                const uint32_t m = (uint32_t)(dE < 0 ? -dE : dE) >> 2;
                const uint32_t thr = (m < strideX) ? thrX[(size_t)t * strideX + m] : 0u;
                const bool acc = ((long long)sgn[t] * dE <= 0) || (u < thr);
                if (acc) {
                    Et[t] = eb; so[t] = rb;                 // position t is final; (ea, ra) is carried up to t + 1
                    if (accepts) accepts[(size_t)chain * (T - 1) + t] += 1ull;
                } else {
                    Et[t] = ea; so[t] = ra;
                    ea = eb; ra = rb;
                }
            }
        }
    }
    if (lane == 0) { Et[T - 1] = ea; so[T - 1] = ra; }
    __syncwarp();
    for (int t = lane; t < T; t += 32) tos[base + so[t]] = t;
}

}  // namespace

extern "C" int pt_exchange_noalloc(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed,
                                   uint32_t sample_offset, uint32_t step, const int32_t *E_dev, int32_t *slot_of_temp_dev,
                                   int32_t *temp_of_slot_dev, uint64_t *accepts_dev, void *cuda_stream)
{
    if (d != 2 && d != 3) return fail(PT_ERR_ARG, "pt_exchange_noalloc: d must be 2 or 3 (got %d)", d);
    if (L < 2 || (L & 1)) return fail(PT_ERR_ARG, "pt_exchange_noalloc: L must be even and >= 2 (got %d)", L);
    if (n_samples < 1 || n_samples > 65535) return fail(PT_ERR_ARG, "pt_exchange_noalloc: n_samples must be in [1, 65535] (got %d)", n_samples);
    if (n_temps < 1 || n_temps > 65535) return fail(PT_ERR_ARG, "pt_exchange_noalloc: n_temps must be in [1, 65535] (got %d)", n_temps);
    const double Nd = std::pow((double)L, d) * d;
    if (Nd > 2147483647.0) return fail(PT_ERR_ARG, "pt_exchange_noalloc: N*d overflows int32");
    if (!betas) return fail(PT_ERR_ARG, "pt_exchange_noalloc: betas is NULL");
    for (int t = 0; t < n_temps; ++t)
        if (!std::isfinite(betas[t]) || betas[t] < 0.0)
            return fail(PT_ERR_ARG, "pt_exchange_noalloc: betas[%d] is negative or not finite", t);
    if ((uint64_t)sample_offset + (uint64_t)n_samples > 4294967296ull)
        return fail(PT_ERR_ARG, "pt_exchange_noalloc: sample_offset + n_samples overflows 2^32");
    if (!E_dev || !slot_of_temp_dev || !temp_of_slot_dev)
        return fail(PT_ERR_ARG, "pt_exchange_noalloc: E_dev, slot_of_temp_dev and temp_of_slot_dev must not be NULL");

    // layout of the scratch area: threshold table | signs | energies by temperature, each 256-byte aligned
    const long N = (d == 2) ? (long)L * L : (long)L * L * L;
    const std::vector<double> b(betas, betas + n_temps);
    const uint32_t strideX = swap_stride(b, d, N);
    const size_t n_chains = (size_t)n_samples * 2;
    const size_t table_bytes = align_up((size_t)(n_temps - 1) * strideX * 4);
    const size_t sgn_bytes = align_up((size_t)n_temps * 4);
    const size_t et_bytes = align_up(n_chains * (size_t)n_temps * 4);
    const size_t need = table_bytes + sgn_bytes + et_bytes;
    if (need > (size_t)PT_NOALLOC_SCRATCH_BYTES)
        return fail(PT_ERR_ARG,
                    "pt_exchange_noalloc: this problem needs %zu bytes of scratch (threshold table %zu + signs %zu + energies by "
                    "temperature %zu) but the built-in area holds %zu: use pt_bind + pt_exchange with a caller-allocated workspace",
                    need, table_bytes, sgn_bytes, et_bytes, (size_t)PT_NOALLOC_SCRATCH_BYTES);

    // set-up, once per device, with that device current: where does this device keep the area?
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kNoAllocMaxDevices) return fail(PT_ERR_CUDA, "pt_exchange_noalloc: device ordinal %d not supported", dev);
    if (!g_noalloc_addr[dev]) {
        void *addr = nullptr;
        CK(cudaGetSymbolAddress(&addr, g_noalloc_scratch));
        if (!addr) return fail(PT_ERR_CUDA, "pt_exchange_noalloc: the runtime returned no address for the scratch area");
        g_noalloc_addr[dev] = addr;
    }
    char *area = (char *)g_noalloc_addr[dev];
    uint32_t *thrX_d = (uint32_t *)area;
    int32_t *sgn_d = (int32_t *)(area + table_bytes);
    int32_t *Et_d = (int32_t *)(area + table_bytes + sgn_bytes);
    cudaStream_t st = (cudaStream_t)cuda_stream;

    // tables on the host in double, as pt_init computes them (R5, R6); pageable source: the copies have left these
    // vectors when cudaMemcpyAsync returns
    std::vector<int32_t> sgn((size_t)n_temps, 0);
    std::vector<uint32_t> thrX((size_t)(n_temps - 1) * strideX, 0u);
    for (int t = 0; t + 1 < n_temps; ++t) {
        sgn[t] = (b[t + 1] > b[t]) - (b[t + 1] < b[t]);
        for (uint32_t m = 0; m < strideX; ++m) thrX[(size_t)t * strideX + m] = THR(thrX_arg(b, t, m));
    }
    if (!thrX.empty()) CK(cudaMemcpyAsync(thrX_d, thrX.data(), thrX.size() * 4, cudaMemcpyHostToDevice, st));
    CK(cudaMemcpyAsync(sgn_d, sgn.data(), sgn.size() * 4, cudaMemcpyHostToDevice, st));

    const int wpb = 4;
    k_exchange_noalloc<<<(unsigned)((n_chains + wpb - 1) / wpb), wpb * 32, 0, st>>>(
        (int)n_chains, n_temps, sample_offset, step, strideX,
        make_round_keys((uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)), thrX_d, sgn_d, Et_d, E_dev, slot_of_temp_dev,
        temp_of_slot_dev, (unsigned long long *)accepts_dev);
    ++G.launches;
    CK(cudaGetLastError());
    return PT_OK;
}
