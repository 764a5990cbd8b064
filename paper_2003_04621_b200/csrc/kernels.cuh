// CUDA kernels of the hot path.  sm_100a; integer only; no tensor cores (nothing here is
// a dense contraction).  Every kernel is written once over the lattice interface of lattice.cuh and
// instantiated for FastLat<D, LOG2L> (word-parallel) and GenLat<D> (general L).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "lattice.cuh"
#include "philox.cuh"
#include "houdayer_rows.cuh"

namespace ptg {

// Device arrays, all carved from the caller's workspace (ptglass.cu: carve()).
struct DevPtrs {
    uint32_t *spin;             // [S][2][T][2][W]   slot order; colour; word.  bit = 1 <=> s = -1
    uint32_t *Jn;               // [S][2][2D][W]     colour; direction k; word. bit = 1 <=> J = -1
    int32_t *E;                 // [S][2][T]         slot order
    int32_t *tos;               // temp_of_slot [S][2][T]
    int32_t *sot;               // slot_of_temp [S][2][T]
    uint32_t *thrM;             // [T][4]            k = 1..D at [t][k-1]
    uint32_t *thrX;             // [T-1][strideX]    entry m = |dE|/4; entries >= strideX are 0
    int32_t *sgn;               // [T-1]
    unsigned long long *accepts;// [S][2][T-1]
    uint32_t *last;             // [S][T]
    unsigned long long *cum;    // [S][T]
    int32_t *outE;              // [S][2][T] scratch for observables
    int32_t *outQ, *outQL;      // [S][T]
    int *mismatch;              // [1]
    int8_t *stage;              // int8 staging for get/set: max(S*2*T*N, S*D*N) bytes
    // fixed-point couplings (NEXT-3, R33-R35)
    int32_t *JqNat;             // [S][D][N] natural order (staging / read-back)
    int32_t *Jdev;              // [S][2][2D][32 W] per colour and direction
    double *betasD;             // [T]
    double *absdb;              // [T-1] |beta_{t+1} - beta_t|
    float *swapSlope;           // [T-1] (float)(-|dbeta| 2^-fbits log2 e): slope of the swap test's float bracket
    // round-trip bookkeeping (NEXT-1, R27-R29)
    uint32_t *rtLabel, *rtStart, *rtTrips;      // [S][2][T] per slot
    unsigned long long *rtSum, *rtCnt;          // [S][2][32] per (sample, chain), bin = floor(log2 pass)
    // cluster-move variants (NEXT-4, R36): single-cluster moves per houdayer_step at temperature index t
    int32_t *nclu;              // [T]
    int32_t *tcold;             // [T] temperature indices by descending beta: the pairs with the largest clusters first
    unsigned long long *phaseClk;   // [4] SM clocks summed over the CTAs of k_mcs: sweeps | Houdayer | PT pass | rest (pt_set_phase_clocks)
};

struct Params {
    int L, D, S, T, N, NH, W;
    uint32_t g0;                // sample_offset: global sample index = g0 + s
    uint32_t strideX;
    int track;                  // 1: round-trip bookkeeping after every PT pass
    int gauss, fbits;           // 1: couplings are fixed-point numbers Jq * 2^-fbits (gauss.cuh)
    unsigned long long thrJ;    // J = +1 iff Philox word < thrJ = floor(p * 2^32)  (Eq. (2), R32); 2^31 for p = 1/2
    RoundKeys rk;
    DevPtrs d;
};

__device__ __forceinline__ size_t rep_index(const Params &P, int s, int c, int r) { return ((size_t)s * 2 + c) * P.T + r; }
__device__ __forceinline__ uint32_t *spin_words(const Params &P, size_t rep, int p) { return P.d.spin + (rep * 2 + p) * P.W; }
__device__ __forceinline__ const uint32_t *J_words(const Params &P, int s, int p, int k)
{
    return P.d.Jn + (((size_t)s * 2 + p) * (2 * P.D) + k) * P.W;
}

__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c) { return (a & b) | (c & (a | b)); }

// =========================================================================================================
// init / pack / unpack (general coordinate arithmetic; not on the timed path)
// =========================================================================================================

// couplings from Philox domain 1 into the int8 staging area [S][D][N]   (Eq. (2), p = 1/2 P:195)
__global__ void k_draw_couplings(Params P)
{
    const int n4 = P.N / 4;
    const long total = (long)P.S * P.D * n4;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int i4 = (int)(id % n4);
        const int mu = (int)((id / n4) % P.D);
        const int s = (int)(id / ((long)n4 * P.D));
        uint32_t w[4];
        philox4x32_10((uint32_t)i4, 0u, P.g0 + (uint32_t)s, make_tag(DOM_J, mu, 0, 0), P.rk, w[0], w[1], w[2], w[3]);
        int8_t *dst = P.d.stage + ((size_t)s * P.D + mu) * P.N + 4 * (size_t)i4;
#pragma unroll
        for (int j = 0; j < 4; ++j) dst[j] = ((unsigned long long)w[j] < P.thrJ) ? 1 : -1;
    }
}

// spins from Philox domain 2 into staging [S][2][T][N]   (R17)
__global__ void k_draw_spins(Params P)
{
    const int n4 = P.N / 4;
    const long total = (long)P.S * 2 * P.T * n4;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int i4 = (int)(id % n4);
        const long rep = id / n4;
        const int r = (int)(rep % P.T);
        const int c = (int)((rep / P.T) & 1);
        const int s = (int)(rep / (2L * P.T));
        uint32_t w[4];
        philox4x32_10((uint32_t)i4, 0u, P.g0 + (uint32_t)s, make_tag(DOM_SPIN, 0, c, r), P.rk, w[0], w[1], w[2], w[3]);
        int8_t *dst = P.d.stage + (size_t)rep * P.N + 4 * (size_t)i4;
#pragma unroll
        for (int j = 0; j < 4; ++j) dst[j] = (w[j] >> 31) ? -1 : 1;
    }
}

// staging int8 J[S][D][N] -> per-colour, per-direction bit arrays (Jn must be zeroed first)
__global__ void k_pack_couplings(Params P)
{
    const long total = (long)P.S * P.D * P.N;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int i = (int)(id % P.N);
        const int mu = (int)((id / P.N) % P.D);
        const int s = (int)(id / ((long)P.N * P.D));
        if (P.d.stage[id] >= 0) continue;
        const int pi = colour_of_site(i, P.L, P.D);
        const int j = neighbour_site(i, 2 * mu, P.L, P.D);
        const int hi = i >> 1, hj = j >> 1;
        uint32_t *Ji = P.d.Jn + (((size_t)s * 2 + pi) * (2 * P.D) + 2 * mu) * P.W;            // +mu seen from i
        uint32_t *Jj = P.d.Jn + (((size_t)s * 2 + (1 - pi)) * (2 * P.D) + 2 * mu + 1) * P.W;  // -mu seen from j
        atomicOr(Ji + (hi >> 5), 1u << (hi & 31));
        atomicOr(Jj + (hj >> 5), 1u << (hj & 31));
    }
}

__global__ void k_unpack_couplings(Params P)
{
    const long total = (long)P.S * P.D * P.N;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int i = (int)(id % P.N);
        const int mu = (int)((id / P.N) % P.D);
        const int s = (int)(id / ((long)P.N * P.D));
        const int pi = colour_of_site(i, P.L, P.D), hi = i >> 1;
        const uint32_t *Ji = P.d.Jn + (((size_t)s * 2 + pi) * (2 * P.D) + 2 * mu) * P.W;
        P.d.stage[id] = ((Ji[hi >> 5] >> (hi & 31)) & 1u) ? -1 : 1;
    }
}

// staging int8 spins [S][2][T][N] -> bit words; one thread per (replica, colour, word)
__global__ void k_pack_spins(Params P)
{
    const long total = (long)P.S * 2 * P.T * 2 * P.W;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int w = (int)(id % P.W);
        const int p = (int)((id / P.W) & 1);
        const long rep = id / (2L * P.W);
        const int8_t *src = P.d.stage + (size_t)rep * P.N;
        uint32_t word = 0;
        for (int b = 0; b < 32; ++b) {
            const int h = 32 * w + b;
            if (h >= P.NH) break;
            if (src[site_of(h, p, P.L, P.D)] < 0) word |= 1u << b;
        }
        P.d.spin[id] = word;
    }
}

__global__ void k_unpack_spins(Params P)
{
    const long total = (long)P.S * 2 * P.T * P.N;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int i = (int)(id % P.N);
        const long rep = id / P.N;
        const int p = colour_of_site(i, P.L, P.D), h = i >> 1;
        const uint32_t *sw = P.d.spin + ((size_t)rep * 2 + p) * P.W;
        P.d.stage[id] = ((sw[h >> 5] >> (h & 31)) & 1u) ? -1 : 1;
    }
}

// ---- word-parallel pack / unpack on the power-of-two lattices: one thread = 64 consecutive sites of one replica = one
// word of EACH colour.  Four 16-byte loads, sign bits gathered four at a time by a multiply (byte k's sign lands on bit
// 24 + k of m * 0x01020408: the ten partial products fall on distinct bits, no carries), the natural-order 64-bit map is
// split by colour with the de-interleave of houdayer.cuh.  No division, no byte loads.
// bad (may be null): counts bytes that are neither +1 nor -1 (they are taken by their sign).
template <class LAT>
__global__ void k_pack_spins_fast(Params P, const int8_t *src, int *bad)
{
    using NL = NatLat<LAT::D, LAT::kLog2L>;
    constexpr int W = NL::W;
    const long total = (long)P.S * 2 * P.T * W;
    int nbad = 0;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int w = (int)(id % W);
        const long rep = id / W;
        const uint4 *p = (const uint4 *)(src + (size_t)rep * P.N + 64 * (size_t)w);
        uint32_t nat[2] = {0u, 0u};
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const uint4 v = __ldg(p + q);
            const uint32_t x[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t m = (x[j] >> 7) & 0x01010101u;
                nbad += (x[j] != 0x01010101u + m * 0xFEu);
                nat[q >> 1] |= ((m * 0x01020408u) >> 24) << (16 * (q & 1) + 4 * j);
            }
        }
        uint32_t a0, a1, b0, b1;
        NL::deinterleave(2 * w, nat[0], a0, a1);
        NL::deinterleave(2 * w + 1, nat[1], b0, b1);
        uint32_t *dst = P.d.spin + (size_t)rep * 2 * W;
        dst[w] = a0 | (b0 << 16);
        dst[W + w] = a1 | (b1 << 16);
    }
    if (bad && nbad) atomicAdd(bad, nbad);
}

template <class LAT>
__global__ void k_unpack_spins_fast(Params P, int8_t *dst)
{
    using NL = NatLat<LAT::D, LAT::kLog2L>;
    constexpr int W = NL::W;
    const long total = (long)P.S * 2 * P.T * W;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int w = (int)(id % W);
        const long rep = id / W;
        const uint32_t *sw = P.d.spin + (size_t)rep * 2 * W;
        const uint32_t c0 = sw[w], c1 = sw[W + w];
        const uint32_t nat[2] = {NL::interleave(2 * w, c0, c1), NL::interleave(2 * w + 1, c0 >> 16, c1 >> 16)};
        uint4 *o = (uint4 *)(dst + (size_t)rep * P.N + 64 * (size_t)w);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            uint32_t x[4];
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const uint32_t nib = (nat[q >> 1] >> (16 * (q & 1) + 4 * j)) & 0xFu;
                const uint32_t m = (nib * 0x00204081u) & 0x01010101u;          // bit k -> byte k
                x[j] = 0x01010101u + m * 0xFEu;                               // 0 -> +1, 1 -> -1
            }
            o[q] = make_uint4(x[0], x[1], x[2], x[3]);
        }
    }
}

// ---- bit-packed boundary (pt_set_spins_packed / pt_get_spins_packed): natural-order bit maps [rep][ceil(N/32)] <-> the two
// colour arrays.  Word-parallel lattices: one thread = the two natural words 2w, 2w+1 = word w of each colour.
template <class LAT>
__global__ void k_nat_to_colour_fast(Params P, const uint32_t *nat)
{
    using NL = NatLat<LAT::D, LAT::kLog2L>;
    constexpr int W = NL::W;
    const long total = (long)P.S * 2 * P.T * W;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int w = (int)(id % W);
        const long rep = id / W;
        const uint2 v = *(const uint2 *)(nat + (size_t)rep * 2 * W + 2 * w);
        uint32_t a0, a1, b0, b1;
        NL::deinterleave(2 * w, v.x, a0, a1);
        NL::deinterleave(2 * w + 1, v.y, b0, b1);
        uint32_t *dst = P.d.spin + (size_t)rep * 2 * W;
        dst[w] = a0 | (b0 << 16);
        dst[W + w] = a1 | (b1 << 16);
    }
}

template <class LAT>
__global__ void k_colour_to_nat_fast(Params P, uint32_t *nat)
{
    using NL = NatLat<LAT::D, LAT::kLog2L>;
    constexpr int W = NL::W;
    const long total = (long)P.S * 2 * P.T * W;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int w = (int)(id % W);
        const long rep = id / W;
        const uint32_t *sw = P.d.spin + (size_t)rep * 2 * W;
        const uint32_t c0 = sw[w], c1 = sw[W + w];
        *(uint2 *)(nat + (size_t)rep * 2 * W + 2 * w) =
            make_uint2(NL::interleave(2 * w, c0, c1), NL::interleave(2 * w + 1, c0 >> 16, c1 >> 16));
    }
}

// general L: one thread per natural word, bit by bit (the colour arrays must be zero before k_nat_to_colour_gen)
__global__ void k_nat_to_colour_gen(Params P, const uint32_t *nat)
{
    const int NWn = (P.N + 31) / 32;
    const long total = (long)P.S * 2 * P.T * NWn;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int n = (int)(id % NWn);
        const long rep = id / NWn;
        const uint32_t x = nat[id];
        for (int b = 0; b < 32; ++b) {
            const int i = 32 * n + b;
            if (i >= P.N) break;
            if ((x >> b) & 1u) {
                const int p = colour_of_site(i, P.L, P.D), h = i >> 1;
                atomicOr(P.d.spin + ((size_t)rep * 2 + p) * P.W + (h >> 5), 1u << (h & 31));
            }
        }
    }
}

__global__ void k_colour_to_nat_gen(Params P, uint32_t *nat)
{
    const int NWn = (P.N + 31) / 32;
    const long total = (long)P.S * 2 * P.T * NWn;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int n = (int)(id % NWn);
        const long rep = id / NWn;
        uint32_t x = 0;
        for (int b = 0; b < 32; ++b) {
            const int i = 32 * n + b;
            if (i >= P.N) break;
            const int p = colour_of_site(i, P.L, P.D), h = i >> 1;
            x |= ((P.d.spin[((size_t)rep * 2 + p) * P.W + (h >> 5)] >> (h & 31)) & 1u) << b;
        }
        nat[id] = x;
    }
}

// counts staged bytes that are not +1/-1 (input validation of pt_set_spins / pt_set_couplings)
__global__ void k_check_pm1(const int8_t *a, size_t n, int *bad)
{
    int local = 0;
    for (size_t i = (blockIdx.x * (size_t)blockDim.x + threadIdx.x) * 16; i < n; i += (size_t)gridDim.x * blockDim.x * 16)
        for (size_t j = i; j < i + 16 && j < n; ++j) local += (a[j] != 1 && a[j] != -1);
    if (local) atomicAdd(bad, local);
}

__global__ void k_identity_perm(Params P)
{
    const long total = (long)P.S * 2 * P.T;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        P.d.tos[id] = (int32_t)(id % P.T);
        P.d.sot[id] = (int32_t)(id % P.T);
        P.d.rtLabel[id] = (id % P.T == 0) ? 1u : 0u;        // the slot that starts at index 0 starts its first trip (R28)
        P.d.rtStart[id] = 0u;
        P.d.rtTrips[id] = 0u;
    }
}

__global__ void k_philox_selftest(RoundKeys rk, const uint32_t *ctr, uint32_t *out, int n)
{
    const int id = blockIdx.x * blockDim.x + threadIdx.x;
    if (id >= n) return;
    uint32_t o0, o1, o2, o3;
    philox4x32_10(ctr[4 * id], ctr[4 * id + 1], ctr[4 * id + 2], ctr[4 * id + 3], rk, o0, o1, o2, o3);
    out[4 * id] = o0; out[4 * id + 1] = o1; out[4 * id + 2] = o2; out[4 * id + 3] = o3;
}

// =========================================================================================================
// energy from scratch:  E = -sum J s s = 2 * #unsatisfied - D*N   (Eq. (1)).  Each bond has exactly one
// black endpoint, so summing the 2D directions over black sites counts every bond once (also at L = 2, R3).
// One warp per replica.  mode 0: write E;  mode 1: write outE (slot order) and count mismatches against E.
// =========================================================================================================
template <class LAT>
__global__ void k_energy(LAT lat, Params P, int mode)
{
    const int warps_per_block = blockDim.x >> 5;
    const long rep = (long)blockIdx.x * warps_per_block + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (rep >= (long)P.S * 2 * P.T) return;
    const int s = (int)(rep / (2L * P.T));
    const uint32_t *Sb = spin_words(P, (size_t)rep, 0), *Sw = spin_words(P, (size_t)rep, 1);
    int unsat = 0;
    for (int w = lane; w < lat.words(); w += 32) {
        uint32_t nb[2 * LAT::D];
        lat.gather(Sw, w, 0, nb);
        const uint32_t sb = Sb[w], v = lat.valid(w);
#pragma unroll
        for (int k = 0; k < 2 * LAT::D; ++k) unsat += __popc((sb ^ nb[k] ^ J_words(P, s, 0, k)[w]) & v);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) unsat += __shfl_xor_sync(0xFFFFFFFFu, unsat, o);
    if (lane == 0) {
        const int32_t e = 2 * unsat - P.D * P.N;
        if (mode == 0) {
            P.d.E[rep] = e;
        } else {
            P.d.outE[rep] = e;
            if (P.d.E[rep] != e) atomicAdd(P.d.mismatch, 1);
        }
    }
}

// E in temperature order: outE[s][c][t] = E[s][c][slot_of_temp[t]]
__global__ void k_energy_by_temp(Params P, int32_t *out)
{
    const long total = (long)P.S * 2 * P.T;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const long base = (id / P.T) * P.T;
        out[id] = P.d.E[base + P.d.sot[id]];
    }
}

// =========================================================================================================
// a1-a3  Metropolis sweeps
//
// One CTA = R replicas of one sample, resident in shared memory together with the sample's coupling bits for
// n_sweeps sweeps.  Work item = one 32-bit word = 32 same-colour sites of one replica:
//   * local fields bit-sliced: unsat_k = s ^ nbr_k ^ Jneg_k (1 LOP3 per direction per 32 sites), then a
//     carry-save adder tree gives the number n_u of unsatisfied bonds per site as bit planes;
//     a = s_i h_i = 2D - 2 n_u, so "a <= 0" <=> n_u >= D and threshold class k = a/2 = D - n_u;
//   * 8 Philox4x32-10 blocks = 32 words u_j; per site one unsigned compare per class, packed into words C_k;
//   * flip = always | OR_k (class_k & C_k); s ^= flip; dE = 4 * sum_flipped (D - n_u) by popcounts.
// =========================================================================================================
template <int D>
struct Classes {
    uint32_t always;        // n_u >= D
    uint32_t m[D];          // m[k-1]: n_u == D - k  (threshold thrM[t][k])
    uint32_t b0, b1, b2;    // bit planes of n_u
};

template <int D>
__device__ __forceinline__ Classes<D> classify(const uint32_t un[2 * D])
{
    Classes<D> c;
    if constexpr (D == 2) {
        const uint32_t s1 = un[0] ^ un[1] ^ un[2];
        const uint32_t c1 = maj3(un[0], un[1], un[2]);
        const uint32_t c2 = s1 & un[3];
        c.b0 = s1 ^ un[3];
        c.b1 = c1 ^ c2;
        c.b2 = c1 & c2;
        c.always = c1 | c2;                 // n_u >= 2
        c.m[0] = c.b0 & ~c.always;          // n_u == 1 -> k = 1
        c.m[1] = ~(c.b0 | c.always);        // n_u == 0 -> k = 2
    } else {
        const uint32_t sA = un[0] ^ un[1] ^ un[2], cA = maj3(un[0], un[1], un[2]);
        const uint32_t sB = un[3] ^ un[4] ^ un[5], cB = maj3(un[3], un[4], un[5]);
        const uint32_t c0 = sA & sB;
        c.b0 = sA ^ sB;
        c.b1 = cA ^ cB ^ c0;
        c.b2 = maj3(cA, cB, c0);
        c.always = c.b2 | (c.b1 & c.b0);    // n_u >= 3
        c.m[0] = c.b1 & ~c.b0 & ~c.b2;      // n_u == 2 -> k = 1
        c.m[1] = c.b0 & ~c.b1 & ~c.b2;      // n_u == 1 -> k = 2
        c.m[2] = ~(c.b0 | c.b1 | c.b2);     // n_u == 0 -> k = 3
    }
    return c;
}

// C |= BIT iff u < thr: one unsigned compare + one predicated OR of an immediate.  Both issue on the alu pipe and
// leave the fma pipe, which IMAD.WIDE saturates, to Philox (an add-with-carry chain compiles to IMAD.X there).
template <uint32_t BIT>
__device__ __forceinline__ void or_if_less(uint32_t &C, uint32_t u, uint32_t thr)
{
    asm("{\n\t.reg .pred p;\n\tsetp.lt.u32 p, %1, %2;\n\t@p or.b32 %0, %0, %3;\n\t}" : "+r"(C) : "r"(u), "r"(thr), "n"(BIT));
}

// Philox block B of word w: accept bits of sites 4B..4B+3
template <int D, int B>
__device__ __forceinline__ void accept_block(uint32_t w, const Round0Shared &r0, const RoundKeys &rk, const uint32_t thr[D],
                                             uint32_t C[D])
{
    uint32_t u0, u1, u2, u3;
    philox4x32_10_shared(8u * w + (uint32_t)B, r0, rk, u0, u1, u2, u3);
#pragma unroll
    for (int k = 0; k < D; ++k) {
        or_if_less<1u << (4 * B + 0)>(C[k], u0, thr[k]);
        or_if_less<1u << (4 * B + 1)>(C[k], u1, thr[k]);
        or_if_less<1u << (4 * B + 2)>(C[k], u2, thr[k]);
        or_if_less<1u << (4 * B + 3)>(C[k], u3, thr[k]);
    }
}

// Accept bits for the 32 sites of word w: bit j of C[k-1] = (u_j < thr[k-1]), u_j = word (j & 3) of Philox block
// 8w + (j >> 2) of the Metropolis stream (domain 3).
template <int D>
__device__ __forceinline__ void accept_bits(uint32_t w, uint32_t step, uint32_t g, uint32_t tag, const RoundKeys &rk,
                                            const uint32_t thr[D], uint32_t C[D])
{
#pragma unroll
    for (int k = 0; k < D; ++k) C[k] = 0;
    const Round0Shared r0 = philox_round0_shared(step, g, tag, rk);
    accept_block<D, 0>(w, r0, rk, thr, C);
    accept_block<D, 1>(w, r0, rk, thr, C);
    accept_block<D, 2>(w, r0, rk, thr, C);
    accept_block<D, 3>(w, r0, rk, thr, C);
    accept_block<D, 4>(w, r0, rk, thr, C);
    accept_block<D, 5>(w, r0, rk, thr, C);
    accept_block<D, 6>(w, r0, rk, thr, C);
    accept_block<D, 7>(w, r0, rk, thr, C);
}

// One work item.  Returns the energy change of the replica caused by this word's flips.
template <class LAT>
__device__ __forceinline__ int update_word(const LAT &lat, uint32_t *Sown, const uint32_t *Soth, const uint32_t *Jp,
                                           int W, int w, int p, const uint32_t thr[LAT::D], uint32_t step, uint32_t g,
                                           uint32_t tag, const RoundKeys &rk)
{
    constexpr int D = LAT::D;
    uint32_t nb[2 * D], un[2 * D];
    lat.gather(Soth, w, p, nb);
    const uint32_t s = Sown[w];
#pragma unroll
    for (int k = 0; k < 2 * D; ++k) un[k] = s ^ nb[k] ^ Jp[k * W + w];
    const Classes<D> cl = classify<D>(un);
    uint32_t C[D];
    accept_bits<D>((uint32_t)w, step, g, tag, rk, thr, C);
    uint32_t flip = cl.always;
#pragma unroll
    for (int k = 0; k < D; ++k) flip |= cl.m[k] & C[k];
    flip &= lat.valid(w);
    Sown[w] = s ^ flip;
    // dE = sum_flipped 2a = 4 * sum_flipped (D - n_u)
    return 4 * (D * __popc(flip) - __popc(flip & cl.b0) - 2 * __popc(flip & cl.b1) - 4 * __popc(flip & cl.b2));
}

// grid: (2T/R groups, S).  dynamic smem: [2][2D][W] couplings | [R][2][W] spins | [R][4] thresholds | [R] dE
template <class LAT>
__global__ void __launch_bounds__(128, 7) k_sweep(LAT lat, Params P, int R, uint32_t step0, int n_sweeps)
{
    constexpr int D = LAT::D;
    extern __shared__ uint32_t smem[];
    const int W = lat.words();
    uint32_t *sJ = smem;                       // [2][2D][W]
    uint32_t *sS = sJ + 2 * 2 * D * W;         // [R][2][W]
    uint32_t *sThr = sS + R * 2 * W;           // [R][4]
    int *sdE = (int *)(sThr + R * 4);          // [R]
    const int s = blockIdx.y;
    const int q0 = blockIdx.x * R;             // first replica (q = c*T + r) of this CTA
    const size_t rep0 = (size_t)s * 2 * P.T + q0;
    const uint32_t g = P.g0 + (uint32_t)s;

    for (int i = threadIdx.x; i < 2 * 2 * D * W; i += blockDim.x) sJ[i] = P.d.Jn[(size_t)s * 2 * 2 * D * W + i];
    for (int i = threadIdx.x; i < R * 2 * W; i += blockDim.x) sS[i] = P.d.spin[rep0 * 2 * W + i];
    for (int i = threadIdx.x; i < R; i += blockDim.x) {
        const int t = P.d.tos[rep0 + i];
#pragma unroll
        for (int k = 0; k < 4; ++k) sThr[4 * i + k] = P.d.thrM[4 * t + k];
        sdE[i] = 0;
    }
    __syncthreads();

    const int items = R * W;
    for (int it = 0; it < n_sweeps; ++it) {
        for (int p = 0; p < 2; ++p) {
            for (int item = threadIdx.x; item < items; item += blockDim.x) {
                const int qi = item / W, w = item - qi * W;
                const int q = q0 + qi;
                const int c = (q >= P.T) ? 1 : 0, r = q - c * P.T;
                uint32_t thr[D];
#pragma unroll
                for (int k = 0; k < D; ++k) thr[k] = sThr[4 * qi + k];
                const int dE = update_word(lat, sS + (qi * 2 + p) * W, sS + (qi * 2 + (1 - p)) * W, sJ + p * 2 * D * W,
                                           W, w, p, thr, step0 + (uint32_t)it, g, make_tag(DOM_METRO, p, c, r), P.rk);
                atomicAdd(sdE + qi, dE);
            }
            __syncthreads();
        }
    }
    for (int i = threadIdx.x; i < R * 2 * W; i += blockDim.x) P.d.spin[rep0 * 2 * W + i] = sS[i];
    for (int i = threadIdx.x; i < R; i += blockDim.x) P.d.E[rep0 + i] += sdE[i];
}

// =========================================================================================================
// a4  parallel-tempering pass (Eq. (5)).  One warp per (sample, chain):
// the lanes draw the T-1 Philox words in parallel, lane 0 walks the ladder sequentially on a temperature-ordered
// copy of the energies in shared memory.  Only the two index arrays change.
// =========================================================================================================
// Round-trip bookkeeping after PT pass number n (1-based) of chain `chain` = s*2 + c (R27-R29): r0 / r1 = the slots now
// at temperature index 0 / T-1.  Called by one thread per chain.
__device__ __forceinline__ void round_trip_update(const Params &P, size_t chain, int r0, int r1, uint32_t n)
{
    uint32_t *lab = P.d.rtLabel + chain * P.T, *st = P.d.rtStart + chain * P.T;
    if (lab[r1] == 1u) lab[r1] = 2u;
    const uint32_t l0 = lab[r0];
    if (l0 == 2u) {
        const int b = 31 - __clz(n);
        P.d.rtTrips[chain * P.T + r0] += 1u;
        P.d.rtSum[chain * 32 + b] += (unsigned long long)(n - st[r0]);
        P.d.rtCnt[chain * 32 + b] += 1ull;
        lab[r0] = 1u;
        st[r0] = n;
    } else if (l0 == 0u) {
        lab[r0] = 1u;
        st[r0] = n;
    }
}

__device__ __forceinline__ uint32_t thrX_lookup(const Params &P, int t, uint32_t m)
{
    return (m < P.strideX) ? __ldg(P.d.thrX + (size_t)t * P.strideX + m) : 0u;
}

// swap threshold for |dE| = absdE at pair t: the +-J table entry m = |dE|/4, or, with fixed-point couplings (R34),
// THR(-(|dbeta| * ldexp(|dE|, -fbits))) evaluated in double
__device__ __forceinline__ uint32_t swap_threshold(const Params &P, int t, uint32_t absdE)
{
    if (!P.gauss) return thrX_lookup(P, t, absdE >> 2);
    const double v = floor(ldexp(exp(-(P.d.absdb[t] * ldexp((double)absdE, -P.fbits))), 32));
    if (v >= 4294967295.0) return 4294967295u;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// PT decision for an unfavourable swap with |dE| = absdE at pair t: u < swap_threshold, decided exactly.  +-J: the table.
// Fixed point: the float bracket of gauss.cuh (accept_site) around Y / 512 = 2^(23 + |dE| slope_t): (float)|dE| and the slope
// carry 2^-24 relative each of an exponent below 150 in magnitude, the fma rounds once (2^-18), ex2.approx is good to 2^-22
// -- under 2e-5 relative in all, against a bracket of 1e-4 -- and only a draw inside the bracket pays for the double exp.
__device__ __forceinline__ bool swap_accept(const Params &P, int t, uint32_t u, uint32_t absdE)
{
    if (!P.gauss) return u < thrX_lookup(P, t, absdE >> 2);
    const float t9 = ex2_approx(fmaf((float)absdE, __ldg(P.d.swapSlope + t), 23.0f));
    const float uf9 = __uint_as_float(0x4B000000u | (u >> 9)) - 8388608.0f;    // exact: 23 bits fill the mantissa
    if (uf9 + 2.0f < t9 * 0.9999f) return true;
    if (uf9 > fmaf(t9, 1.0001f, 1.0f)) return false;
    return u < swap_threshold(P, t, absdE);
}

constexpr int kExchangeTableT = 64;     // ladders up to this length evaluate all (carried, rung) decisions in parallel

// dynamic smem: per warp [T] energies by temperature + [T] slot_of_temp + [T] draws + [T] signs / accept flags.  GLOBAL_SCRATCH (very long ladders):
// the same walk on outE / slot_of_temp in global memory.
template <bool GLOBAL_SCRATCH>
__global__ void k_exchange(Params P, uint32_t step)
{
    extern __shared__ int32_t xsm[];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const long chain = (long)blockIdx.x * wpb + wib;
    if (chain >= (long)P.S * 2) return;
    const int s = (int)(chain >> 1), c = (int)(chain & 1);
    const uint32_t g = P.g0 + (uint32_t)s;
    const int T = P.T;
    const size_t base = (size_t)chain * T;
    int32_t *Et = GLOBAL_SCRATCH ? P.d.outE + base : xsm + (size_t)wib * 4 * T;
    int32_t *so = GLOBAL_SCRATCH ? P.d.sot + base : Et + T;
    for (int t = lane; t < T; t += 32) {
        const int r = P.d.sot[base + t];
        if (!GLOBAL_SCRATCH) so[t] = r;
        Et[t] = P.d.E[base + r];
    }
    __syncwarp();
    int32_t ea = 0, ra = 0;
    if constexpr (!GLOBAL_SCRATCH) {
        // draws and signs staged in shared memory by all lanes; lane 0 walks with the next rung prefetched; accept
        // flags are left in the sign array (value 2) and counted by all lanes afterwards
        uint32_t *U = (uint32_t *)(so + T);
        int32_t *SG = (int32_t *)(U + T);
        for (int t = lane; t < T - 1; t += 32) {
            uint32_t u, o1, o2, o3;
            philox4x32_10((uint32_t)t, step, g, make_tag(DOM_SWAP, 0, c, 0), P.rk, u, o1, o2, o3);
            U[t] = u;
            SG[t] = P.d.sgn[t];
        }
        __syncwarp();
        if (T > 1 && T <= kExchangeTableT) {
            // Short ladders: the walk is one dependent chain per (sample, chain) and the threshold lookup from L2 per rung
            // is half of its stall samples.  The replica carried up to rung t is the ORIGINAL resident of some position
            // j <= t, so every decision the walk can meet is one of the T (T-1) / 2 pairs (j, t): all lanes evaluate them
            // side by side, eight independent lookups in flight per lane, then lane 0 walks with one byte load per rung.
            uint8_t *ACC = (uint8_t *)(xsm + (size_t)wpb * 4 * T) + (size_t)wib * T * T;       // ACC[t * T + j]
            for (int j = lane; j < T - 1; j += 32) {
                const int32_t ej = Et[j];
                for (int t0 = j; t0 < T - 1; t0 += 8) {
                    if (!P.gauss) {
                        uint32_t thr[8];
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const int t = min(t0 + k, T - 2);
                            const int32_t dE = ej - Et[t + 1];
                            const uint32_t m = (uint32_t)(dE < 0 ? -dE : dE) >> 2;
                            thr[k] = __ldg(P.d.thrX + (size_t)t * P.strideX + min(m, P.strideX - 1u));
                            if (m >= P.strideX) thr[k] = 0u;
                        }
#pragma unroll
                        for (int k = 0; k < 8; ++k) {
                            const int t = t0 + k;
                            if (t < T - 1) {
                                const int32_t dE = ej - Et[t + 1];
                                ACC[t * T + j] = ((long long)SG[t] * dE <= 0 || U[t] < thr[k]) ? 1 : 0;
                            }
                        }
                    } else {
                        for (int t = t0; t < min(t0 + 8, T - 1); ++t) {
                            const int32_t dE = ej - Et[t + 1];
                            bool acc = (long long)SG[t] * dE <= 0;
                            if (!acc) acc = swap_accept(P, t, U[t], (uint32_t)(dE < 0 ? -dE : dE));
                            ACC[t * T + j] = acc ? 1 : 0;
                        }
                    }
                }
            }
            __syncwarp();
            if (lane == 0) {
                ra = so[0];
                int j = 0;
                int32_t rb = so[1];
                for (int t = 0; t < T - 1; ++t) {
                    const int32_t rbn = (t + 2 < T) ? so[t + 2] : 0;       // positions > t + 1 are not modified before they are read
                    const bool acc = ACC[t * T + j] != 0;
                    so[t] = acc ? rb : ra;                                  // position t is final
                    if (acc) SG[t] = 2;
                    ra = acc ? ra : rb;
                    j = acc ? j : t + 1;
                    rb = rbn;
                }
            }
        } else if (lane == 0 && T > 1) {
            ea = Et[0]; ra = so[0];
            int32_t eb = Et[1], rb = so[1];
            for (int t = 0; t < T - 1; ++t) {
                int32_t ebn = 0, rbn = 0;
                if (t + 2 < T) { ebn = Et[t + 2]; rbn = so[t + 2]; }     // positions > t + 1 are not modified before they are read
                const int32_t dE = ea - eb;
                bool acc = (long long)SG[t] * dE <= 0;
                if (!acc) acc = swap_accept(P, t, U[t], (uint32_t)(dE < 0 ? -dE : dE));
                if (acc) { Et[t] = eb; so[t] = rb; SG[t] = 2; }          // position t is final; (ea, ra) moves up to t+1
                else     { Et[t] = ea; so[t] = ra; ea = eb; ra = rb; }
                eb = ebn; rb = rbn;
            }
        } else if (lane == 0) { ea = Et[0]; ra = so[0]; }
        __syncwarp();
        for (int t = lane; t < T - 1; t += 32)
            if (SG[t] == 2) P.d.accepts[(size_t)chain * (T - 1) + t] += 1ull;
    } else {
    if (lane == 0) { ea = Et[0]; ra = so[0]; }
    for (int tb = 0; tb < T - 1; tb += 32) {
        const int tl = tb + lane;
        uint32_t u_l = 0, o1, o2, o3;
        if (tl < T - 1) philox4x32_10((uint32_t)tl, step, g, make_tag(DOM_SWAP, 0, c, 0), P.rk, u_l, o1, o2, o3);
        const int nstep = min(32, T - 1 - tb);
        for (int j = 0; j < nstep; ++j) {
            const uint32_t u = __shfl_sync(0xFFFFFFFFu, u_l, j);
            if (lane == 0) {
                const int t = tb + j;
                const int32_t eb = Et[t + 1], rb = so[t + 1];
                const int32_t dE = ea - eb;
                const int sg = P.d.sgn[t];
                const bool acc = ((long long)sg * dE <= 0) || swap_accept(P, t, u, (uint32_t)(dE < 0 ? -dE : dE));
                if (acc) {
                    Et[t] = eb; so[t] = rb;                 // position t is final; (ea, ra) moves up to t+1
                    P.d.accepts[(size_t)chain * (T - 1) + t] += 1ull;
                } else {
                    Et[t] = ea; so[t] = ra;
                    ea = eb; ra = rb;
                }
            }
        }
    }
    }
    if (lane == 0) {
        Et[T - 1] = ea; so[T - 1] = ra;
        if (P.track && T > 1) round_trip_update(P, (size_t)chain, so[0], ra, step + 1u);
    }
    __syncwarp();
    for (int t = lane; t < T; t += 32) {
        const int r = so[t];
        P.d.sot[base + t] = r;
        P.d.tos[base + r] = t;
    }
}

// =========================================================================================================
// a5  Houdayer cluster exchange, GENERAL path (Eq. (10)): any lattice
// implementation, one CTA per (sample, t), one neighbour step per iteration on the colour layout.
// The q = -1 cluster is grown on bit maps: C_p |= (OR of the neighbour bits of C_{1-p}) & Neg_p, alternating
// colours until nothing changes -- the fixed point is exactly the connected component of the seed.
// =========================================================================================================
// dynamic smem: Neg[2][W] | Cl[2][W] | scan[blockDim/32 + 2]
// Tail shared by the one-CTA-per-pair kernels: Cl[2][W] holds a union of q = -1 components in the colour layout.
// size, delta = 2 * sum over boundary bonds of J A_i A_j = 2 * (#boundary - 2 #boundary&unsatisfied) (old spins), each
// bond seen from its black endpoint; then the set is negated in both configurations and E, last, cum are updated.
// red: 2 * nwarps ints of shared memory.  Every thread of the CTA must call.
template <class LAT>
__device__ __forceinline__ void cta_exchange_set(const LAT &lat, const Params &P, int s, int t, size_t repA, size_t repB,
                                                 uint32_t *const A[2], uint32_t *const B[2], const uint32_t *Cl, int *red)
{
    constexpr int D = LAT::D;
    const int W = lat.words();
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nwarps = blockDim.x >> 5;
    int size = 0, delta = 0;
    for (int w = tid; w < W; w += blockDim.x) {
        const uint32_t cb = Cl[w], cwh = Cl[W + w], v = lat.valid(w);
        size += __popc(cb) + __popc(cwh);
        uint32_t nbC[2 * D], nbA[2 * D];
        lat.gather(Cl + W, w, 0, nbC);
        lat.gather(A[1], w, 0, nbA);
        const uint32_t ab = A[0][w];
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) {
            const uint32_t bnd = (cb ^ nbC[k]) & v;
            const uint32_t uns = ab ^ nbA[k] ^ J_words(P, s, 0, k)[w];
            delta += 2 * (__popc(bnd) - 2 * __popc(bnd & uns));
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        size += __shfl_xor_sync(0xFFFFFFFFu, size, o);
        delta += __shfl_xor_sync(0xFFFFFFFFu, delta, o);
    }
    __syncthreads();                 // all reads of the old A done before anyone writes; red[] reusable
    if (lane == 0) { red[wid] = size; red[nwarps + wid] = delta; }
    __syncthreads();
    for (int p = 0; p < 2; ++p)
        for (int w = tid; w < W; w += blockDim.x) {
            const uint32_t c = Cl[p * W + w];
            if (c) { A[p][w] ^= c; B[p][w] ^= c; }
        }
    if (tid == 0) {
        int sz = 0, dl = 0;
        for (int i = 0; i < nwarps; ++i) { sz += red[i]; dl += red[nwarps + i]; }
        P.d.E[repA] += dl;
        P.d.E[repB] -= dl;
        P.d.last[(size_t)s * P.T + t] = (uint32_t)sz;
        P.d.cum[(size_t)s * P.T + t] += (unsigned long long)sz;
    }
}

// move: number of this single-cluster move within the step (R36); pairs with nclu[t] <= move do nothing.
template <class LAT>
__global__ void __launch_bounds__(128) k_houdayer_gen(LAT lat, Params P, uint32_t step, uint32_t move)
{
    constexpr int D = LAT::D;
    extern __shared__ uint32_t hsm[];
    const int W = lat.words();
    uint32_t *Neg = hsm, *Cl = hsm + 2 * W;
    int *scan = (int *)(Cl + 2 * W);           // [0..nwarps): warp totals; [nwarps]: seed word; [nwarps+1]: seed colour|bit
    const int t = blockIdx.x, s = blockIdx.y;
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5, nwarps = blockDim.x >> 5;
    if (move >= (uint32_t)P.d.nclu[t]) {
        if (move == 0 && tid == 0) P.d.last[(size_t)s * P.T + t] = 0;
        return;
    }
    const size_t repA = rep_index(P, s, 0, P.d.sot[rep_index(P, s, 0, t)]);
    const size_t repB = rep_index(P, s, 1, P.d.sot[rep_index(P, s, 1, t)]);
    uint32_t *A[2] = {spin_words(P, repA, 0), spin_words(P, repA, 1)};
    uint32_t *B[2] = {spin_words(P, repB, 0), spin_words(P, repB, 1)};

    // q_i = -1 bits; per-thread chunk of consecutive words for the prefix count in site-index order
    const int cpt = (W + blockDim.x - 1) / blockDim.x;
    const int w_lo = min(W, tid * cpt), w_hi = min(W, w_lo + cpt);
    int local = 0;
    for (int w = w_lo; w < w_hi; ++w) {
        const uint32_t v = lat.valid(w);
        const uint32_t n0 = (A[0][w] ^ B[0][w]) & v, n1 = (A[1][w] ^ B[1][w]) & v;
        Neg[w] = n0; Neg[W + w] = n1;
        Cl[w] = 0; Cl[W + w] = 0;
        local += __popc(n0) + __popc(n1);
    }
    int incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
        if (lane >= o) incl += v;
    }
    if (lane == 31) scan[wid] = incl;
    __syncthreads();
    int warp_off = 0, n_neg = 0;
    for (int i = 0; i < nwarps; ++i) {
        if (i < wid) warp_off += scan[i];
        n_neg += scan[i];
    }
    const int excl = warp_off + incl - local;
    if (n_neg == 0) {
        if (tid == 0) P.d.last[(size_t)s * P.T + t] = 0;
        return;
    }
    uint32_t u, o1, o2, o3;
    philox4x32_10(move, step, P.g0 + (uint32_t)s, make_tag(DOM_HOUD, 0, 0, t), P.rk, u, o1, o2, o3);
    const int kth = (int)(((unsigned long long)u * (unsigned long long)n_neg) >> 32);
    if (kth >= excl && kth < excl + local) {
        // this thread's chunk holds the seed: walk words, then the 32 half-indices of the word in site order
        int rem = kth - excl;
        for (int w = w_lo; w < w_hi; ++w) {
            const int cw = __popc(Neg[w]) + __popc(Neg[W + w]);
            if (rem >= cw) { rem -= cw; continue; }
            for (int b = 0; b < 32; ++b) {
                const int h = 32 * w + b;
                const int first = colour_of_site(2 * h, P.L, P.D);     // colour of site 2h; site 2h+1 has the other
                const uint32_t f = (Neg[first * W + w] >> b) & 1u, g2 = (Neg[(1 - first) * W + w] >> b) & 1u;
                if (f) { if (rem == 0) { Cl[first * W + w] = 1u << b; break; } --rem; }
                if (g2) { if (rem == 0) { Cl[(1 - first) * W + w] = 1u << b; break; } --rem; }
            }
            break;
        }
    }
    __syncthreads();

    // grow to the fixed point
    for (;;) {
        int changed = 0;
#pragma unroll 1
        for (int p = 0; p < 2; ++p) {
            for (int w = tid; w < W; w += blockDim.x) {
                const uint32_t neg = Neg[p * W + w], cur = Cl[p * W + w];
                if (neg & ~cur) {
                    uint32_t nb[2 * D];
                    lat.gather(Cl + (1 - p) * W, w, p, nb);
                    uint32_t any = 0;
#pragma unroll
                    for (int k = 0; k < 2 * D; ++k) any |= nb[k];
                    const uint32_t nw = cur | (any & neg);
                    if (nw != cur) { Cl[p * W + w] = nw; changed = 1; }
                }
            }
            __syncthreads();
        }
        if (!__syncthreads_or(changed)) break;
    }

    cta_exchange_set(lat, P, s, t, repA, repB, A, B, Cl, scan);
}

// =========================================================================================================
// a5  Houdayer cluster exchange, FAST path: one warp per (sample, t) pair (houdayer.cuh).
// grid: ceil(S*T / warps per CTA); dynamic smem: kPairScratchWords<LAT> words per warp.
// =========================================================================================================
template <class LAT>
__global__ void __launch_bounds__(128, 6) k_houdayer(LAT lat, Params P, uint32_t step, uint32_t move)
{
    extern __shared__ uint32_t hsm[];
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    // Launch order: coldest temperature first, all samples of one temperature next to each other.  Cluster sizes (and with
    // them the rounds a pair needs) grow with beta, so the long pairs start first and the four pairs of a CTA take alike.
    const long gw = (long)blockIdx.x * wpb + wib;
    if (gw >= (long)P.S * P.T) return;
    const int t = P.d.tcold[gw / P.S], s = (int)(gw % P.S);
    const long pair = (long)s * P.T + t;
    if (move >= (uint32_t)P.d.nclu[t]) {                    // R36: this temperature makes no move number `move`
        if (move == 0 && lane == 0) P.d.last[pair] = 0;
        return;
    }
    const size_t repA = rep_index(P, s, 0, P.d.sot[rep_index(P, s, 0, t)]);
    const size_t repB = rep_index(P, s, 1, P.d.sot[rep_index(P, s, 1, t)]);
    uint32_t u, o1, o2, o3;
    philox4x32_10(move, step, P.g0 + (uint32_t)s, make_tag(DOM_HOUD, 0, 0, t), P.rk, u, o1, o2, o3);
    int delta;
    const int size = houdayer_warp(lat, spin_words(P, repA, 0), spin_words(P, repA, 1), spin_words(P, repB, 0),
                                   spin_words(P, repB, 1), J_words(P, s, 0, 0), hsm + (size_t)wib * kPairScratchWords<LAT>, u, lane, delta);
    if (lane == 0) {
        if (delta) { P.d.E[repA] += delta; P.d.E[repB] -= delta; }
        P.d.last[pair] = (uint32_t)size;
        P.d.cum[pair] += (unsigned long long)size;
    }
}

// =========================================================================================================
// a6  two-replica measurement (Eq. (4); link overlap R14).  One CTA per (sample, t).
//   Q = N - 2 #(q_i = -1);   QL = D*N - 2 #(bonds with q_i != q_j), each bond seen from its black endpoint.
// dynamic smem: NegW[W] | red[2]
// =========================================================================================================
template <class LAT>
__global__ void __launch_bounds__(128) k_measure(LAT lat, Params P, int32_t *outQ, int32_t *outQL)
{
    constexpr int D = LAT::D;
    extern __shared__ uint32_t msm[];
    const int W = lat.words();
    uint32_t *NegW = msm;
    int *red = (int *)(msm + W);
    const int t = blockIdx.x, s = blockIdx.y, tid = threadIdx.x;
    const size_t repA = rep_index(P, s, 0, P.d.sot[rep_index(P, s, 0, t)]);
    const size_t repB = rep_index(P, s, 1, P.d.sot[rep_index(P, s, 1, t)]);
    const uint32_t *Ab = spin_words(P, repA, 0), *Aw = spin_words(P, repA, 1);
    const uint32_t *Bb = spin_words(P, repB, 0), *Bw = spin_words(P, repB, 1);
    if (tid < 2) red[tid] = 0;
    for (int w = tid; w < W; w += blockDim.x) NegW[w] = (Aw[w] ^ Bw[w]) & lat.valid(w);
    __syncthreads();
    int nneg = 0, ndiff = 0;
    for (int w = tid; w < W; w += blockDim.x) {
        const uint32_t v = lat.valid(w), nbk = (Ab[w] ^ Bb[w]) & v;
        nneg += __popc(nbk) + __popc(NegW[w]);
        uint32_t nb[2 * D];
        lat.gather(NegW, w, 0, nb);
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) ndiff += __popc((nbk ^ nb[k]) & v);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nneg += __shfl_xor_sync(0xFFFFFFFFu, nneg, o);
        ndiff += __shfl_xor_sync(0xFFFFFFFFu, ndiff, o);
    }
    if ((tid & 31) == 0) { atomicAdd(red, nneg); atomicAdd(red + 1, ndiff); }
    __syncthreads();
    if (tid == 0) {
        outQ[(size_t)s * P.T + t] = P.N - 2 * red[0];
        if (outQL) outQL[(size_t)s * P.T + t] = P.D * P.N - 2 * red[1];
    }
}

// Same measurement with one WARP per (sample, t) pair and several pairs per CTA: on small lattices (W words per
// colour <= 128) a CTA per pair is mostly launch overhead.  dynamic smem: W words per warp.
template <class LAT>
__global__ void __launch_bounds__(128) k_measure_warp(LAT lat, Params P, int32_t *outQ, int32_t *outQL)
{
    constexpr int D = LAT::D;
    extern __shared__ uint32_t msm[];
    const int W = lat.words();
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const long pair = (long)blockIdx.x * wpb + wib;
    if (pair >= (long)P.S * P.T) return;
    const int s = (int)(pair / P.T), t = (int)(pair - (long)s * P.T);
    uint32_t *NegW = msm + (size_t)wib * W;
    const size_t repA = rep_index(P, s, 0, P.d.sot[rep_index(P, s, 0, t)]);
    const size_t repB = rep_index(P, s, 1, P.d.sot[rep_index(P, s, 1, t)]);
    const uint32_t *Ab = spin_words(P, repA, 0), *Aw = spin_words(P, repA, 1);
    const uint32_t *Bb = spin_words(P, repB, 0), *Bw = spin_words(P, repB, 1);
    for (int w = lane; w < W; w += 32) NegW[w] = (Aw[w] ^ Bw[w]) & lat.valid(w);
    __syncwarp();
    int nneg = 0, ndiff = 0;
    for (int w = lane; w < W; w += 32) {
        const uint32_t v = lat.valid(w), nbk = (Ab[w] ^ Bb[w]) & v;
        nneg += __popc(nbk) + __popc(NegW[w]);
        if (outQL) {
            uint32_t nb[2 * D];
            lat.gather(NegW, w, 0, nb);
#pragma unroll
            for (int k = 0; k < 2 * D; ++k) ndiff += __popc((nbk ^ nb[k]) & v);
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        nneg += __shfl_xor_sync(0xFFFFFFFFu, nneg, o);
        ndiff += __shfl_xor_sync(0xFFFFFFFFu, ndiff, o);
    }
    if (lane == 0) {
        outQ[pair] = P.N - 2 * nneg;
        if (outQL) outQL[pair] = P.D * P.N - 2 * ndiff;
    }
}

// =========================================================================================================
// NEXT-2  overlap profiles (R31): prof[s][t][mu][x] = sum of q_i over the plane x_mu = x
//         = L^(D-1) - 2 #(q_i = -1 in that plane).  One CTA per (sample, t); any even L (coordinates from the
// half-index); only the q = -1 sites touch the shared counters.  dynamic smem: D*L counters.
// =========================================================================================================
template <class LAT>
__global__ void __launch_bounds__(128) k_profile(LAT lat, Params P, int32_t *out)
{
    extern __shared__ int pneg[];
    const int t = blockIdx.x, s = blockIdx.y, tid = threadIdx.x;
    const int DL = P.D * P.L;
    for (int i = tid; i < DL; i += blockDim.x) pneg[i] = 0;
    __syncthreads();
    const size_t repA = rep_index(P, s, 0, P.d.sot[rep_index(P, s, 0, t)]);
    const size_t repB = rep_index(P, s, 1, P.d.sot[rep_index(P, s, 1, t)]);
    for (int id = tid; id < 2 * P.W; id += blockDim.x) {
        const int p = id / P.W, w = id - p * P.W;
        uint32_t x = spin_words(P, repA, p)[w] ^ spin_words(P, repB, p)[w];
        const int left = P.NH - 32 * w;
        if (left < 32) x &= (1u << left) - 1u;
        while (x) {
            const int b = __ffs(x) - 1;
            x &= x - 1;
            int cx, cy, cz;
            nat_coords<LAT>(nat_site_of<LAT>(32 * w + b, p, P.L, P.D), P.L, P.D, cx, cy, cz);
            atomicAdd(pneg + cx, 1);
            atomicAdd(pneg + P.L + cy, 1);
            if (LAT::D == 3) atomicAdd(pneg + 2 * P.L + cz, 1);
        }
    }
    __syncthreads();
    const int plane = P.N / P.L;
    int32_t *o = out + ((size_t)s * P.T + t) * DL;
    for (int i = tid; i < DL; i += blockDim.x) o[i] = plane - 2 * pneg[i];
}

// Same profiles on the power-of-two lattices, by popcounts on the natural-order bit map (bit i = site i) of q = -1 sites:
// one WARP per (sample, t) pair, four pairs per CTA.  Planes of constant y (z): popcount of a row, one shared-memory add per
// WORD (the per-site version above makes one per q = -1 site).  Planes of constant x: the column sums of a block of 32 words
// are the popcounts of the 32 x 32 bit TRANSPOSE of the block, five shuffle-and-mask butterfly stages across the lanes,
// after which lane b holds bit b of all 32 words.  dynamic smem: D*L counters per warp.
template <class LAT>
__global__ void __launch_bounds__(128) k_profile_fast(LAT lat, Params P, int32_t *out)
{
    using NL = NatLat<LAT::D, LAT::kLog2L>;
    constexpr int D = LAT::D, L = NL::L, LG = LAT::kLog2L, NW = NL::NW, W = NL::W;
    constexpr bool SMALL = NL::kSmall;                 // several rows per word (L < 32)
    constexpr int CLS = SMALL ? 1 : NL::WR;            // classes of words that hold the same x range
    constexpr int RPW = SMALL ? 32 / L : 1;            // rows per word
    constexpr int DL = D * L;
    extern __shared__ int pcnt[];
    const unsigned FULL = 0xFFFFFFFFu;
    const int wib = threadIdx.x >> 5, lane = threadIdx.x & 31, wpb = blockDim.x >> 5;
    const long pair = (long)blockIdx.x * wpb + wib;
    if (pair >= (long)P.S * P.T) return;
    const int s = (int)(pair / P.T), t = (int)(pair - (long)s * P.T);
    int *cnt = pcnt + wib * DL;
    for (int i = lane; i < DL; i += 32) cnt[i] = 0;
    __syncwarp();
    const size_t repA = rep_index(P, s, 0, P.d.sot[rep_index(P, s, 0, t)]);
    const size_t repB = rep_index(P, s, 1, P.d.sot[rep_index(P, s, 1, t)]);
    const uint32_t *A0 = spin_words(P, repA, 0), *A1 = A0 + W, *B0 = spin_words(P, repB, 0), *B1 = B0 + W;
    (void)lat;
    if constexpr (!SMALL && NL::WR >= 2) {
        // L >= 64: a colour word holds 32 same-colour sites of one row, x = 64 jc + 2 k + x0 with x0 = (colour + y) & 1, so the
        // words of one class (jc, x0) -- colour 0 on rows y = x0 (mod 2), colour 1 on the others -- share their x positions and
        // are transposed as they are: no colour -> natural interleave at all.
        constexpr int WRC = NL::WR / 2;                 // colour words per row
        constexpr int ROWS = NW / NL::WR;               // lattice rows
#pragma unroll 1
        for (int cls = 0; cls < 2 * WRC; ++cls) {
            const int jc = cls >> 1, x0 = cls & 1;
            int acc = 0;                                // lane b: q = -1 sites with x = 64 jc + 2 b + x0
#pragma unroll 1
            for (int base = 0; base < ROWS; base += 32) {               // ROWS words of the class: one per row
                const int y = base + lane;
                uint32_t x = 0;
                if (y < ROWS) {
                    const int p = (x0 + y) & 1;                         // the colour whose sites of row y start at x0
                    const int w = y * WRC + jc;
                    x = (p ? A1[w] ^ B1[w] : A0[w] ^ B0[w]);
                    const int c = __popc(x);
                    if (c) atomicAdd(cnt + L + (y & (L - 1)), c);
                }
#pragma unroll
                for (int k = 16; k >= 1; k >>= 1) {
                    const uint32_t m = (k == 16) ? 0x0000FFFFu : (k == 8) ? 0x00FF00FFu : (k == 4) ? 0x0F0F0F0Fu : (k == 2) ? 0x33333333u : 0x55555555u;
                    const uint32_t o = __shfl_xor_sync(FULL, x, k);
                    x = (lane & k) ? ((x & ~m) | ((o >> k) & m)) : ((x & m) | ((o << k) & ~m));
                }
                acc += __popc(x);
            }
            cnt[64 * jc + 2 * lane + x0] = acc;
        }
    } else
#pragma unroll 1
    for (int j = 0; j < CLS; ++j) {
        int acc = 0;                                   // lane b: number of q = -1 sites on bit b of the words of class j
#pragma unroll 1
        for (int base = 0; base < NW / CLS; base += 32) {
            const int idx = base + lane;
            uint32_t x = 0;
            if (idx < NW / CLS) {
                const int n = idx * CLS + j, w = n >> 1;
                const uint32_t x0 = A0[w] ^ B0[w], x1 = A1[w] ^ B1[w];
                x = (n & 1) ? NL::interleave(n, x0 >> 16, x1 >> 16) : NL::interleave(n, x0, x1);
#pragma unroll
                for (int q = 0; q < RPW; ++q) {
                    const int r = SMALL ? n * RPW + q : idx;                    // row index y + L z
                    const int c = SMALL ? __popc(x & (((L < 32 ? (1u << (L & 31)) : 0u) - 1u) << (q * L))) : __popc(x);
                    if (c) {
                        atomicAdd(cnt + L + (r & (L - 1)), c);
                        if (D == 3) atomicAdd(cnt + 2 * L + (r >> LG), c);
                    }
                }
            }
            // 32 x 32 bit transpose across the lanes (row = lane, column = bit, LSB = column 0)
#pragma unroll
            for (int k = 16; k >= 1; k >>= 1) {
                const uint32_t m = (k == 16) ? 0x0000FFFFu : (k == 8) ? 0x00FF00FFu : (k == 4) ? 0x0F0F0F0Fu : (k == 2) ? 0x33333333u : 0x55555555u;
                const uint32_t o = __shfl_xor_sync(FULL, x, k);
                // lanes with bit k clear keep their low part and take the partner's low part into their high part;
                // lanes with bit k set keep their high part and take the partner's high part into their low part
                x = (lane & k) ? ((x & ~m) | ((o >> k) & m)) : ((x & m) | ((o << k) & ~m));
            }
            acc += __popc(x);
        }
        if (SMALL) atomicAdd(cnt + (lane & (L - 1)), acc);
        else cnt[32 * j + lane] = acc;
    }
    __syncwarp();
    const int plane = P.N / L;
    int32_t *o = out + (size_t)pair * DL;
    for (int i = lane; i < DL; i += 32) o[i] = plane - 2 * cnt[i];
}

}  // namespace ptg
