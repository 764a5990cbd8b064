// a5  Houdayer cluster exchange inside the fused kernel, FOUR LANES PER PAIR (Eq. (10)).
// 2D L = 32 (a lattice row = one 32-bit natural word, 32 rows), the shape of BASELINE config 2.
//
// The lane-per-pair phase (houdayer_lanes.cuh) runs on ONE warp of the CTA for as many Gauss-Seidel passes as the slowest
// of its 32 pairs needs (C2 states: 9-11, mean 4.4) while the other three warps wait at the barrier: it is 23 % of the
// kernel's instructions but 60 % of a CTA's time, and with at most 7 CTAs per SM the schedulers run out of eligible warps
// (ncu: 0.98 eligible warps per cycle, issue active 52 %).  Here every pair gets four lanes, each owning a strip of 8 rows
// in REGISTERS, so all four warps of the CTA work (8 pairs each) and a warp waits only for the slowest of 8 pairs.  One
// round = fetch the neighbour strips' boundary rows by shuffle, sweep the strip down and up (Gauss-Seidel inside the
// strip, Jacobi across strips); odd strips are held in reverse row order, so the same index sweep runs down the lattice
// on even strips and up on odd ones and membership crosses two strips per round in either direction (houdayer_rows.cuh).
// A row step closes the row along x with the carry trick.  Offline replay of the oracle's C2 states: 3.4 rounds per pair
// on average, 4.8 for the slowest of 8.  Same least fixed point = the connected component of the seed (bit-exact parity).
#pragma once
#include "houdayer_rows.cuh"
#include "philox.cuh"

namespace ptg {

template <class LAT, bool FAST = LAT::kFast>
struct QuadHoudayer { static constexpr bool kEligible = false; static constexpr int kScratchWords = 0; };

template <class LAT>
struct QuadHoudayer<LAT, true> {
    static constexpr bool kEligible = (LAT::D == 2 && LAT::kLog2L == 5);
    static constexpr int kPairStride = 33;                      // 2W + 1 words of cluster map per pair (odd: conflict-free)
    static constexpr int kScratchWords = 32 * kPairStride;      // per CTA: the 32 pairs of one temperature group
};

// One pair per 4 consecutive lanes; ALL lanes of the warp must call (inactive pairs pass active = false).
// A0/A1, B0/B1: the pair's colour-0 / colour-1 words (shared memory); Jb: the sample's colour-0 couplings [2D][W];
// CC: the pair's kPairStride words of scratch; u: the pair's Philox word (domain 5).
// Returns the cluster size; delta = change of E_A (E_B changes by -delta); the same on the four lanes of the pair.
template <class LAT>
__device__ __forceinline__ int houdayer_quad(const LAT &lat, uint32_t *A0, uint32_t *A1, uint32_t *B0, uint32_t *B1,
                                             const uint32_t *Jb, uint32_t *CC, uint32_t u, bool active, int lane, int &delta)
{
    constexpr int D = LAT::D;
    using NL = NatLat<D, LAT::kLog2L>;
    constexpr int W = NL::W;                    // 16 colour words per colour
    constexpr int RPL = 8, CPL = 4;             // rows / colour words (per colour) per lane
    const unsigned FULL = 0xFFFFFFFFu;
    const int k = lane & 3;                     // strip: lattice rows 8k .. 8k+7 = colour words 4k .. 4k+3
    const bool odd = k & 1;
    const int qbase = lane & ~3;

    // q = -1 map of my rows, natural order
    uint32_t neg[RPL], rng[RPL], cl[RPL];
    int local = 0;
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const int w = CPL * k + i;
        uint32_t n0 = 0, n1 = 0;
        if (active) {
            const uint32_t x0 = A0[w] ^ B0[w], x1 = A1[w] ^ B1[w];
            n0 = NL::interleave(2 * w, x0, x1);
            n1 = NL::interleave(2 * w + 1, x0 >> 16, x1 >> 16);
        }
        neg[2 * i] = n0; neg[2 * i + 1] = n1;
        local += __popc(n0) + __popc(n1);
    }
    // seed: the kth q = -1 site of the pair in index order, kth = (u * n_neg) >> 32   (R13)
    int incl = local;
#pragma unroll
    for (int o = 1; o < 4; o <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, o, 4);
        if (k >= o) incl += v;
    }
    const int n_neg = __shfl_sync(FULL, incl, 3, 4);
    int rem = (int)(((unsigned long long)u * (unsigned long long)n_neg) >> 32) - (incl - local);
    bool mine = n_neg > 0 && rem >= 0 && rem < local;
#pragma unroll
    for (int i = 0; i < RPL; ++i) {
        const uint32_t x = neg[i];
        const int c = __popc(x);
        const bool here = mine && rem < c;
        cl[i] = here ? (1u << select_bit(x, here ? rem : 0)) : 0u;
        mine = mine && !here;
        rem -= c;
    }
    // odd strips in reverse row order
#pragma unroll
    for (int i = 0; i < RPL / 2; ++i) {
        cswap(neg[i], neg[RPL - 1 - i], odd);
        cswap(cl[i], cl[RPL - 1 - i], odd);
    }
#pragma unroll
    for (int i = 0; i < RPL; ++i) rng[i] = __brev(neg[i]);

    // grow to the fixed point
    const int src0 = qbase | ((odd ? k + 1 : k - 1) & 3);      // holds the row beyond my index 0 (its index 0)
    const int srcL = qbase | ((odd ? k - 1 : k + 1) & 3);      // ... beyond my index RPL-1 (its index RPL-1)
    auto row_step = [](uint32_t ng, uint32_t rg, uint32_t cur, uint32_t up, uint32_t dn) {
        const uint32_t s = cur | __funnelshift_l(cur, cur, 1) | __funnelshift_r(cur, cur, 1) | up | dn;   // not yet masked
        const uint32_t f = ng & (~(ng + (s & ng)) | s);                                                   // upward fill
        const uint32_t rs = __brev(s) & rg;
        const uint32_t g = rg & (~(rg + rs) | rs);                                                        // downward fill, reversed
        return f | __brev(g);
    };
    for (;;) {
        uint32_t diff = 0;
        uint32_t b0 = __shfl_sync(FULL, cl[0], src0), bL = __shfl_sync(FULL, cl[RPL - 1], srcL);
#pragma unroll
        for (int i = 0; i < RPL; ++i) {
            const uint32_t nw = row_step(neg[i], rng[i], cl[i], i > 0 ? cl[i - 1] : b0, i < RPL - 1 ? cl[i + 1] : bL);
            diff |= nw ^ cl[i];
            cl[i] = nw;
        }
        b0 = __shfl_sync(FULL, cl[0], src0);
        bL = __shfl_sync(FULL, cl[RPL - 1], srcL);
#pragma unroll
        for (int i = RPL - 1; i >= 0; --i) {
            const uint32_t nw = row_step(neg[i], rng[i], cl[i], i > 0 ? cl[i - 1] : b0, i < RPL - 1 ? cl[i + 1] : bL);
            diff |= nw ^ cl[i];
            cl[i] = nw;
        }
        if (!__any_sync(FULL, diff != 0)) break;
    }
#pragma unroll
    for (int i = 0; i < RPL / 2; ++i) cswap(cl[i], cl[RPL - 1 - i], odd);

    // cluster in the colour layout -> the pair's scratch CC[2][W]
    int size = 0;
    uint32_t c0[CPL], c1[CPL];
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const uint32_t a = cl[2 * i], b = cl[2 * i + 1];
        size += __popc(a) + __popc(b);
        uint32_t a0, a1, bb0, bb1;
        NL::deinterleave(2 * (CPL * k + i), a, a0, a1);
        NL::deinterleave(2 * (CPL * k + i) + 1, b, bb0, bb1);
        c0[i] = a0 | (bb0 << 16);
        c1[i] = a1 | (bb1 << 16);
        CC[CPL * k + i] = c0[i];
        CC[W + CPL * k + i] = c1[i];
    }
    __syncwarp();
    // delta = 2 * sum over boundary bonds of J A_i A_j = 2 * (#boundary - 2 #(boundary & unsatisfied)), old spins, each bond
    // seen from its black endpoint
    int dl = 0;
    if (active) {
#pragma unroll
        for (int i = 0; i < CPL; ++i) {
            const int w = CPL * k + i;
            uint32_t nbC[2 * D], nbA[2 * D];
            lat.gather(CC + W, w, 0, nbC);
            lat.gather(A1, w, 0, nbA);
            const uint32_t ab = A0[w];
#pragma unroll
            for (int q = 0; q < 2 * D; ++q) {
                const uint32_t bnd = nbC[q] ^ c0[i];
                const uint32_t uns = ab ^ nbA[q] ^ Jb[q * W + w];
                dl += __popc(bnd) - 2 * __popc(bnd & uns);
            }
        }
    }
    __syncwarp();                        // every read of the old A is done before anyone writes
    if (active) {
#pragma unroll
        for (int i = 0; i < CPL; ++i) {
            const int w = CPL * k + i;
            A0[w] ^= c0[i]; B0[w] ^= c0[i];
            A1[w] ^= c1[i]; B1[w] ^= c1[i];
        }
    }
#pragma unroll
    for (int o = 2; o > 0; o >>= 1) {
        size += __shfl_xor_sync(FULL, size, o, 4);
        dl += __shfl_xor_sync(FULL, dl, o, 4);
    }
    __syncwarp();
    delta = 2 * dl;
    return size;
}

// NEXT-4, R37: the MULTI-cluster exchange on the same four-lane register strips (2D L = 32, fused kernel).  Every connected
// component of q = -1 sites is exchanged iff the top bit of the Philox word of its SMALLEST site index is set.  On bit maps:
//   (1) the roots, by a tournament over the 10 index bits from the top: among the survivors S (at first every q = -1 site),
//       Z = those whose index bit b is 0; G = all components that contain a site of Z (one multi-seed growth); in those
//       components the survivors with bit b = 1 are out.  After the last bit S holds exactly the minimum of every component;
//   (2) one Philox block per root gives its coin (the roots of a lane's 8 rows are walked bit by bit);
//   (3) one more growth from the roots whose coin is set gives the exchanged set.
// Eleven growths where the single-cluster move makes one; all of it in registers, on all four warps.  Same set as the
// oracle's component labelling (bit-exact parity, tests/test_gpu_next4.py).  Contract as houdayer_quad; `step`, `g`, `t`
// name the move's Philox stream (domain 5, aux = 1).  Returns the number of exchanged sites.
template <class LAT>
__device__ __forceinline__ int houdayer_multi_quad(const LAT &lat, uint32_t *A0, uint32_t *A1, uint32_t *B0, uint32_t *B1,
                                                   const uint32_t *Jb, uint32_t *CC, uint32_t step, uint32_t g, int t,
                                                   const RoundKeys &rk, bool active, int lane, int &delta)
{
    constexpr int D = LAT::D;
    using NL = NatLat<D, LAT::kLog2L>;
    constexpr int W = NL::W;
    constexpr int RPL = 8, CPL = 4;
    const unsigned FULL = 0xFFFFFFFFu;
    const int k = lane & 3;
    const bool odd = k & 1;
    const int qbase = lane & ~3;

    uint32_t neg[RPL], rng[RPL], cl[RPL], S[RPL];
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const int w = CPL * k + i;
        uint32_t n0 = 0, n1 = 0;
        if (active) {
            const uint32_t x0 = A0[w] ^ B0[w], x1 = A1[w] ^ B1[w];
            n0 = NL::interleave(2 * w, x0, x1);
            n1 = NL::interleave(2 * w + 1, x0 >> 16, x1 >> 16);
        }
        neg[2 * i] = n0; neg[2 * i + 1] = n1;
    }
#pragma unroll
    for (int i = 0; i < RPL / 2; ++i) cswap(neg[i], neg[RPL - 1 - i], odd);        // odd strips in reverse row order
#pragma unroll
    for (int i = 0; i < RPL; ++i) { rng[i] = __brev(neg[i]); S[i] = neg[i]; }
    const int src0 = qbase | ((odd ? k + 1 : k - 1) & 3);
    const int srcL = qbase | ((odd ? k - 1 : k + 1) & 3);
    auto row_step = [](uint32_t ng, uint32_t rg, uint32_t cur, uint32_t up, uint32_t dn) {
        const uint32_t s = cur | __funnelshift_l(cur, cur, 1) | __funnelshift_r(cur, cur, 1) | up | dn;
        const uint32_t f = ng & (~(ng + (s & ng)) | s);
        const uint32_t rs = __brev(s) & rg;
        const uint32_t gg = rg & (~(rg + rs) | rs);
        return f | __brev(gg);
    };
    auto grow = [&]() {                 // cl <- all components of neg that contain a bit of cl
        for (;;) {
            uint32_t diff = 0;
            uint32_t b0 = __shfl_sync(FULL, cl[0], src0), bL = __shfl_sync(FULL, cl[RPL - 1], srcL);
#pragma unroll
            for (int i = 0; i < RPL; ++i) {
                const uint32_t nw = row_step(neg[i], rng[i], cl[i], i > 0 ? cl[i - 1] : b0, i < RPL - 1 ? cl[i + 1] : bL);
                diff |= nw ^ cl[i];
                cl[i] = nw;
            }
            b0 = __shfl_sync(FULL, cl[0], src0);
            bL = __shfl_sync(FULL, cl[RPL - 1], srcL);
#pragma unroll
            for (int i = RPL - 1; i >= 0; --i) {
                const uint32_t nw = row_step(neg[i], rng[i], cl[i], i > 0 ? cl[i - 1] : b0, i < RPL - 1 ? cl[i + 1] : bL);
                diff |= nw ^ cl[i];
                cl[i] = nw;
            }
            if (!__any_sync(FULL, diff != 0)) break;
        }
    };
    // (1) tournament over the index bits: site index = 32 y + x, y = the lattice row of storage index i
#pragma unroll 1
    for (int b = 9; b >= 0; --b) {
        const uint32_t xone = (b == 0) ? 0xAAAAAAAAu : (b == 1) ? 0xCCCCCCCCu : (b == 2) ? 0xF0F0F0F0u : (b == 3) ? 0xFF00FF00u : 0xFFFF0000u;
        uint32_t one[RPL];              // sites of my rows whose index bit b is 1
#pragma unroll
        for (int i = 0; i < RPL; ++i) {
            const int y = 8 * k + (odd ? RPL - 1 - i : i);
            one[i] = (b >= 5) ? (((y >> (b - 5)) & 1) ? 0xFFFFFFFFu : 0u) : xone;
            cl[i] = S[i] & ~one[i];
        }
        grow();
#pragma unroll
        for (int i = 0; i < RPL; ++i) S[i] &= ~(cl[i] & one[i]);
    }
    // (2) coins of the roots, (3) the exchanged set
#pragma unroll
    for (int i = 0; i < RPL; ++i) {
        const int y = 8 * k + (odd ? RPL - 1 - i : i);
        uint32_t x = S[i], keep = 0;
        while (x) {
            const int bit = __ffs(x) - 1;
            x &= x - 1;
            const uint32_t site = 32u * (uint32_t)y + (uint32_t)bit;
            uint32_t w4[4];
            philox4x32_10(site >> 2, step, g, make_tag(DOM_HOUD, 1, 0, t), rk, w4[0], w4[1], w4[2], w4[3]);
            const uint32_t wsel = (site & 2) ? ((site & 1) ? w4[3] : w4[2]) : ((site & 1) ? w4[1] : w4[0]);
            if (wsel >> 31) keep |= 1u << bit;
        }
        cl[i] = keep;
    }
    grow();
#pragma unroll
    for (int i = 0; i < RPL / 2; ++i) cswap(cl[i], cl[RPL - 1 - i], odd);

    // the exchanged set in the colour layout -> the pair's scratch, boundary-bond sum, negation (as houdayer_quad)
    int size = 0;
    uint32_t c0[CPL], c1[CPL];
#pragma unroll
    for (int i = 0; i < CPL; ++i) {
        const uint32_t a = cl[2 * i], b = cl[2 * i + 1];
        size += __popc(a) + __popc(b);
        uint32_t a0, a1, bb0, bb1;
        NL::deinterleave(2 * (CPL * k + i), a, a0, a1);
        NL::deinterleave(2 * (CPL * k + i) + 1, b, bb0, bb1);
        c0[i] = a0 | (bb0 << 16);
        c1[i] = a1 | (bb1 << 16);
        CC[CPL * k + i] = c0[i];
        CC[W + CPL * k + i] = c1[i];
    }
    __syncwarp();
    int dl = 0;
    if (active) {
#pragma unroll
        for (int i = 0; i < CPL; ++i) {
            const int w = CPL * k + i;
            uint32_t nbC[2 * D], nbA[2 * D];
            lat.gather(CC + W, w, 0, nbC);
            lat.gather(A1, w, 0, nbA);
            const uint32_t ab = A0[w];
#pragma unroll
            for (int q = 0; q < 2 * D; ++q) {
                const uint32_t bnd = nbC[q] ^ c0[i];
                const uint32_t uns = ab ^ nbA[q] ^ Jb[q * W + w];
                dl += __popc(bnd) - 2 * __popc(bnd & uns);
            }
        }
    }
    __syncwarp();
    if (active) {
#pragma unroll
        for (int i = 0; i < CPL; ++i) {
            const int w = CPL * k + i;
            A0[w] ^= c0[i]; B0[w] ^= c0[i];
            A1[w] ^= c1[i]; B1[w] ^= c1[i];
        }
    }
#pragma unroll
    for (int o = 2; o > 0; o >>= 1) {
        size += __shfl_xor_sync(FULL, size, o, 4);
        dl += __shfl_xor_sync(FULL, dl, o, 4);
    }
    __syncwarp();
    delta = 2 * dl;
    return size;
}

}  // namespace ptg
