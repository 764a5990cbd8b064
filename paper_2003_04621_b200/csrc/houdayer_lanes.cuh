// a5  Houdayer cluster exchange, LANE-PER-PAIR path (Eq. (10)).
//
// One LANE owns one (sample, temperature) pair; a warp therefore runs 32 temperatures of a sample side by side
// with no communication between lanes.  The q_i = -1 map and the growing cluster are natural-order bit maps
// (bit i = site i) in shared memory, word n of lane l at scratch[n * kLaneStride + l] (conflict-free).  Growth to
// the least fixed point (= the connected component of the seed, which the paper's breadth-first search also
// finds) is SEQUENTIAL per lane: Gauss-Seidel passes over the words, alternately downwards and upwards, each word
// pulling in its +-y (+-z) neighbours' cluster bits and filling whole runs along x in O(1) with the carry trick of
// houdayer.cuh.  A downward pass carries membership through any number of rows at once, so a pair converges in a
// few passes (C2 states: mean 5, worst 13) where the row-parallel iteration of houdayer.cuh needs ~20-40 rounds.
// Used inside the fused MCS kernel when the lattice has at most 32 natural words (2D L <= 32, 3D L = 8).
#pragma once
#include "houdayer.cuh"

namespace ptg {

constexpr int kLaneStride = 33;        // odd: lanes hit distinct banks for any word index

template <class LAT>
struct LaneHoudayer {
    static constexpr int D = LAT::D;
    using NL = NatLat<D, LAT::kLog2L>;
    static constexpr int W = NL::W, NW = NL::NW;
    static constexpr bool kEligible = (NW <= 32);
    static constexpr int kScratchWords = 2 * NW * kLaneStride;     // per warp: Neg[NW] | Cl[NW], 32 lanes each
};

// One pair per lane; ALL 32 lanes of the warp must call (inactive lanes pass active = false and any pointers).
// A0/A1, B0/B1: this lane's colour-0 / colour-1 words of the two configurations; Jb: the sample's colour-0 couplings
// [2D][W]; col: this lane's column of the warp's scratch (scratch + lane); u: the pair's Philox word (domain 5).
// Returns the cluster size; delta = change of E_A (E_B changes by -delta).
template <class LAT>
__device__ __forceinline__ int houdayer_lane(const LAT &lat, uint32_t *A0, uint32_t *A1, uint32_t *B0, uint32_t *B1,
                                             const uint32_t *Jb, uint32_t *col, uint32_t u, bool active, int &delta)
{
    constexpr int D = LAT::D;
    using NL = NatLat<D, LAT::kLog2L>;
    constexpr int W = NL::W, NW = NL::NW, SP = kLaneStride;
    const unsigned FULL = 0xFFFFFFFFu;
    uint32_t *Neg = col, *Cl = col + NW * SP;

    // q = -1 map in natural order
    int n_neg = 0;
    if (active) {
#pragma unroll 2
        for (int w = 0; w < W; ++w) {
            const uint32_t x0 = A0[w] ^ B0[w], x1 = A1[w] ^ B1[w];
            const uint32_t n0 = NL::interleave(2 * w, x0, x1), n1 = NL::interleave(2 * w + 1, x0 >> 16, x1 >> 16);
            Neg[(2 * w) * SP] = n0; Neg[(2 * w + 1) * SP] = n1;
            Cl[(2 * w) * SP] = 0;   Cl[(2 * w + 1) * SP] = 0;
            n_neg += __popc(n0) + __popc(n1);
        }
    } else {
        for (int n = 0; n < NW; ++n) { Neg[n * SP] = 0; Cl[n * SP] = 0; }
    }
    // seed: the k-th q = -1 site in index order, k = (u * n_neg) >> 32   (R13)
    if (n_neg > 0) {
        int rem = (int)(((unsigned long long)u * (unsigned long long)n_neg) >> 32);
        for (int n = 0; n < NW; ++n) {
            const uint32_t x = Neg[n * SP];
            const int c = __popc(x);
            if (rem < c) { Cl[n * SP] = 1u << select_bit(x, rem); break; }
            rem -= c;
        }
    }

    // grow to the fixed point: alternate downward / upward Gauss-Seidel passes until no lane changes anything
    if constexpr (D == 2 && !NL::kSmall && NL::WR == 1) {
        // 2D, one row per word (L = 32): branch-free row steps with the previous row's new value carried in a
        // register, so the only serial dependency of a pass is ~10 ALU operations per row; the loads of the rows
        // ahead do not depend on it and are issued early.  fill_runs(neg, seeds) with seeds containing cur is
        // monotone (result contains cur), so computing it unconditionally is the same iteration.
        for (int pass = 0;; ++pass) {
            uint32_t diff = 0;
            if (!(pass & 1)) {
                uint32_t prev = Cl[(NW - 1) * SP];
#pragma unroll 8
                for (int n = 0; n < NW; ++n) {
                    const uint32_t neg = Neg[n * SP], cur = Cl[n * SP], nxt = Cl[((n + 1) & (NW - 1)) * SP];
                    const uint32_t seeds = (cur | __funnelshift_l(cur, cur, 1) | __funnelshift_r(cur, cur, 1) | prev | nxt) & neg;
                    const uint32_t nw = NL::fill_runs(neg, seeds);
                    diff |= nw ^ cur;
                    Cl[n * SP] = nw;
                    prev = nw;
                }
            } else {
                uint32_t prev = Cl[0];
#pragma unroll 8
                for (int n = NW - 1; n >= 0; --n) {
                    const uint32_t neg = Neg[n * SP], cur = Cl[n * SP], nxt = Cl[((n - 1) & (NW - 1)) * SP];
                    const uint32_t seeds = (cur | __funnelshift_l(cur, cur, 1) | __funnelshift_r(cur, cur, 1) | prev | nxt) & neg;
                    const uint32_t nw = NL::fill_runs(neg, seeds);
                    diff |= nw ^ cur;
                    Cl[n * SP] = nw;
                    prev = nw;
                }
            }
            if (!__any_sync(FULL, diff != 0)) break;
        }
    } else
    for (int pass = 0;; ++pass) {
        bool changed = false;
        for (int k = 0; k < NW; ++k) {
            const int n = (pass & 1) ? NW - 1 - k : k;
            const uint32_t neg = Neg[n * SP], cur = Cl[n * SP];
            if (neg & ~cur) {
                const uint32_t seeds = (cur | NL::neighbour_union_f([Cl](int i) { return Cl[i * SP]; }, n, cur)) & neg;
                if (seeds & ~cur) {
                    const uint32_t nw = NL::fill_runs(neg, seeds);
                    Cl[n * SP] = nw;
                    changed = true;
                }
            }
        }
        if (!__any_sync(FULL, changed)) break;
    }
    delta = 0;
    if (n_neg == 0) return 0;

    // cluster in the colour layout, over the (no longer needed) q map: CC0[w] = Neg[w], CC1[w] = Neg[W + w]
    uint32_t *CC0 = Neg, *CC1 = Neg + W * SP;
    int size = 0;
    for (int w = 0; w < W; ++w) {
        const uint32_t a = Cl[(2 * w) * SP], b = Cl[(2 * w + 1) * SP];
        size += __popc(a) + __popc(b);
        uint32_t a0, a1, b0, b1;
        NL::deinterleave(2 * w, a, a0, a1);
        NL::deinterleave(2 * w + 1, b, b0, b1);
        CC0[w * SP] = a0 | (b0 << 16);
        CC1[w * SP] = a1 | (b1 << 16);
    }
    // delta = 2 * sum over boundary bonds of J A_i A_j = 2 * (#boundary - 2 #(boundary & unsatisfied)), old spins,
    // each bond seen from its black endpoint
    int dl = 0;
    for (int w = 0; w < W; ++w) {
        uint32_t nbC[2 * D];
        lat.gather_f([CC1](int i) { return CC1[i * SP]; }, w, 0, nbC);
        const uint32_t cb = CC0[w * SP];
        // no test for "no boundary bond in this word": with 32 pairs side by side some lane always has one
        uint32_t nbA[2 * D];
        lat.gather(A1, w, 0, nbA);
        const uint32_t ab = A0[w];
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) {
            const uint32_t bnd = nbC[k] ^ cb;
            const uint32_t uns = ab ^ nbA[k] ^ Jb[k * W + w];
            dl += __popc(bnd) - 2 * __popc(bnd & uns);
        }
    }
    // every read of the old A is done (same lane, program order): negate the cluster in both configurations
    for (int w = 0; w < W; ++w) {
        const uint32_t x0 = CC0[w * SP], x1 = CC1[w * SP];
        A0[w] ^= x0; B0[w] ^= x0;
        A1[w] ^= x1; B1[w] ^= x1;
    }
    delta = 2 * dl;
    return size;
}

}  // namespace ptg
