// a5  Houdayer cluster exchange, warp-per-pair path with REGISTER-RESIDENT ROW STRIPS (Eq. (10) P:136-138, P:143;
// DESIGN.md 7.3c).  2D lattices with L >= 32 whose natural bit map fits 16 words per lane (L = 32, 64, 128).
//
// Every lane keeps a strip of RPL consecutive lattice rows (WR words each) of the q = -1 map and of the growing
// cluster in registers.  One round = fetch the neighbour lanes' boundary rows with shuffles, then sweep the strip down
// and up (Gauss-Seidel inside the strip, Jacobi across strips).  A row step closes the WHOLE row along x at once:
// the carry trick of houdayer.cuh on the row as one WR-word integer (add-with-carry chain), upwards and, bit-reversed,
// downwards.  Nothing but the two shuffles per word and round leaves the register file, so a round costs a few hundred
// cycles and the hard pairs (hundreds of row-Jacobi rounds) no longer set the kernel time.
// Same least fixed point as every other path = the connected component of the seed (bit-exact parity).
#pragma once
#include "houdayer.cuh"

namespace ptg {

template <class LAT>
struct RowStrip {
    using NL = NatLat<LAT::D, LAT::kLog2L>;
    static constexpr int W = NL::W, WR = NL::WR;
    static constexpr int CPT = (W + 31) / 32;          // colour words per lane
    static constexpr int CHN = 2 * CPT;                // natural words per lane
    static constexpr int RPL = CHN / WR;               // rows per lane
    static constexpr int LANES = W / CPT;              // lanes that hold rows (a power of two <= 32)
    static constexpr bool kEligible = (LAT::D == 2) && !NL::kSmall && CHN <= 16 && RPL >= 2 && RPL * WR == CHN;
};

// close one row: cur <- all runs of neg (along x, whole row) that touch cur, its x-neighbours (periodic) or up / dn
template <int WR>
__device__ __forceinline__ bool row_close(const uint32_t (&neg)[WR], const uint32_t (&rneg)[WR], uint32_t (&cur)[WR],
                                          const uint32_t (&up)[WR], const uint32_t (&dn)[WR])
{
    uint32_t seeds[WR], f[WR];
#pragma unroll
    for (int j = 0; j < WR; ++j) {
        const uint32_t lft = cur[(j + WR - 1) % WR], rgt = cur[(j + 1) % WR];
        seeds[j] = (cur[j] | __funnelshift_l(lft, cur[j], 1) | __funnelshift_r(cur[j], rgt, 1) | up[j] | dn[j]) & neg[j];
    }
    // upward fill: (neg + seeds) as one WR-word integer
    unsigned long long carry = 0;
#pragma unroll
    for (int j = 0; j < WR; ++j) {
        const unsigned long long t = (unsigned long long)neg[j] + seeds[j] + carry;
        carry = t >> 32;
        f[j] = ((((uint32_t)t) ^ neg[j]) & neg[j]) | seeds[j];
    }
    // downward fill: the same on the bit-reversed row (word order reversed too); rneg[j] = brev(neg[WR-1-j])
    carry = 0;
#pragma unroll
    for (int j = 0; j < WR; ++j) {
        const uint32_t rs = __brev(seeds[WR - 1 - j]);
        const unsigned long long t = (unsigned long long)rneg[j] + rs + carry;
        carry = t >> 32;
        f[WR - 1 - j] |= __brev(((((uint32_t)t) ^ rneg[j]) & rneg[j]) | rs);
    }
    uint32_t diff = 0;
#pragma unroll
    for (int j = 0; j < WR; ++j) { diff |= f[j] ^ cur[j]; cur[j] = f[j]; }
    return diff != 0;
}

__device__ __forceinline__ void cswap(uint32_t &a, uint32_t &b, bool c)
{
    const uint32_t t = c ? a : b;
    a = c ? b : a;
    b = t;
}

// Same contract as houdayer_pair (houdayer.cuh); scratch: 2W words of the warp's shared memory.
template <class LAT>
__device__ __forceinline__ int houdayer_pair_rows(const LAT &lat, uint32_t *A0, uint32_t *A1, uint32_t *B0, uint32_t *B1,
                                                  const uint32_t *Jb, uint32_t *scratch, uint32_t u, int lane, int &delta)
{
    using RSx = RowStrip<LAT>;
    using NL = typename RSx::NL;
    constexpr int W = RSx::W, WR = RSx::WR, CPT = RSx::CPT, CHN = RSx::CHN, RPL = RSx::RPL, LANES = RSx::LANES;
    const unsigned FULL = 0xFFFFFFFFu;
    const int w_lo = min(W, lane * CPT), w_hi = min(W, w_lo + CPT);

    // q = -1 map of this lane's rows, natural order: word i of the strip = natural word 2 w_lo + i = row i / WR, word i % WR
    uint32_t neg[RPL][WR], rneg[RPL][WR], cl[RPL][WR];
    int local = 0;
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const int w = w_lo + i;
        uint32_t n0 = 0, n1 = 0;
        if (w < w_hi) {
            const uint32_t x0 = A0[w] ^ B0[w], x1 = A1[w] ^ B1[w];
            n0 = NL::interleave(2 * w, x0, x1);
            n1 = NL::interleave(2 * w + 1, x0 >> 16, x1 >> 16);
        }
        neg[(2 * i) / WR][(2 * i) % WR] = n0;
        neg[(2 * i + 1) / WR][(2 * i + 1) % WR] = n1;
        local += __popc(n0) + __popc(n1);
    }
#pragma unroll
    for (int r = 0; r < RPL; ++r)
#pragma unroll
        for (int j = 0; j < WR; ++j) { rneg[r][j] = __brev(neg[r][WR - 1 - j]); cl[r][j] = 0; }

    int incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += v;
    }
    const int n_neg = __shfl_sync(FULL, incl, 31);
    delta = 0;
    if (n_neg == 0) return 0;
    // seed: the k-th q = -1 site in index order (R13)
    const int kth = (int)(((unsigned long long)u * (unsigned long long)n_neg) >> 32);
    int rem = kth - (incl - local);
    bool mine = rem >= 0 && rem < local;
#pragma unroll
    for (int i = 0; i < CHN; ++i) {
        const uint32_t x = neg[i / WR][i % WR];
        const int c = __popc(x);
        if (mine && rem < c) { cl[i / WR][i % WR] = 1u << select_bit(x, rem); mine = false; }
        rem -= c;
    }

    // grow to the fixed point.  ODD lanes keep their strip in REVERSE row order, so the same index sweep 0 -> RPL-1 runs
    // down the lattice on even lanes and up on odd lanes: with the boundary rows exchanged before each of the two sweeps of
    // a round, membership crosses TWO strips per round in either direction (even: down then up, odd: up then down) instead
    // of one.  The row beyond index 0 is the neighbour lane's index-0 row, the row beyond index RPL-1 its index-(RPL-1) row
    // (row_close is symmetric in its two vertical neighbours).  Any order of monotone row closures reaches the same least
    // fixed point; a round that changes nothing has evaluated every row against final values.
    const bool odd = lane & 1;
#pragma unroll
    for (int r = 0; r < RPL / 2; ++r)
#pragma unroll
        for (int j = 0; j < WR; ++j) {
            cswap(neg[r][j], neg[RPL - 1 - r][j], odd);
            cswap(rneg[r][j], rneg[RPL - 1 - r][j], odd);
            cswap(cl[r][j], cl[RPL - 1 - r][j], odd);
        }
    const int lane_up = (lane - 1) & (LANES - 1), lane_dn = (lane + 1) & (LANES - 1);
    const int src0 = odd ? lane_dn : lane_up;          // holds the row beyond my index 0
    const int srcL = odd ? lane_up : lane_dn;          // holds the row beyond my index RPL-1
    for (;;) {
        uint32_t b0[WR], bL[WR];
#pragma unroll
        for (int j = 0; j < WR; ++j) {
            b0[j] = __shfl_sync(FULL, cl[0][j], src0);
            bL[j] = __shfl_sync(FULL, cl[RPL - 1][j], srcL);
        }
        bool changed = false;
#pragma unroll
        for (int r = 0; r < RPL; ++r)
            changed |= row_close<WR>(neg[r], rneg[r], cl[r], r > 0 ? cl[r - 1] : b0, r < RPL - 1 ? cl[r + 1] : bL);
#pragma unroll
        for (int j = 0; j < WR; ++j) {
            b0[j] = __shfl_sync(FULL, cl[0][j], src0);
            bL[j] = __shfl_sync(FULL, cl[RPL - 1][j], srcL);
        }
#pragma unroll
        for (int r = RPL - 1; r >= 0; --r)
            changed |= row_close<WR>(neg[r], rneg[r], cl[r], r > 0 ? cl[r - 1] : b0, r < RPL - 1 ? cl[r + 1] : bL);
        if (!__any_sync(FULL, changed)) break;
    }
#pragma unroll
    for (int r = 0; r < RPL / 2; ++r)
#pragma unroll
        for (int j = 0; j < WR; ++j) cswap(cl[r][j], cl[RPL - 1 - r][j], odd);

    // cluster in the colour layout
    int size = 0;
    uint32_t c0[CPT], c1[CPT];
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const uint32_t a = cl[(2 * i) / WR][(2 * i) % WR], b = cl[(2 * i + 1) / WR][(2 * i + 1) % WR];
        size += __popc(a) + __popc(b);
        uint32_t a0, a1, b0, b1;
        NL::deinterleave(2 * (w_lo + i), a, a0, a1);
        NL::deinterleave(2 * (w_lo + i) + 1, b, b0, b1);
        c0[i] = a0 | (b0 << 16);
        c1[i] = a1 | (b1 << 16);
    }
    return houdayer_apply<LAT, CPT>(lat, A0, A1, B0, B1, Jb, scratch, c0, c1, w_lo, w_hi, size, lane, delta);
}

// warp-per-pair entry point: register-resident row strips where the lattice allows, else the shared-memory strips
template <class LAT>
__device__ __forceinline__ int houdayer_warp(const LAT &lat, uint32_t *A0, uint32_t *A1, uint32_t *B0, uint32_t *B1,
                                             const uint32_t *Jb, uint32_t *scratch, uint32_t u, int lane, int &delta)
{
    if constexpr (RowStrip<LAT>::kEligible) return houdayer_pair_rows(lat, A0, A1, B0, B1, Jb, scratch, u, lane, delta);
    else return houdayer_pair(lat, A0, A1, B0, B1, Jb, scratch, u, lane, delta);
}

}  // namespace ptg
