// a5  Houdayer cluster exchange, fast path (Eq. (10)).
//
// ONE WARP per (sample, temperature) pair.  The q_i = -1 map and the growing cluster live in per-warp shared
// memory as NATURAL-order bit maps (bit i = site i, so a lattice row is L consecutive bits):
//   * seed site = k-th set bit of the q = -1 map in index order: word popcounts + warp scan + select;
//   * growth to the least fixed point = connected component of the seed (the paper's breadth-first search finds
//     the same set): per word, OR in the cluster bits of the +-y (+-z) neighbour words and of the +-x wrap /
//     cross-word neighbours, then fill whole runs of q = -1 sites along x in O(1) with the carry trick
//     ((neg + seeds) ^ neg) & neg (upwards) and its bit-reversed twin (downwards).  Words are updated in place
//     (chaotic relaxation of a monotone map reaches the same least fixed point in any order) until a full pass
//     changes nothing;
//   * delta = 2 * sum over boundary bonds of J A_i A_j (old spins) and the size come from popcounts on the colour
//     layout; the cluster is de-interleaved and XORed into both configurations.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "lattice.cuh"

namespace ptg {

// bits 0..15 -> even bit positions
__device__ __forceinline__ uint32_t spread16(uint32_t x)
{
    x &= 0xFFFFu;
    x = (x | (x << 8)) & 0x00FF00FFu;
    x = (x | (x << 4)) & 0x0F0F0F0Fu;
    x = (x | (x << 2)) & 0x33333333u;
    x = (x | (x << 1)) & 0x55555555u;
    return x;
}

// even bit positions -> bits 0..15
__device__ __forceinline__ uint32_t squeeze16(uint32_t x)
{
    x &= 0x55555555u;
    x = (x | (x >> 1)) & 0x33333333u;
    x = (x | (x >> 2)) & 0x0F0F0F0Fu;
    x = (x | (x >> 4)) & 0x00FF00FFu;
    x = (x | (x >> 8)) & 0x0000FFFFu;
    return x;
}

// position of the r-th (0-based) set bit of x; r < popc(x)
__device__ __forceinline__ int select_bit(uint32_t x, int r)
{
    int pos = 0;
#pragma unroll
    for (int sh = 16; sh > 0; sh >>= 1) {
        const int c = __popc(x & ((1u << sh) - 1u));
        if (r >= c) { r -= c; x >>= sh; pos += sh; }
    }
    return pos;
}

// Natural-order view of FastLat<D, LOG2L>: NW = N/32 words; natural words 2w and 2w+1 hold the sites of the colour
// words w (both colours): site 2h has colour (y+z)&1, site 2h+1 the other.
template <int D_, int LOG2L>
struct NatLat {
    static constexpr int D = D_;
    static constexpr int L = 1 << LOG2L;
    static constexpr int N = (D_ == 2) ? L * L : L * L * L;
    static constexpr int NW = N / 32;
    static constexpr int W = NW / 2;
    static constexpr bool kSmall = (L < 32);                     // several rows per word
    static constexpr int WR = kSmall ? 1 : L / 32;               // words per row        (L >= 32)
    static constexpr int PWN = (L * L) / 32;                     // words per xy-plane   (>= 2 for L >= 8)

    __host__ __device__ static constexpr uint32_t rep_mask(uint32_t pat, int period)
    {
        uint32_t m = 0;
        for (int s = 0; s < 32; s += period) m |= pat << s;
        return m;
    }
    static constexpr uint32_t SEG_LSB = kSmall ? rep_mask(1u, kSmall ? L : 32) : 1u;
    static constexpr uint32_t SEG_MSB = kSmall ? (SEG_LSB << (L - 1)) : 0x80000000u;
    // half-word (16 same-colour sites = 32 consecutive sites) bits that lie in rows of odd y
    static constexpr uint32_t ODD16 = kSmall ? (rep_mask(((1u << (L / 2)) - 1u) << (L / 2), L) & 0xFFFFu) : 0u;

    // 16-bit mask of the half-word positions whose EVEN-x site has colour 1, for natural word n
    __device__ __forceinline__ static uint32_t colour1_even_mask(int n)
    {
        if constexpr (kSmall) {
            const int z = (D_ == 3) ? n / PWN : 0;
            return (z & 1) ? (~ODD16 & 0xFFFFu) : ODD16;
        } else {
            const int row = n / WR;
            const int y = row & (L - 1), z = row >> LOG2L;
            return ((y + z) & 1) ? 0xFFFFu : 0u;
        }
    }

    // natural word n from the two colour half-words (16 bits each)
    __device__ __forceinline__ static uint32_t interleave(int n, uint32_t h0, uint32_t h1)
    {
        const uint32_t m1 = colour1_even_mask(n);
        const uint32_t ev = (h0 & ~m1) | (h1 & m1), od = (h1 & ~m1) | (h0 & m1);
        return spread16(ev) | (spread16(od) << 1);
    }
    // colour half-words (16 bits each) from natural word n
    __device__ __forceinline__ static void deinterleave(int n, uint32_t nat, uint32_t &h0, uint32_t &h1)
    {
        const uint32_t m1 = colour1_even_mask(n);
        const uint32_t ev = squeeze16(nat), od = squeeze16(nat >> 1);
        h0 = (ev & ~m1) | (od & m1);
        h1 = (od & ~m1) | (ev & m1);
    }

    // OR of the cluster bits of the 2D neighbours of the 32 sites of word n (cur = Cl[n]); ld(i) returns Cl[i]
    template <class F>
    __device__ __forceinline__ static uint32_t neighbour_union_f(F ld, int n, uint32_t cur)
    {
        uint32_t u;
        if constexpr (kSmall) {
            const int base = (D_ == 3) ? (n / PWN) * PWN : 0, j = n - base;
            u = ((cur << 1) & ~SEG_LSB) | ((cur >> (L - 1)) & SEG_LSB) | ((cur >> 1) & ~SEG_MSB) | ((cur << (L - 1)) & SEG_MSB);
            const uint32_t nxt = ld(base + ((j + 1) & (PWN - 1))), prv = ld(base + ((j - 1) & (PWN - 1)));
            u |= __funnelshift_r(cur, nxt, L) | __funnelshift_l(prv, cur, L);
        } else {
            const int row = n / WR, j = n - row * WR;
            if constexpr (WR == 1) {
                u = __funnelshift_l(cur, cur, 1) | __funnelshift_r(cur, cur, 1);
            } else {
                const uint32_t pw = ld(row * WR + ((j - 1) & (WR - 1))), nw = ld(row * WR + ((j + 1) & (WR - 1)));
                u = __funnelshift_l(pw, cur, 1) | __funnelshift_r(cur, nw, 1);
            }
            const int base = (D_ == 3) ? (n / PWN) * PWN : 0, jj = n - base;
            u |= ld(base + ((jj + WR) & (PWN - 1))) | ld(base + ((jj - WR) & (PWN - 1)));
        }
        if constexpr (D_ == 3) u |= ld((n + PWN) & (NW - 1)) | ld((n - PWN) & (NW - 1));
        return u;
    }
    __device__ __forceinline__ static uint32_t neighbour_union(const uint32_t *Cl, int n, uint32_t cur)
    {
        return neighbour_union_f([Cl](int i) { return Cl[i]; }, n, cur);
    }

    // upward fill of the runs of `neg` (within row segments) that contain a bit of `seeds` (seeds subset of neg)
    __device__ __forceinline__ static uint32_t fill_up(uint32_t neg, uint32_t seeds)
    {
        if constexpr (kSmall) {
            const uint32_t nm = neg & ~SEG_MSB;                  // the carry stops at the segment's top bit
            uint32_t f = (((nm + (seeds & nm)) ^ nm) & nm) | seeds;
            f |= (f << 1) & neg & SEG_MSB;
            return f;
        } else {
            return (((neg + seeds) ^ neg) & neg) | seeds;
        }
    }
    __device__ __forceinline__ static uint32_t fill_runs(uint32_t neg, uint32_t seeds)
    {
        return fill_up(neg, seeds) | __brev(fill_up(__brev(neg), __brev(seeds)));
    }
};

// One pair, one warp.  A0/A1 and B0/B1: the colour-0 / colour-1 words of the two configurations (global or shared
// memory); Jb: the sample's colour-0 couplings [2D][W]; scratch: kPairScratchWords<LAT> words of this warp's shared memory; u: the
// pair's Philox word (domain 5).  Returns the cluster size; delta = change of E_A (E_B changes by -delta).
// All lanes return the same values.
// Common tail of the warp-per-pair paths: the lane holds the cluster bits of its colour words [w_lo, w_hi) in c0 / c1
// (colour 0 / 1) and its share of the size.  Publishes the cluster in the colour layout to CC (2W words of the warp's
// shared memory), computes delta = 2 * sum over boundary bonds of J A_i A_j (old spins; each bond seen from its black
// endpoint) = 2 * (#boundary - 2 #(boundary & unsatisfied)), then negates the cluster in both configurations.
template <class LAT, int CPT>
__device__ __forceinline__ int houdayer_apply(const LAT &lat, uint32_t *A0, uint32_t *A1, uint32_t *B0, uint32_t *B1,
                                              const uint32_t *Jb, uint32_t *CC, const uint32_t (&c0)[CPT],
                                              const uint32_t (&c1)[CPT], int w_lo, int w_hi, int size, int lane, int &delta)
{
    constexpr int D = LAT::D, W = LAT::W;
    const unsigned FULL = 0xFFFFFFFFu;
    __syncwarp();
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const int w = w_lo + i;
        if (w < w_hi) { CC[w] = c0[i]; CC[W + w] = c1[i]; }
    }
    __syncwarp();
    int dl = 0;
    for (int w = lane; w < W; w += 32) {
        uint32_t nbC[2 * D];
        lat.gather(CC + W, w, 0, nbC);
        const uint32_t cb = CC[w];
        uint32_t any = 0;
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) { nbC[k] ^= cb; any |= nbC[k]; }
        if (any) {
            uint32_t nbA[2 * D];
            lat.gather(A1, w, 0, nbA);
            const uint32_t ab = A0[w];
#pragma unroll
            for (int k = 0; k < 2 * D; ++k) {
                const uint32_t uns = ab ^ nbA[k] ^ Jb[k * W + w];
                dl += __popc(nbC[k]) - 2 * __popc(nbC[k] & uns);
            }
        }
    }
    __syncwarp();                        // every read of the old A is done before anyone writes
    for (int w = lane; w < W; w += 32) {
        const uint32_t x0 = CC[w], x1 = CC[W + w];
        if (x0) { A0[w] ^= x0; B0[w] ^= x0; }
        if (x1) { A1[w] ^= x1; B1[w] ^= x1; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        size += __shfl_xor_sync(FULL, size, o);
        dl += __shfl_xor_sync(FULL, dl, o);
    }
    __syncwarp();
    delta = 2 * dl;
    return size;
}

// scratch words per warp of houdayer_pair: two padded natural bit maps (NW + one pad word per lane chunk, each)
template <class LAT>
constexpr int kPairScratchWords = 2 * (4 * LAT::W / 2 + 32);      // 2 * (NW + NW / CHN) <= 2 * (2W + 32)

template <class LAT>
__device__ __forceinline__ int houdayer_pair(const LAT &lat, uint32_t *A0, uint32_t *A1, uint32_t *B0, uint32_t *B1,
                                             const uint32_t *Jb, uint32_t *scratch, uint32_t u, int lane, int &delta)
{
    constexpr int D = LAT::D;
    using NL = NatLat<D, LAT::kLog2L>;
    constexpr int W = NL::W, NW = NL::NW;
    constexpr int CPT = (W + 31) / 32;                 // colour words per lane (contiguous chunk)
    constexpr int CHN = 2 * CPT;                       // natural words per lane
    // Neg / Cl: natural word n lives at pos(n) = n + n / CHN: one pad word per lane chunk makes the chunk stride odd,
    // so the 32 lanes walking their chunks in step hit 32 different banks.
    constexpr int PADDED = NW + NW / CHN;
    auto pos = [](int n) { return n + n / CHN; };
    uint32_t *Neg = scratch, *Cl = scratch + PADDED;
    const unsigned FULL = 0xFFFFFFFFu;

    // q = -1 map in natural order; lane's chunk = colour words [w_lo, w_hi) = natural words [2 w_lo, 2 w_hi)
    const int w_lo = min(W, lane * CPT), w_hi = min(W, w_lo + CPT);
    int local = 0;
    for (int w = w_lo; w < w_hi; ++w) {
        const uint32_t x0 = A0[w] ^ B0[w], x1 = A1[w] ^ B1[w];
        const uint32_t n0 = NL::interleave(2 * w, x0, x1), n1 = NL::interleave(2 * w + 1, x0 >> 16, x1 >> 16);
        Neg[pos(2 * w)] = n0; Neg[pos(2 * w + 1)] = n1;
        Cl[pos(2 * w)] = 0; Cl[pos(2 * w + 1)] = 0;
        local += __popc(n0) + __popc(n1);
    }
    int incl = local;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(FULL, incl, o);
        if (lane >= o) incl += v;
    }
    const int n_neg = __shfl_sync(FULL, incl, 31);
    delta = 0;
    if (n_neg == 0) return 0;
    const int kth = (int)(((unsigned long long)u * (unsigned long long)n_neg) >> 32);
    const int excl = incl - local;
    if (kth >= excl && kth < incl) {
        int rem = kth - excl;
        for (int n = 2 * w_lo; n < 2 * w_hi; ++n) {
            const uint32_t x = Neg[pos(n)];
            const int c = __popc(x);
            if (rem < c) { Cl[pos(n)] = 1u << select_bit(x, rem); break; }
            rem -= c;
        }
    }
    __syncwarp();

    // grow to the fixed point.  Every lane owns a contiguous strip of natural words (whole rows where a row spans
    // several words) and sweeps it down, then up, in place (Gauss-Seidel inside the strip: membership crosses the whole
    // strip, and along x the whole row, in one round), reading its neighbours' strips as they are (Jacobi across
    // strips; chaotic relaxation of a monotone map reaches the same least fixed point in any order).
    const int n_lo = 2 * w_lo, n_hi = 2 * w_hi;
    auto ldCl = [Cl](int i) { return Cl[i + i / CHN]; };
    // Even lanes sweep their strip down then up, odd lanes up then down, and the second sweep starts on the word the first
    // one ended on: a front that reaches the bottom of an even strip is picked up by the odd strip below at the start of
    // its downward sweep in the same round (and the mirror image upwards), so membership crosses two strips per round in
    // either direction instead of one (as in houdayer_rows.cuh).
    const int len = n_hi - n_lo;
    const bool odd = lane & 1;
    for (;;) {
        bool changed = false;
        for (int k = 0; k < 2 * len; ++k) {
            const int j = (k < len) ? k : 2 * len - 1 - k;          // 0 .. len-1, len-1 .. 0
            const int n = odd ? n_hi - 1 - j : n_lo + j;
            const uint32_t neg = Neg[pos(n)], cur = Cl[pos(n)];
            if (neg & ~cur) {
                const uint32_t seeds = (cur | NL::neighbour_union_f(ldCl, n, cur)) & neg;
                if (seeds & ~cur) {
                    Cl[pos(n)] = NL::fill_runs(neg, seeds);
                    changed = true;
                }
            }
        }
        __syncwarp();
        if (!__any_sync(FULL, changed)) break;
    }

    // cluster in the colour layout, over the (no longer needed) q map: CC[p][w]
    uint32_t *CC = Neg;
    int size = 0;
    uint32_t c0[CPT], c1[CPT];
#pragma unroll
    for (int i = 0; i < CPT; ++i) {
        const int w = w_lo + i;
        c0[i] = 0; c1[i] = 0;
        if (w < w_hi) {
            const uint32_t a = Cl[pos(2 * w)], b = Cl[pos(2 * w + 1)];
            size += __popc(a) + __popc(b);
            uint32_t a0, a1, b0, b1;
            NL::deinterleave(2 * w, a, a0, a1);
            NL::deinterleave(2 * w + 1, b, b0, b1);
            c0[i] = a0 | (b0 << 16);
            c1[i] = a1 | (b1 << 16);
        }
    }
    return houdayer_apply<LAT, CPT>(lat, A0, A1, B0, B1, Jb, CC, c0, c1, w_lo, w_hi, size, lane, delta);
}

}  // namespace ptg
