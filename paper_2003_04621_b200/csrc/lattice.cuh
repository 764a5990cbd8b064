// Device-internal lattice layout and neighbour gathers.
//
// A configuration is stored as two bit arrays, one per checkerboard colour p, indexed by the half-index
// h = i >> 1 (L is even, so sites 2h and 2h+1 share a row and have opposite colours: h enumerates the N/2
// sites of one colour bijectively, in site-index order).  bit = 1 <=> spin = -1.  A 32-bit word therefore
// holds 32 same-colour sites = 8 Philox blocks of the Metropolis stream, in order.  Couplings are stored
// per colour and per direction k (k = 2mu: +e_mu, k = 2mu+1: -e_mu) in the same indexing: bit = 1 <=> J = -1.
//
// "gather(O, w, p, nb)" returns, for the 32 sites of word w of colour p, the bits of their 2D neighbours
// taken from the OTHER colour's array O.  Two implementations with one interface:
//   FastLat<D, LOG2L>  L = 2^LOG2L >= 8: whole-word shifts / funnel shifts, everything compile-time;
//   GenLat<D>          any even L >= 2: bit-by-bit from coordinates (slow, general).
#pragma once
#include <stdint.h>

namespace ptg {

// -------------------------------------------------------------------------------------------------------
// coordinates from the half-index (runtime L); used by the general path and by the pack/unpack kernels
struct Coord { int x, y, z; };

__host__ __device__ __forceinline__ int words_per_colour(int N) { return (N / 2 + 31) / 32; }

// site of colour p with half-index h:  i = 2h + x0,  x0 = (p + y + z) & 1
__host__ __device__ __forceinline__ int site_of(int h, int p, int L, int D, Coord *c = nullptr)
{
    const int i2 = 2 * h;
    const int xe = i2 % L;
    const int y = (i2 / L) % L;
    const int z = (D == 3) ? i2 / (L * L) : 0;
    const int x0 = (p + y + z) & 1;
    if (c) { c->x = xe + x0; c->y = y; c->z = z; }
    return i2 + x0;
}

__host__ __device__ __forceinline__ int colour_of_site(int i, int L, int D)
{
    const int x = i % L, y = (i / L) % L, z = (D == 3) ? i / (L * L) : 0;
    return (x + y + z) & 1;
}

// neighbour of site i in direction k (k = 2mu: +e_mu, 2mu+1: -e_mu), periodic
__host__ __device__ __forceinline__ int neighbour_site(int i, int k, int L, int D)
{
    (void)D;
    const int mu = k >> 1;
    const int stride = (mu == 0) ? 1 : (mu == 1 ? L : L * L);
    const int xmu = (i / stride) % L;
    if ((k & 1) == 0) return (xmu == L - 1) ? i - (L - 1) * stride : i + stride;
    return (xmu == 0) ? i + (L - 1) * stride : i - stride;
}

// -------------------------------------------------------------------------------------------------------
template <int D_>
struct GenLat {
    static constexpr int D = D_;
    static constexpr bool kFast = false;
    int L, NH, W;
    __host__ __device__ GenLat(int L_) : L(L_)
    {
        const int N = (D == 2) ? L * L : L * L * L;
        NH = N / 2;
        W = words_per_colour(N);
    }
    __device__ __forceinline__ int words() const { return W; }
    __device__ __forceinline__ uint32_t valid(int w) const
    {
        const int left = NH - 32 * w;
        return left >= 32 ? 0xFFFFFFFFu : ((1u << left) - 1u);
    }
    __device__ void gather(const uint32_t *O, int w, int p, uint32_t nb[2 * D_]) const
    {
#pragma unroll
        for (int k = 0; k < 2 * D_; ++k) nb[k] = 0;
        for (int b = 0; b < 32; ++b) {
            const int h = 32 * w + b;
            if (h >= NH) break;
            const int i = site_of(h, p, L, D_);
#pragma unroll
            for (int k = 0; k < 2 * D_; ++k) {
                const int hj = neighbour_site(i, k, L, D_) >> 1;
                nb[k] |= ((O[hj >> 5] >> (hj & 31)) & 1u) << b;
            }
        }
    }
};

// -------------------------------------------------------------------------------------------------------
template <int D_, int LOG2L>
struct FastLat {
    static constexpr int D = D_;
    static constexpr bool kFast = true;
    static constexpr int kLog2L = LOG2L;
    static constexpr int L = 1 << LOG2L;
    static constexpr int Lh = L / 2;
    static constexpr int N = (D_ == 2) ? L * L : L * L * L;
    static constexpr int NH = N / 2;
    static constexpr int W = NH / 32;
    static_assert(LOG2L >= 3, "fast path needs L >= 8");

    __device__ __forceinline__ int words() const { return W; }
    __device__ __forceinline__ uint32_t valid(int) const { return 0xFFFFFFFFu; }

    // replicate a pattern of `period` bits across the word
    __host__ __device__ static constexpr uint32_t rep_mask(uint32_t pat, int period)
    {
        uint32_t m = 0;
        for (int s = 0; s < 32; s += period) m |= pat << s;
        return m;
    }

    __device__ __forceinline__ void gather(const uint32_t *O, int w, int p, uint32_t nb[2 * D_]) const
    {
        gather_f([O](int i) { return O[i]; }, w, p, nb);
    }

    // same, the other colour's words read through ld(i) (strided or padded layouts)
    template <class F>
    __device__ __forceinline__ void gather_f(F ld, int w, int p, uint32_t nb[2 * D_]) const
    {
        if constexpr (Lh < 32) {
            constexpr int PW = (L * Lh) / 32;                       // words per xy-plane (>= 1)
            constexpr uint32_t SEG_LSB = rep_mask(1u, Lh);          // bit 0 of every row segment
            constexpr uint32_t SEG_MSB = SEG_LSB << (Lh - 1);
            constexpr uint32_t ODD = rep_mask(((1u << Lh) - 1u) << Lh, 2 * Lh);   // bits in rows of odd y
            const int z = (D_ == 3) ? (w / PW) : 0;
            const int base = z * PW, j = w - base;
            const uint32_t same = ld(w);
            const uint32_t rl = ((same << 1) & ~SEG_LSB) | ((same >> (Lh - 1)) & SEG_LSB);   // bit k <- k-1
            const uint32_t rr = ((same >> 1) & ~SEG_MSB) | ((same << (Lh - 1)) & SEG_MSB);   // bit k <- k+1
            const uint32_t x0m = ((p + z) & 1) ? ~ODD : ODD;        // sites with odd x
            nb[0] = (same & ~x0m) | (rr & x0m);                     // +x
            nb[1] = (rl & ~x0m) | (same & x0m);                     // -x
            const uint32_t wn = ld(base + ((j + 1) & (PW - 1)));
            const uint32_t wp = ld(base + ((j - 1) & (PW - 1)));
            nb[2] = __funnelshift_r(same, wn, Lh);                  // +y: bit b <- bit b + Lh (cyclic in plane)
            nb[3] = __funnelshift_l(wp, same, Lh);                  // -y
            if constexpr (D_ == 3) {
                nb[4] = ld((w + PW) & (W - 1));
                nb[5] = ld((w - PW) & (W - 1));
            }
        } else {
            constexpr int WR = Lh / 32;                             // words per row
            constexpr int PW = L * WR;                              // words per plane
            const int row = w / WR, j = w - row * WR;
            const int y = row & (L - 1), z = row >> LOG2L;
            const uint32_t same = ld(w);
            // sites with odd x (row parity p + y + z odd) have their +x neighbour one bit up, the others their -x neighbour one
            // bit down; the other neighbour has the same half-index.  Branch-free: threads of a warp differ in row parity.
            const bool oddx = (p + y + z) & 1;
            const uint32_t side = ld(row * WR + ((oddx ? j + 1 : j - 1) & (WR - 1)));
            nb[0] = oddx ? __funnelshift_r(same, side, 1) : same;
            nb[1] = oddx ? same : __funnelshift_l(side, same, 1);
            const int base = z * PW, jj = w - base;
            nb[2] = ld(base + ((jj + WR) & (PW - 1)));
            nb[3] = ld(base + ((jj - WR) & (PW - 1)));
            if constexpr (D_ == 3) {
                nb[4] = ld((w + PW) & (W - 1));
                nb[5] = ld((w - PW) & (W - 1));
            }
        }
    }
};

// natural-order neighbour / colour / site helpers: shifts and masks on the power-of-two lattices, coordinates otherwise
template <class LAT, int K>
__device__ __forceinline__ int nat_neighbour(int i, int L, int D)
{
    if constexpr (LAT::kFast) {
        constexpr int LG = LAT::kLog2L, mu = K >> 1;
        constexpr int st = 1 << (LG * mu), M = (LAT::L - 1) << (LG * mu);
        return (i & ~M) | ((i + ((K & 1) ? -st : st)) & M);
    } else {
        return neighbour_site(i, K, L, D);
    }
}

template <class LAT>
__device__ __forceinline__ int nat_colour(int i, int L, int D)
{
    if constexpr (LAT::kFast) {
        constexpr int LG = LAT::kLog2L;
        return (i ^ (i >> LG) ^ (LAT::D == 3 ? (i >> (2 * LG)) : 0)) & 1;
    } else {
        return colour_of_site(i, L, D);
    }
}

template <class LAT>
__device__ __forceinline__ int nat_site_of(int h, int p, int L, int D)
{
    if constexpr (LAT::kFast) {
        constexpr int LG = LAT::kLog2L;
        const int i2 = 2 * h;
        return i2 + ((p ^ (i2 >> LG) ^ (LAT::D == 3 ? (i2 >> (2 * LG)) : 0)) & 1);
    } else {
        return site_of(h, p, L, D);
    }
}

// coordinates of natural site index i
template <class LAT>
__device__ __forceinline__ void nat_coords(int i, int L, int D, int &x, int &y, int &z)
{
    if constexpr (LAT::kFast) {
        constexpr int LG = LAT::kLog2L;
        x = i & (LAT::L - 1);
        y = (i >> LG) & (LAT::L - 1);
        z = (LAT::D == 3) ? (i >> (2 * LG)) : 0;
    } else {
        x = i % L;
        y = (i / L) % L;
        z = (D == 3) ? i / (L * L) : 0;
    }
}

}  // namespace ptg
