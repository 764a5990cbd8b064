// NEXT-3  Fixed-point (Gaussian) couplings (readings R33-R35, section 9b).
//
// J = Jq * 2^-fbits with Jq int32: local fields, energies and energy differences are exact integers in units of 2^-fbits,
// so every reduction is order-free and the path stays bit-exact against the oracle; acceptance probabilities are
// evaluated per decision in double (R34).  Spins stay bit-packed per colour as in the +-J path and the Philox mapping,
// the checkerboard order, the PT pass and the cluster growth are unchanged; only the kernels that need the VALUE of a
// coupling are new: the sweep and the energy.  Couplings live as Jdev[s][colour p][direction k][B][w][j] int32 with
// half-index h = 32 w + 4 B + j (each bond stored from both endpoints, like the +-J bit arrays): the four couplings of
// Philox block B of word w are one int4, and threads that own consecutive words read consecutive int4s (coalesced).
#pragma once
#include "kernels.cuh"

namespace ptg {

// THR(x) = min(2^32-1, floor(2^32 exp(x))), x <= 0, in double (R5, R34)
__device__ __forceinline__ uint32_t thr_double(double x)
{
    const double v = floor(ldexp(exp(x), 32));
    if (v >= 4294967295.0) return 4294967295u;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

// test hook (pt_threshold_selftest): the DEVICE evaluation of THR for a list of arguments, to be compared with the host libm's
__global__ void k_threshold_selftest(const double *x, uint32_t *out, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = thr_double(x[i]);
}

// Uphill move with a = s_i h_i > 0 (units of 2^-fbits): accept iff u < THR(x), x = -(beta * ldexp(2a, -fbits)) (R34), decided
// EXACTLY but cheaply.  Let Y = 2^32 e^x; u < floor(Y) <=> u + 1 <= Y.  A float estimate t9 of y9 = Y / 512 = 2^(23 + a c2),
// c2 = (float)(-2 beta 2^-fbits log2 e), is off by at most 1e-5 relative: (float)a is exact below 2^23, the fma rounds once
// (<= 2^-18 absolute in the exponent for |exponent| < 128), c2 carries 2^-24 relative of an exponent of magnitude < 150, and
// ex2.approx is good to 2^-22.  With u9 = u >> 9 (512 u9 <= u < 512 (u9 + 1); 23 bits, exactly representable in float):
//   u9 + 2 < 0.9999 t9   =>  u + 1 <= 512 (u9 + 1) < 512 (y9 - 1) < Y            => accept;
//   u9 > 1.0001 t9 + 1   =>  u >= 512 u9 > Y                                      => reject
// (the float products add < 2e-7 relative, far inside the 1e-4 bracket; the oracle's double exp is within 1e-16 of Y).
// Only a draw inside the bracket (probability ~2e-4 of an uphill attempt) or a >= 2^23 pays for the double evaluation,
// which is the oracle's formula.  Same decision as u < thr_double(x) always.
// the rare exact evaluation, kept out of line so the 32 unrolled site decisions stay small
__device__ __noinline__ bool accept_exact(uint32_t u, int a, const double *beta_ptr, int fbits)
{
    return u < thr_double(-(*beta_ptr * ldexp((double)(2LL * a), -fbits)));
}

// Decision for one site, branch-free: returns the sure part of the decision (a <= 0 always flips; an uphill move
// whose draw is below the bracket flips) and sets `need` when the draw fell inside the bracket (or a >= 2^23) and the exact
// evaluation (accept_exact) has to decide.  u9 + 2 is formed directly by the magic subtraction (exact below 2^24).
// SMALL: the host has checked 2 D max|Jq| < 2^23, so every a is below 2^23 and the range test is dropped.
template <bool SMALL>
__device__ __forceinline__ bool accept_site(uint32_t u, int a, float c2, bool &need)
{
    const float af = __int_as_float(0x4B000000 + a) - 8388608.0f;              // exact for 0 <= a < 2^23 (unused otherwise)
    const float t9 = ex2_approx(fmaf(af, c2, 23.0f));
    const float uf9p2 = __uint_as_float(0x4B000000u | (u >> 9)) - 8388606.0f;  // u9 + 2, exact: 23 bits fill the mantissa
    const bool up = a > 0;
    const bool small = SMALL || (uint32_t)a < (1u << 23);
    const bool sure_acc = small && (uf9p2 < t9 * 0.9999f);
    const bool sure_rej = small && (uf9p2 > fmaf(t9, 1.0001f, 3.0f));
    need = up && !sure_acc && !sure_rej;
    return !up || sure_acc;
}

// s -= J if bit j of un is set: one LOP3 with predicate output + one predicated add
template <int J>
__device__ __forceinline__ void sub_if_bit(int &s, uint32_t un, int Jv)
{
    asm("{\n\t.reg .pred p;\n\t.reg .b32 t;\n\tand.b32 t, %1, %3;\n\tsetp.ne.u32 p, t, 0;\n\t@p sub.s32 %0, %0, %2;\n\t}"
        : "+r"(s) : "r"(un), "r"(Jv), "n"(1u << J));
}

// natural-order int32 couplings JqNat[S][D][N] -> Jdev[S][2][2D][NHP]
__device__ __forceinline__ size_t jdev_index(int W, int k, int B, int w) { return ((size_t)(k * 8 + B) * W + w) * 4; }

__global__ void k_pack_jq(Params P)
{
    const int NHP = 32 * P.W;
    const long total = (long)P.S * 2 * (2 * P.D) * NHP;
    for (long id = blockIdx.x * (long)blockDim.x + threadIdx.x; id < total; id += (long)gridDim.x * blockDim.x) {
        const int h = (int)(id % NHP);
        const int k = (int)((id / NHP) % (2 * P.D));
        const int p = (int)((id / ((long)NHP * 2 * P.D)) & 1);
        const int s = (int)(id / ((long)NHP * 2 * P.D * 2));
        int32_t v = 0;
        if (h < P.NH) {
            const int i = site_of(h, p, P.L, P.D);
            const int mu = k >> 1;
            const int b = (k & 1) ? neighbour_site(i, k, P.L, P.D) : i;      // bond (mu, b): b -> b + e_mu
            v = P.d.JqNat[((size_t)s * P.D + mu) * P.N + b];
        }
        const int w = h >> 5, B = (h >> 2) & 7, j = h & 3;
        P.d.Jdev[((size_t)s * 2 + p) * (2 * P.D) * NHP + jdev_index(P.W, k, B, w) + j] = v;
    }
}

// E = -sum_bonds J s_i s_j, every bond seen from its black endpoint.  One warp per replica.
// mode 0: write E;  mode 1: write outE (slot order) and count mismatches against E.
template <class LAT>
__global__ void k_energy_q(LAT lat, Params P, int mode)
{
    const int warps_per_block = blockDim.x >> 5;
    const long rep = (long)blockIdx.x * warps_per_block + (threadIdx.x >> 5);
    const int lane = threadIdx.x & 31;
    if (rep >= (long)P.S * 2 * P.T) return;
    const int s = (int)(rep / (2L * P.T));
    const int NHP = 32 * P.W;
    const uint32_t *Sb = spin_words(P, (size_t)rep, 0), *Sw = spin_words(P, (size_t)rep, 1);
    const int32_t *Jb = P.d.Jdev + ((size_t)s * 2 + 0) * (2 * LAT::D) * NHP;
    long long e = 0;
    for (int w = lane; w < lat.words(); w += 32) {
        uint32_t nb[2 * LAT::D];
        lat.gather(Sw, w, 0, nb);
        const uint32_t sb = Sb[w], v = lat.valid(w);
#pragma unroll
        for (int k = 0; k < 2 * LAT::D; ++k) {
            const uint32_t uns = sb ^ nb[k];                   // 1 <=> s_i s_j = -1
            for (int B = 0; B < 8; ++B) {
                const int4 J4 = *(const int4 *)(Jb + jdev_index(lat.words(), k, B, w));
                const uint32_t u4 = uns >> (4 * B), v4 = v >> (4 * B);
                int part = 0;
                if (v4 & 1u) part += (u4 & 1u) ? J4.x : -J4.x;
                if (v4 & 2u) part += (u4 & 2u) ? J4.y : -J4.y;
                if (v4 & 4u) part += (u4 & 4u) ? J4.z : -J4.z;
                if (v4 & 8u) part += (u4 & 8u) ? J4.w : -J4.w;
                e += part;
            }
        }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xFFFFFFFFu, e, o);
    if (lane == 0) {
        const int32_t ei = (int32_t)e;
        if (mode == 0) {
            P.d.E[rep] = ei;
        } else {
            P.d.outE[rep] = ei;
            if (P.d.E[rep] != ei) atomicAdd(P.d.mismatch, 1);
        }
    }
}

template <int J> __device__ __forceinline__ int comp(const int4 &v) { return J == 0 ? v.x : J == 1 ? v.y : J == 2 ? v.z : v.w; }

// Site J (0..3) of the current Philox block: un[k] has the block's four sign bits in bits 0..3.  The sure decisions go
// into nib / dE at once; a site whose draw fell inside the bracket sets bit J of needmask and is settled by the caller.
template <class LAT, bool SMALL, int J>
__device__ __forceinline__ int sweep_site_q(const uint32_t (&un)[2 * LAT::D], const int4 (&Jv)[2 * LAT::D], uint32_t u, uint32_t vv,
                                            float c2, uint32_t &nib, int &dE, uint32_t &needmask)
{
    constexpr int D = LAT::D;
    int tot = 0, lost = 0;                       // a = sum_k J_k - 2 sum_{k: s_i s_k = -1} J_k
#pragma unroll
    for (int k = 0; k < 2 * D; ++k) tot += comp<J>(Jv[k]);
#pragma unroll
    for (int k = 0; k < 2 * D; ++k) sub_if_bit<J>(lost, un[k], comp<J>(Jv[k]));
    const int a = tot + 2 * lost;
    bool need;
    bool acc = accept_site<SMALL>(u, a, c2, need);
    if constexpr (!LAT::kFast) { const bool ok = vv & (1u << J); acc = acc && ok; need = need && ok; }
    if (acc) { nib |= 1u << J; dE += 2 * a; }
    if (need) needmask |= 1u << J;
    return a;
}

// One work item of the fixed-point sweep = one word = 32 same-colour sites of one replica, walked Philox block by Philox
// block (4 sites): a = s_i h_i = sum_k J_k (s_i s_k) (integer) starts from sum_k J_k and loses 2 J_k for every
// unsatisfied-sign bit of un_k = s ^ nb_k; flip iff a <= 0 or the exact bracket test.  Same Philox words as the +-J sweep
// (domain 3).  Sown / Soth: the replica's words of colour p / 1-p (shared memory); Jp: the sample's colour-p block of Jdev
// (global, read through L1).  Returns the energy change of the replica.
template <class LAT, bool SMALL>
__device__ __forceinline__ int update_word_q(const LAT &lat, uint32_t *Sown, const uint32_t *Soth, const int32_t *Jp, int W,
                                             int w, int p, float c2, const double *beta_ptr, int fbits, uint32_t step,
                                             uint32_t g, uint32_t tag, const RoundKeys &rk)
{
    constexpr int D = LAT::D;
    uint32_t un[2 * D];
    lat.gather(Soth, w, p, un);
    const uint32_t sw = Sown[w];
    uint32_t vv = lat.valid(w);
#pragma unroll
    for (int k = 0; k < 2 * D; ++k) un[k] ^= sw;                   // bit = 1 <=> s_i s_k = -1
    const Round0Shared r0 = philox_round0_shared(step, g, tag, rk);
    uint32_t flip = 0;
    int dE = 0;
#pragma unroll 4        // measured: 2 -> 4 is +1.3 % on the fused Gaussian MCS, 8 is -14 % (instruction cache)
    for (int B = 0; B < 8; ++B) {
        if (LAT::kFast || (vv & 0xFu) != 0u) {          // the word-parallel lattices have no partial words
            uint32_t u[4];
            philox4x32_10_shared(8u * (uint32_t)w + (uint32_t)B, r0, rk, u[0], u[1], u[2], u[3]);
            int4 Jv[2 * D];
#pragma unroll
            for (int k = 0; k < 2 * D; ++k) Jv[k] = __ldg((const int4 *)(Jp + jdev_index(W, k, B, w)));
            uint32_t nib = 0, needmask = 0;
            int av[4];
            av[0] = sweep_site_q<LAT, SMALL, 0>(un, Jv, u[0], vv, c2, nib, dE, needmask);
            av[1] = sweep_site_q<LAT, SMALL, 1>(un, Jv, u[1], vv, c2, nib, dE, needmask);
            av[2] = sweep_site_q<LAT, SMALL, 2>(un, Jv, u[2], vv, c2, nib, dE, needmask);
            av[3] = sweep_site_q<LAT, SMALL, 3>(un, Jv, u[3], vv, c2, nib, dE, needmask);
            if (needmask) {                      // rare (~1e-3 of the blocks): the oracle's double formula decides
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    if (((needmask >> j) & 1u) && accept_exact(u[j], av[j], beta_ptr, fbits)) { nib |= 1u << j; dE += 2 * av[j]; }
            }
            flip |= nib << (4 * B);
        }
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) un[k] >>= 4;
        vv >>= 4;
    }
    Sown[w] = sw ^ flip;
    return dE;
}

// Energy of a replica from the couplings' values, every bond seen from its black endpoint:
//   E = -sum_bonds J s_i s_j = -(sum_bonds J) + 2 * sum over the bonds with s_i s_j = -1 of J.
// bond_sum_word_q: sum over the 32 black sites of word w and their 2D directions of J (a constant of the sample);
// unsat_sum_word_q: the same sum restricted to the bonds with s_i s_j = -1 (one predicate-setting LOP3 and one predicated
// subtract per bond; returns minus the sum).  Sb / Sw: the replica's black / white words; Jb: colour-0 block of Jdev.
template <class LAT>
__device__ __forceinline__ int bond_sum_word_q(const LAT &lat, const int32_t *Jb, int W, int w)
{
    constexpr int D = LAT::D;
    uint32_t vv = lat.valid(w);
    int sum = 0;
    for (int B = 0; B < 8; ++B) {
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) {
            const int4 J4 = __ldg((const int4 *)(Jb + jdev_index(W, k, B, w)));
            if (vv & 1u) sum += J4.x;
            if (vv & 2u) sum += J4.y;
            if (vv & 4u) sum += J4.z;
            if (vv & 8u) sum += J4.w;
        }
        vv >>= 4;
    }
    return sum;
}

template <class LAT>
__device__ __forceinline__ int unsat_sum_word_q(const LAT &lat, const uint32_t *Sb, const uint32_t *Sw, const int32_t *Jb, int W,
                                                int w)
{
    constexpr int D = LAT::D;
    uint32_t un[2 * D];
    lat.gather(Sw, w, 0, un);
    const uint32_t sb = Sb[w], v = lat.valid(w);
#pragma unroll
    for (int k = 0; k < 2 * D; ++k) un[k] = (un[k] ^ sb) & v;
    int lost = 0;                                   // = -(sum of J over the unsatisfied-sign bonds)
#pragma unroll 2
    for (int B = 0; B < 8; ++B) {
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) {
            const int4 J4 = __ldg((const int4 *)(Jb + jdev_index(W, k, B, w)));
            sub_if_bit<0>(lost, un[k], J4.x);
            sub_if_bit<1>(lost, un[k], J4.y);
            sub_if_bit<2>(lost, un[k], J4.z);
            sub_if_bit<3>(lost, un[k], J4.w);
        }
#pragma unroll
        for (int k = 0; k < 2 * D; ++k) un[k] >>= 4;
    }
    return lost;
}

// c2 of accept_site for inverse temperature beta: (float)(-2 beta 2^-fbits log2 e)
__device__ __forceinline__ float bracket_slope(double beta, int fbits) { return (float)(-(2.0 * beta) * ldexp(1.4426950408889634, -fbits)); }

// Metropolis sweeps with fixed-point couplings, separate kernel.  CTA = R replicas of one sample in shared memory.
// grid: (2T/R groups, S).  dynamic smem: [R][2][W] spins | [R] dE | [R] temperature index | [R] c2 (float)
template <class LAT, bool SMALL>
__global__ void __launch_bounds__(128) k_sweep_q(LAT lat, Params P, int R, uint32_t step0, int n_sweeps)
{
    constexpr int D = LAT::D;
    extern __shared__ uint32_t smem[];
    const int W = lat.words(), NHP = 32 * W;
    uint32_t *sS = smem;                       // [R][2][W]
    int *sdE = (int *)(sS + R * 2 * W);        // [R]
    int *sT = sdE + R;                         // [R]
    float *sC2 = (float *)(sT + R);            // [R]
    const int s = blockIdx.y;
    const int q0 = blockIdx.x * R;
    const size_t rep0 = (size_t)s * 2 * P.T + q0;
    const uint32_t g = P.g0 + (uint32_t)s;
    for (int i = threadIdx.x; i < R * 2 * W; i += blockDim.x) sS[i] = P.d.spin[rep0 * 2 * W + i];
    for (int i = threadIdx.x; i < R; i += blockDim.x) {
        const int t = P.d.tos[rep0 + i];
        sdE[i] = 0;
        sT[i] = t;
        sC2[i] = bracket_slope(P.d.betasD[t], P.fbits);
    }
    __syncthreads();

    for (int it = 0; it < n_sweeps; ++it) {
        for (int p = 0; p < 2; ++p) {
            const int32_t *Jp = P.d.Jdev + ((size_t)s * 2 + p) * (2 * D) * NHP;
            for (int item = threadIdx.x; item < R * W; item += blockDim.x) {
                const int qi = item / W, w = item - qi * W;
                const int q = q0 + qi;
                const int c = (q >= P.T) ? 1 : 0, r = q - c * P.T;
                const int dE = update_word_q<LAT, SMALL>(lat, sS + (qi * 2 + p) * W, sS + (qi * 2 + (1 - p)) * W, Jp, W, w, p, sC2[qi],
                                                         P.d.betasD + sT[qi], P.fbits, step0 + (uint32_t)it, g,
                                                         make_tag(DOM_METRO, p, c, r), P.rk);
                atomicAdd(sdE + qi, dE);
            }
            __syncthreads();
        }
    }
    for (int i = threadIdx.x; i < R * 2 * W; i += blockDim.x) P.d.spin[rep0 * 2 * W + i] = sS[i];
    for (int i = threadIdx.x; i < R; i += blockDim.x) P.d.E[rep0 + i] += sdE[i];
}

}  // namespace ptg
