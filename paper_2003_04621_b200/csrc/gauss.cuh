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

// u < THR(x) decided exactly, cheaply: a float estimate of 2^32 e^x brackets the double threshold (the error of __expf
// for |x| <= 23 is below 4e-6 relative, (float)x and (float)u add 2e-6; the bracket is 1e-4 wide), and only a draw that
// falls inside the bracket (probability ~2e-4 p) pays for the double evaluation.  Same decision as thr_double(x) always.
__device__ __forceinline__ bool accept_exp(uint32_t u, double x)
{
    const float t = __expf((float)x) * 4294967296.0f;
    const float uf = (float)u;
    if (uf < t * 0.9999f - 1.0f) return true;
    if (uf > t * 1.0001f + 1.0f) return false;
    return u < thr_double(x);
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

// Metropolis sweeps with fixed-point couplings.  CTA = R replicas of one sample in shared memory; work item = one word =
// 32 same-colour sites of one replica, walked site by site: h = sum_k J_k s_k (integer), a = s_i h, flip iff a <= 0 or
// u < THR(-(beta * ldexp(2a, -fbits))).  Same Philox words as the +-J sweep (domain 3).
// grid: (2T/R groups, S).  dynamic smem: [R][2][W] spins | [R] dE | [R] temperature index
template <class LAT>
__global__ void __launch_bounds__(128) k_sweep_q(LAT lat, Params P, int R, uint32_t step0, int n_sweeps)
{
    constexpr int D = LAT::D;
    extern __shared__ uint32_t smem[];
    const int W = lat.words(), NHP = 32 * W;
    uint32_t *sS = smem;                       // [R][2][W]
    int *sdE = (int *)(sS + R * 2 * W);        // [R]
    int *sT = sdE + R;                         // [R]
    const int s = blockIdx.y;
    const int q0 = blockIdx.x * R;
    const size_t rep0 = (size_t)s * 2 * P.T + q0;
    const uint32_t g = P.g0 + (uint32_t)s;
    for (int i = threadIdx.x; i < R * 2 * W; i += blockDim.x) sS[i] = P.d.spin[rep0 * 2 * W + i];
    for (int i = threadIdx.x; i < R; i += blockDim.x) { sdE[i] = 0; sT[i] = P.d.tos[rep0 + i]; }
    __syncthreads();

    for (int it = 0; it < n_sweeps; ++it) {
        for (int p = 0; p < 2; ++p) {
            const int32_t *Jp = P.d.Jdev + ((size_t)s * 2 + p) * (2 * D) * NHP;
            for (int item = threadIdx.x; item < R * W; item += blockDim.x) {
                const int qi = item / W, w = item - qi * W;
                const int q = q0 + qi;
                const int c = (q >= P.T) ? 1 : 0, r = q - c * P.T;
                const double beta = P.d.betasD[sT[qi]];
                uint32_t *Sown = sS + (qi * 2 + p) * W;
                uint32_t nb[2 * D];
                lat.gather(sS + (qi * 2 + (1 - p)) * W, w, p, nb);
                const uint32_t sw = Sown[w], valid = lat.valid(w);
                const Round0Shared r0 = philox_round0_shared(step0 + (uint32_t)it, g, make_tag(DOM_METRO, p, c, r), P.rk);
                uint32_t flip = 0;
                int dE = 0;
#pragma unroll 1
                for (int B = 0; B < 8; ++B) {
                    if (((valid >> (4 * B)) & 0xFu) == 0u) continue;
                    uint32_t u[4];
                    philox4x32_10_shared(8u * (uint32_t)w + (uint32_t)B, r0, P.rk, u[0], u[1], u[2], u[3]);
                    int4 Jv[2 * D];
#pragma unroll
                    for (int k = 0; k < 2 * D; ++k) Jv[k] = *(const int4 *)(Jp + jdev_index(W, k, B, w));
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int b = 4 * B + j;
                        if (!((valid >> b) & 1u)) continue;
                        int h = 0;
#pragma unroll
                        for (int k = 0; k < 2 * D; ++k) {
                            const int Jk = (j == 0) ? Jv[k].x : (j == 1) ? Jv[k].y : (j == 2) ? Jv[k].z : Jv[k].w;
                            h += ((nb[k] >> b) & 1u) ? -Jk : Jk;
                        }
                        const int a = ((sw >> b) & 1u) ? -h : h;
                        bool acc = a <= 0;
                        if (!acc) acc = accept_exp(u[j], -(beta * ldexp((double)(2LL * a), -P.fbits)));
                        if (acc) { flip |= 1u << b; dE += 2 * a; }
                    }
                }
                Sown[w] = sw ^ flip;
                if (dE != 0) atomicAdd(sdE + qi, dE);
            }
            __syncthreads();
        }
    }
    for (int i = threadIdx.x; i < R * 2 * W; i += blockDim.x) P.d.spin[rep0 * 2 * W + i] = sS[i];
    for (int i = threadIdx.x; i < R; i += blockDim.x) P.d.E[rep0 + i] += sdE[i];
}

}  // namespace ptg
