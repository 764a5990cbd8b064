// NEXT-4  Multi-cluster variant of the Houdayer exchange ("a formal conversion to a multi-cluster
// variant", :247; reading R37): EVERY connected component of q = -1 sites is exchanged between the two
// configurations with probability 1/2, decided by the top bit of the Philox word of the component's smallest site
// index (domain 5, aux = 1: block i_min >> 2, word i_min & 3).
//
// One CTA per (sample, temperature); any lattice (coordinates in natural site order).  Components are found by
// label propagation in shared memory -- the scheme north_star names for the cluster kernel: lab[i] starts as i on the
// q = -1 sites, every pass takes the minimum over the q = -1 neighbours and then follows the label chain to its
// current root (pointer jumping; a label is always the index of a site of the same component with a smaller or
// equal index, so chains end at a site that is its own label).  Only the owner thread of site i writes lab[i] and
// labels only decrease, so stale reads are harmless; at the fixed point every site of a component carries the
// component's smallest index, which makes the decision independent of the thread mapping.
#pragma once
#include "kernels.cuh"

namespace ptg {

constexpr uint32_t kNoLabel = 0x7FFFFFFFu;      // q = +1 site (never a valid site index: N*d < 2^31)
constexpr uint32_t kFlagBit = 0x80000000u;      // set on a root's own label once its coin says "exchange"

// dynamic smem: Neg[2][W] | Cl[2][W] | red[2 * nwarps + 2] | lab[N]
template <class LAT>
__global__ void __launch_bounds__(256) k_houdayer_multi(LAT lat, Params P, uint32_t step)
{
    extern __shared__ uint32_t hsm[];
    const int W = lat.words();
    const int nwarps = blockDim.x >> 5;
    uint32_t *Neg = hsm, *Cl = hsm + 2 * W;
    int *red = (int *)(Cl + 2 * W);
    uint32_t *lab = (uint32_t *)(red + 2 * nwarps + 2);
    const int t = blockIdx.x, s = blockIdx.y, tid = threadIdx.x;
    const int L = P.L, D = P.D, N = P.N;
    const size_t repA = rep_index(P, s, 0, P.d.sot[rep_index(P, s, 0, t)]);
    const size_t repB = rep_index(P, s, 1, P.d.sot[rep_index(P, s, 1, t)]);
    uint32_t *A[2] = {spin_words(P, repA, 0), spin_words(P, repA, 1)};
    uint32_t *B[2] = {spin_words(P, repB, 0), spin_words(P, repB, 1)};

    for (int w = tid; w < W; w += blockDim.x) {
        const uint32_t v = lat.valid(w);
        Neg[w] = (A[0][w] ^ B[0][w]) & v;
        Neg[W + w] = (A[1][w] ^ B[1][w]) & v;
        Cl[w] = 0; Cl[W + w] = 0;
    }
    __syncthreads();
    for (int i = tid; i < N; i += blockDim.x) {
        const int p = colour_of_site(i, L, D), h = i >> 1;
        lab[i] = ((Neg[p * W + (h >> 5)] >> (h & 31)) & 1u) ? (uint32_t)i : kNoLabel;
    }
    __syncthreads();

    // label propagation to the fixed point
    for (;;) {
        int changed = 0;
        for (int i = tid; i < N; i += blockDim.x) {
            const uint32_t cur = lab[i];
            if (cur == kNoLabel) continue;
            uint32_t m = cur;
            for (int k = 0; k < 2 * D; ++k) m = min(m, lab[neighbour_site(i, k, L, D)]);     // kNoLabel never wins
            for (uint32_t up = lab[m]; up < m; up = lab[m]) m = up;                          // follow the chain to its root
            if (m < cur) { lab[i] = m; changed = 1; }
        }
        if (!__syncthreads_or(changed)) break;
    }

    // one coin per component, thrown by its root (the site that is its own label)
    for (int i = tid; i < N; i += blockDim.x) {
        if (lab[i] != (uint32_t)i) continue;
        uint32_t w4[4];
        philox4x32_10((uint32_t)(i >> 2), step, P.g0 + (uint32_t)s, make_tag(DOM_HOUD, 1, 0, t), P.rk, w4[0], w4[1], w4[2], w4[3]);
        const uint32_t wsel = (i & 2) ? ((i & 1) ? w4[3] : w4[2]) : ((i & 1) ? w4[1] : w4[0]);
        if (wsel >> 31) lab[i] = (uint32_t)i | kFlagBit;
    }
    __syncthreads();

    // the exchanged set in the colour layout: one thread per (colour, word)
    for (int id = tid; id < 2 * W; id += blockDim.x) {
        const int p = id / W, w = id - p * W;
        uint32_t x = Neg[id], out = 0;
        while (x) {
            const int b = __ffs(x) - 1;
            x &= x - 1;
            const int i = site_of(32 * w + b, p, L, D);
            const uint32_t r = lab[i] & ~kFlagBit;
            if (lab[r] & kFlagBit) out |= 1u << b;
        }
        Cl[id] = out;
    }
    __syncthreads();
    cta_exchange_set(lat, P, s, t, repA, repB, A, B, Cl, red);
}

}  // namespace ptg
