// NEXT-4  Multi-cluster variant of the Houdayer exchange ("a formal conversion to a multi-cluster
// variant", :247; reading R37): EVERY connected component of q = -1 sites is exchanged between the two
// configurations with probability 1/2, decided by the top bit of the Philox word of the component's smallest site
// index (domain 5, aux = 1: block i_min >> 2, word i_min & 3).
//
// One CTA per (sample, temperature); any lattice (coordinates in natural site order).  Components are found by
// label equivalence in shared memory -- the scheme north_star names for the cluster kernel: lab[i] starts as i on the
// q = -1 sites; a pass is (scan) every site takes the minimum label m over its q = -1 neighbours and, if m is smaller
// than its own label l, lowers the label OF SITE l to m with an atomicMin (it merges the two trees at their roots,
// not just the site), then (flatten) every site follows its label chain to the root (a label is always the index of
// a site of the same component with a smaller or equal index, so chains end at a site that is its own label).
// Merging at the roots converges in a handful of passes where plain neighbour propagation needs one per lattice
// step.  At the fixed point every site of a component carries the component's smallest index, which makes the
// decision independent of the thread mapping.
#pragma once
#include "kernels.cuh"

namespace ptg {

constexpr uint32_t kNoLabel = 0x7FFFFFFFu;      // q = +1 site (never a valid site index: N*d < 2^31)
constexpr uint32_t kFlagBit = 0x80000000u;      // set on a root's own label once its coin says "exchange"

template <class LAT, int K>
__device__ __forceinline__ uint32_t min_neighbour_label(const uint32_t *lab, int i, int L, int D, uint32_t m)
{
    if constexpr (K < 2 * LAT::D) {
        m = min(m, lab[nat_neighbour<LAT, K>(i, L, D)]);          // kNoLabel never wins
        return min_neighbour_label<LAT, K + 1>(lab, i, L, D, m);
    } else {
        return m;
    }
}

// dynamic smem: Neg[2][W] | Cl[2][W] | red[2 * nwarps + 2] | lab[N] | act[N] (uint16: list of the q = -1 sites, N <= 65536)
template <class LAT>
__global__ void __launch_bounds__(512) k_houdayer_multi(LAT lat, Params P, uint32_t step)
{
    extern __shared__ uint32_t hsm[];
    const int W = lat.words();
    const int nwarps = blockDim.x >> 5;
    uint32_t *Neg = hsm, *Cl = hsm + 2 * W;
    int *red = (int *)(Cl + 2 * W);
    uint32_t *lab = (uint32_t *)(red + 2 * nwarps + 2);
    uint16_t *act = (uint16_t *)(lab + P.N);
    int *n_act_s = red + 2 * nwarps;                 // red[2 nwarps]: number of q = -1 sites (red[0 .. 2 nwarps) is used by the tail only)
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
    if (tid == 0) *n_act_s = 0;
    __syncthreads();
    // labels, and the compact list of the q = -1 sites (any order) that every later loop walks: about half of the sites
    // have q = +1 and would only idle their lanes.  Warp-aggregated append: one atomicAdd per 32 sites.
    for (int i0 = (tid & ~31); i0 < N; i0 += blockDim.x) {
        const int i = i0 + (tid & 31);
        bool on = false;
        if (i < N) {
            const int p = nat_colour<LAT>(i, L, D), h = i >> 1;
            on = (Neg[p * W + (h >> 5)] >> (h & 31)) & 1u;
            lab[i] = on ? (uint32_t)i : kNoLabel;
        }
        const unsigned m = __ballot_sync(0xFFFFFFFFu, on);
        int base = 0;
        if ((tid & 31) == 0 && m) base = atomicAdd(n_act_s, __popc(m));
        base = __shfl_sync(0xFFFFFFFFu, base, 0);
        if (on) act[base + __popc(m & ((1u << (tid & 31)) - 1u))] = (uint16_t)i;
    }
    __syncthreads();
    const int n_act = *n_act_s;

    // label equivalence to the fixed point
    for (;;) {
        int changed = 0;
        for (int k = tid; k < n_act; k += blockDim.x) {                  // scan: merge trees at their roots
            const int i = act[k];
            const uint32_t l = lab[i];
            const uint32_t m = min_neighbour_label<LAT, 0>(lab, i, L, D, l);
            if (m < l) { atomicMin(lab + l, m); changed = 1; }
        }
        if (!__syncthreads_or(changed)) break;
        for (int k = tid; k < n_act; k += blockDim.x) {                  // flatten: every site points at its root
            const int i = act[k];
            uint32_t l = lab[i];
            for (uint32_t up = lab[l]; up != l; up = lab[l]) l = up;
            lab[i] = l;
        }
        __syncthreads();
    }

    // one coin per component, thrown by its root (the site that is its own label)
    for (int k = tid; k < n_act; k += blockDim.x) {
        const int i = act[k];
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
            const int i = nat_site_of<LAT>(32 * w + b, p, L, D);
            const uint32_t r = lab[i] & ~kFlagBit;
            if (lab[r] & kFlagBit) out |= 1u << b;
        }
        Cl[id] = out;
    }
    __syncthreads();
    cta_exchange_set(lat, P, s, t, repA, repB, A, B, Cl, red);
}

}  // namespace ptg
