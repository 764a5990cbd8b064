// a7  Fused Monte Carlo steps: ONE CTA keeps ONE SAMPLE -- the bit-packed spins of all
// its 2T replicas, its couplings, tracked energies, both index maps and the per-slot thresholds -- resident in
// shared memory for n_mcs whole MCS:  [ n_metro sweeps -> Houdayer exchange per temperature -> PT pass ] x n_mcs.
// Samples never interact (P:7), so there is no grid-wide synchronisation; the state is read from and
// written back to global memory once per call.  The phases are the same device functions the separate kernels
// use (update_word, houdayer_pair) and the exchange walk of k_exchange, so the results are bit-identical.
#pragma once
#include "kernels.cuh"

namespace ptg {

struct McsArgs {
    int n_mcs, n_metro, do_houdayer, do_exchange;
    uint32_t sweep0, houd0, exch0;          // counter values at the start of the call
};

// shared-memory carve-up, shared by host (size) and device (pointers); all offsets in 32-bit words
struct McsSmem {
    int oJ, oS, oE, oTos, oSot, oThr, oAcc, oLast, oCum, oScr, words;
    __host__ __device__ McsSmem(int D, int W, int T, int nwarps)
    {
        int o = 0;
        oJ = o;    o += 2 * 2 * D * W;
        oS = o;    o += 2 * T * 2 * W;
        oE = o;    o += 2 * T;
        oTos = o;  o += 2 * T;
        oSot = o;  o += 2 * T;
        oThr = o;  o += 2 * T * 4;
        oAcc = o;  o += 2 * T;              // accepted swaps of this call per (chain, pair)
        oLast = o; o += T;
        o = (o + 1) & ~1;
        oCum = o;  o += 2 * T;              // 64-bit
        oScr = o;  o += nwarps * 4 * W;
        words = o;
    }
};

template <class LAT, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) k_mcs(LAT lat, Params P, McsArgs a)
{
    constexpr int D = LAT::D, W = LAT::W, NWARPS = NT / 32;
    extern __shared__ __align__(16) uint32_t msm[];
    const int T = P.T, R = 2 * T;
    const McsSmem L(D, W, T, NWARPS);
    uint32_t *sJ = msm + L.oJ, *sS = msm + L.oS, *sThr = msm + L.oThr, *sAcc = msm + L.oAcc, *sLast = msm + L.oLast;
    int *sE = (int *)(msm + L.oE), *sTos = (int *)(msm + L.oTos), *sSot = (int *)(msm + L.oSot);
    unsigned long long *sCum = (unsigned long long *)(msm + L.oCum);
    uint32_t *scratch = msm + L.oScr + (threadIdx.x >> 5) * 4 * W;
    const int s = blockIdx.x, tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const uint32_t g = P.g0 + (uint32_t)s;
    const size_t rep0 = (size_t)s * R;

    for (int i = tid; i < 2 * 2 * D * W; i += NT) sJ[i] = P.d.Jn[(size_t)s * 2 * 2 * D * W + i];
    for (int i = tid; i < R * 2 * W; i += NT) sS[i] = P.d.spin[rep0 * 2 * W + i];
    for (int i = tid; i < R; i += NT) {
        const int t = P.d.tos[rep0 + i];
        sTos[i] = t;
        sSot[i] = P.d.sot[rep0 + i];
        sE[i] = P.d.E[rep0 + i];
        sAcc[i] = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) sThr[4 * i + k] = P.d.thrM[4 * t + k];
    }
    for (int i = tid; i < T; i += NT) { sLast[i] = P.d.last[(size_t)s * T + i]; sCum[i] = 0ull; }
    __syncthreads();

    for (int m = 0; m < a.n_mcs; ++m) {
        // ---- a1-a3: n_metro checkerboard sweeps
        for (int it = 0; it < a.n_metro; ++it) {
            const uint32_t step = a.sweep0 + (uint32_t)m * (uint32_t)a.n_metro + (uint32_t)it;
            for (int p = 0; p < 2; ++p) {
#pragma unroll 1
                for (int item = tid; item < R * W; item += NT) {
                    const int q = item / W, w = item - q * W;
                    const int c = (q >= T) ? 1 : 0, r = q - c * T;
                    uint32_t thr[D];
#pragma unroll
                    for (int k = 0; k < D; ++k) thr[k] = sThr[4 * q + k];
                    const int dE = update_word(lat, sS + (q * 2 + p) * W, sS + (q * 2 + (1 - p)) * W, sJ + p * 2 * D * W, W, w,
                                               p, thr, step, g, make_tag(DOM_METRO, p, c, r), P.rk);
                    if (dE != 0) atomicAdd(sE + q, dE);
                }
                __syncthreads();
            }
        }
        // ---- a5: Houdayer exchange, one warp per temperature
        if (a.do_houdayer) {
            const uint32_t step = a.houd0 + (uint32_t)m;
            for (int t = wid; t < T; t += NWARPS) {
                const int ra = sSot[t], rb = T + sSot[T + t];
                uint32_t u, o1, o2, o3;
                philox4x32_10(0u, step, g, make_tag(DOM_HOUD, 0, 0, t), P.rk, u, o1, o2, o3);
                int delta;
                const int size = houdayer_pair(lat, sS + (ra * 2) * W, sS + (ra * 2 + 1) * W, sS + (rb * 2) * W,
                                               sS + (rb * 2 + 1) * W, sJ, scratch, u, lane, delta);
                if (lane == 0) {
                    sE[ra] += delta;
                    sE[rb] -= delta;
                    sLast[t] = (uint32_t)size;
                    sCum[t] += (unsigned long long)size;
                }
            }
            __syncthreads();
        }
        // ---- a4: PT pass, one warp per chain (R9: sequential walk, each step seeing the previous)
        if (a.do_exchange && T > 1) {
            const uint32_t step = a.exch0 + (uint32_t)m;
            for (int c = wid; c < 2; c += NWARPS) {
                int *so = sSot + c * T;
                const int *Ec = sE + c * T;
                int ea = 0, ra = 0;
                if (lane == 0) { ra = so[0]; ea = Ec[ra]; }
                for (int tb = 0; tb < T - 1; tb += 32) {
                    const int tl = tb + lane;
                    uint32_t u_l = 0, o1, o2, o3;
                    int rb_l = 0, eb_l = 0, sg_l = 0;
                    if (tl < T - 1) {
                        philox4x32_10((uint32_t)tl, step, g, make_tag(DOM_SWAP, 0, c, 0), P.rk, u_l, o1, o2, o3);
                        rb_l = so[tl + 1];              // positions > t are not modified before they are read
                        eb_l = Ec[rb_l];
                        sg_l = P.d.sgn[tl];
                    }
                    __syncwarp();
                    const int nstep = min(32, T - 1 - tb);
                    uint32_t accmask = 0;
                    for (int j = 0; j < nstep; ++j) {
                        const uint32_t u = __shfl_sync(0xFFFFFFFFu, u_l, j);
                        const int rb = __shfl_sync(0xFFFFFFFFu, rb_l, j), eb = __shfl_sync(0xFFFFFFFFu, eb_l, j);
                        const int sg = __shfl_sync(0xFFFFFFFFu, sg_l, j);
                        if (lane == 0) {
                            const int t = tb + j;
                            const int dE = ea - eb;
                            const uint32_t mm = (uint32_t)(dE < 0 ? -dE : dE) >> 2;
                            const bool acc = ((long long)sg * dE <= 0) || (u < thrX_lookup(P, t, mm));
                            if (acc) { so[t] = rb; accmask |= 1u << j; }
                            else     { so[t] = ra; ea = eb; ra = rb; }
                        }
                    }
                    accmask = __shfl_sync(0xFFFFFFFFu, accmask, 0);
                    if (tl < T - 1 && ((accmask >> lane) & 1u)) sAcc[c * T + tl] += 1u;
                }
                if (lane == 0) so[T - 1] = ra;
                __syncwarp();
                for (int t = lane; t < T; t += 32) sTos[c * T + so[t]] = t;
            }
            __syncthreads();
            for (int i = tid; i < R; i += NT) {
                const int t = sTos[i];
#pragma unroll
                for (int k = 0; k < 4; ++k) sThr[4 * i + k] = P.d.thrM[4 * t + k];
            }
            __syncthreads();
        }
    }

    for (int i = tid; i < R * 2 * W; i += NT) P.d.spin[rep0 * 2 * W + i] = sS[i];
    for (int i = tid; i < R; i += NT) {
        P.d.E[rep0 + i] = sE[i];
        P.d.tos[rep0 + i] = sTos[i];
        P.d.sot[rep0 + i] = sSot[i];
    }
    if (T > 1)
        for (int i = tid; i < R; i += NT) {
            const int c = i / T, t = i - c * T;
            if (t < T - 1 && sAcc[i]) P.d.accepts[((size_t)s * 2 + c) * (T - 1) + t] += (unsigned long long)sAcc[i];
        }
    for (int i = tid; i < T; i += NT) {
        P.d.last[(size_t)s * T + i] = sLast[i];
        P.d.cum[(size_t)s * T + i] += sCum[i];
    }
}

}  // namespace ptg
