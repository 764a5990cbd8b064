// a7  Fused Monte Carlo steps: ONE CTA keeps ONE SAMPLE -- the bit-packed spins of all
// its 2T replicas, its couplings, tracked energies, both index maps and the per-slot thresholds -- resident in
// shared memory for n_mcs whole MCS:  [ n_metro sweeps -> Houdayer exchange per temperature -> PT pass ] x n_mcs.
// Samples never interact (P:7), so there is no grid-wide synchronisation; the state is read from and
// written back to global memory once per call.  The sweep is the device function the separate kernel uses
// (update_word); the Houdayer phase runs one LANE per temperature where the lattice allows it
// (houdayer_lanes.cuh), else one warp per temperature (houdayer.cuh); the exchange walk is done by one lane per
// chain.  All of them compute exactly what the separate kernels compute, so the results are bit-identical.
#pragma once
#include "kernels.cuh"
#include "houdayer_lanes.cuh"
#include "houdayer_quad.cuh"
#include "gauss.cuh"

namespace ptg {

struct McsArgs {
    int n_mcs, n_metro, do_houdayer, do_exchange;
    int split_chains;                       // 1: one CTA per (sample, chain) -- only without Houdayer moves (the chains never meet)
    int max_clu;                            // max over t of nclu[t] (R36); 1 in a default run
    uint32_t sweep0, houd0, exch0;          // counter values at the start of the call
    int measure_every;                      // > 0: overlap record after every measure_every-th MCS of the call (whole-sample CTAs only)
    int32_t *recQ, *recQL;                  // device records [n_mcs / measure_every][S][T]; recQL may be null
    int phase_clocks;                       // 1: thread 0 of every CTA sums clock64() per phase into P.d.phaseClk (Eq. (11) split of the fused launch)
    int rec_S, rec_s0;                      // records are [rec][rec_S][T]; this launch holds samples rec_s0 ... (a launch per sample group)
};

// shared-memory carve-up, shared by host (size) and device (pointers); all offsets in 32-bit words.
// A replica occupies RS = 2W + 1 words (colour 0 | colour 1 | pad): the odd stride lets 32 lanes that each own a
// different replica (lane-per-pair Houdayer) hit 32 different banks.
struct McsSmem {
    int RS, oJ, oS, oE, oTos, oSot, oThr, oAcc, oLast, oCum, oU, oSgn, oC2, oPair, oTot, oMeas, oScr, oPh, words;
    // nch: chains held by the CTA (2 = the whole sample, 1 = one chain)
    // extras: the arrays only the fixed-point (GAUSS) and fused-measurement (MEAS) variants use, placed after the scratch so
    // that the plain +-J kernel keeps its layout
    __host__ __device__ McsSmem(int D, int W, int T, int nwarps, bool lanes, int nch, bool extras)
    {
        RS = 2 * W + 1;
        int o = 0;
        oJ = o;    o += 2 * 2 * D * W;
        oS = o;    o += nch * T * RS;
        oE = o;    o += 2 * T;
        oTos = o;  o += 2 * T;
        oSot = o;  o += 2 * T;
        o = (o + 3) & ~3;
        oThr = o;  o += 2 * T * 4;          // 16-byte aligned rows
        oAcc = o;  o += 2 * T;              // accepted swaps of this call per (chain, pair)
        oLast = o; o += T;
        o = (o + 1) & ~1;
        oCum = o;  o += 2 * T;              // 64-bit
        oU = o;    o += 2 * T;              // PT draws of the current pass, [chain][pair]
        oSgn = o;  o += T;
        o = (o + 1) & ~1;
        oPh = o;   o += 10;                 // 64-bit: last time stamp | clocks in sweeps, Houdayer, PT pass, rest
        oScr = o;
        if (nch < 2) {
            // no Houdayer phase, no scratch
        } else if (lanes) {
            const int groups = (T + 31) / 32;
            o += (groups < nwarps ? groups : nwarps) * 2 * (2 * W) * kLaneStride;
        } else {
            o += nwarps * (4 * W + 64);         // kPairScratchWords
        }
        oC2 = oPair = oTot = oMeas = o;
        if (extras) {
            oC2 = o;   o += 2 * T;          // fixed-point couplings: bracket slope per replica (float)
            oPair = o; o += T;              //   E_A + E_B of the pair at temperature t before the cluster moves
            oTot = o;  o += 1;              //   sum of all couplings of the sample
            oMeas = o; o += 2 * T;          // overlap accumulators of a fused measurement: #(q = -1) | #(bonds with q_i != q_j)
        }
        words = o;
    }
};

// a6 inside the fused kernel: overlap record (Eq. (4), link overlap R14) of the pairs now at equal temperature, from
// the resident state: what pt_measure_overlap would return after this MCS.  gather() is a bit permutation, so the
// neighbour bits of q = A ^ B are gather(A) ^ gather(B).  Kept out of line: inlined into the MCS loop it cost the sweep
// loop 9 % on C3 (register allocation), although it runs once per measure_every steps.  Every thread of the CTA calls.
template <class LAT, int NT>
__device__ __noinline__ void mcs_overlap_record(LAT lat, const Params &P, const uint32_t *sS, const int *sSot, int *sQ, int s, size_t rec,
                                                size_t rec_S, int32_t *recQ, int32_t *recQL)
{
    constexpr int D = LAT::D, W = LAT::W, RS = 2 * W + 1;
    const int T = P.T, tid = threadIdx.x;
    int *sQL = sQ + T;
    for (int i = tid; i < 2 * T; i += NT) sQ[i] = 0;
    __syncthreads();
#pragma unroll 1
    for (int item = tid; item < T * W; item += NT) {
        const int t = item / W, w = item - t * W;
        const uint32_t *A0 = sS + sSot[t] * RS, *B0 = sS + (T + sSot[T + t]) * RS;
        const uint32_t nbk = A0[w] ^ B0[w];
        atomicAdd(sQ + t, __popc(nbk) + __popc(A0[W + w] ^ B0[W + w]));
        if (recQL) {
            uint32_t nbA[2 * D], nbB[2 * D];
            lat.gather(A0 + W, w, 0, nbA);
            lat.gather(B0 + W, w, 0, nbB);
            int nd = 0;
#pragma unroll
            for (int k = 0; k < 2 * D; ++k) nd += __popc(nbk ^ nbA[k] ^ nbB[k]);
            atomicAdd(sQL + t, nd);
        }
    }
    __syncthreads();
    for (int t = tid; t < T; t += NT) {
        recQ[(rec * rec_S + s) * T + t] = P.N - 2 * sQ[t];
        if (recQL) recQL[(rec * rec_S + s) * T + t] = P.D * P.N - 2 * sQL[t];
    }
}

// Phase clocks (Eq. (11) P:189 asks for the time per spin of each update; inside ONE fused launch CUDA events cannot
// separate them): thread 0 adds the SM clocks since the last stamp to phase `k`.  Called right after a CTA barrier.
__device__ __forceinline__ void phase_stamp(unsigned long long *sPh, int k)
{
    const unsigned long long now = (unsigned long long)clock64();
    sPh[1 + k] += now - sPh[0];
    sPh[0] = now;
}

// GAUSS: 0 = +-J bit couplings; 1 / 2 = fixed-point couplings (gauss.cuh) with / without the host's range guarantee
// 2 D max|Jq| < 2^23.  With fixed-point couplings the sweep walks its word site by site (update_word_q), the energies are
// recomputed from scratch after the cluster moves (field_sum_word_q; the cluster itself depends on q only) and the PT walk
// evaluates its thresholds in double (swap_threshold).
// MEAS: overlap records after every a.measure_every-th MCS from the resident state (pt_mcs_measure_device).
// MULTI: the cluster phase is the multi-cluster exchange (R37; a.do_houdayer == 2) on the four-lane strips -- a separate
// instantiation (2D L = 32 only), so that the kernel of the paper's MCS keeps its code.
template <class LAT, int NT, int MINB, int GAUSS, bool MEAS, bool MULTI = false>
__global__ void __launch_bounds__(NT, MINB) k_mcs(LAT lat, Params P, McsArgs a)
{
    constexpr int D = LAT::D, W = LAT::W, NWARPS = NT / 32;
    constexpr bool LANES = LaneHoudayer<LAT>::kEligible;
    extern __shared__ __align__(16) uint32_t msm[];
    const int T = P.T;
    const int NCH = a.split_chains ? 1 : 2;         // chains in this CTA
    const int R = NCH * T;                          // replicas in this CTA
    const McsSmem L(D, W, T, NWARPS, LANES, NCH, GAUSS != 0 || MEAS);
    constexpr int RS = 2 * W + 1;
    uint32_t *sJ = msm + L.oJ, *sS = msm + L.oS, *sThr = msm + L.oThr, *sAcc = msm + L.oAcc, *sLast = msm + L.oLast;
    uint32_t *sU = msm + L.oU;
    float *sC2 = (float *)(msm + L.oC2);
    int *sPair = (int *)(msm + L.oPair), *sTot = (int *)(msm + L.oTot);
    int *sE = (int *)(msm + L.oE), *sTos = (int *)(msm + L.oTos), *sSot = (int *)(msm + L.oSot), *sSgn = (int *)(msm + L.oSgn);
    unsigned long long *sCum = (unsigned long long *)(msm + L.oCum);
    unsigned long long *sPh = (unsigned long long *)(msm + L.oPh);
    const bool clk = a.phase_clocks && threadIdx.x == 0;
    if (clk) { sPh[0] = (unsigned long long)clock64(); sPh[1] = sPh[2] = sPh[3] = sPh[4] = 0ull; }
    const int s = a.split_chains ? (int)(blockIdx.x >> 1) : (int)blockIdx.x;
    const int c0 = a.split_chains ? (int)(blockIdx.x & 1) : 0;      // first chain of this CTA
    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    const uint32_t g = P.g0 + (uint32_t)s;
    const size_t rep0 = ((size_t)s * 2 + c0) * T;

    for (int i = tid; i < 2 * 2 * D * W; i += NT) sJ[i] = P.d.Jn[(size_t)s * 2 * 2 * D * W + i];
    for (int i = tid; i < R * 2 * W; i += NT) {
        const int q = i / (2 * W), j = i - q * (2 * W);
        sS[q * RS + j] = P.d.spin[rep0 * 2 * W + i];
    }
    for (int i = tid; i < R; i += NT) {
        const int t = P.d.tos[rep0 + i];
        sTos[i] = t;
        sSot[i] = P.d.sot[rep0 + i];
        sE[i] = P.d.E[rep0 + i];
        sAcc[i] = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) sThr[4 * i + k] = P.d.thrM[4 * t + k];
        if constexpr (GAUSS != 0) sC2[i] = bracket_slope(P.d.betasD[t], P.fbits);
    }
    if constexpr (GAUSS != 0) {
        if (tid == 0) *sTot = 0;
        __syncthreads();
        if (a.do_houdayer && NCH == 2) {
            int part = 0;
            for (int w = tid; w < W; w += NT) part += bond_sum_word_q(lat, P.d.Jdev + (size_t)s * 2 * (2 * D) * (32 * W), W, w);
            if (part != 0) atomicAdd(sTot, part);
        }
    }
    for (int i = tid; i < T; i += NT) {
        sLast[i] = P.d.last[(size_t)s * T + i];
        sCum[i] = 0ull;
        sSgn[i] = (i < T - 1) ? P.d.sgn[i] : 0;
    }
    __syncthreads();

    if (clk) phase_stamp(sPh, 3);
    for (int m = 0; m < a.n_mcs; ++m) {
        // ---- a1-a3: n_metro checkerboard sweeps
#pragma unroll 1
        for (int it = 0; it < a.n_metro; ++it) {
            const uint32_t step = a.sweep0 + (uint32_t)m * (uint32_t)a.n_metro + (uint32_t)it;
#pragma unroll 1
            for (int p = 0; p < 2; ++p) {
#pragma unroll 1
                for (int item = tid; item < R * W; item += NT) {
                    const int q = item / W, w = item - q * W;
                    const int cl = (q >= T) ? 1 : 0, r = q - cl * T, c = c0 + cl;
                    int dE;
                    if constexpr (GAUSS != 0) {
                        dE = update_word_q<LAT, GAUSS == 1>(lat, sS + q * RS + p * W, sS + q * RS + (1 - p) * W,
                                                            P.d.Jdev + ((size_t)s * 2 + p) * (2 * D) * (32 * W), W, w, p, sC2[q],
                                                            P.d.betasD + sTos[q], P.fbits, step, g, make_tag(DOM_METRO, p, c, r), P.rk);
                    } else {
                        uint32_t thr[D];
#pragma unroll
                        for (int k = 0; k < D; ++k) thr[k] = sThr[4 * q + k];
                        dE = update_word(lat, sS + q * RS + p * W, sS + q * RS + (1 - p) * W, sJ + p * 2 * D * W, W, w,
                                         p, thr, step, g, make_tag(DOM_METRO, p, c, r), P.rk);
                    }
                    atomicAdd(sE + q, dE);
                }
                __syncthreads();
            }
        }
        if (clk) phase_stamp(sPh, 0);
        // ---- a5: Houdayer exchange
        if (a.do_houdayer && NCH == 2) {
            const uint32_t step = a.houd0 + (uint32_t)m;
            if constexpr (GAUSS != 0) {
                for (int t = tid; t < T; t += NT) sPair[t] = sE[sSot[t]] + sE[T + sSot[T + t]];
                __syncthreads();
            }
            if constexpr (MULTI && QuadHoudayer<LAT>::kEligible && NT == 128) {
                // multi-cluster exchange, four lanes per temperature (houdayer_multi_quad); R36's move counts do not apply
                uint32_t *cc = msm + L.oScr + (tid >> 2) * QuadHoudayer<LAT>::kPairStride;
                for (int t0 = 0; t0 < T; t0 += 32) {
                    const int t = t0 + (tid >> 2);
                    const bool active = t < T;
                    const int ra = active ? sSot[t] : 0, rb = active ? T + sSot[T + t] : T;
                    int delta;
                    const int size = houdayer_multi_quad(lat, sS + ra * RS, sS + ra * RS + W, sS + rb * RS, sS + rb * RS + W, sJ, cc,
                                                         step, g, active ? t : 0, P.rk, active, lane, delta);
                    if (active && (tid & 3) == 0) {
                        sE[ra] += delta;
                        sE[rb] -= delta;
                        sLast[t] = (uint32_t)size;
                        sCum[t] += (unsigned long long)size;
                    }
                }
            } else if constexpr (QuadHoudayer<LAT>::kEligible && NT == 128) {
                // FOUR lanes per temperature, all warps of the CTA at work: 32 temperatures at a time (houdayer_quad.cuh)
                uint32_t *cc = msm + L.oScr + (tid >> 2) * QuadHoudayer<LAT>::kPairStride;
                for (int t0 = 0; t0 < T; t0 += 32) {
                    const int t = t0 + (tid >> 2);
                    const int moves = (t < T) ? P.d.nclu[t] : 0;                // R36; 1 everywhere in a default run
                    if (t < T && moves == 0 && (tid & 3) == 0) sLast[t] = 0u;
                    for (int mv = 0; mv < a.max_clu; ++mv) {
                        const bool active = mv < moves;
                        int ra = 0, rb = T;
                        uint32_t u = 0, o1, o2, o3;
                        if (active) {
                            ra = sSot[t];
                            rb = T + sSot[T + t];
                            philox4x32_10((uint32_t)mv, step, g, make_tag(DOM_HOUD, 0, 0, t), P.rk, u, o1, o2, o3);
                        }
                        int delta;
                        const int size = houdayer_quad(lat, sS + ra * RS, sS + ra * RS + W, sS + rb * RS, sS + rb * RS + W, sJ, cc, u,
                                                       active, lane, delta);
                        if (active && (tid & 3) == 0) {
                            sE[ra] += delta;
                            sE[rb] -= delta;
                            sLast[t] = (uint32_t)size;
                            sCum[t] += (unsigned long long)size;
                        }
                    }
                }
            } else if constexpr (LANES) {
                // one LANE per temperature: warp k takes temperatures [32k, 32k+32), then strides by the warps in use
                const int groups = (T + 31) / 32, hw = groups < NWARPS ? groups : NWARPS;
                if (wid < hw) {
                    uint32_t *col = msm + L.oScr + wid * LaneHoudayer<LAT>::kScratchWords + lane;
                    for (int t0 = wid * 32; t0 < T; t0 += hw * 32) {
                        const int t = t0 + lane;
                        const int moves = (t < T) ? P.d.nclu[t] : 0;            // R36; 1 everywhere in a default run
                        if (t < T && moves == 0) sLast[t] = 0u;
                        for (int mv = 0; mv < a.max_clu; ++mv) {
                            const bool active = mv < moves;
                            int ra = 0, rb = T;
                            uint32_t u = 0, o1, o2, o3;
                            if (active) {
                                ra = sSot[t];
                                rb = T + sSot[T + t];
                                philox4x32_10((uint32_t)mv, step, g, make_tag(DOM_HOUD, 0, 0, t), P.rk, u, o1, o2, o3);
                            }
                            int delta;
                            const int size = houdayer_lane(lat, sS + ra * RS, sS + ra * RS + W, sS + rb * RS, sS + rb * RS + W,
                                                           sJ, col, u, active, delta);
                            if (active) {
                                sE[ra] += delta;
                                sE[rb] -= delta;
                                sLast[t] = (uint32_t)size;
                                sCum[t] += (unsigned long long)size;
                            }
                        }
                    }
                }
            } else {
                // one WARP per temperature
                uint32_t *scratch = msm + L.oScr + wid * kPairScratchWords<LAT>;
                for (int t = wid; t < T; t += NWARPS) {
                    const int ra = sSot[t], rb = T + sSot[T + t];
                    const int moves = P.d.nclu[t];                              // R36
                    if (moves == 0 && lane == 0) sLast[t] = 0u;
                    for (int mv = 0; mv < moves; ++mv) {
                        uint32_t u, o1, o2, o3;
                        philox4x32_10((uint32_t)mv, step, g, make_tag(DOM_HOUD, 0, 0, t), P.rk, u, o1, o2, o3);
                        int delta;
                        const int size = houdayer_warp(lat, sS + ra * RS, sS + ra * RS + W, sS + rb * RS, sS + rb * RS + W, sJ,
                                                       scratch, u, lane, delta);
                        if (lane == 0) {
                            sE[ra] += delta;
                            sE[rb] -= delta;
                            sLast[t] = (uint32_t)size;
                            sCum[t] += (unsigned long long)size;
                        }
                        __syncwarp();
                    }
                }
            }
            __syncthreads();
            if constexpr (GAUSS != 0) {
                // the cluster phase counted +-1 bonds: recompute the energies of chain 0 from the couplings' values
                // (E = -sum J + 2 sum_unsatisfied J, every bond seen from its black endpoint); the move conserves
                // E_A + E_B of a pair exactly, which gives chain 1
                for (int i = tid; i < T; i += NT) sE[i] = -*sTot;
                __syncthreads();
                const int32_t *Jb = P.d.Jdev + (size_t)s * 2 * (2 * D) * (32 * W);          // colour-0 block
#pragma unroll 1
                for (int item = tid; item < T * W; item += NT) {
                    const int q = item / W, w = item - q * W;
                    const int lost = unsat_sum_word_q(lat, sS + q * RS, sS + q * RS + W, Jb, W, w);
                    if (lost != 0) atomicAdd(sE + q, -2 * lost);
                }
                __syncthreads();
                for (int t = tid; t < T; t += NT) sE[T + sSot[T + t]] = sPair[t] - sE[sSot[t]];
                __syncthreads();
            }
        }
        if (clk) phase_stamp(sPh, 1);
        // ---- a4: PT pass (R9: sequential walk, each step seeing the previous).  Warp 0: all lanes draw the Philox
        // words, then one lane per chain walks its ladder; only the two index maps change.
        // Measured and rejected on B200: a decision table over all (carried, rung) pairs built
        // by the whole CTA (2.6 K instructions per sample and MCS against 1.6 K for this walk; C2 929 against 961 flips/ns),
        // the rungs' own-resident decisions evaluated side by side with a warp per chain (939), and a banded table with a
        // speculative accept-bit walk and a parallel rebuild of the map (PT phase 12.4 -> 9.5 us of CTA time, but C2 952,
        // C3 977 against 1011): the walk costs ~500 cycles per rung whatever its instruction count.  Last, the pass as a SCAN
        // (a rung = a map on the number of rungs the arriving replica was carried, composed over the ladder in 5 shuffle
        // steps, the map rebuilt in parallel from the accept mask): PT phase 12.4 -> 7.8 us of CTA time, bit-exact, and C2 969,
        // C3 1005, C4 1153 against 959 / 1011 / 1152 -- the phase is no longer what limits the kernel, so the walk stays.
        // Round 3: the threshold of rung t + 1 fetched one rung ahead for both replicas that can arrive there (two independent
        // loads in flight, selected by the decision at t): bit-exact, and SLOWER -- C2 943 / C3 918 / C4 1133 against 958 / 950 /
        // 1151 flips/ns (same box, three alternating runs, plain pt_mcs): twice the loads and six more live registers on the
        // one lane that walks cost more than the shorter dependency chain returns.
        if (a.do_exchange && T > 1) {
            const uint32_t step = a.exch0 + (uint32_t)m;
            if (wid == 0) {
                for (int i = lane; i < NCH * (T - 1); i += 32) {
                    const int c = i / (T - 1), t = i - c * (T - 1);        // c: chain index within the CTA
                    uint32_t u, o1, o2, o3;
                    philox4x32_10((uint32_t)t, step, g, make_tag(DOM_SWAP, 0, c0 + c, 0), P.rk, u, o1, o2, o3);
                    sU[c * T + t] = u;
                }
                __syncwarp();
                if (lane < NCH) {
                    const int c = lane;
                    int *so = sSot + c * T;
                    const int *Ec = sE + c * T;
                    int ra = so[0], ea = Ec[ra];
                    int rb = so[1], eb = Ec[rb];
                    const uint32_t *Uc = sU + c * T;
                    uint32_t *Ac = sAcc + c * T;
                    const uint32_t *trow = P.d.thrX;                            // row of rung t of the +-J swap table
#pragma unroll 1
                    for (int t = 0; t < T - 1; ++t, trow += P.strideX) {
                        const int tn = min(t + 2, T - 1);                       // positions > t are not modified before they are read
                        const int rbn = so[tn], ebn = Ec[rbn];
                        const int dE = ea - eb;
                        bool acc = sSgn[t] * dE <= 0;
                        if constexpr (GAUSS != 0) {
                            if (!acc) acc = swap_accept(P, t, Uc[t], (uint32_t)(dE < 0 ? -dE : dE));
                        } else {                                                // branch-free: the lookup is issued for every rung
                            const uint32_t mm = (uint32_t)(dE < 0 ? -dE : dE) >> 2;
                            const uint32_t thr = __ldg(trow + min(mm, P.strideX - 1u));
                            acc = acc || (mm < P.strideX && Uc[t] < thr);
                        }
                        so[t] = acc ? rb : ra;                                  // position t is final; on accept (ea, ra) moves up
                        Ac[t] += acc ? 1u : 0u;
                        ea = acc ? ea : eb;
                        ra = acc ? ra : rb;
                        rb = rbn; eb = ebn;
                    }
                    so[T - 1] = ra;
                    if (P.track) round_trip_update(P, (size_t)s * 2 + c0 + c, so[0], ra, step + 1u);
                }
                __syncwarp();
                for (int i = lane; i < R; i += 32) {
                    const int c = i / T, t = i - c * T;
                    sTos[c * T + sSot[i]] = t;
                }
            }
            __syncthreads();
            for (int i = tid; i < R; i += NT) {
                if constexpr (GAUSS != 0) sC2[i] = bracket_slope(P.d.betasD[sTos[i]], P.fbits);
                else *(uint4 *)(sThr + 4 * i) = __ldg((const uint4 *)(P.d.thrM + 4 * sTos[i]));
            }
            __syncthreads();
        }
        if (clk) phase_stamp(sPh, 2);
        // ---- a6: overlap record (Eq. (4), link overlap R14) of the pairs now at equal temperature, from the resident
        // state: what pt_measure_overlap would return after this MCS.  gather() is a bit permutation, so the neighbour
        // bits of q = A ^ B are gather(A) ^ gather(B).
        if constexpr (MEAS)
            if (a.measure_every > 0 && NCH == 2 && (m + 1) % a.measure_every == 0)
                mcs_overlap_record<LAT, NT>(lat, P, sS, sSot, (int *)(msm + L.oMeas), a.rec_s0 + s, (size_t)((m + 1) / a.measure_every - 1),
                                            (size_t)a.rec_S, a.recQ, a.recQL);
        if (clk) phase_stamp(sPh, 3);
    }

    for (int i = tid; i < R * 2 * W; i += NT) {
        const int q = i / (2 * W), j = i - q * (2 * W);
        P.d.spin[rep0 * 2 * W + i] = sS[q * RS + j];
    }
    for (int i = tid; i < R; i += NT) {
        P.d.E[rep0 + i] = sE[i];
        P.d.tos[rep0 + i] = sTos[i];
        P.d.sot[rep0 + i] = sSot[i];
    }
    if (T > 1)
        for (int i = tid; i < R; i += NT) {
            const int c = i / T, t = i - c * T;
            if (t < T - 1 && sAcc[i]) P.d.accepts[((size_t)s * 2 + c0 + c) * (T - 1) + t] += (unsigned long long)sAcc[i];
        }
    if (NCH == 2)
        for (int i = tid; i < T; i += NT) {
            P.d.last[(size_t)s * T + i] = sLast[i];
            P.d.cum[(size_t)s * T + i] += sCum[i];
        }
    if (clk) {
        phase_stamp(sPh, 3);
        for (int k = 0; k < 4; ++k) atomicAdd(P.d.phaseClk + k, sPh[1 + k]);
    }
}

}  // namespace ptg
