/*
 * ref_ptglass.h -- CPU ORACLE for the parallel-tempering +-J Edwards-Anderson hot path of
 * arXiv 2003.04621.  TEST INFRASTRUCTURE ONLY.
 *
 * This is a plain, slow, single-threaded C restatement of the method, written from the paper and the
 * readings R1..R26 listed in DESIGN.md.  It shares no code with the CUDA library (own Philox, own lattice
 * code) and is used only by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs.  The product never calls it.
 *
 * Notation:  S samples, T temperatures, C = 2 chains,
 * N = L^d sites, site i = x + L*y (+ L*L*z), colour p(i) = (x+y+z)&1, bond (mu,i) joins i and i+e_mu
 * (periodic) with coupling J[mu][i] in {-1,+1} (Eq. (1)-(2)).
 * A "slot" r is a fixed spin configuration of chain c of sample s; temp_of_slot / slot_of_temp are the two
 * arrays of PAPER.md:169.
 *
 * Every function returns 0 on success, a negative value on a bad argument.
 */
#ifndef REF_PTGLASS_H
#define REF_PTGLASS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ref_ctx ref_ctx;

/* Philox4x32-10 (paper ref. [70]); out[0..3] in the order the round function writes. */
void ref_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4]);

/* THR(x) = min(2^32-1, floor(2^32 * exp(x))), x <= 0, C double exp (reading R5/R6). */
uint32_t ref_threshold(double x);

/* Init (8(c).2): couplings, spins, identity permutations, energies.  NULL on invalid arguments
 * (d not in {2,3}, L odd or < 2, S < 1, T < 1 or > 65535, betas NULL / negative / non-finite). */
ref_ctx *ref_create(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed,
                    uint32_t sample_offset);
/* Same with the bimodal distribution of Eq. (2) for general p = P(J = +1) (NEXT-4, reading R32):
 * J = +1 iff the bond's Philox word w < floor(p * 2^32); p = 1/2 is ref_create exactly.  NULL unless 0 <= p <= 1. */
ref_ctx *ref_create_p(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed,
                      uint32_t sample_offset, double p_ferro);
void ref_destroy(ref_ctx *c);

/* Updates: Metropolis sweeps, PT pass (Eq. (5)),
 * Houdayer cluster exchange (Eq. (10)), MCS in the paper's order. */
int ref_sweep(ref_ctx *c, int n);
int ref_exchange(ref_ctx *c);
int ref_houdayer(ref_ctx *c);
int ref_mcs(ref_ctx *c, int n_mcs, int n_metro, int do_houdayer /* 0 none, 1 single-cluster, 2 multi-cluster */,
            int do_exchange);
/* NEXT-4 cluster-move variants (readings R36, R37).
 * ref_set_cluster_moves: n_clu[t] in [0, 65535] single-cluster moves per ref_houdayer call at temperature index t
 * (move j draws its seed from Philox counter index j; n_clu = NULL restores one move everywhere; 0 switches the move
 * off at that temperature -- the temperature window of ref. [39]).
 * ref_houdayer_multi: every q = -1 component is exchanged with probability 1/2, decided by the Philox bit of its
 * smallest site index; the cluster-size observables then count exchanged sites. */
int ref_set_cluster_moves(ref_ctx *c, const int32_t *n_clu /* [T] or NULL */);
int ref_houdayer_multi(ref_ctx *c);

/* Observables, indexed by TEMPERATURE t. */
int ref_get_energy(const ref_ctx *c, int32_t *E /* [S][2][T] */);
int ref_measure_overlap(const ref_ctx *c, int32_t *Q /* [S][T] */, int32_t *QL /* [S][T] or NULL */);
/* NEXT-2 (reading R31): prof[s][t][mu][x] = sum of q_i over the plane x_mu = x. */
int ref_measure_overlap_profile(const ref_ctx *c, int32_t *prof /* [S][T][d][L] */);
int ref_get_swap_counts(const ref_ctx *c, uint64_t *attempts, uint64_t *accepts /* [S][2][T-1] */);
int ref_get_cluster_sizes(const ref_ctx *c, uint32_t *last, uint64_t *cumulative /* [S][T], may be NULL */);
int ref_get_perm(const ref_ctx *c, int32_t *temp_of_slot, int32_t *slot_of_temp /* [S][2][T] */);

/* Temperature-schedule family of Eq. (6)-(7): T_i = i^phi * T_norm + T_min,
 * T_norm = (T_max - T_min) / (N_T - 1)^phi, in double with C pow(); betas[i] = 1 / T_i.  temps / betas may be NULL. */
int ref_schedule_family(double T_min, double T_max, int n_temps, double phi, double *temps, double *betas);

/* Round trips in temperature space (tunnelling time; readings R27-R29): per slot the number of
 * completed trips index 0 -> index T-1 -> index 0 (slot order); per (sample, chain) the sum and the number of
 * round-trip times (in exchange passes) completed at pass n, binned by floor(log2 n) (logarithmic binning, Fig. 4). */
int ref_get_round_trips(const ref_ctx *c, uint32_t *trips /* [S][2][T] */, uint64_t *tau_sum /* [S][2][32] */,
                        uint64_t *tau_cnt /* [S][2][32] */);

/* State in SLOT order. */
int ref_get_spins(const ref_ctx *c, int8_t *spins /* [S][2][T][N] */);
int ref_get_couplings(const ref_ctx *c, int8_t *J /* [S][d][N] */);
int ref_get_thresholds(const ref_ctx *c, uint32_t *thrM /* [T][d], k = 1..d at [t][k-1] */,
                       uint32_t *thrX /* [T-1][stride], entry m = |dE|/4 */, size_t thrX_stride);
int ref_get_counters(const ref_ctx *c, uint32_t *n_sweep, uint32_t *n_exchange, uint32_t *n_houdayer);
int ref_set_spins(ref_ctx *c, const int8_t *spins);
int ref_set_couplings(ref_ctx *c, const int8_t *J);
/* NEXT-3 (readings R33-R35): couplings as fixed-point numbers J = Jq * 2^-fbits, [S][d][N].
 * -1 if fbits not in [0, 24] or d*N*max|Jq| >= 2^31. */
int ref_set_couplings_fixed(ref_ctx *c, const int32_t *Jq, int fbits);
int ref_get_couplings_fixed(const ref_ctx *c, int32_t *Jq, int *fbits);
int ref_recompute_energy(const ref_ctx *c, int32_t *E_slot_order /* [S][2][T] or NULL */, int *mismatch_count);

#ifdef __cplusplus
}
#endif
#endif
