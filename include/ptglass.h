/*
 * ptglass.h -- C ABI of the B200-native parallel-tempering Monte Carlo library for Edwards-Anderson +-J Ising
 * spin glasses: the data-parallel hot path of arXiv 2003.04621 (Kumar, Gross, Janke, Weigel).
 *
 * "P:n" cites line n of the paper text; "Rk" a reading listed in DESIGN.md section 3.
 *
 * MODEL (Eq. (1)-(2)): H = -sum_<ij> J_ij s_i s_j, s_i = +-1, J_ij = +-1 with p = 1/2, zero field,
 * d-dimensional (d = 2 square, d = 3 simple cubic) periodic lattice of linear size L (even, R3), N = L^d sites,
 * site index i = x + L*y (+ L*L*z), colour p(i) = (x+y+z)&1, bond (mu,i) joins i and i+e_mu.
 * ENSEMBLE: S disorder samples x T temperatures x C = 2 replica chains.  A "slot" r in [0,T) is a
 * fixed spin configuration of chain c of sample s; its current temperature index is temp_of_slot[s][c][r], the
 * inverse map is slot_of_temp[s][c][t] (the "two arrays" of P:169).
 * RANDOM NUMBERS (R11): Philox4x32-10, key = seed, counter = (index, step, global sample, tag); every
 * result is a pure function of (L, d, S, T, betas, seed, sample_offset, sequence of calls), independent of how
 * the work is mapped to threads, CTAs or GPUs.
 *
 * CONVENTIONS
 *  - Every call returns 0 (PT_OK) or a negative PT_ERR_* code; nothing throws or aborts.  pt_last_error()
 *    returns a static NUL-terminated message describing the last failing call.
 *  - One process-global simulation context (the calls carry no handle).  Calling an update / observable before
 *    pt_init or after pt_free returns PT_ERR_STATE.
 *  - DEVICE MEMORY IS CALLER-OWNED: the caller (PyTorch) allocates one workspace of pt_workspace_bytes() bytes,
 *    256-byte aligned, and passes its raw device pointer and a cudaStream_t to pt_bind(); the library never
 *    allocates or frees device memory.  Work is queued on that stream, with one exception: where pt_mcs or
 *    pt_set_spins_async cut the samples into groups (pt_set_sample_groups), groups 1.. run on up to 7 library-owned
 *    non-blocking side streams, created on first use and kept until the process exits.  They start after everything queued
 *    on the bound stream so far and the bound stream waits for them before the call returns (after pt_set_spins_async: at
 *    the next call that touches the state), so to the caller every call is still ordered on the bound stream; pt_bind,
 *    pt_init and pt_free synchronise them.
 *  - All `const T *` inputs are HOST pointers, caller-owned, copied during the call.  All output pointers are
 *    HOST buffers, caller-allocated with the documented shape (C order), filled after a stream synchronise.
 *    The *_device variants take DEVICE pointers instead and do not synchronise.
 *  - There is no CPU fallback: without a CUDA device every compute call returns PT_ERR_CUDA.
 */
#ifndef PTGLASS_H
#define PTGLASS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PT_OK            0
#define PT_ERR_ARG      -1   /* invalid argument (see each call) */
#define PT_ERR_STATE    -2   /* not bound / not initialised / workspace too small */
#define PT_ERR_OVERFLOW -3   /* a uint32 step counter would pass 2^32-1 (R21); state unchanged */
#define PT_ERR_CUDA     -4   /* CUDA runtime failure; message carries cudaGetErrorString */

/* ---- sizes & binding ------------------------------------------------------------------------------------ */

/* Bytes of device workspace needed for a problem of this shape (includes a bounded int8 staging area, 16 MiB or one sample's state if that is more, for the
 * state get/set calls and the init draws).  PT_ERR_ARG for shapes pt_init would reject. */
int pt_workspace_bytes(int L, int d, int n_samples, int n_temps, size_t *bytes_out);
/* The same with optional parts (flags OR-ed):
 *  PT_WS_FIXED_COUPLINGS  the int32 coupling arrays of the fixed-point (Gaussian) model, 24 bytes per bond (NEXT-3), which
 *                         pt_set_couplings_fixed needs (PT_ERR_STATE without them);
 *  PT_WS_FULL_STAGING     a staging area of the whole int8 state (S*2*T*N bytes) instead of the bounded 16 MiB through
 *                         which the int8 get / set calls otherwise pass in chunks of samples: pt_set_spins_async can then
 *                         copy a whole sample group at a time.
 * pt_workspace_bytes_ex only SIZES the workspace; tell pt_init which parts it was sized for with pt_set_workspace_flags
 * (same flags; after pt_bind, before pt_init; pt_bind resets them to 0).  pt_init never guesses from spare bytes: it lays
 * out the int32 couplings iff PT_WS_FIXED_COUPLINGS is set, returns PT_ERR_STATE if the bound workspace is too small for
 * the parts asked for, and gives every byte bound beyond the minimum to the staging area (up to one whole int8 state).
 * pt_get_stage_bytes: the size the staging area ended up with (after pt_init). */
#define PT_WS_FIXED_COUPLINGS 1
#define PT_WS_FULL_STAGING    2
int pt_workspace_bytes_ex(int L, int d, int n_samples, int n_temps, int flags, size_t *bytes_out);
int pt_set_workspace_flags(int flags);
int pt_get_stage_bytes(size_t *bytes);

/* Bind the caller's device workspace (device pointer, >= pt_workspace_bytes, 256-byte aligned) and CUDA stream
 * (a cudaStream_t passed as void*; NULL = default stream).  Must precede pt_init.  Re-binding frees the context. */
int pt_bind(void *device_workspace, size_t bytes, void *cuda_stream);

/* ---- life cycle ----------------------------------------------------------------------------------------- */

/* Initialise: couplings J[s][mu][i] and spins from Philox (domains 1, 2), identity permutations,
 * energies E = -sum J s s (Eq. (1)), zero counters; acceptance tables computed HERE ON THE HOST in double
 * (R5, R6):  thrM[t][k] = THR(-(betas[t]*4k)), k = 1..d;  thrX[t][m] = THR(-(|betas[t+1]-betas[t]|*4m));
 * THR(x) = min(2^32-1, floor(2^32 exp(x))).
 * betas: HOST array [n_temps], any order, duplicates allowed (R7); index t = position in this array.
 * PT_ERR_ARG: d not in {2,3}; L < 2 or odd (checkerboard needs a bipartite periodic lattice, R3); n_samples < 1 or
 * > 65535 per context (larger sets: several shards through pt_init_shard); n_temps < 1 or > 65535; betas NULL, negative
 * or non-finite; N*d > 2^31-1; a lattice whose coupling bits (4 d N / 8 bytes per sample) plus one replica exceed the
 * 227 KiB of shared memory of a CTA (2D: L > 608, 3D: L > 64); sample_offset+n_samples > 2^32.
 * PT_ERR_STATE: no workspace bound or workspace too small. */
int pt_init(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed);
/* Same, for a shard holding global samples [sample_offset, sample_offset + n_samples) (multi-GPU). */
int pt_init_shard(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed,
                  uint32_t sample_offset);
int pt_free(void);
/* NEXT-4: the bimodal distribution of Eq. (2) for general p = P(J = +1) (R32).  J[s][mu][i] = +1
 * iff the bond's Philox word (domain 1) w < floor(p * 2^32); the default p = 1/2 is the sign-bit rule above, bit for bit.
 * Call after pt_bind and BEFORE pt_init (PT_ERR_STATE otherwise); PT_ERR_ARG unless 0 <= p <= 1. */
int pt_set_coupling_probability(double p_ferro);

/* ---- updates -------------------------------------------------------------------------------- */

/* n >= 0 checkerboard Metropolis sweeps of every replica (R1, R2, R4): for colour p = 0 then 1, for
 * every site i of colour p: a = s_i * sum_{2d nbrs} J s_j; flip iff a <= 0 or u < thrM[temp][a/2], u = the
 * site's Philox word (domain 3: index i>>3, step = sweep number, tag (p, chain, slot), word (i>>1)&3).
 * E[slot] is updated by 2a per accepted flip.  Asynchronous on the bound stream. */
int pt_sweep(int n);

/* One parallel-tempering pass (Eq. (5); R9, R10): for every (sample, chain), for t = 0..T-2 in
 * order, each step seeing the previous: dE = E[slot_of_temp[t]] - E[slot_of_temp[t+1]]; accept iff
 * sgn(beta[t+1]-beta[t])*dE <= 0 or u < thrX[t][|dE|/4]; on accept swap the entries of both maps.  Spins and
 * E[slot] are untouched (only temperatures are exchanged). */
int pt_exchange(void);

/* One Houdayer cluster exchange per (sample, temperature) (Eq. (10); R12, R13): the two slots at
 * temperature t (one per chain); q_i = s1_i s2_i; the k-th q = -1 site in index order, k = (u*n_neg)>>32; its
 * connected component among q = -1 sites is negated in both configurations; E1 += delta, E2 -= delta. */
int houdayer_step(void);

/* Cluster-move variants the paper proposes against idle threads and for three dimensions (P:140,
 * ref. [39]), readings R36, R37.
 *
 * pt_set_cluster_moves: n_clu[t] in [0, 65535] single-cluster moves per houdayer_step (and per MCS of pt_mcs with
 * do_houdayer = 1) at temperature index t -- "several cluster updates in the high-temperature copies"; 0 switches the
 * move off at that temperature (a temperature window).  n_clu: host array [T], copied; NULL restores one move
 * everywhere (the state after pt_init).  Move j at a temperature draws its seed from the domain-5 Philox block with
 * counter index j, so the default (all ones) is bit-identical to the plain move.  last = size of the last move (0 where
 * n_clu[t] = 0), cumulative adds every move.  PT_ERR_ARG on a count outside the range; call after pt_init.
 *
 * houdayer_multi_step: the multi-cluster variant -- EVERY connected component of q = -1 sites is exchanged with
 * probability 1/2: the component whose smallest site index is i_min is exchanged iff the top bit of word (i_min & 3) of
 * the Philox block ctr = (i_min >> 2, step, g, tag(5, aux 1, 0, t)) is set.  E1 + E2 is conserved for any such union
 * (P:138).  last / cumulative count exchanged sites; the Houdayer step counter advances by one.  Components are found by
 * label propagation in shared memory, one CTA per (sample, temperature): PT_ERR_ARG if 6 N bytes of labels and site list do not
 * fit (N <= ~36000 sites: up to 2D L = 128, 3D L = 32).  In pt_mcs it is do_houdayer = 2: inside the fused launch on the 2D
 * L = 32 lattice with +-J couplings (components by a tournament on bit maps), separate kernels on every other lattice. */
int pt_set_cluster_moves(const int32_t *n_clu);
int houdayer_multi_step(void);

/* Fused Monte Carlo steps in the paper's order (R15): n_mcs x [ pt_sweep(n_metro);
 * houdayer_step() if do_houdayer = 1, houdayer_multi_step() if do_houdayer = 2; pt_exchange() if do_exchange ].
 * Bit-identical to the separate calls.  PT_ERR_ARG if do_houdayer is not 0, 1 or 2.
 * Where a sample's whole state fits in shared memory this is ONE kernel launch that keeps each
 * sample resident in one CTA for all n_mcs steps; otherwise it issues the separate kernels in order. */
int pt_mcs(int n_mcs, int n_metro, int do_houdayer, int do_exchange);
/* pt_mcs with the two-replica measurement of Eq. (4) fused in: n_mcs steps as pt_mcs, and after every measure_every-th
 * step of the call the overlaps Q and (if QL_rec_dev is not NULL) link overlaps QL of all (sample, temperature) pairs are
 * written to record r = 0, 1, ... of the DEVICE buffers Q_rec_dev / QL_rec_dev, [n_mcs / measure_every][S][T] int32 each,
 * caller-owned -- exactly what pt_mcs(measure_every, ...) followed by pt_measure_overlap_device(record r) would leave
 * there (BASELINE config 3: "overlap q and link overlap measured every 10 sweeps").  Where a CTA of the fused kernel
 * holds both chains of a sample the whole call is ONE launch and the records come from the resident state; otherwise the
 * library issues those calls.  PT_ERR_ARG: measure_every < 1, Q_rec_dev NULL, negative counts, bad do_houdayer. */
int pt_mcs_measure_device(int n_mcs, int n_metro, int do_houdayer, int do_exchange, int measure_every, int32_t *Q_rec_dev,
                          int32_t *QL_rec_dev);
/* mode -1 (default): pt_mcs uses the fused kernel where eligible; 0: always the separate kernels (tests, profiling).
 * pt_get_fused: 1 if pt_mcs of the bound problem runs fused. */
int pt_set_fused(int mode);
int pt_get_fused(int *fused);

/* ---- NEXT-1: temperature-schedule family and tunnelling times --------------------------------- */

/* Temperature-schedule family of Eq. (6)-(7) (R30): T_i = i^phi * T_norm + T_min with
 * T_norm = (T_max - T_min) / (n_temps - 1)^phi, in double with pow(); betas_out[i] = 1 / T_i.  Index 0 is T_min (the
 * paper's numbering T_0 < T_1 < ...); phi = 1 is the linear ladder.  HOST arrays [n_temps], either may be NULL.
 * Pure host function: needs no device and no context.  PT_ERR_ARG unless 0 < T_min <= T_max < inf, n_temps >= 1,
 * 0 < phi < inf.  Pass betas_out to pt_init like any ladder. */
int pt_schedule_family(double T_min, double T_max, int n_temps, double phi, double *temps_out, double *betas_out);

/* Round trips in temperature space, the paper's tunnelling time tau_tunnel (R27-R29): "the expected time
 * it takes for a replica to move from the lowest to the highest temperature and back".  When tracking is on, after
 * every PT pass n (1-based count of passes since pt_init) of every (sample, chain): the slot now at index T-1 is
 * marked as having reached the far end; the slot now at index 0 completes a round trip if it was so marked since its
 * trip began (tau = n - start; start <- n), or begins its first trip.  The slot that starts at index 0 begins at
 * pass 0.  pt_set_round_trip_tracking must be called after pt_bind and BEFORE pt_init (PT_ERR_STATE otherwise);
 * default off.  pt_get_round_trips: trips[S][2][T] completed trips per SLOT; tau_sum / tau_cnt [S][2][32]: sum and
 * number of the round-trip times completed at pass n, in bin floor(log2 n) (logarithmic binning, Fig. 4); any pointer
 * may be NULL; PT_ERR_STATE if tracking is off.  Time is counted in PT passes (= MCS in pt_mcs). */
int pt_set_round_trip_tracking(int on);
int pt_get_round_trips(uint32_t *trips, uint64_t *tau_sum, uint64_t *tau_cnt);

/* ---- observables: all integer, indexed by TEMPERATURE index t ------------------------------------------- */

int pt_get_energy(int32_t *E /* [S][2][T]: E of the configuration currently at temperature t (Eq. (3) x N) */);
/* Q = sum_i s1_i s2_i (Eq. (4) x N), QL = sum_{mu,i} q_i q_{i+e_mu} (R14); [S][T] each; QL may be NULL.
 * Consumes no random numbers and advances no counter (R26). */
int pt_measure_overlap(int32_t *Q, int32_t *QL);
/* NEXT-2 ("the modes for the correlation length"; R31): overlap profiles
 * prof[s][t][mu][x] = sum of q_i = s1_i s2_i over the lattice plane x_mu = x, for the two configurations at temperature
 * t; shape [S][T][d][L], int32.  Every axis sums to Q.  The Fourier modes of the overlap field with wave vector along
 * an axis, q(k e_mu) = sum_x prof[mu][x] exp(i k x) (k = 2 pi / L for the second-moment correlation length), are a
 * length-L transform left to the caller; chi_SG = <Q^2>/N from pt_measure_overlap.  Integer only; consumes no random
 * numbers, advances no counter.  The _device variant takes a DEVICE pointer and does not synchronise. */
int pt_measure_overlap_profile(int32_t *prof);
int pt_measure_overlap_profile_device(int32_t *prof_dev);
int pt_get_swap_counts(uint64_t *attempts, uint64_t *accepts /* [S][2][T-1] since init; either may be NULL */);
int pt_get_cluster_sizes(uint32_t *last, uint64_t *cumulative /* [S][T]; either may be NULL */);
int pt_get_perm(int32_t *temp_of_slot, int32_t *slot_of_temp /* [S][2][T] each; either may be NULL */);

/* Device-resident variants (DEVICE pointers, same shapes, no host synchronisation): for callers that keep
 * observables on the GPU. */
int pt_get_energy_device(int32_t *E_dev);
int pt_measure_overlap_device(int32_t *Q_dev, int32_t *QL_dev);

/* ---- state access in SLOT order (parity tests, checkpointing) ------------------------------------------- */

int pt_get_spins(int8_t *spins /* [S][2][T(slot)][N], +1/-1 */);
int pt_get_couplings(int8_t *J /* [S][d][N], J[mu][i] = bond i -> i+e_mu, +1/-1 */);
int pt_get_thresholds(uint32_t *thrM /* [T][d], k=1..d at [t][k-1]; may be NULL */,
                      uint32_t *thrX /* [T-1][thrX_stride], entry m = |dE|/4; may be NULL */, size_t thrX_stride);
int pt_get_counters(uint32_t *n_sweep, uint32_t *n_exchange, uint32_t *n_houdayer);
int pt_set_spins(const int8_t *spins);      /* values must be +1/-1 (PT_ERR_ARG otherwise); recomputes E */
/* Same upload WITHOUT waiting for it: the samples are cut into groups; every group's host-to-device copy (~16 MiB), its
 * packing kernel and its energy kernel are queued on that group's stream and the call returns at once.  A pt_mcs /
 * pt_mcs_measure_device call that follows runs group by group on the same streams, so the Monte Carlo steps of the first
 * groups overlap the copies of the later ones; every other call first makes the bound stream wait for all groups.
 * spins: HOST [S][2][T(slot)][N], +1/-1; use pinned memory (a pageable buffer makes the copies synchronous) and do not
 * modify it before the next call that synchronises (pt_synchronize or any call that fills a host buffer).  Values are not
 * validated up front: a byte that is neither +1 nor -1 is taken by its sign and counted, and the next pt_synchronize()
 * then returns PT_ERR_ARG. */
int pt_set_spins_async(const int8_t *spins);
/* The same state through a BIT-PACKED boundary, one eighth of the bytes: HOST uint32 [S][2][T(slot)][ceil(N/32)], bit
 * (i & 31) of word (i >> 5) of a replica = site i in natural order, 1 <=> spin -1 (bits beyond site N-1 are ignored on
 * input and zero on output).  This is a boundary format; the device-internal layout is different.
 * pt_set_spins_packed queues copy + conversion + energies on the bound stream and returns without waiting (keep the buffer
 * unchanged until the next synchronising call; use pinned memory); pt_get_spins_packed synchronises. */
int pt_set_spins_packed(const uint32_t *bits);
int pt_get_spins_packed(uint32_t *bits);
/* Checkpoint / resume.  The RNG is counter-based, so the complete state of a run is: the couplings (or the
 * seed), the spins, the slot_of_temp maps and the three step counters; energies follow from the spins.  A run resumed with
 * pt_init (same arguments) + pt_set_spins + pt_set_perm + pt_set_counters continues bit-identically (the observables that
 * count since init -- swap counts, cumulative cluster sizes, round trips -- restart from zero).
 * pt_set_perm: HOST [S][2][T]; every row must be a permutation of 0..T-1 (PT_ERR_ARG otherwise); temp_of_slot is its
 * inverse.  pt_set_counters also lets a caller place a run anywhere in the Philox streams; a later call that would pass
 * 2^32 - 1 returns PT_ERR_OVERFLOW and leaves the state unchanged. */
int pt_set_perm(const int32_t *slot_of_temp);
int pt_set_counters(uint32_t n_sweep, uint32_t n_exchange, uint32_t n_houdayer);
int pt_set_couplings(const int8_t *J);      /* values must be +1/-1; recomputes E */
/* NEXT-3 (R33-R35): replace the couplings by fixed-point numbers J = Jq * 2^-frac_bits
 * (HOST int32 [S][d][N], Jq[mu][i] = bond i -> i+e_mu; e.g. a rounded standard-normal sample -- the couplings are an input
 * of the run) and recompute E.  From then on local fields, energies (in units of 2^-frac_bits, int32 as before) and energy
 * differences are exact integers and the acceptance probabilities are evaluated per decision in double:
 * flip with a = s_i h_i > 0: u < THR(-(beta_t * ldexp(2a, -frac_bits))); swap: u < THR(-(|dbeta| * ldexp(|dE|, -frac_bits))).
 * (the kernels settle a decision with a float bracket of 2^32 e^x that is provably on one side of the double threshold and
 * evaluate the double exp only for a draw inside the bracket: the decision is the double one always).
 * Philox mapping, sweep order, PT pass and cluster move are unchanged; pt_mcs is fused where the +-J path is.
 * PT_ERR_ARG: NULL, frac_bits outside [0, 24], or d*N*max|Jq| >= 2^31.  pt_set_couplings returns to the +-J model. */
int pt_set_couplings_fixed(const int32_t *Jq, int frac_bits);
int pt_get_couplings_fixed(int32_t *Jq /* [S][d][N] or NULL */, int *frac_bits /* or NULL */);   /* PT_ERR_STATE in the +-J model */
/* Recompute every E from scratch and count slots whose tracked E differs (invariant check; must be 0). */
int pt_recompute_energy(int32_t *E_slot_order /* [S][2][T] or NULL */, int *mismatch_count /* or NULL */);

/* ---- one PT pass for callers that must not allocate device memory ------------------------------------------ */

/* Everything above works inside a workspace the caller allocates and hands to pt_bind().  Some callers cannot do that:
 * an analysis hook that runs inside somebody else's GPU job after that job's memory pool (a framework's caching
 * allocator, a simulation sized to fill the card) has taken the device memory, so a fresh cudaMalloc fails or is against
 * the host program's rules; a latency-critical loop that cannot afford the device-wide synchronisation that
 * cudaMalloc / cudaFree imply while other streams are busy.  For them this ONE call needs no workspace, no pt_bind
 * and no pt_init, and allocates no device memory, neither itself nor through a library routine: its scratch is a fixed
 * area of PT_NOALLOC_SCRATCH_BYTES (4 MiB) that is part of libptglass.so's device image (every GPU on which the
 * library's code is loaded holds that area until the process exits).
 *
 * pt_exchange_noalloc makes the decisions of pt_exchange() (Eq. (5); R9, R10) -- pass number `step`
 * of a +-J problem of n_samples samples of an L^d lattice on the ladder betas, keyed by (seed, sample_offset) exactly as
 * after pt_init_shard -- on arrays the CALLER holds:
 *   E_dev             DEVICE const int32 [n_samples][2][n_temps], energy of every slot (slot order), read only;
 *   slot_of_temp_dev  DEVICE int32, same shape, every row a permutation of 0..n_temps-1 (NOT checked: an entry out of
 *                     range makes the kernel read outside E_dev), updated in place;
 *   temp_of_slot_dev  DEVICE int32, same shape, overwritten with the inverse of the new slot_of_temp;
 *   accepts_dev       DEVICE uint64 [n_samples][2][n_temps-1] or NULL: += 1 for every accepted pair;
 *   betas             HOST double [n_temps], as for pt_init;  step = the value pt_get_counters() reports as n_exchange
 *                     for the pass to reproduce;  cuda_stream: a cudaStream_t of the CURRENT device (NULL = default).
 * With these, maps and counts come out bit-identical to pt_exchange() on the same state.  The call returns once the work
 * is queued on cuda_stream; it does not synchronise.  The bound context (if any) is neither needed nor touched.
 * What the scratch holds: the swap-threshold table of the ladder and the sign of every beta step, computed on the host
 * in double and copied in on EVERY call (O(n_temps * table stride) exp() evaluations: meant for the occasional pass, not
 * for the inner loop), and the energies in temperature order on which the walk runs.
 * PT_ERR_ARG, nothing queued: an argument pt_init would reject (the shared-memory limit on L does not apply here), a
 * NULL array other than accepts_dev, or a problem whose tables and energies need more than PT_NOALLOC_SCRATCH_BYTES (the
 * message states both numbers; such problems need pt_bind + pt_exchange).  PT_ERR_CUDA: a CUDA call failed.
 * SET-UP: the first call on each device asks the CUDA runtime where that device keeps the scratch area (no allocation,
 * but a runtime query that may load the library's device code); make that first call before any stream capture begins
 * on the device.  Later calls on the device skip it.
 * SHARING: there is one scratch area per device and every call writes it, leaving its contents behind.  Each call
 * rewrites all it will read, so nothing has to be cleared and the order of earlier calls does not matter -- but two calls
 * whose work can overlap on the GPU (different streams without an event between them, or two host threads) race on it and
 * give garbage.  Put them on one stream or order them with events.  Like the rest of the library, not thread-safe. */
#define PT_NOALLOC_SCRATCH_BYTES (4u << 20)
int pt_exchange_noalloc(int L, int d, int n_samples, int n_temps, const double *betas, uint64_t seed,
                        uint32_t sample_offset, uint32_t step, const int32_t *E_dev, int32_t *slot_of_temp_dev,
                        int32_t *temp_of_slot_dev, uint64_t *accepts_dev, void *cuda_stream);

/* ---- diagnostics ---------------------------------------------------------------------------------------- */

int pt_synchronize(void);                          /* cudaStreamSynchronize on the bound stream */
int pt_get_launch_count(uint64_t *n_launches);     /* kernels launched by this library since pt_bind */
/* Per-kernel-class device times: when on, every launch of the sweep (class 0), Houdayer (1), exchange (2),
 * measurement (3) and fused-MCS (4) kernels is bracketed by CUDA events on the bound stream.  pt_set_profiling resets the sums;
 * pt_get_kernel_times synchronises and returns the summed milliseconds and launch counts since then. */
int pt_set_profiling(int on);
int pt_get_kernel_times(double ms[5], uint64_t launches[5]);
/* Where pt_mcs runs the three separate kernels per MCS (a sample does not fit a CTA's shared memory: BASELINE config 5),
 * the samples are cut into n groups, each issuing its sweep -> cluster -> exchange chain on its own stream (group 0 on the
 * bound stream, the others on library-owned side streams that fork from and join the bound stream inside the call), so
 * that the low-occupancy tail of one group's cluster kernel and its latency-bound exchange kernel overlap another group's
 * sweep.  Samples never interact (P:7), so results are bit-identical for every n.  n = -1: automatic (one group per wave
 * of sweep CTAs -- SMs x resident CTAs per SM, both asked from the runtime -- at most 8 and at most S; BASELINE config 5
 * runs 6); n in 1..8 (larger values are taken as 8): that many groups; n = 1: one stream (used for per-kernel timing). */
int pt_set_sample_groups(int n);
/* Phase split of the FUSED launch (pt_mcs where one CTA keeps a sample resident): CUDA events cannot separate the
 * Metropolis sweeps, the Houdayer moves and the PT pass inside one kernel, so when on, thread 0 of every CTA sums the SM
 * clocks it spends in each phase (a clock64() read after the CTA barrier that ends the phase) and adds them to four
 * device counters at the end of the launch: clocks[0] sweeps, [1] Houdayer, [2] PT pass, [3] the rest (load / store of
 * the state, overlap records).  clocks[k] / sum = the share of the launch time a CTA spends in phase k, which gives the
 * per-spin update times of Eq. (11) P:189 for the cluster move and the PT pass on the fused path.
 * pt_set_phase_clocks zeroes the counters; off by default (the timed bench region runs without it). */
int pt_set_phase_clocks(int on);
int pt_get_phase_clocks(uint64_t clocks[4]);
/* Which code path the bound problem uses: 1 = word-parallel kernels specialised for L a power of two >= 8,
 * 0 = general-L kernels. */
int pt_get_path(int *fast);
/* Test and measurement probes (device Philox / exp self-tests, the INT32 issue-rate microbenchmark, forcing the general-L
 * path, the development-build flag) are exported by the same library but declared in ptglass_diag.h: they are not part of
 * the method's interface. */
const char *pt_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
