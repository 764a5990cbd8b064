/*
 * ref_ptglass.c -- CPU ORACLE (TEST INFRASTRUCTURE ONLY; see ref_ptglass.h).
 *
 * Plain single-threaded C, int8 spins and couplings, one site at a time, in the paper's order and
 * notation.  No blocking, no bit tricks, no shared code with the CUDA path.  Each function cites the
 * passage of /root/reference/PAPER.md ("P:n") or the DESIGN.md reading ("Rk") it follows.
 *
 * Pins (tests/test_oracle_*.py): Philox known answers; gauge / ferromagnet / brute-force energy; beta=0 and
 * beta=50 sweeps; incremental == recomputed energy; PT cyclic shift and Eq. (5) decision grid; Houdayer
 * E1+E2, Q, QL conservation, involution, union-find component; exact enumeration of <E>, <q^2> at 2D L=4
 * and <E> at 3D L=2; sharding invariance; the survey's worked examples W1-W3.  The 10^4-MCS trajectories of
 * configs C2-C5 themselves are "parity unpinned" beyond oracle == GPU.
 */
#include "ref_ptglass.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

struct ref_ctx {
    int L, d, S, T, N;
    uint64_t seed;
    uint32_t sample_offset;
    double *betas;        /* [T] */
    int8_t *J;            /* [S][d][N]       J[mu][i] = bond i -> i+e_mu */
    int32_t *Jq;          /* [S][d][N]       fixed-point couplings J = Jq * 2^-fbits (NEXT-3, R33), or NULL */
    int fbits;            /* fractional bits of Jq; -1 in the +-J model */
    int8_t *spin;         /* [S][2][T][N]    slot order */
    int32_t *E;           /* [S][2][T]       slot order */
    int32_t *temp_of_slot;/* [S][2][T] */
    int32_t *slot_of_temp;/* [S][2][T] */
    uint32_t *thrM;       /* [T][d] */
    int *sgn;             /* [T-1] */
    uint64_t *attempts, *accepts; /* [S][2][T-1] */
    uint32_t *last_size;  /* [S][T] */
    uint64_t *cum_size;   /* [S][T] */
    uint32_t n_sweep, n_exchange, n_houdayer;
    int32_t *n_clu;       /* [T] single-cluster moves per ref_houdayer call (NEXT-4, R36), or NULL = 1 each */
    /* round-trip bookkeeping (readings R27-R29), per slot / per (sample, chain) */
    uint32_t *rt_label;   /* [S][2][T] 0 = never at index 0 yet, 1 = last end visited is index 0, 2 = index T-1 */
    uint32_t *rt_start;   /* [S][2][T] pass number at which the current trip started */
    uint32_t *rt_trips;   /* [S][2][T] completed round trips 0 -> T-1 -> 0 */
    uint64_t *rt_tau_sum; /* [S][2][32] sum of round-trip times completed at pass n, bin = floor(log2 n) */
    uint64_t *rt_tau_cnt; /* [S][2][32] */
    int *nbr;             /* [N][2d]: nbr[i][2mu] = i+e_mu, nbr[i][2mu+1] = i-e_mu */
    int *queue;           /* [N] BFS queue */
    uint8_t *mark;        /* [N] */
};

/* ---------------------------------------------------------------- Philox4x32-10, ref. [70] */

void ref_philox4x32_10(const uint32_t key[2], const uint32_t ctr[4], uint32_t out[4])
{
    const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)M0 * c0;
        uint64_t p1 = (uint64_t)M1 * c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;          /* key bumped after each round; round r uses key + r*W */
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Counter convention 8(c).1 (R11): key = seed, ctr = (index, step, global sample, TAG). */
static uint32_t draw(const ref_ctx *c, uint32_t index, uint32_t step, uint32_t g, int domain, int aux,
                     int chain, int idx16, int word)
{
    uint32_t key[2] = { (uint32_t)(c->seed & 0xFFFFFFFFu), (uint32_t)(c->seed >> 32) };
    uint32_t ctr[4] = { index, step, g,
                        ((uint32_t)domain << 28) | ((uint32_t)aux << 24) | ((uint32_t)chain << 16) |
                            (uint32_t)idx16 };
    uint32_t out[4];
    ref_philox4x32_10(key, ctr, out);
    return out[word];
}

static int8_t sign_of(uint32_t w) { return (w >> 31) == 0 ? (int8_t)1 : (int8_t)-1; }

/* ---------------------------------------------------------------- thresholds (R5, R6) */

uint32_t ref_threshold(double x)
{
    double v = floor(ldexp(exp(x), 32));
    if (v >= 4294967295.0) return 4294967295u;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

static uint32_t thrX_of(const ref_ctx *c, int t, long m)
{
    return ref_threshold(-(fabs(c->betas[t + 1] - c->betas[t]) * (double)(4 * m)));
}

/* coupling of bond (mu, i) of sample s as an integer: +-1, or Jq in the fixed-point model (NEXT-3, R33) */
static long jval(const ref_ctx *c, int s, int mu, int i)
{
    size_t k = ((size_t)s * c->d + mu) * c->N + i;
    return c->Jq ? (long)c->Jq[k] : (long)c->J[k];
}

/* Metropolis threshold for a flip with a = s_i h_i > 0 (Delta E = 2a) at temperature index t:
 * +-J: the table thrM[t][a/2];  fixed point (R34): THR(-(beta_t * ldexp((double)(2a), -fbits))), double exp. */
static uint32_t thr_flip(const ref_ctx *c, int t, long a)
{
    if (!c->Jq) return c->thrM[t * c->d + (a / 2 - 1)];
    return ref_threshold(-(c->betas[t] * ldexp((double)(2 * a), -c->fbits)));
}

/* swap threshold for |dE| at pair t: +-J: THR(-(|dbeta| * 4m)), m = |dE|/4;  fixed point (R34): THR(-(|dbeta| * ldexp(|dE|, -fbits))) */
static uint32_t thr_swap(const ref_ctx *c, int t, long absdE)
{
    if (!c->Jq) return thrX_of(c, t, absdE / 4);
    return ref_threshold(-(fabs(c->betas[t + 1] - c->betas[t]) * ldexp((double)absdE, -c->fbits)));
}

/* ---------------------------------------------------------------- lattice */

static void build_neighbours(ref_ctx *c)
{
    int L = c->L, d = c->d;
    for (int i = 0; i < c->N; ++i) {
        int x[3] = { i % L, (i / L) % L, d == 3 ? i / (L * L) : 0 };
        int stride = 1;
        for (int mu = 0; mu < d; ++mu) {
            int up = (x[mu] + 1) % L, dn = (x[mu] + L - 1) % L;
            c->nbr[i * 2 * d + 2 * mu]     = i + (up - x[mu]) * stride;
            c->nbr[i * 2 * d + 2 * mu + 1] = i + (dn - x[mu]) * stride;
            stride *= L;
        }
    }
}

static int colour_of(const ref_ctx *c, int i)
{
    int L = c->L;
    return ((i % L) + (i / L) % L + (c->d == 3 ? i / (L * L) : 0)) & 1;
}

/* E = -sum_{mu<d} sum_i J[mu][i] s_i s_{i+e_mu}   (Eq. (1) with H = 0; R3: both bonds counted at L=2) */
static int32_t energy_of(const ref_ctx *c, int smp, const int8_t *s)
{
    long e = 0;
    for (int mu = 0; mu < c->d; ++mu)
        for (int i = 0; i < c->N; ++i)
            e -= jval(c, smp, mu, i) * s[i] * s[c->nbr[i * 2 * c->d + 2 * mu]];
    return (int32_t)e;
}

static int8_t *spins_of(const ref_ctx *c, int s, int ch, int r)
{
    return c->spin + (((size_t)s * 2 + ch) * c->T + r) * c->N;
}
static size_t rep(const ref_ctx *c, int s, int ch, int r) { return ((size_t)s * 2 + ch) * c->T + r; }

static void recompute_all(ref_ctx *c)
{
    for (int s = 0; s < c->S; ++s)
        for (int ch = 0; ch < 2; ++ch)
            for (int r = 0; r < c->T; ++r)
                c->E[rep(c, s, ch, r)] = energy_of(c, s, spins_of(c, s, ch, r));
}

/* ---------------------------------------------------------------- init (8(c).2) */

ref_ctx *ref_create(int L, int d, int S, int T, const double *betas, uint64_t seed, uint32_t sample_offset)
{
    return ref_create_p(L, d, S, T, betas, seed, sample_offset, 0.5);
}

/* Eq. (2) with general p (reading R32): J = +1 iff w < floor(p * 2^32) for the bond's Philox word w. */
ref_ctx *ref_create_p(int L, int d, int S, int T, const double *betas, uint64_t seed, uint32_t sample_offset, double p_ferro)
{
    if (!(p_ferro >= 0.0) || !(p_ferro <= 1.0)) return NULL;
    const uint64_t thrJ = (uint64_t)floor(ldexp(p_ferro, 32));
    if (d != 2 && d != 3) return NULL;
    if (L < 2 || (L & 1)) return NULL;
    if (S < 1 || T < 1 || T > 65535 || betas == NULL) return NULL;
    for (int t = 0; t < T; ++t)
        if (!isfinite(betas[t]) || betas[t] < 0.0) return NULL;
    double Nd = pow((double)L, d) * d;
    if (Nd > 2147483647.0) return NULL;
    if ((uint64_t)sample_offset + (uint64_t)S > 4294967296ull) return NULL;

    ref_ctx *c = (ref_ctx *)calloc(1, sizeof(ref_ctx));
    c->L = L; c->d = d; c->S = S; c->T = T; c->seed = seed; c->sample_offset = sample_offset;
    c->N = (d == 2) ? L * L : L * L * L;
    c->Jq = NULL; c->fbits = -1;
    size_t R = (size_t)S * 2 * T, N = (size_t)c->N;
    c->betas = (double *)malloc(sizeof(double) * T);
    memcpy(c->betas, betas, sizeof(double) * T);
    c->J = (int8_t *)malloc((size_t)S * d * N);
    c->spin = (int8_t *)malloc(R * N);
    c->E = (int32_t *)malloc(R * sizeof(int32_t));
    c->temp_of_slot = (int32_t *)malloc(R * sizeof(int32_t));
    c->slot_of_temp = (int32_t *)malloc(R * sizeof(int32_t));
    c->thrM = (uint32_t *)malloc(sizeof(uint32_t) * T * d);
    c->sgn = (int *)calloc((size_t)T, sizeof(int));
    c->attempts = (uint64_t *)calloc((size_t)S * 2 * T, sizeof(uint64_t));
    c->accepts = (uint64_t *)calloc((size_t)S * 2 * T, sizeof(uint64_t));
    c->last_size = (uint32_t *)calloc((size_t)S * T, sizeof(uint32_t));
    c->cum_size = (uint64_t *)calloc((size_t)S * T, sizeof(uint64_t));
    c->rt_label = (uint32_t *)calloc(R, sizeof(uint32_t));
    c->rt_start = (uint32_t *)calloc(R, sizeof(uint32_t));
    c->rt_trips = (uint32_t *)calloc(R, sizeof(uint32_t));
    c->rt_tau_sum = (uint64_t *)calloc((size_t)S * 2 * 32, sizeof(uint64_t));
    c->rt_tau_cnt = (uint64_t *)calloc((size_t)S * 2 * 32, sizeof(uint64_t));
    c->nbr = (int *)malloc(sizeof(int) * N * 2 * d);
    c->queue = (int *)malloc(sizeof(int) * N);
    c->mark = (uint8_t *)malloc(N);
    build_neighbours(c);

    for (int s = 0; s < S; ++s) {
        uint32_t g = sample_offset + (uint32_t)s;
        /* 1. couplings: domain 1, p = 1/2 exactly (Eq. (2)) */
        for (int mu = 0; mu < d; ++mu)
            for (int i = 0; i < c->N; ++i)
                c->J[((size_t)s * d + mu) * N + i] =
                    ((uint64_t)draw(c, (uint32_t)i >> 2, 0, g, 1, mu, 0, 0, i & 3) < thrJ) ? (int8_t)1 : (int8_t)-1;
        /* 2. spins: domain 2 (R17);  3. identity permutations */
        for (int ch = 0; ch < 2; ++ch)
            for (int r = 0; r < T; ++r) {
                int8_t *sp = spins_of(c, s, ch, r);
                for (int i = 0; i < c->N; ++i)
                    sp[i] = sign_of(draw(c, (uint32_t)i >> 2, 0, g, 2, 0, ch, r, i & 3));
                c->temp_of_slot[rep(c, s, ch, r)] = r;
                c->slot_of_temp[rep(c, s, ch, r)] = r;
            }
        /* the slot that starts at temperature index 0 starts its first trip at pass 0 (R28) */
        for (int ch = 0; ch < 2; ++ch) c->rt_label[rep(c, s, ch, 0)] = 1;
    }
    /* 4. energies */
    recompute_all(c);
    /* 5. Metropolis thresholds thrM[t][k] = THR(-(beta_t * 4k)), k = 1..d */
    for (int t = 0; t < T; ++t)
        for (int k = 1; k <= d; ++k)
            c->thrM[t * d + (k - 1)] = ref_threshold(-(betas[t] * (double)(4 * k)));
    /* 6. swap sign sgn[t] = sign(beta_{t+1} - beta_t); thrX evaluated on demand */
    for (int t = 0; t + 1 < T; ++t)
        c->sgn[t] = (betas[t + 1] > betas[t]) - (betas[t + 1] < betas[t]);
    return c;
}

void ref_destroy(ref_ctx *c)
{
    if (!c) return;
    free(c->Jq);
    free(c->betas); free(c->J); free(c->spin); free(c->E); free(c->temp_of_slot); free(c->slot_of_temp);
    free(c->thrM); free(c->sgn); free(c->attempts); free(c->accepts); free(c->last_size); free(c->cum_size); free(c->n_clu);
    free(c->rt_label); free(c->rt_start); free(c->rt_trips); free(c->rt_tau_sum); free(c->rt_tau_cnt);
    free(c->nbr); free(c->queue); free(c->mark);
    free(c);
}

/* ---------------------------------------------------------------- Metropolis sweep (8(c).3, R1, R2, R4) */

int ref_sweep(ref_ctx *c, int n)
{
    if (!c || n < 0) return -1;
    if ((uint64_t)c->n_sweep + (uint64_t)n > 4294967295ull) return -3;
    int d = c->d, N = c->N;
    for (int it = 0; it < n; ++it) {
        for (int p = 0; p < 2; ++p)                       /* black (x+y+z even) first, then white */
            for (int s = 0; s < c->S; ++s) {
                uint32_t g = c->sample_offset + (uint32_t)s;
                for (int ch = 0; ch < 2; ++ch)
                    for (int r = 0; r < c->T; ++r) {
                        int8_t *sp = spins_of(c, s, ch, r);
                        int t = c->temp_of_slot[rep(c, s, ch, r)];
                        for (int i = 0; i < N; ++i) {
                            if (colour_of(c, i) != p) continue;
                            long h = 0;
                            for (int mu = 0; mu < d; ++mu) {
                                int up = c->nbr[i * 2 * d + 2 * mu], dn = c->nbr[i * 2 * d + 2 * mu + 1];
                                h += jval(c, s, mu, i) * sp[up] + jval(c, s, mu, dn) * sp[dn];
                            }
                            long a = sp[i] * h;           /* Delta E = 2a */
                            uint32_t u = draw(c, (uint32_t)i >> 3, c->n_sweep, g, 3, p, ch, r, (i >> 1) & 3);
                            if (a <= 0 || u < thr_flip(c, t, a)) {
                                sp[i] = (int8_t)-sp[i];
                                c->E[rep(c, s, ch, r)] += (int32_t)(2 * a);
                            }
                        }
                    }
            }
        c->n_sweep += 1;
    }
    return 0;
}

/* ---------------------------------------------------------------- PT pass (8(c).4; Eq. (5), R9, R10) */

int ref_exchange(ref_ctx *c)
{
    if (!c) return -1;
    if (c->n_exchange == 4294967295u) return -3;
    int T = c->T;
    for (int s = 0; s < c->S; ++s) {
        uint32_t g = c->sample_offset + (uint32_t)s;
        for (int ch = 0; ch < 2; ++ch) {
            int32_t *sot = c->slot_of_temp + rep(c, s, ch, 0);
            int32_t *tos = c->temp_of_slot + rep(c, s, ch, 0);
            int32_t *E = c->E + rep(c, s, ch, 0);
            for (int t = 0; t + 1 < T; ++t) {
                int ra = sot[t], rb = sot[t + 1];
                long dE = (long)E[ra] - (long)E[rb];      /* multiple of 4 (R22b) */
                if (!c->Jq && dE % 4 != 0) abort();
                uint32_t u = draw(c, (uint32_t)t, c->n_exchange, g, 4, 0, ch, 0, 0);
                size_t k = ((size_t)s * 2 + ch) * (T - 1) + t;
                c->attempts[k] += 1;
                if (c->sgn[t] * dE <= 0 || u < thr_swap(c, t, labs(dE))) {
                    sot[t] = rb; sot[t + 1] = ra; tos[ra] = t + 1; tos[rb] = t;
                    c->accepts[k] += 1;
                }
            }
            /* round-trip bookkeeping after the pass (R27-R29): n = number of passes done, this one included.
             * The replica now at index T-1 has reached the far end; the replica now at index 0 completes a
             * round trip 0 -> T-1 -> 0 if it has been at the far end since its trip started. */
            if (T > 1) {
                uint32_t n = c->n_exchange + 1u;
                size_t base = rep(c, s, ch, 0);
                int r1 = sot[T - 1], r0 = sot[0];
                if (c->rt_label[base + r1] == 1u) c->rt_label[base + r1] = 2u;
                if (c->rt_label[base + r0] == 2u) {
                    uint32_t tau = n - c->rt_start[base + r0];
                    int b = 0;
                    while ((n >> (b + 1)) != 0u) ++b;           /* b = floor(log2 n), n >= 1 */
                    c->rt_trips[base + r0] += 1u;
                    c->rt_tau_sum[((size_t)s * 2 + ch) * 32 + b] += tau;
                    c->rt_tau_cnt[((size_t)s * 2 + ch) * 32 + b] += 1u;
                    c->rt_label[base + r0] = 1u;
                    c->rt_start[base + r0] = n;
                } else if (c->rt_label[base + r0] == 0u) {
                    c->rt_label[base + r0] = 1u;
                    c->rt_start[base + r0] = n;
                }
            }
        }
    }
    c->n_exchange += 1;
    return 0;
}

/* ---------------------------------------------------------------- temperature-schedule family, Eq. (6)-(7) */
int ref_schedule_family(double T_min, double T_max, int n_temps, double phi, double *temps, double *betas)
{
    if (!(T_min > 0.0) || !(T_max >= T_min) || n_temps < 1 || !(phi > 0.0) || !isfinite(T_max) || !isfinite(phi)) return -1;
    double T_norm = (n_temps > 1) ? (T_max - T_min) / pow((double)(n_temps - 1), phi) : 0.0;     /* Eq. (7) */
    for (int i = 0; i < n_temps; ++i) {
        double Ti = pow((double)i, phi) * T_norm + T_min;                                        /* Eq. (6) */
        if (temps) temps[i] = Ti;
        if (betas) betas[i] = 1.0 / Ti;
    }
    return 0;
}

int ref_get_round_trips(const ref_ctx *c, uint32_t *trips, uint64_t *tau_sum, uint64_t *tau_cnt)
{
    if (!c) return -1;
    size_t R = (size_t)c->S * 2 * c->T, B = (size_t)c->S * 2 * 32;
    if (trips) memcpy(trips, c->rt_trips, R * sizeof(uint32_t));
    if (tau_sum) memcpy(tau_sum, c->rt_tau_sum, B * sizeof(uint64_t));
    if (tau_cnt) memcpy(tau_cnt, c->rt_tau_cnt, B * sizeof(uint64_t));
    return 0;
}

/* ---------------------------------------------------------------- Houdayer cluster exchange (8(c).5; Eq. (10), R12, R13) */

/* Exchange the sites with mark[i] = 1 between the two configurations at temperature t of sample s: since q_i = -1 there,
 * both spins are negated; the marked set must be a union of q = -1 components.  Energies are updated by
 * delta = 2 * sum over boundary bonds (i marked, j not) of J_ij A_i A_j, old spins. */
static void exchange_marked(ref_ctx *c, int s, int t)
{
    int d = c->d, N = c->N;
    int ra = c->slot_of_temp[rep(c, s, 0, t)], rb = c->slot_of_temp[rep(c, s, 1, t)];
    int8_t *A = spins_of(c, s, 0, ra), *B = spins_of(c, s, 1, rb);
    int32_t delta = 0;
    for (int i = 0; i < N; ++i) {
        if (!c->mark[i]) continue;
        for (int mu = 0; mu < d; ++mu) {
            int up = c->nbr[i * 2 * d + 2 * mu], dn = c->nbr[i * 2 * d + 2 * mu + 1];
            if (!c->mark[up]) delta += (int32_t)(2 * jval(c, s, mu, i) * A[i] * A[up]);
            if (!c->mark[dn]) delta += (int32_t)(2 * jval(c, s, mu, dn) * A[i] * A[dn]);
        }
    }
    for (int i = 0; i < N; ++i)
        if (c->mark[i]) { A[i] = (int8_t)-A[i]; B[i] = (int8_t)-B[i]; }
    c->E[rep(c, s, 0, ra)] += delta;
    c->E[rep(c, s, 1, rb)] -= delta;
}

/* One single-cluster move of pair (s, t): move number j of this step (j = 0 is the paper's one move per MCS, P:143;
 * j > 0 only with ref_set_cluster_moves, R36).  Returns the cluster size (0 if no site has q = -1). */
static uint32_t houdayer_move(ref_ctx *c, int s, int t, uint32_t j)
{
    int d = c->d, N = c->N;
    uint32_t g = c->sample_offset + (uint32_t)s;
    int ra = c->slot_of_temp[rep(c, s, 0, t)], rb = c->slot_of_temp[rep(c, s, 1, t)];
    int8_t *A = spins_of(c, s, 0, ra), *B = spins_of(c, s, 1, rb);
    int n_neg = 0;
    for (int i = 0; i < N; ++i) n_neg += (A[i] * B[i] == -1);
    uint32_t u = draw(c, j, c->n_houdayer, g, 5, 0, 0, t, 0);
    if (n_neg == 0) return 0;
    int k = (int)(((uint64_t)u * (uint64_t)n_neg) >> 32), i0 = -1;
    for (int i = 0, seen = 0; i < N; ++i)
        if (A[i] * B[i] == -1) { if (seen == k) { i0 = i; break; } ++seen; }
    /* breadth-first search over q = -1 sites */
    memset(c->mark, 0, (size_t)N);
    int head = 0, tail = 0;
    c->queue[tail++] = i0; c->mark[i0] = 1;
    while (head < tail) {
        int i = c->queue[head++];
        for (int k2 = 0; k2 < 2 * d; ++k2) {
            int jn = c->nbr[i * 2 * d + k2];
            if (!c->mark[jn] && A[jn] * B[jn] == -1) { c->mark[jn] = 1; c->queue[tail++] = jn; }
        }
    }
    exchange_marked(c, s, t);
    return (uint32_t)tail;
}

int ref_houdayer(ref_ctx *c)
{
    if (!c) return -1;
    if (c->n_houdayer == 4294967295u) return -3;
    int T = c->T;
    for (int s = 0; s < c->S; ++s)
        for (int t = 0; t < T; ++t) {
            int moves = c->n_clu ? c->n_clu[t] : 1;
            uint32_t size = 0;
            for (int j = 0; j < moves; ++j) {
                size = houdayer_move(c, s, t, (uint32_t)j);
                c->cum_size[(size_t)s * T + t] += (uint64_t)size;
            }
            c->last_size[(size_t)s * T + t] = size;        /* the last move's; 0 where n_clu[t] = 0 */
        }
    c->n_houdayer += 1;
    return 0;
}

/* NEXT-4 ("perform several cluster updates in the high-temperature copies"; P:140 / ref. [39]: cluster moves
 * only where they help; reading R36): n_clu[t] >= 0 single-cluster moves per ref_houdayer call at temperature index t;
 * NULL restores one move everywhere. */
int ref_set_cluster_moves(ref_ctx *c, const int32_t *n_clu)
{
    if (!c) return -1;
    if (!n_clu) { free(c->n_clu); c->n_clu = NULL; return 0; }
    for (int t = 0; t < c->T; ++t) if (n_clu[t] < 0 || n_clu[t] > 65535) return -1;
    if (!c->n_clu) c->n_clu = (int32_t *)malloc((size_t)c->T * sizeof(int32_t));
    if (!c->n_clu) return -2;
    memcpy(c->n_clu, n_clu, (size_t)c->T * sizeof(int32_t));
    return 0;
}

/* NEXT-4 ("a formal conversion to a multi-cluster variant"; reading R37): EVERY connected component of
 * q = -1 sites is exchanged between the two configurations independently with probability 1/2.  The component whose
 * smallest site index is i_min is exchanged iff the top bit of word (i_min & 3) of the Philox block
 * ctr = (i_min >> 2, step, g, tag(5, aux = 1, 0, t)) is set.  Exchanging any union of q = -1 components leaves
 * E1 + E2 unchanged (every boundary bond has a q = +1 end).  last_size = number of exchanged sites. */
int ref_houdayer_multi(ref_ctx *c)
{
    if (!c) return -1;
    if (c->n_houdayer == 4294967295u) return -3;
    int d = c->d, N = c->N, T = c->T;
    uint8_t *seen = (uint8_t *)malloc((size_t)N);
    if (!seen) return -2;
    for (int s = 0; s < c->S; ++s) {
        uint32_t g = c->sample_offset + (uint32_t)s;
        for (int t = 0; t < T; ++t) {
            int ra = c->slot_of_temp[rep(c, s, 0, t)], rb = c->slot_of_temp[rep(c, s, 1, t)];
            int8_t *A = spins_of(c, s, 0, ra), *B = spins_of(c, s, 1, rb);
            memset(seen, 0, (size_t)N);
            memset(c->mark, 0, (size_t)N);
            uint32_t total = 0;
            for (int i0 = 0; i0 < N; ++i0) {
                if (seen[i0] || A[i0] * B[i0] != -1) continue;
                /* i0 is the smallest index of a component not seen yet: collect it by BFS */
                int head = 0, tail = 0;
                c->queue[tail++] = i0; seen[i0] = 1;
                while (head < tail) {
                    int i = c->queue[head++];
                    for (int k2 = 0; k2 < 2 * d; ++k2) {
                        int jn = c->nbr[i * 2 * d + k2];
                        if (!seen[jn] && A[jn] * B[jn] == -1) { seen[jn] = 1; c->queue[tail++] = jn; }
                    }
                }
                uint32_t w = draw(c, (uint32_t)(i0 >> 2), c->n_houdayer, g, 5, 1, 0, t, i0 & 3);
                if (w >> 31) {
                    for (int k = 0; k < tail; ++k) c->mark[c->queue[k]] = 1;
                    total += (uint32_t)tail;
                }
            }
            if (total) exchange_marked(c, s, t);
            c->last_size[(size_t)s * T + t] = total;
            c->cum_size[(size_t)s * T + t] += (uint64_t)total;
        }
    }
    free(seen);
    c->n_houdayer += 1;
    return 0;
}

/* ---------------------------------------------------------------- MCS in the paper's order (8(c).7, R15) */

int ref_mcs(ref_ctx *c, int n_mcs, int n_metro, int do_houdayer, int do_exchange)
{
    if (!c || n_mcs < 0 || n_metro < 0 || do_houdayer < 0 || do_houdayer > 2) return -1;
    for (int m = 0; m < n_mcs; ++m) {
        int rc = ref_sweep(c, n_metro);
        if (rc) return rc;
        if (do_houdayer == 1 && (rc = ref_houdayer(c))) return rc;
        if (do_houdayer == 2 && (rc = ref_houdayer_multi(c))) return rc;
        if (do_exchange && (rc = ref_exchange(c))) return rc;
    }
    return 0;
}

/* ---------------------------------------------------------------- observables (8(c).6) */

int ref_get_energy(const ref_ctx *c, int32_t *E)
{
    if (!c || !E) return -1;
    for (int s = 0; s < c->S; ++s)
        for (int ch = 0; ch < 2; ++ch)
            for (int t = 0; t < c->T; ++t)
                E[rep(c, s, ch, t)] = c->E[rep(c, s, ch, c->slot_of_temp[rep(c, s, ch, t)])];
    return 0;
}

/* Q = sum_i q_i (Eq. (4) x N);  QL = sum_{mu,i} q_i q_{i+e_mu} (R14) */
int ref_measure_overlap(const ref_ctx *c, int32_t *Q, int32_t *QL)
{
    if (!c || !Q) return -1;
    for (int s = 0; s < c->S; ++s)
        for (int t = 0; t < c->T; ++t) {
            const int8_t *A = spins_of(c, s, 0, c->slot_of_temp[rep(c, s, 0, t)]);
            const int8_t *B = spins_of(c, s, 1, c->slot_of_temp[rep(c, s, 1, t)]);
            int32_t q = 0, ql = 0;
            for (int i = 0; i < c->N; ++i) {
                q += A[i] * B[i];
                for (int mu = 0; mu < c->d; ++mu) {
                    int j = c->nbr[i * 2 * c->d + 2 * mu];
                    ql += A[i] * B[i] * A[j] * B[j];
                }
            }
            Q[(size_t)s * c->T + t] = q;
            if (QL) QL[(size_t)s * c->T + t] = ql;
        }
    return 0;
}

/* Overlap profiles (NEXT-2; "the modes for the correlation length"; reading R31): for every axis mu and every
 * coordinate x along it, the sum of q_i = A_i B_i over the lattice plane x_mu = x.  The Fourier modes of the overlap
 * field with wave vector along an axis, q(k e_mu) = sum_x prof[mu][x] exp(i k x), are a length-L transform of this. */
int ref_measure_overlap_profile(const ref_ctx *c, int32_t *prof)
{
    if (!c || !prof) return -1;
    int L = c->L, d = c->d;
    for (int s = 0; s < c->S; ++s)
        for (int t = 0; t < c->T; ++t) {
            const int8_t *A = spins_of(c, s, 0, c->slot_of_temp[rep(c, s, 0, t)]);
            const int8_t *B = spins_of(c, s, 1, c->slot_of_temp[rep(c, s, 1, t)]);
            int32_t *out = prof + ((size_t)s * c->T + t) * d * L;
            for (int k = 0; k < d * L; ++k) out[k] = 0;
            for (int i = 0; i < c->N; ++i) {
                int coord[3] = { i % L, (i / L) % L, i / (L * L) };
                for (int mu = 0; mu < d; ++mu) out[mu * L + coord[mu]] += A[i] * B[i];
            }
        }
    return 0;
}

int ref_get_swap_counts(const ref_ctx *c, uint64_t *attempts, uint64_t *accepts)
{
    if (!c) return -1;
    size_t n = (size_t)c->S * 2 * (c->T - 1);
    if (attempts) memcpy(attempts, c->attempts, n * sizeof(uint64_t));
    if (accepts) memcpy(accepts, c->accepts, n * sizeof(uint64_t));
    return 0;
}

int ref_get_cluster_sizes(const ref_ctx *c, uint32_t *last, uint64_t *cumulative)
{
    if (!c) return -1;
    size_t n = (size_t)c->S * c->T;
    if (last) memcpy(last, c->last_size, n * sizeof(uint32_t));
    if (cumulative) memcpy(cumulative, c->cum_size, n * sizeof(uint64_t));
    return 0;
}

int ref_get_perm(const ref_ctx *c, int32_t *temp_of_slot, int32_t *slot_of_temp)
{
    if (!c) return -1;
    size_t n = (size_t)c->S * 2 * c->T;
    if (temp_of_slot) memcpy(temp_of_slot, c->temp_of_slot, n * sizeof(int32_t));
    if (slot_of_temp) memcpy(slot_of_temp, c->slot_of_temp, n * sizeof(int32_t));
    return 0;
}

int ref_get_spins(const ref_ctx *c, int8_t *spins)
{
    if (!c || !spins) return -1;
    memcpy(spins, c->spin, (size_t)c->S * 2 * c->T * c->N);
    return 0;
}

int ref_get_couplings(const ref_ctx *c, int8_t *J)
{
    if (!c || !J) return -1;
    memcpy(J, c->J, (size_t)c->S * c->d * c->N);
    return 0;
}

int ref_get_thresholds(const ref_ctx *c, uint32_t *thrM, uint32_t *thrX, size_t stride)
{
    if (!c) return -1;
    if (thrM) memcpy(thrM, c->thrM, sizeof(uint32_t) * c->T * c->d);
    if (thrX)
        for (int t = 0; t + 1 < c->T; ++t)
            for (size_t m = 0; m < stride; ++m)
                thrX[(size_t)t * stride + m] = thrX_of(c, t, (long)m);
    return 0;
}

int ref_get_counters(const ref_ctx *c, uint32_t *n_sweep, uint32_t *n_exchange, uint32_t *n_houdayer)
{
    if (!c) return -1;
    if (n_sweep) *n_sweep = c->n_sweep;
    if (n_exchange) *n_exchange = c->n_exchange;
    if (n_houdayer) *n_houdayer = c->n_houdayer;
    return 0;
}

int ref_set_spins(ref_ctx *c, const int8_t *spins)
{
    if (!c || !spins) return -1;
    size_t n = (size_t)c->S * 2 * c->T * c->N;
    for (size_t k = 0; k < n; ++k)
        if (spins[k] != 1 && spins[k] != -1) return -1;
    memcpy(c->spin, spins, n);
    recompute_all(c);
    return 0;
}

int ref_set_couplings(ref_ctx *c, const int8_t *J)
{
    if (!c || !J) return -1;
    size_t n = (size_t)c->S * c->d * c->N;
    for (size_t k = 0; k < n; ++k)
        if (J[k] != 1 && J[k] != -1) return -1;
    memcpy(c->J, J, n);
    recompute_all(c);
    return 0;
}

/* NEXT-3 (readings R33-R35): replace the couplings by fixed-point values J = Jq * 2^-fbits (e.g. a
 * rounded standard normal sample, an INPUT of the run) and recompute the energies.  From here on the sweeps, the PT pass
 * and the cluster move use integer fields / energy differences in units of 2^-fbits and evaluate the acceptance
 * probabilities with double exp (thr_flip, thr_swap).  d * N * max|Jq| must stay below 2^31 (int32 energies). */
int ref_set_couplings_fixed(ref_ctx *c, const int32_t *Jq, int fbits)
{
    if (!c || !Jq || fbits < 0 || fbits > 24) return -1;
    size_t n = (size_t)c->S * c->d * c->N;
    long maxabs = 0;
    for (size_t k = 0; k < n; ++k) {
        long v = Jq[k] < 0 ? -(long)Jq[k] : (long)Jq[k];
        if (v > maxabs) maxabs = v;
    }
    if ((double)maxabs * (double)c->d * (double)c->N >= 2147483648.0) return -1;
    if (!c->Jq) c->Jq = (int32_t *)malloc(n * sizeof(int32_t));
    memcpy(c->Jq, Jq, n * sizeof(int32_t));
    c->fbits = fbits;
    recompute_all(c);
    return 0;
}

int ref_get_couplings_fixed(const ref_ctx *c, int32_t *Jq, int *fbits)
{
    if (!c || !c->Jq) return -1;
    if (Jq) memcpy(Jq, c->Jq, (size_t)c->S * c->d * c->N * sizeof(int32_t));
    if (fbits) *fbits = c->fbits;
    return 0;
}

int ref_recompute_energy(const ref_ctx *c, int32_t *E_slot_order, int *mismatch_count)
{
    if (!c) return -1;
    int bad = 0;
    for (int s = 0; s < c->S; ++s)
        for (int ch = 0; ch < 2; ++ch)
            for (int r = 0; r < c->T; ++r) {
                int32_t e = energy_of(c, s, spins_of(c, s, ch, r));
                if (E_slot_order) E_slot_order[rep(c, s, ch, r)] = e;
                bad += (e != c->E[rep(c, s, ch, r)]);
            }
    if (mismatch_count) *mismatch_count = bad;
    return 0;
}
