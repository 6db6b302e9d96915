/* olsm.c -- ORACLE for the lattice-spring-model hot path of arXiv 2201.04565 ("ImageMech" / CuLSM).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  It shares no code with paper_2201_04565_b200/ (the CUDA path)
 * and neither includes the other.  Plain C11, fp64, serial, no blocking / fusion / reordering: every loop below can
 * be checked against the paper by eye.  Build: gcc -O2 -ffp-contract=off -fPIC -shared (see oracle/olsm.py).
 *
 * What it computes (citations are PAPER.md line numbers):
 *   force_eval()  Eq. 1 (L45) energy and Eq. 2 (L53-L55) force of the truncated harmonic springs, with the
 *                 irreversible breakage test of the kernel listing (L98: `if (r_ij > rc[i]) k[i] = 0;`, L196),
 *                 as ONE serial loop over the spring list in caller order (the paper's parallel-over-springs loop,
 *                 L88-L111, run serially: this fixes the summation order).
 *   olsm_step()   velocity Verlet, Eq. 3-5 (L64-L74), in the half-step-velocity form the paper says it uses (L76):
 *                 kick - drift - force - kick; boundary displacement applied first (L88).
 *   samples       U and KE (L113), boundary reaction sums and broken count (BASELINE.json north_star item 4).
 *   olsm_read_virial()  per-particle virial stress, Eq. 7 (L147), pinned by P13 (virial = Cauchy stress in a homogeneous
 *                 static state; kinetic term; sum over particles = sum over springs of g d (x) d).
 *   olsm_read_strain()  per-particle Lagrangian strain, Eq. 8 (L150, L156), reading Q21; pinned by P15 (homogeneous
 *                 deformation gives exactly (F^T F - I)/2, rigid rotation gives 0, small-strain limit of P3's state,
 *                 rank-deficient neighbourhoods are flagged, a transposed J fails).
 * Readings where the paper is silent are those of SURVEY.md 8(c) / DESIGN.md "Readings" (Q1..Q21), named inline.
 *
 * Pins (tests/test_oracle_pins.py, all run without a GPU): P1 paper's worked oscillator example (L123-L127) against
 * the closed form of velocity Verlet and the analytic ODE solution; P2 two free particles (reduced mass period);
 * P3 affine uniaxial-stress state of a full triangular lattice (Young's modulus 2k/sqrt3, Poisson ratio 1/3, energy);
 * P4 zero net force / torque; P5 brute-force all-pairs; P6 energy conservation; P7 strict '>' with dyadic numbers;
 * P8 irreversibility; P9 time reversibility (L76); P10 F = -grad U by finite differences; P12 damping closed form.
 * Mass != 1 (Eq. 4), olsm_write_state, the stored velocity of kinematic particles and olsm_set_boundary between steps
 * have their own closed-form pins (P1 with m = 4, P2 with unequal masses, P12 with m = 2, restart on the closed form).
 * Unpinned: the fracture path AFTER the first breakage has no closed form (statistics only) -- "parity unpinned"
 * for that part; see DESIGN.md.
 *
 * olsm_set_threads(n > 1) switches the force evaluation to force_eval_threads(): the same arithmetic per spring, summed
 * per particle in the same ascending spring order, run over OpenMP threads.  It exists only so that bench.py can time
 * the oracle on all host cores; the serial loop stays the reference every parity test compares with,
 * and tests/test_oracle_pins.py asserts the threaded variant is bit-equal to it through a fracture run.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define OLSM_MAX_GROUPS 8

typedef struct {
    int64_t n;          /* number of ids */
    int32_t *ids;
    int32_t mode;       /* 0 FIXED, 1 MOVE */
    double du[3];       /* displacement per step (0 for FIXED) */
    double *x0;         /* [n*D] origin snapshot */
    int64_t n0;         /* step at which the group was set */
} ogroup;

typedef struct olsm_sim {
    int32_t D;
    int64_t N, M;
    int32_t B;                      /* n_batch */
    int64_t *poff, *soff;           /* [B+1] */
    double *x, *v, *f, *fd, *m;     /* [N*D] x4, [N] */
    double *xref;                   /* [N*D] positions at olsm_create: the reference configuration of Eq. 8 (Q21) */
    int32_t *si, *sj;
    double *k, *r0, *rc;
    uint8_t *alive;
    int64_t *break_step;
    int64_t *nbroken;               /* [B] cumulative */
    double *U;                      /* [B] of the last force evaluation */
    int32_t *spec_of_spring;        /* [M] specimen index */
    int32_t *spec_of_particle;      /* [N] */
    int8_t *group_of;               /* [N], -1 = free */
    ogroup g[OLSM_MAX_GROUPS];
    double dt, gamma;
    int64_t step;
    int32_t sample_every;
    /* history */
    int64_t ns, cap;
    int64_t *h_step;
    double *h_R;                    /* [cap][B][8][D] */
    double *h_U, *h_KE;             /* [cap][B] */
    int64_t *h_nb;                  /* [cap][B] */
    /* all-cores variant (olsm_set_threads): per-particle incidence lists in ascending spring id, per-spring scratch */
    int32_t threads;                /* 0 / 1 = the serial loop */
    int64_t *adj_off;               /* [N+1] */
    int32_t *adj_e;                 /* [2M] spring ids, ascending inside each particle's list */
    double *gs, *ue;                /* [M] k (r - r0)/r and the energy of each spring in the last evaluation */
    uint8_t *act;                   /* [M] 1 if the spring contributed to the last evaluation */
    int32_t U_stale;                /* per-specimen U not yet summed from ue[] */
} olsm_sim;

/* Eq. 1 / Eq. 2 / listing L91-L107.  Serial loop, caller spring order. */
static void force_eval(olsm_sim *s)
{
    const int D = s->D;
    memset(s->f, 0, sizeof(double) * (size_t)(s->N * D));
    for (int b = 0; b < s->B; ++b) s->U[b] = 0.0;
    s->U_stale = 0;                                       /* U[] is summed right here: nothing left over from force_eval_threads() */
    for (int64_t e = 0; e < s->M; ++e) {
        if (!s->alive[e]) continue;                       /* irreversible: L98, L196 (Q2) */
        const int64_t i = s->si[e], j = s->sj[e];
        double d[3] = {0.0, 0.0, 0.0};
        double r2 = 0.0;
        for (int c = 0; c < D; ++c) {
            d[c] = s->x[j * D + c] - s->x[i * D + c];     /* r_j - r_i */
            r2 = r2 + d[c] * d[c];                        /* L95-L97; no FMA contraction (-ffp-contract=off) */
        }
        const double r = sqrt(r2);                        /* L95 */
        if (r > s->rc[e]) {                               /* strict '>' as in L98 (Q1) */
            s->alive[e] = 0;
            s->break_step[e] = s->step;
            s->nbroken[s->spec_of_spring[e]] += 1;
            continue;                                     /* zero force and energy in the same evaluation (Q3) */
        }
        if (r == 0.0) continue;                           /* direction undefined (Q4) */
        const double ext = r - s->r0[e];
        const double g = s->k[e] * ext / r;               /* k (r - r0) / r : L99-L101 */
        for (int c = 0; c < D; ++c) {
            const double gd = g * d[c];
            s->f[i * D + c] += gd;                        /* f_i = -k(r-r0)(r_i-r_j)/r  (Eq. 2; L99, L102) */
            s->f[j * D + c] -= gd;                        /* L105-L107 */
        }
        s->U[s->spec_of_spring[e]] += 0.5 * s->k[e] * ext * ext;   /* Eq. 1 (L45); broken springs add 0 (Q18) */
    }
}

/* The same evaluation over OpenMP threads (all-cores timing leg only).  Pass 1, one iteration per spring: the same
 * expressions as force_eval() for r, the breakage test, g and the energy, stored per spring.  Pass 2, one iteration per
 * particle: add its springs' g*d in ascending spring id -- the order, and hence every rounding, of the serial loop
 * (which does f[i] += gd, f[j] -= gd spring by spring).  U is summed serially in spring order when it is next read. */
static void sum_U(olsm_sim *s)
{
    if (!s->U_stale) return;
    for (int b = 0; b < s->B; ++b) s->U[b] = 0.0;
    for (int64_t e = 0; e < s->M; ++e)
        if (s->act[e]) s->U[s->spec_of_spring[e]] += s->ue[e];
    s->U_stale = 0;
}

static void force_eval_threads(olsm_sim *s)
{
    const int D = s->D;
    #pragma omp parallel for schedule(static) num_threads(s->threads)
    for (int64_t e = 0; e < s->M; ++e) {
        s->act[e] = 0;
        if (!s->alive[e]) continue;
        const int64_t i = s->si[e], j = s->sj[e];
        double d[3] = {0.0, 0.0, 0.0};
        double r2 = 0.0;
        for (int c = 0; c < D; ++c) {
            d[c] = s->x[j * D + c] - s->x[i * D + c];
            r2 = r2 + d[c] * d[c];
        }
        const double r = sqrt(r2);
        if (r > s->rc[e]) {
            s->alive[e] = 0;
            s->break_step[e] = s->step;
            #pragma omp atomic
            s->nbroken[s->spec_of_spring[e]] += 1;
            continue;
        }
        if (r == 0.0) continue;
        const double ext = r - s->r0[e];
        s->gs[e] = s->k[e] * ext / r;
        s->ue[e] = 0.5 * s->k[e] * ext * ext;
        s->act[e] = 1;
    }
    #pragma omp parallel for schedule(static) num_threads(s->threads)
    for (int64_t p = 0; p < s->N; ++p) {
        double fp[3] = {0.0, 0.0, 0.0};
        for (int64_t q = s->adj_off[p]; q < s->adj_off[p + 1]; ++q) {
            const int64_t e = s->adj_e[q];
            if (!s->act[e]) continue;
            const int64_t i = s->si[e], j = s->sj[e];
            for (int c = 0; c < D; ++c) {
                const double gd = s->gs[e] * (s->x[j * D + c] - s->x[i * D + c]);
                if (p == i) fp[c] += gd; else fp[c] -= gd;
            }
        }
        for (int c = 0; c < D; ++c) s->f[p * D + c] = fp[c];
    }
    s->U_stale = 1;
}

static void damp(olsm_sim *s)
{
    /* Q7: viscous force -gamma*v, v = the velocity held at force time. gamma = 0 reproduces the paper. */
    const int64_t n = s->N * s->D;
    #pragma omp parallel for schedule(static) num_threads(s->threads) if (s->threads > 1)
    for (int64_t q = 0; q < n; ++q) s->fd[q] = s->f[q] - s->gamma * s->v[q];
}

static void record_sample(olsm_sim *s)
{
    const int D = s->D;
    if (s->ns == s->cap) {
        int64_t nc = s->cap ? 2 * s->cap : 64;
        s->h_step = realloc(s->h_step, sizeof(int64_t) * (size_t)nc);
        s->h_R = realloc(s->h_R, sizeof(double) * (size_t)(nc * s->B * OLSM_MAX_GROUPS * D));
        s->h_U = realloc(s->h_U, sizeof(double) * (size_t)(nc * s->B));
        s->h_KE = realloc(s->h_KE, sizeof(double) * (size_t)(nc * s->B));
        s->h_nb = realloc(s->h_nb, sizeof(int64_t) * (size_t)(nc * s->B));
        s->cap = nc;
    }
    sum_U(s);
    const int64_t t = s->ns++;
    s->h_step[t] = s->step;
    double *R = s->h_R + t * s->B * OLSM_MAX_GROUPS * D;
    memset(R, 0, sizeof(double) * (size_t)(s->B * OLSM_MAX_GROUPS * D));
    for (int gi = 0; gi < OLSM_MAX_GROUPS; ++gi)          /* reaction: sum of spring forces on the group's particles */
        for (int64_t q = 0; q < s->g[gi].n; ++q) {
            const int64_t p = s->g[gi].ids[q];
            const int b = s->spec_of_particle[p];
            for (int c = 0; c < D; ++c) R[(b * OLSM_MAX_GROUPS + gi) * D + c] += s->f[p * D + c];
        }
    for (int b = 0; b < s->B; ++b) {
        double ke = 0.0;
        for (int64_t p = s->poff[b]; p < s->poff[b + 1]; ++p) {
            if (s->group_of[p] >= 0) continue;            /* kinematic particles carry no KE (Q6) */
            double v2 = 0.0;
            for (int c = 0; c < D; ++c) v2 = v2 + s->v[p * D + c] * s->v[p * D + c];
            ke += 0.5 * s->m[p] * v2;                     /* L113 */
        }
        s->h_U[t * s->B + b] = s->U[b];
        s->h_KE[t * s->B + b] = ke;
        s->h_nb[t * s->B + b] = s->nbroken[b];
    }
}

olsm_sim *olsm_create(int32_t D, int64_t N, int64_t M, int32_t B, const int64_t *poff, const int64_t *soff,
                      const double *x, const double *v, const double *mass, double mass_uniform,
                      const int32_t *si, const int32_t *sj, const double *k, const double *r0, const double *rc,
                      double dt, double gamma, int32_t sample_every)
{
    if ((D != 2 && D != 3) || N <= 0 || M < 0 || B < 1 || !x || dt <= 0.0 || gamma < 0.0) return NULL;
    olsm_sim *s = calloc(1, sizeof(*s));
    s->D = D; s->N = N; s->M = M; s->B = B; s->dt = dt; s->gamma = gamma; s->sample_every = sample_every;
    s->poff = malloc(sizeof(int64_t) * (size_t)(B + 1));
    s->soff = malloc(sizeof(int64_t) * (size_t)(B + 1));
    if (B == 1 && !poff) { s->poff[0] = 0; s->poff[1] = N; s->soff[0] = 0; s->soff[1] = M; }
    else { memcpy(s->poff, poff, sizeof(int64_t) * (size_t)(B + 1)); memcpy(s->soff, soff, sizeof(int64_t) * (size_t)(B + 1)); }
    const size_t nd = (size_t)(N * D);
    s->x = malloc(sizeof(double) * nd); memcpy(s->x, x, sizeof(double) * nd);
    s->xref = malloc(sizeof(double) * nd); memcpy(s->xref, x, sizeof(double) * nd);
    s->v = calloc(nd, sizeof(double)); if (v) memcpy(s->v, v, sizeof(double) * nd);
    s->f = calloc(nd, sizeof(double)); s->fd = calloc(nd, sizeof(double));
    s->m = malloc(sizeof(double) * (size_t)N);
    for (int64_t p = 0; p < N; ++p) s->m[p] = mass ? mass[p] : mass_uniform;
    s->si = malloc(sizeof(int32_t) * (size_t)(M + 1)); s->sj = malloc(sizeof(int32_t) * (size_t)(M + 1));
    s->k = malloc(sizeof(double) * (size_t)(M + 1)); s->r0 = malloc(sizeof(double) * (size_t)(M + 1));
    s->rc = malloc(sizeof(double) * (size_t)(M + 1));
    memcpy(s->si, si, sizeof(int32_t) * (size_t)M); memcpy(s->sj, sj, sizeof(int32_t) * (size_t)M);
    memcpy(s->k, k, sizeof(double) * (size_t)M); memcpy(s->r0, r0, sizeof(double) * (size_t)M);
    memcpy(s->rc, rc, sizeof(double) * (size_t)M);
    s->alive = malloc((size_t)(M + 1)); memset(s->alive, 1, (size_t)(M + 1));
    s->break_step = malloc(sizeof(int64_t) * (size_t)(M + 1));
    for (int64_t e = 0; e < M; ++e) s->break_step[e] = -1;
    s->nbroken = calloc((size_t)B, sizeof(int64_t));
    s->U = calloc((size_t)B, sizeof(double));
    s->spec_of_spring = malloc(sizeof(int32_t) * (size_t)(M + 1));
    s->spec_of_particle = malloc(sizeof(int32_t) * (size_t)N);
    for (int b = 0; b < B; ++b) {
        for (int64_t p = s->poff[b]; p < s->poff[b + 1]; ++p) s->spec_of_particle[p] = b;
        for (int64_t e = s->soff[b]; e < s->soff[b + 1]; ++e) s->spec_of_spring[e] = b;
    }
    s->group_of = malloc((size_t)N); memset(s->group_of, -1, (size_t)N);
    s->step = 0;
    force_eval(s);            /* f, U defined at step 0; a spring already longer than rc breaks at step 0 */
    damp(s);
    return s;              /* samples are recorded at steps n > 0 with n % sample_every == 0 */
}

int32_t olsm_set_boundary(olsm_sim *s, int32_t gi, const int32_t *ids, int64_t n, int32_t mode, const double *du)
{
    if (!s || gi < 0 || gi >= OLSM_MAX_GROUPS || n < 0 || (mode != 0 && mode != 1)) return -1;
    ogroup *g = &s->g[gi];
    for (int64_t q = 0; q < g->n; ++q) s->group_of[g->ids[q]] = -1;      /* release the old members */
    free(g->ids); free(g->x0);
    g->n = n; g->mode = mode; g->n0 = s->step;
    g->ids = malloc(sizeof(int32_t) * (size_t)(n + 1));
    g->x0 = malloc(sizeof(double) * (size_t)(n * s->D + 1));
    for (int c = 0; c < 3; ++c) g->du[c] = (mode == 1 && du && c < s->D) ? du[c] : 0.0;
    for (int64_t q = 0; q < n; ++q) {
        const int64_t p = ids[q];
        if (p < 0 || p >= s->N || (s->group_of[p] >= 0 && s->group_of[p] != gi)) return -2;
        g->ids[q] = (int32_t)p;
        s->group_of[p] = (int8_t)gi;
        for (int c = 0; c < s->D; ++c) {
            g->x0[q * s->D + c] = s->x[p * s->D + c];                    /* origin = current position (Q6) */
            s->v[p * s->D + c] = g->du[c] / s->dt;                       /* stored velocity of a kinematic particle */
        }
    }
    return 0;
}

/* One call = n_steps velocity-Verlet steps (Eq. 3-5, half-step-velocity form, L76). */
int32_t olsm_step(olsm_sim *s, int64_t n_steps)
{
    if (!s || n_steps < 0) return -1;
    const int D = s->D;
    const double dt = s->dt, hdt = 0.5 * s->dt;
    for (int64_t it = 0; it < n_steps; ++it) {
        /* 1-2. first half kick (Eq. 5, first half) and drift (Eq. 3) of the free particles */
        #pragma omp parallel for schedule(static) num_threads(s->threads) if (s->threads > 1)
        for (int64_t p = 0; p < s->N; ++p) {
            if (s->group_of[p] >= 0) continue;
            for (int c = 0; c < D; ++c) {
                const double a = s->fd[p * D + c] / s->m[p];             /* Eq. 4: a = F/m */
                s->v[p * D + c] = s->v[p * D + c] + hdt * a;
                s->x[p * D + c] = s->x[p * D + c] + dt * s->v[p * D + c];
            }
        }
        /* boundary displacement ("first applied", L88): closed form origin + steps*du, no accumulation drift (Q6) */
        for (int gi = 0; gi < OLSM_MAX_GROUPS; ++gi) {
            const ogroup *g = &s->g[gi];
            const double ns = (double)(s->step + 1 - g->n0);
            for (int64_t q = 0; q < g->n; ++q)
                for (int c = 0; c < D; ++c) {
                    s->x[g->ids[q] * D + c] = g->x0[q * D + c] + ns * g->du[c];
                    s->v[g->ids[q] * D + c] = g->du[c] / dt;
                }
        }
        /* 3. forces at the new positions (Eq. 4) + breakage (L98) */
        s->step += 1;
        if (s->threads > 1) force_eval_threads(s); else force_eval(s);
        /* 4. damping with the half-step velocity (Q7) */
        damp(s);
        /* 5. second half kick (Eq. 5, second half) */
        #pragma omp parallel for schedule(static) num_threads(s->threads) if (s->threads > 1)
        for (int64_t p = 0; p < s->N; ++p) {
            if (s->group_of[p] >= 0) continue;
            for (int c = 0; c < D; ++c) {
                const double a = s->fd[p * D + c] / s->m[p];
                s->v[p * D + c] = s->v[p * D + c] + hdt * a;
            }
        }
        /* 6. samples */
        if (s->sample_every > 0 && s->step % s->sample_every == 0) record_sample(s);
    }
    return 0;
}

/* Overwrite x and v (restart / perturbation), re-evaluate forces at the current step. Kinematic particles keep
 * their group; their origin is re-snapshotted from the new positions. */
int32_t olsm_write_state(olsm_sim *s, const double *x, const double *v)
{
    if (!s || !x) return -1;
    const size_t nd = (size_t)(s->N * s->D);
    memcpy(s->x, x, sizeof(double) * nd);
    if (v) memcpy(s->v, v, sizeof(double) * nd); else memset(s->v, 0, sizeof(double) * nd);
    for (int gi = 0; gi < OLSM_MAX_GROUPS; ++gi) {
        ogroup *g = &s->g[gi];
        g->n0 = s->step;
        for (int64_t q = 0; q < g->n; ++q)
            for (int c = 0; c < s->D; ++c) {
                g->x0[q * s->D + c] = s->x[g->ids[q] * s->D + c];
                s->v[g->ids[q] * s->D + c] = g->du[c] / s->dt;
            }
    }
    if (s->threads > 1) force_eval_threads(s); else force_eval(s);
    damp(s);
    return 0;
}

/* Run the following steps on n OpenMP threads (n <= 1: the serial loop).  Builds the per-particle incidence lists. */
int32_t olsm_set_threads(olsm_sim *s, int32_t n)
{
    if (!s) return -1;
    if (n > 1 && !s->adj_off) {
        s->adj_off = calloc((size_t)(s->N + 1), sizeof(int64_t));
        s->adj_e = malloc(sizeof(int32_t) * (size_t)(2 * s->M + 1));
        s->gs = calloc((size_t)(s->M + 1), sizeof(double));
        s->ue = calloc((size_t)(s->M + 1), sizeof(double));
        s->act = calloc((size_t)(s->M + 1), 1);
        for (int64_t e = 0; e < s->M; ++e) { s->adj_off[s->si[e] + 1]++; s->adj_off[s->sj[e] + 1]++; }
        for (int64_t p = 0; p < s->N; ++p) s->adj_off[p + 1] += s->adj_off[p];
        int64_t *fill = malloc(sizeof(int64_t) * (size_t)(s->N + 1));
        memcpy(fill, s->adj_off, sizeof(int64_t) * (size_t)(s->N + 1));
        for (int64_t e = 0; e < s->M; ++e) {               /* ascending e -> every list is ascending */
            s->adj_e[fill[s->si[e]]++] = (int32_t)e;
            s->adj_e[fill[s->sj[e]]++] = (int32_t)e;
        }
        free(fill);
    }
    s->threads = n > 1 ? n : 0;
    return 0;
}

int32_t olsm_read_state(const olsm_sim *s, double *x, double *v)
{
    if (!s) return -1;
    if (x) memcpy(x, s->x, sizeof(double) * (size_t)(s->N * s->D));
    if (v) memcpy(v, s->v, sizeof(double) * (size_t)(s->N * s->D));
    return 0;
}

int32_t olsm_read_forces(const olsm_sim *s, double *f)
{
    if (!s || !f) return -1;
    memcpy(f, s->f, sizeof(double) * (size_t)(s->N * s->D));
    return 0;
}

int32_t olsm_read_broken(const olsm_sim *s, uint8_t *broken, int64_t *break_step, int64_t *n_broken)
{
    if (!s) return -1;
    int64_t nb = 0;
    for (int64_t e = 0; e < s->M; ++e) {
        if (broken) broken[e] = !s->alive[e];
        if (break_step) break_step[e] = s->break_step[e];
        nb += !s->alive[e];
    }
    if (n_broken) *n_broken = nb;
    return 0;
}

/* Current per-specimen energies: U of the last force evaluation, KE of the current velocities. */
int32_t olsm_read_energy(olsm_sim *s, double *U, double *KE)
{
    if (!s) return -1;
    sum_U(s);
    for (int b = 0; b < s->B; ++b) {
        if (U) U[b] = s->U[b];
        if (KE) {
            double ke = 0.0;
            for (int64_t p = s->poff[b]; p < s->poff[b + 1]; ++p) {
                if (s->group_of[p] >= 0) continue;
                double v2 = 0.0;
                for (int c = 0; c < s->D; ++c) v2 = v2 + s->v[p * s->D + c] * s->v[p * s->D + c];
                ke += 0.5 * s->m[p] * v2;
            }
            KE[b] = ke;
        }
    }
    return 0;
}

/* Per-particle virial, Eq. 7 without the 1/Omega factor (the caller divides by a volume):
 *   S^k_ij = 1/2 sum_l (x^l_i - x^k_i) f^kl_j  -  m^k v^k_i v^k_j ,   f^kl = force on k from its spring to l (Eq. 2).
 * Serial loop over the alive springs in caller order; out[k] = {S_xx, S_yy, S_xy} in 2-D, {S_xx, S_yy, S_zz, S_xy, S_yz,
 * S_zx} in 3-D (symmetric: central forces).
 * Tension is positive.  Broken springs and coincident endpoints contribute nothing (Q3, Q4). */
int32_t olsm_read_virial(const olsm_sim *s, double *out)
{
    if (!s || !out) return -1;
    const int D = s->D, C = D == 2 ? 3 : 6;   /* D = 3: out[k] = {S_xx, S_yy, S_zz, S_xy, S_yz, S_zx} */
    for (int64_t q = 0; q < C * s->N; ++q) out[q] = 0.0;
    for (int64_t e = 0; e < s->M; ++e) {
        if (!s->alive[e]) continue;
        const int64_t i = s->si[e], j = s->sj[e];
        double d[3] = {0.0, 0.0, 0.0}, r2 = 0.0;
        for (int c = 0; c < D; ++c) { d[c] = s->x[D * j + c] - s->x[D * i + c]; r2 = r2 + d[c] * d[c]; }
        const double r = sqrt(r2);
        if (r == 0.0) continue;
        const double g = s->k[e] * (r - s->r0[e]) / r;      /* f^ij = g d,  f^ji = -g (-d): same dyad on both ends */
        const double h = 0.5 * g;
        double t[6];
        if (D == 2) { t[0] = h * d[0] * d[0]; t[1] = h * d[1] * d[1]; t[2] = h * d[0] * d[1]; }
        else { t[0] = h * d[0] * d[0]; t[1] = h * d[1] * d[1]; t[2] = h * d[2] * d[2]; t[3] = h * d[0] * d[1]; t[4] = h * d[1] * d[2]; t[5] = h * d[2] * d[0]; }
        for (int c = 0; c < C; ++c) { out[C * i + c] += t[c]; out[C * j + c] += t[c]; }
    }
    for (int64_t p = 0; p < s->N; ++p) {
        const double *v = s->v + D * p;
        const double m = s->m[p];
        if (D == 2) { out[3 * p] -= m * v[0] * v[0]; out[3 * p + 1] -= m * v[1] * v[1]; out[3 * p + 2] -= m * v[0] * v[1]; }
        else {
            out[6 * p] -= m * v[0] * v[0]; out[6 * p + 1] -= m * v[1] * v[1]; out[6 * p + 2] -= m * v[2] * v[2];
            out[6 * p + 3] -= m * v[0] * v[1]; out[6 * p + 4] -= m * v[1] * v[2]; out[6 * p + 5] -= m * v[2] * v[0];
        }
    }
    return 0;
}

/* Per-particle Lagrangian strain, Eq. 8: eps^L = (J J^T - delta) / 2 with "J the locally affine
 * transformation matrix considering the relative displacement of particle with its first nearest neighbors" (L156; the
 * method of Shimizu et al. 2007 cited at L145).  The printed index form "J_ij J_ji" has lost its summation: reading Q21.
 *   neighbours of p   the particles joined to p by a spring that is alive now (its "first nearest neighbours" in a
 *                     spring network are the particles it is bonded to; a broken bond is no longer one);
 *   reference         the positions given to olsm_create, d0 = xref_l - xref_p;  current d = x_l - x_p;
 *   J                 Shimizu's row-vector map d0 J ~ d in the least-squares sense: J = V^-1 W, V = sum d0^T d0,
 *                     W = sum d0^T d.  In column-vector language F = J^T = (sum d (x) d0) V^-1 is the deformation
 *                     gradient and J J^T = F^T F, so eps = (F^T F - I)/2, the Green-Lagrange strain; symmetric.
 *   rank deficiency   fewer than D independent reference bonds (det V <= 1e-12 (tr V / D)^D): eps = 0 and ok[p] = 0.
 * out[p] = {e_xx, e_yy, e_xy} in 2-D, {e_xx, e_yy, e_zz, e_xy, e_yz, e_zx} in 3-D (the layout of olsm_read_virial);
 * ok may be NULL.  Serial loop over the alive springs in caller order, then one solve per particle. */
int32_t olsm_read_strain(const olsm_sim *s, double *out, uint8_t *ok)
{
    if (!s || !out) return -1;
    const int D = s->D, C = D == 2 ? 3 : 6;
    double *V = calloc((size_t)(s->N * 9), sizeof(double)), *W = calloc((size_t)(s->N * 9), sizeof(double));
    if (!V || !W) { free(V); free(W); return -2; }
    for (int64_t e = 0; e < s->M; ++e) {
        if (!s->alive[e]) continue;
        const int64_t i = s->si[e], j = s->sj[e];
        double d0[3] = {0.0, 0.0, 0.0}, d[3] = {0.0, 0.0, 0.0};
        for (int c = 0; c < D; ++c) { d0[c] = s->xref[D * j + c] - s->xref[D * i + c]; d[c] = s->x[D * j + c] - s->x[D * i + c]; }
        /* the bond seen from j is (-d0, -d): the same dyads, so both ends add the same terms */
        for (int a = 0; a < D; ++a)
            for (int b = 0; b < D; ++b) {
                V[9 * i + 3 * a + b] += d0[a] * d0[b]; V[9 * j + 3 * a + b] += d0[a] * d0[b];
                W[9 * i + 3 * a + b] += d[a] * d0[b];  W[9 * j + 3 * a + b] += d[a] * d0[b];      /* W = sum d (x) d0 */
            }
    }
    for (int64_t p = 0; p < s->N; ++p) {
        const double *v = V + 9 * p, *w = W + 9 * p;
        double inv[9], F[9], det, tr;
        for (int c = 0; c < C; ++c) out[C * p + c] = 0.0;
        if (ok) ok[p] = 0;
        if (D == 2) {
            det = v[0] * v[4] - v[1] * v[3];
            tr = 0.5 * (v[0] + v[4]);
            if (!(det > 1e-12 * tr * tr)) continue;
            inv[0] = v[4] / det; inv[1] = -v[1] / det; inv[3] = -v[3] / det; inv[4] = v[0] / det;
        } else {
            const double c00 = v[4] * v[8] - v[5] * v[7], c01 = v[5] * v[6] - v[3] * v[8], c02 = v[3] * v[7] - v[4] * v[6];
            det = v[0] * c00 + v[1] * c01 + v[2] * c02;
            tr = (v[0] + v[4] + v[8]) / 3.0;
            if (!(det > 1e-12 * tr * tr * tr)) continue;
            inv[0] = c00 / det; inv[1] = (v[2] * v[7] - v[1] * v[8]) / det; inv[2] = (v[1] * v[5] - v[2] * v[4]) / det;
            inv[3] = c01 / det; inv[4] = (v[0] * v[8] - v[2] * v[6]) / det; inv[5] = (v[2] * v[3] - v[0] * v[5]) / det;
            inv[6] = c02 / det; inv[7] = (v[1] * v[6] - v[0] * v[7]) / det; inv[8] = (v[0] * v[4] - v[1] * v[3]) / det;
        }
        for (int a = 0; a < D; ++a)
            for (int b = 0; b < D; ++b) {
                double t = 0.0;
                for (int c = 0; c < D; ++c) t += w[3 * a + c] * inv[3 * c + b];                   /* F = W V^-1 */
                F[3 * a + b] = t;
            }
        double E[9];
        for (int a = 0; a < D; ++a)
            for (int b = 0; b < D; ++b) {
                double t = 0.0;
                for (int c = 0; c < D; ++c) t += F[3 * c + a] * F[3 * c + b];                     /* (F^T F)_ab = (J J^T)_ab */
                E[3 * a + b] = 0.5 * (t - (a == b ? 1.0 : 0.0));
            }
        if (D == 2) { out[3 * p] = E[0]; out[3 * p + 1] = E[4]; out[3 * p + 2] = E[1]; }
        else { out[6 * p] = E[0]; out[6 * p + 1] = E[4]; out[6 * p + 2] = E[8]; out[6 * p + 3] = E[1]; out[6 * p + 4] = E[5]; out[6 * p + 5] = E[6]; }
        if (ok) ok[p] = 1;
    }
    free(V); free(W);
    return 0;
}

int64_t olsm_n_samples(const olsm_sim *s) { return s ? s->ns : -1; }
int64_t olsm_current_step(const olsm_sim *s) { return s ? s->step : -1; }

/* Copies (and clears) the recorded samples: step[ns], R[ns][B][8][D], U[ns][B], KE[ns][B], nb[ns][B]. */
int32_t olsm_read_stress(olsm_sim *s, int64_t capacity, int64_t *n_out, int64_t *step, double *R, double *U,
                         double *KE, int64_t *nb)
{
    if (!s || !n_out) return -1;
    const int64_t n = s->ns < capacity ? s->ns : capacity;
    const int64_t first = s->ns - n;                       /* keep the latest */
    const size_t rs = (size_t)(s->B * OLSM_MAX_GROUPS * s->D);
    if (step) memcpy(step, s->h_step + first, sizeof(int64_t) * (size_t)n);
    if (R) memcpy(R, s->h_R + first * rs, sizeof(double) * (size_t)n * rs);
    if (U) memcpy(U, s->h_U + first * s->B, sizeof(double) * (size_t)(n * s->B));
    if (KE) memcpy(KE, s->h_KE + first * s->B, sizeof(double) * (size_t)(n * s->B));
    if (nb) memcpy(nb, s->h_nb + first * s->B, sizeof(int64_t) * (size_t)(n * s->B));
    *n_out = n;
    s->ns = 0;
    return 0;
}

void olsm_destroy(olsm_sim *s)
{
    if (!s) return;
    for (int gi = 0; gi < OLSM_MAX_GROUPS; ++gi) { free(s->g[gi].ids); free(s->g[gi].x0); }
    free(s->poff); free(s->soff); free(s->x); free(s->xref); free(s->v); free(s->f); free(s->fd); free(s->m);
    free(s->si); free(s->sj); free(s->k); free(s->r0); free(s->rc); free(s->alive); free(s->break_step);
    free(s->nbroken); free(s->U); free(s->spec_of_spring); free(s->spec_of_particle); free(s->group_of);
    free(s->h_step); free(s->h_R); free(s->h_U); free(s->h_KE); free(s->h_nb);
    free(s->adj_off); free(s->adj_e); free(s->gs); free(s->ue); free(s->act);
    free(s);
}
