/*
 * ca_oracle.c -- ORACLE (test infrastructure, NOT the product).  See ca_oracle.h.
 *
 * One simulation, one thread, plain nested loops, fields in `real` (double for
 * the oracle proper).  No tiling, no fusion, no reordering: each stage is the
 * algorithm of DESIGN.md section 4 written out in its order and notation.
 *
 * Pinned by tests/test_oracle_*.py (pins P1..P15 of DESIGN.md section 5).
 * Parity unpinned (stated here as the contract requires): absolute tumour sizes /
 * growth rates / the paper's Tables 1-4 -- PAPER.md gives no rule or constant for
 * the CA (l.240 defers to refs 7, 14-16), so the model below is this build's
 * concretisation and only its internal consistency is pinned (pin P12 is
 * qualitative).
 */
#include "ca_oracle.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

struct car_ctx {
    int nx, ny, nz;
    int64_t n;                 /* nx*ny*nz, WALL layer included */
    car_params p;
    uint8_t  *state;
    uint16_t *clock;
    uint16_t *damage;
    real *f[3];                /* current fields: O2, glucose, H+ */
    real *g[3];                /* Jacobi scratch */
    int64_t step;
    uint32_t key[2];
    uint32_t sim_id;
    int seeded;
    /* protocol */
    int nfrac;
    int64_t *fire;             /* S_j */
    double  *dose;
    /* division scratch */
    int64_t *tgt;              /* per parent site: chosen target, -1 none */
    int64_t *win;              /* per target site: winning parent, -1 none */
    uint32_t *wkey;
};

/* ------------------------------------------------------------------ RNG -- */
/* Philox4x32-10, Salmon et al., SC'11 (pin P1: published known answers). */
void car_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; ++r) {
        uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* word 0 of philox(site, step, sim, purpose | aux << 8) */
static uint32_t rnd(const car_ctx *c, int64_t site, int64_t step, uint32_t sim, uint32_t purpose, uint32_t aux)
{
    uint32_t ctr[4] = { (uint32_t)site, (uint32_t)step, sim, purpose | (aux << 8) };
    uint32_t out[4];
    car_philox4x32_10(ctr, c->key, out);
    return out[0];
}

/* G23: uniform integer in [0, m) and Bernoulli threshold from one 32-bit word */
uint32_t car_uniform_int(uint32_t x, uint32_t m) { return (uint32_t)(((uint64_t)x * m) >> 32); }

uint32_t car_bernoulli_threshold(double p)
{
    double t = floor(p * 4294967296.0);
    if (t >= 4294967295.0) return 4294967295u;
    if (t <= 0.0) return 0u;
    return (uint32_t)t;
}

/* G7: clock drawn at entry of phase `kind` (1..4): T - J + U{0..2J} */
static uint16_t draw_clock(const car_ctx *c, int kind, int64_t site, uint32_t purpose)
{
    int T = c->p.T[kind - 1], J = c->p.J[kind - 1];
    uint32_t x = rnd(c, site, c->step, c->sim_id, purpose, 0);
    return (uint16_t)(T - J + (int)car_uniform_int(x, (uint32_t)(2 * J + 1)));
}

/* ------------------------------------------------------------- lifecycle -- */
static int is_wall(const car_ctx *c, int x, int y, int z)
{
    return x == 0 || y == 0 || z == 0 || x == c->nx - 1 || y == c->ny - 1 || z == c->nz - 1;
}

car_ctx *car_create(int nx, int ny, int nz, const car_params *p)
{
    if (nx < 3 || ny < 3 || nz < 3 || !p) return NULL;
    if (p->n_sub < 1 || p->steps_per_hour < 1) return NULL;
    for (int s = 0; s < 3; ++s)
        if (!(p->lambda[s] >= 0.0f) || (double)p->lambda[s] > 1.0 / 6.0) return NULL;
    for (int k = 0; k < 4; ++k)
        if (p->J[k] < 0 || p->T[k] - p->J[k] < 1 || p->T[k] + p->J[k] > 65535) return NULL;
    if (p->lysis_steps < 1 || p->lysis_steps > 65535 || p->repair_period < 1 ||
        p->repair_shift < 0 || p->repair_shift > 15) return NULL;
    car_ctx *c = (car_ctx *)calloc(1, sizeof(car_ctx));
    c->nx = nx; c->ny = ny; c->nz = nz; c->n = (int64_t)nx * ny * nz; c->p = *p;
    c->state  = (uint8_t *)calloc(c->n, 1);
    c->clock  = (uint16_t *)calloc(c->n, 2);
    c->damage = (uint16_t *)calloc(c->n, 2);
    for (int s = 0; s < 3; ++s) {
        c->f[s] = (real *)calloc(c->n, sizeof(real));
        c->g[s] = (real *)calloc(c->n, sizeof(real));
    }
    c->tgt = (int64_t *)malloc(c->n * sizeof(int64_t));
    c->win = (int64_t *)malloc(c->n * sizeof(int64_t));
    c->wkey = (uint32_t *)malloc(c->n * sizeof(uint32_t));
    return c;
}

void car_destroy(car_ctx *c)
{
    if (!c) return;
    free(c->state); free(c->clock); free(c->damage);
    for (int s = 0; s < 3; ++s) { free(c->f[s]); free(c->g[s]); }
    free(c->tgt); free(c->win); free(c->wkey); free(c->fire); free(c->dose);
    free(c);
}

int car_set_rng(car_ctx *c, uint64_t rng_seed, uint32_t sim_id)
{
    c->key[0] = (uint32_t)rng_seed; c->key[1] = (uint32_t)(rng_seed >> 32);
    c->sim_id = sim_id;
    return 0;
}

/* mode decision of O-S2(i) (G5); returns -1 if starved */
static int decide_mode(const car_ctx *c, int64_t i)
{
    real O = c->f[0][i], G = c->f[1][i], H = c->f[2][i];
    if (G < (real)c->p.G_Q || H > (real)c->p.H_Q) return -1;
    int prolif  = (G >= (real)c->p.G_P) && (H <= (real)c->p.H_P);
    int aerobic = (O >= (real)c->p.O_A);
    return 2 * (!prolif) + (!aerobic);
}

/* O-SEED (BASELINE configs[0]: fields at constant boundary values, Dirichlet faces,
 * cluster at centre, phases uniform from the seed; readings G2, G16, G17) */
int car_seed(car_ctx *c, const car_init *init, uint64_t rng_seed, uint32_t sim_id)
{
    car_set_rng(c, rng_seed, sim_id);
    memset(c->clock, 0, c->n * 2);
    memset(c->damage, 0, c->n * 2);
    c->step = 0;
    for (int z = 0; z < c->nz; ++z)
        for (int y = 0; y < c->ny; ++y)
            for (int x = 0; x < c->nx; ++x) {
                int64_t i = ((int64_t)z * c->ny + y) * c->nx + x;
                c->state[i] = is_wall(c, x, y, z) ? K_WALL : K_EMPTY;
                for (int s = 0; s < 3; ++s) c->f[s][i] = (real)c->p.boundary[s];
            }
    int cx = init->cx >= 0 ? init->cx : c->nx / 2;
    int cy = init->cy >= 0 ? init->cy : c->ny / 2;
    int cz = init->cz >= 0 ? init->cz : c->nz / 2;
    uint32_t sid = init->shared_init ? 0u : sim_id;
    double r2 = (double)init->radius * (double)init->radius;
    for (int z = 1; z < c->nz - 1; ++z)
        for (int y = 1; y < c->ny - 1; ++y)
            for (int x = 1; x < c->nx - 1; ++x) {
                int dx = x - cx, dy = y - cy, dz = z - cz;
                int d2 = dx * dx + dy * dy + dz * dz;
                int place;
                if (init->kind == INIT_SINGLE) place = (d2 == 0);
                else if (init->kind == INIT_CLUSTER7) place = (d2 <= 1);
                else if (init->kind == INIT_BALL) place = ((double)d2 <= r2);
                else return -1;
                if (!place) continue;
                int64_t i = ((int64_t)z * c->ny + y) * c->nx + x;
                int kind = 1 + (int)car_uniform_int(rnd(c, i, 0, sid, P_INIT_PHASE, 0), 4);
                int clk  = 1 + (int)car_uniform_int(rnd(c, i, 0, sid, P_INIT_CLOCK, 0), (uint32_t)c->p.T[kind - 1]);
                c->state[i] = (uint8_t)kind;
                c->clock[i] = (uint16_t)clk;
                int m = decide_mode(c, i);
                if (m < 0) m = 3;          /* boundary medium never starves with sane params */
                c->state[i] = (uint8_t)(kind | (m << 3));
            }
    c->seeded = 1;
    return 0;
}

/* Scheduling (delay = wait since previous fraction, first from the
 * start; l.262: 600 steps/h).  S_j = round((t0 + sum_{m<=j} delay_m) * steps_per_hour), G24. */
int car_set_protocol(car_ctx *c, const double *dose_gy, const double *delay_h, int nfrac, double t0_h)
{
    if (nfrac < 0) return -2;
    int64_t *fire = (int64_t *)malloc((nfrac + 1) * sizeof(int64_t));
    double  *dose = (double *)malloc((nfrac + 1) * sizeof(double));
    double t = t0_h;
    for (int j = 0; j < nfrac; ++j) {
        if (!(dose_gy[j] >= 0.0) || !(delay_h[j] >= 0.0)) { free(fire); free(dose); return -2; }
        double ds = delay_h[j] * c->p.steps_per_hour;
        if (fabs(ds - floor(ds + 0.5)) > 1e-6) { free(fire); free(dose); return -2; }
        t += delay_h[j];
        fire[j] = (int64_t)floor(t * c->p.steps_per_hour + 0.5);
        dose[j] = dose_gy[j];
        if (fire[j] < c->step) { free(fire); free(dose); return -2; }
    }
    free(c->fire); free(c->dose);
    c->fire = fire; c->dose = dose; c->nfrac = nfrac;
    return 0;
}

int car_fire_steps(car_ctx *c, int64_t *out, int cap)
{
    for (int j = 0; j < c->nfrac && j < cap; ++j) out[j] = c->fire[j];
    return c->nfrac;
}

/* ------------------------------------------------------------ O-S0 ------- */
/* Irradiation: LQ with incomplete repair (Lea-Catcheside form), phase- and oxygen-
 * dependent (reading G10; components named in PAPER.md l.32, l.294, l.309-310).
 * All arithmetic in fp64 (in the f32 diagnostic build too). */
void car_stage_irradiate(car_ctx *c)
{
    for (int j = 0; j < c->nfrac; ++j) {
        if (c->fire[j] != c->step) continue;
        double d = c->dose[j];
        if (!(d > 0.0)) continue;
        double m = (double)c->p.oer_m, K = (double)c->p.oer_K;
        for (int64_t i = 0; i < c->n; ++i) {
            int kind = ST_KIND(c->state[i]);
            if (kind < K_G1 || kind > K_M) continue;
            double O   = (double)c->f[0][i];
            double omf = (m * O + K) / ((O + K) * m);
            double de  = d * omf;
            double D   = (double)c->damage[i] / 1024.0;
            double a = (double)c->p.alpha[kind - 1], b = (double)c->p.beta[kind - 1];
            double E = a * de + b * de * de + 2.0 * b * de * D;
            double pk = -expm1(-E);
            uint32_t T = car_bernoulli_threshold(pk);
            if (rnd(c, i, c->step, c->sim_id, P_IRRADIATE, (uint32_t)j) < T)
                c->state[i] |= ST_DOOMED;
            double nd = (double)c->damage[i] + floor(1024.0 * de + 0.5);
            c->damage[i] = (uint16_t)(nd > 65535.0 ? 65535.0 : nd);
        }
    }
}

/* ------------------------------------------------------------ O-S1 ------- */
/* One explicit 7-point Jacobi sub-step of all three species (readings G2-G4).
 * The association of sum6, the un-fused 6*c and the single fma are part of the
 * definition (pin P5: a uniform field is reproduced bit-exactly). */
static void diffuse_once(car_ctx *c)
{
    const int nx = c->nx, ny = c->ny, nz = c->nz;
    const int64_t sx = 1, sy = nx, sz = (int64_t)nx * ny;
    for (int s = 0; s < 3; ++s) {
        const real *a = c->f[s];
        real *b = c->g[s];
        const real lam = (real)c->p.lambda[s];
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    int64_t i = ((int64_t)z * ny + y) * nx + x;
                    if (is_wall(c, x, y, z)) { b[i] = a[i]; continue; }
                    /* alternative reading of G2 ("well-mixed replenished substrate"): an EMPTY site is medium */
                    if (c->p.well_mixed_medium && ST_KIND(c->state[i]) == K_EMPTY) { b[i] = (real)c->p.boundary[s]; continue; }
                    real sum6 = ((a[i - sx] + a[i + sx]) + (a[i - sy] + a[i + sy])) + (a[i - sz] + a[i + sz]);
                    real six  = (real)6 * a[i];
                    real lap  = sum6 - six;
#if defined(CA_REAL_IS_FLOAT)
                    real v = fmaf(lam, lap, a[i]);
#else
                    real v = fma(lam, lap, a[i]);
#endif
                    int kind = ST_KIND(c->state[i]);
                    real r = (kind >= K_G1 && kind <= K_M) ? (real)c->p.rate[s][ST_MODE(c->state[i])] : (real)0;
                    v = v + r;
                    b[i] = v > (real)0 ? v : (real)0;
                }
    }
    for (int s = 0; s < 3; ++s) { real *t = c->f[s]; c->f[s] = c->g[s]; c->g[s] = t; }
}

void car_diffuse_substeps(car_ctx *c, int m) { for (int k = 0; k < m; ++k) diffuse_once(c); }
void car_stage_diffuse(car_ctx *c) { car_diffuse_substeps(c, c->p.n_sub); }

/* ------------------------------------------------------------ O-S2 ------- */
static void make_dead(car_ctx *c, int64_t i)
{
    c->state[i]  = K_DEAD;                       /* flags and mode cleared */
    c->clock[i]  = (uint16_t)c->p.lysis_steps;   /* G12 */
    c->damage[i] = 0;
}

/* Per-site cell-state update (readings G5-G7, G10-G12; components PAPER.md l.240) */
void car_stage_cells(car_ctx *c)
{
    for (int64_t i = 0; i < c->n; ++i) {
        uint8_t st = c->state[i];
        int kind = ST_KIND(st);
        if (kind == K_EMPTY || kind == K_WALL) continue;
        if (kind == K_DEAD) {
            c->clock[i] -= 1;
            if (c->clock[i] == 0) { c->state[i] = K_EMPTY; c->damage[i] = 0; }
            continue;
        }
        /* (i) metabolism */
        int mode = decide_mode(c, i);
        if (mode < 0) { make_dead(c, i); continue; }
        st = (uint8_t)((st & ~0x18) | (mode << 3));
        /* (ii) repair, G11 */
        if ((c->step + 1) % c->p.repair_period == 0 && c->damage[i] > 0) {
            int dec = c->damage[i] >> c->p.repair_shift;
            if (dec < 1) dec = 1;
            c->damage[i] = (uint16_t)(c->damage[i] - dec);
        }
        /* (iii) cycle, G6-G7 */
        if (mode < 2 && !(st & ST_READY)) {
            c->clock[i] -= 1;
            if (c->clock[i] == 0) {
                if (kind == K_G1 || kind == K_S) {
                    kind += 1;
                    st = (uint8_t)((st & ~7) | kind);
                    c->clock[i] = draw_clock(c, kind, i, P_PHASE_CLOCK);
                } else if (kind == K_G2) {
                    if (st & ST_DOOMED) { make_dead(c, i); continue; }   /* mitotic death, G10 */
                    kind = K_M;
                    st = (uint8_t)((st & ~7) | kind);
                    c->clock[i] = draw_clock(c, kind, i, P_PHASE_CLOCK);
                } else {   /* M finished */
                    st |= ST_READY;
                }
            }
        }
        c->state[i] = st;
    }
}

/* ------------------------------------------------------------ O-S3 ------- */
/* Division and placement, synchronous on the post-S2 lattice (readings G8, G9). */
int car_stage_divide(car_ctx *c)
{
    const int64_t off[6] = { -1, +1, -(int64_t)c->nx, +(int64_t)c->nx,
                             -(int64_t)c->nx * c->ny, +(int64_t)c->nx * c->ny };
    for (int64_t i = 0; i < c->n; ++i) { c->tgt[i] = -1; c->win[i] = -1; }
    /* 1-2: each parent picks its target */
    for (int64_t p = 0; p < c->n; ++p) {
        uint8_t st = c->state[p];
        if (ST_KIND(st) != K_M || !(st & ST_READY) || ST_MODE(st) >= 2) continue;
        int best_dir = -1; uint32_t best_key = 0;
        for (int d = 0; d < 6; ++d) {
            int64_t e = p + off[d];
            if (c->state[e] != K_EMPTY) continue;          /* WALL != EMPTY */
            uint32_t k = rnd(c, p, c->step, c->sim_id, P_DIR, (uint32_t)d);
            if (best_dir < 0 || k < best_key) { best_dir = d; best_key = k; }   /* ties -> lower dir */
        }
        if (best_dir >= 0) c->tgt[p] = p + off[best_dir];
    }
    /* 3: each contested site goes to the smallest (claim key, parent index) */
    for (int64_t p = 0; p < c->n; ++p) {
        int64_t e = c->tgt[p];
        if (e < 0) continue;
        uint32_t k = rnd(c, p, c->step, c->sim_id, P_CLAIM, 0);
        if (c->win[e] < 0 || k < c->wkey[e]) { c->win[e] = p; c->wkey[e] = k; }  /* p ascending: ties -> lower p */
    }
    /* 4: apply all winners */
    int births = 0;
    for (int64_t e = 0; e < c->n; ++e) {
        int64_t p = c->win[e];
        if (p < 0) continue;
        uint8_t ps = c->state[p];
        uint8_t keep = (uint8_t)(ps & (0x18 | ST_DOOMED));   /* mode and DOOMED carried (reading G10b) */
        c->state[p] = (uint8_t)(K_G1 | keep);
        c->clock[p] = draw_clock(c, K_G1, p, P_PARENT_CLOCK);
        c->state[e] = (uint8_t)(K_G1 | keep);
        c->clock[e] = draw_clock(c, K_G1, e, P_DAUGHTER_CLOCK);
        c->damage[e] = c->damage[p];
        ++births;
    }
    return births;
}

/* ------------------------------------------------------------ step loop --- */
/* Order inside a step: irradiate, diffuse/react, cell state, divide (reading G15). */
void car_step(car_ctx *c, int64_t nsteps)
{
    for (int64_t k = 0; k < nsteps; ++k) {
        car_stage_irradiate(c);
        car_stage_diffuse(c);
        car_stage_cells(c);
        car_stage_divide(c);
        c->step += 1;
    }
}

int car_run(car_ctx *c, double t_end_h)
{
    int64_t end = (int64_t)floor(t_end_h * c->p.steps_per_hour + 0.5);
    if (end < c->step) return -1;
    car_step(c, end - c->step);
    return 0;
}

int64_t car_get_step(const car_ctx *c) { return c->step; }

/* ------------------------------------------------------------ O-S4 ------- */
void car_counts(const car_ctx *c, int32_t out[C_NCOUNT])
{
    for (int k = 0; k < C_NCOUNT; ++k) out[k] = 0;
    for (int64_t i = 0; i < c->n; ++i) {
        uint8_t st = c->state[i];
        int kind = ST_KIND(st);
        if (kind >= K_G1 && kind <= K_M) {
            out[C_LIVE]++;
            if (st & ST_DOOMED) out[C_DOOMED]++;
            if (st & ST_READY) out[C_READY]++;
            out[C_PHASE0 + kind - 1]++;
            out[C_MODE0 + ST_MODE(st)]++;
        } else if (kind == K_DEAD) out[C_DEAD]++;
    }
    out[C_OCCUPIED] = out[C_LIVE] + out[C_DEAD];      /* G13 */
}

/* Eq. 1: f = N_ref - n_occupied (paper's N_ref = 1500; G14) */
double car_fitness(const car_ctx *c)
{
    int32_t cnt[C_NCOUNT];
    car_counts(c, cnt);
    double nref = c->p.N_ref > 0 ? (double)c->p.N_ref
                                 : (double)(c->nx - 2) * (double)(c->ny - 2) * (double)(c->nz - 2);
    return nref - (double)cnt[C_OCCUPIED];
}

/* ------------------------------------------------------------ state i/o -- */
void car_get_state(const car_ctx *c, uint8_t *state, uint16_t *clock, uint16_t *damage,
                   double *o2, double *glc, double *h)
{
    if (state)  memcpy(state, c->state, c->n);
    if (clock)  memcpy(clock, c->clock, c->n * 2);
    if (damage) memcpy(damage, c->damage, c->n * 2);
    double *dst[3] = { o2, glc, h };
    for (int s = 0; s < 3; ++s)
        if (dst[s]) for (int64_t i = 0; i < c->n; ++i) dst[s][i] = (double)c->f[s][i];
}

int car_set_state(car_ctx *c, const uint8_t *state, const uint16_t *clock, const uint16_t *damage,
                  const double *o2, const double *glc, const double *h, int64_t step)
{
    if (state)  memcpy(c->state, state, c->n);
    if (clock)  memcpy(c->clock, clock, c->n * 2);
    if (damage) memcpy(c->damage, damage, c->n * 2);
    const double *src[3] = { o2, glc, h };
    for (int s = 0; s < 3; ++s)
        if (src[s]) for (int64_t i = 0; i < c->n; ++i) c->f[s][i] = (real)src[s][i];
    if (step >= 0) c->step = step;
    c->seeded = 1;
    return 0;
}

int car_real_bytes(void) { return (int)sizeof(real); }
