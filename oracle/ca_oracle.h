/*
 * ca_oracle.h -- ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, single-threaded CPU simulator of the batched-fitness hot path of
 * arxiv 2303.08123 ("GPU-GA in-silico"): one EMT6/Ro spheroid cellular-automaton
 * simulation under one radiotherapy protocol, fitness f = N_ref - n_occupied
 * (Eq. 1).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may build, load or call this.  It shares NO code with the CUDA
 * path (paper_2303_08123_b200/csrc, include/ca.h): this header is the oracle's
 * own and is never included from there.
 *
 * The paper names the model components but prints no
 * update rule; the rules are this build's readings G1..G24 listed in DESIGN.md
 * section 3 (taken from SURVEY.md section 8(c)).  Every function below cites
 * the passage / reading it follows.
 *
 * Precision: compiled with CA_REAL = double (THE oracle, libca_oracle_f64.so).
 * The same source compiled with CA_REAL = float (libca_oracle_f32.so) is a
 * diagnostic only: it takes every field-dependent decision in the kernel's own
 * precision so that a bit-for-bit comparison over long horizons is possible.
 */
#ifndef CA_ORACLE_H
#define CA_ORACLE_H
#include <stdint.h>

#ifndef CA_REAL
#define CA_REAL double
#endif
typedef CA_REAL real;

/* cell kinds, state bits 0-2 */
enum { K_EMPTY = 0, K_G1 = 1, K_S = 2, K_G2 = 3, K_M = 4, K_DEAD = 5, K_WALL = 7 };
#define ST_KIND(s)   ((s) & 7)
#define ST_MODE(s)   (((s) >> 3) & 3)   /* 0 PA, 1 PN, 2 QA, 3 QN */
#define ST_READY     0x20
#define ST_DOOMED    0x40

/* Philox purposes (counter word 3 low byte) */
enum { P_INIT_PHASE = 0, P_INIT_CLOCK = 1, P_PHASE_CLOCK = 2, P_IRRADIATE = 3,
       P_DIR = 4, P_CLAIM = 5, P_DAUGHTER_CLOCK = 6, P_PARENT_CLOCK = 7 };

/* counts layout */
enum { C_LIVE = 0, C_DOOMED = 1, C_READY = 2, C_DEAD = 3, C_PHASE0 = 4 /* G1,S,G2,M */,
       C_MODE0 = 8 /* PA,PN,QA,QN */, C_OCCUPIED = 12, C_NCOUNT = 13 };

/* Model parameters.  Every constant that takes part in floating-point
 * arithmetic or comparisons is STORED AS fp32 and widened, so oracle and
 * kernel compare against the same real numbers (reading G-FP). */
typedef struct {
    int32_t steps_per_hour;      /* 600 */
    int32_t n_sub;               /* diffusion sub-steps per CA step (G3) */
    float   lambda[3];           /* D*dt_sub/h^2 for O2, glucose, H+ ; each <= 1/6 (G3) */
    float   boundary[3];         /* medium values */
    float   rate[3][4];          /* signed source per sub-step [species][mode] (G4) */
    float   O_A, G_P, G_Q, H_P, H_Q;   /* mode thresholds (G5) */
    int32_t T[4], J[4];          /* phase durations / jitter, steps (G7) */
    float   alpha[4], beta[4];   /* LQ per phase (G10) */
    float   oer_m, oer_K;        /* oxygen modification (G10) */
    int32_t repair_period, repair_shift;   /* G11 */
    int32_t lysis_steps;         /* G12 */
    int32_t N_ref;               /* Eq. 1 constant; 0 => interior sites (G14) */
    int32_t well_mixed_medium;   /* != 0: EMPTY sites are held at the medium values (alternative reading of G2) */
} car_params;

typedef struct { int32_t kind; int32_t cx, cy, cz; float radius; int32_t shared_init; } car_init;
enum { INIT_SINGLE = 0, INIT_CLUSTER7 = 1, INIT_BALL = 2 };

typedef struct car_ctx car_ctx;

#ifdef __cplusplus
extern "C" {
#endif
void     car_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
uint32_t car_uniform_int(uint32_t x, uint32_t m);            /* G23 */
uint32_t car_bernoulli_threshold(double p);                  /* G23 */

car_ctx *car_create(int nx, int ny, int nz, const car_params *p);   /* NULL on invalid args */
void     car_destroy(car_ctx *c);
int      car_seed(car_ctx *c, const car_init *init, uint64_t rng_seed, uint32_t sim_id);
int      car_set_rng(car_ctx *c, uint64_t rng_seed, uint32_t sim_id);
int      car_set_protocol(car_ctx *c, const double *dose_gy, const double *delay_h, int nfrac, double t0_h);
int      car_fire_steps(car_ctx *c, int64_t *out, int cap);  /* returns nfrac */

/* one stage each, at the context's current step counter (does not advance it) */
void     car_stage_irradiate(car_ctx *c);
void     car_stage_diffuse(car_ctx *c);
void     car_stage_cells(car_ctx *c);
int      car_stage_divide(car_ctx *c);                       /* returns births */
void     car_diffuse_substeps(car_ctx *c, int m);            /* m Jacobi sub-steps only (pins P3-P6) */

void     car_step(car_ctx *c, int64_t nsteps);               /* irradiate, diffuse, cells, divide; ++step */
int      car_run(car_ctx *c, double t_end_h);
int64_t  car_get_step(const car_ctx *c);

void     car_counts(const car_ctx *c, int32_t out[C_NCOUNT]);
double   car_fitness(const car_ctx *c);

/* canonical export / import; fields are copied as double; any pointer may be NULL */
void     car_get_state(const car_ctx *c, uint8_t *state, uint16_t *clock, uint16_t *damage,
                       double *o2, double *glc, double *h);
int      car_set_state(car_ctx *c, const uint8_t *state, const uint16_t *clock, const uint16_t *damage,
                       const double *o2, const double *glc, const double *h, int64_t step);
int      car_real_bytes(void);
#ifdef __cplusplus
}
#endif
#endif
