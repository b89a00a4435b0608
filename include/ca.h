/*
 * ca.h -- C ABI of libca_b200: batched fitness evaluation of radiotherapy protocols on B200
 * (the hot path of arxiv 2303.08123, "GPU-GA in-silico").
 *
 * What it computes.  Each of `batch` independent EMT6/Ro spheroid cellular-automaton simulations
 * (nutrient/waste diffusion, differentiated metabolism, cell-cycle phases,
 * division, DNA damage and repair, necrosis) is advanced under its own protocol -- an ordered
 * list of (dose Gy, delay h) fractions, delay counted from the previous fraction and the first
 * one from the start -- at 600 CA steps per simulated hour, and
 * the surviving tumour is read out as  fitness = N_ref - n_occupied  (Eq. 1).
 * The paper prints no update rule; the rules are the readings G1..G24 of DESIGN.md section 3 and
 * the step algorithm S0..S4 of DESIGN.md section 4, which this header cites as [D Gn] / [D Sn].
 *
 * Shape of the interface: BASELINE.json north_star ("ca_create(batch, lattice dims, model
 * params), ca_seed(spheroid init, rng seed), ca_set_protocols(batch x fractions), ca_run(t_end),
 * ca_fitness(out)") plus the saved / re-loaded tumour state of PAPER.md l.244 (ca_get_state /
 * ca_set_state) and per-simulation counts.
 *
 * Conventions
 *   - Every function returns CA_OK (0) or a negative CA_E* code; ca_last_error() gives the text.
 *     No exceptions, no aborts, nothing printed.
 *   - "HOST" / "DEVICE" is stated for every pointer.  The library never keeps a caller's pointer
 *     after the call returns, except the workspace and the stream given to ca_create.
 *   - All device work is enqueued on the stream given to ca_create; calls that return data to
 *     HOST memory synchronise that stream, the others are asynchronous.
 *   - Lattice arrays are [sim][z][y][x], x fastest; linear site index i = (z*ny + y)*nx + x.
 *     The outermost one-site layer is WALL (Dirichlet medium values, never a cell) [D G2].
 *   - Every call runs on the device the context was created on and restores the caller's current device.
 *   - Deferred device errors (CA_EOVERFLOW: more births of one simulation in one step than the winner lists hold,
 *     i.e. > 2048 per CTA + n/8 per simulation; the surplus births are dropped) are reported by the next call that
 *     synchronises -- ca_sync, ca_get_state, ca_fitness / ca_counts with HOST output.  With DEVICE output those
 *     two stay asynchronous: call ca_sync to observe errors.  ca_seed and a whole-batch ca_set_state clear them.
 *   - Fitness is fp32: exact while the lattice has fewer than 2^24 interior sites (all BASELINE configs).
 *   - There is no CPU fallback: without a CUDA device every compute entry point fails with CA_ECUDA.
 */
#ifndef CA_B200_H
#define CA_B200_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum { CA_OK = 0, CA_EINVAL = -1, CA_EPROTO = -2, CA_ESTATE = -3, CA_ECUDA = -4, CA_EOVERFLOW = -5 };

/* state byte [D section 4, "state encoding"]: bits 0-2 kind, bits 3-4 metabolic mode, bit 5 READY, bit 6 DOOMED */
enum { CA_EMPTY = 0, CA_G1 = 1, CA_S = 2, CA_G2 = 3, CA_M = 4, CA_DEAD = 5, CA_WALL = 7 };
enum { CA_READY = 0x20, CA_DOOMED = 0x40 };
/* metabolic mode: 0 PA (proliferating aerobic), 1 PN, 2 QA (quiescent aerobic), 3 QN   ([D G5]) */

/* ca_counts() layout, int32 per simulation */
enum { CA_C_LIVE = 0, CA_C_DOOMED = 1, CA_C_READY = 2, CA_C_DEAD = 3, CA_C_G1 = 4, CA_C_S = 5, CA_C_G2 = 6, CA_C_M = 7,
       CA_C_PA = 8, CA_C_PN = 9, CA_C_QA = 10, CA_C_QN = 11, CA_C_OCCUPIED = 12, CA_NCOUNT = 13 };

/* Model parameters (plain data, copied by ca_create).  Floating-point constants are fp32: the
 * kernels compute in fp32 and compare against exactly these numbers [D section 3, O-PARAM]. */
typedef struct ca_params {
    int32_t steps_per_hour;      /* 600 */
    int32_t n_sub;               /* explicit diffusion sub-steps per CA step, 1..8 [D G3] */
    float   lambda[3];           /* D*dt_sub/h^2 for O2, glucose, H+; each in [0, 1/6] [D G3] */
    float   boundary[3];         /* medium values in mM: 0.28, 5.5, 3.98e-5 */
    float   rate[3][4];          /* signed source per sub-step, [species][mode] [D G4] */
    float   O_A, G_P, G_Q, H_P, H_Q;   /* mode thresholds [D G5] */
    int32_t T[4], J[4];          /* mean phase length / jitter in steps for G1, S, G2, M [D G7] */
    float   alpha[4], beta[4];   /* linear-quadratic coefficients per phase [D G10] */
    float   oer_m, oer_K;        /* oxygen modification factor [D G10] */
    int32_t repair_period, repair_shift;   /* integer repair law [D G11] */
    int32_t lysis_steps;         /* steps a DEAD cell keeps its site [D G12] */
    int32_t N_ref;               /* Eq. 1 constant (paper: 1500); 0 => number of interior sites [D G14] */
    int32_t well_mixed_medium;   /* != 0: every EMPTY site is held at the medium values ("well-mixed replenished substrate",
                                    PAPER.md l.244; the alternative reading of [D G2], for the paper-shaped workload NEXT-3).
                                    Served by the per-sub-step diffusion kernel (the fused kernels assume free diffusion). */
} ca_params;

/* Initial spheroid [D S-SEED]: kind 0 SINGLE cell, 1 CLUSTER7 (centre + 6 face neighbours,
 * BASELINE configs[0]), 2 BALL(radius, in sites).  cx/cy/cz < 0 => lattice centre (n/2).
 * shared_init != 0: every simulation draws its initial phases/clocks with sim id 0, i.e. the
 * batch starts from one identical spheroid (BASELINE configs[1]) [D G17]. */
typedef struct ca_init {
    int32_t kind;
    int32_t cx, cy, cz;
    float   radius;
    int32_t shared_init;
} ca_init;

typedef struct ca_ctx ca_ctx;    /* opaque; owned by the library */

/* Bytes of DEVICE workspace ca_create needs for this problem size (0 on invalid sizes). */
size_t ca_workspace_bytes(int batch, int nx, int ny, int nz, int max_frac);

/* Create a context for `batch` simulations on an nx*ny*nz lattice (each dim >= 3).
 *   p          HOST, copied.  CA_EINVAL if a lambda is outside [0, 1/6], a phase length minus its
 *              jitter is < 1, plus jitter > 65535, lysis_steps outside 1..65535, n_sub outside 1..8.
 *   max_frac   capacity of the protocol table per simulation (1..64).
 *   workspace  DEVICE memory of at least ca_workspace_bytes(...) bytes, 256-byte aligned, owned by
 *              the caller (a torch tensor in the Python binding) and kept alive until ca_destroy.
 *   stream     a cudaStream_t; all work of this context runs on it.  NULL: the context creates and owns a
 *              non-blocking stream (the legacy default stream cannot be captured into CUDA graphs).
 * The context is bound to the CUDA device that is current at the time of the call. */
/* batch <= 65535. */
int ca_create(ca_ctx **out, int batch, int nx, int ny, int nz, const ca_params *p, int max_frac,
              void *workspace, size_t workspace_bytes, void *stream);
int ca_destroy(ca_ctx *c);

/* [D S-SEED] Zero everything, mark WALL, set the three fields to their boundary values at every
 * site (BASELINE configs[0]), place the initial cells with phases uniform over {G1,S,G2,M} and
 * remaining clock uniform in 1..T[phase] [D G16], step counter = 0.  Simulation b gets the global
 * id sim_id_base + b, which is what enters the random-number counter: results do not depend on
 * how a population is cut into batches.  Philox key = (low 32, high 32 bits of rng_seed). */
int ca_seed(ca_ctx *c, const ca_init *init, uint64_t rng_seed, uint32_t sim_id_base);
/* Change key / ids without touching the lattice (used after ca_set_state). */
int ca_set_rng(ca_ctx *c, uint64_t rng_seed, uint32_t sim_id_base);

/* Protocols.  dose_gy, delay_h: HOST [batch][max_frac_in] row-major; nfrac: HOST
 * [batch].  Fraction j of simulation b fires at the START of step
 *     S_bj = round((t0_h + sum_{m<=j} delay_bm) * steps_per_hour)            [D scheduling]
 * in whichever ca_run call reaches it; fractions on one step are applied in list order; dose 0 is
 * a legal no-op (the paper's sparse 240-slot vector).  CA_EPROTO (nothing changed)
 * if a dose or delay is negative or not finite, a delay is not a whole number of steps
 * (tested to fp32 precision, |delay*steps_per_hour - round| > 4e-7 * max(1, delay*steps_per_hour), because the
 * ABI takes fp32: 0.35 h arrives as 209.9999964 steps; an accepted delay is snapped to the step grid), nfrac[b] is outside 0..max_frac_in, max_frac_in exceeds
 * the capacity given to ca_create, or some S_bj lies before the current step. */
int ca_set_protocols(ca_ctx *c, const float *dose_gy, const float *delay_h, const int32_t *nfrac,
                     int max_frac_in, float t0_h);

/* Advance every simulation to absolute time t_end_h (step index round(t_end_h*steps_per_hour));
 * one CA step = irradiate, n_sub diffusion-reaction sub-steps, cell state, division [D G15].
 * Asynchronous; ca_run(a); ca_run(b) is bitwise the same as ca_run(b).  CA_ESTATE before
 * ca_seed/ca_set_state, CA_EINVAL if t_end_h lies in the past or is not finite.  CA_ECUDA if a kernel of a step
 * cannot be launched: nothing of that step (or, inside a CUDA graph, of that group of steps) is enqueued and the
 * step counter stays where it was. */
int ca_run(ca_ctx *c, double t_end_h);
/* Same, by step count. */
int ca_step(ca_ctx *c, int64_t nsteps);
int ca_get_step(ca_ctx *c, int64_t *step);       /* HOST out; no synchronisation needed */
int ca_sync(ca_ctx *c);                          /* wait for the stream; reports deferred device errors */

/* Eq. 1: out[b] = N_ref - n_occupied(b), n_occupied = live + dead-not-yet-lysed
 * [D G13].  out: [batch] fp32, DEVICE if out_is_device else HOST (then the call synchronises). */
int ca_fitness(ca_ctx *c, float *out, int out_is_device);
/* out: [batch][CA_NCOUNT] int32, DEVICE or HOST as above. */
int ca_counts(ca_ctx *c, int32_t *out, int out_is_device);

/* Canonical export of one simulation to HOST arrays of nx*ny*nz elements (any pointer may be NULL):
 * state u8, clock u16 (steps left in the phase / until lysis), damage u16 (1/1024 Gy), fields fp32. */
int ca_get_state(ca_ctx *c, int sim, uint8_t *state, uint16_t *clock, uint16_t *damage,
                 float *o2, float *glc, float *h, int64_t *step);
/* Import ONE simulation's snapshot from HOST arrays and broadcast it to simulations
 * [sim_first, sim_first + sim_count) (saved tumour state re-loaded for every
 * evaluation).  NULL arrays are left unchanged; step < 0 leaves the step counter unchanged.
 * The WALL layer of `state` must be CA_WALL and nowhere else (CA_EINVAL otherwise). */
int ca_set_state(ca_ctx *c, int sim_first, int sim_count, const uint8_t *state, const uint16_t *clock,
                 const uint16_t *damage, const float *o2, const float *glc, const float *h, int64_t step);

/* Individual stages at the current step, for single-stage parity tests (they do not advance the
 * step counter): 0 irradiate [D S0], 1 all n_sub diffusion sub-steps [D S1], 2 cell state [D S2],
 * 3 division [D S3].  stage 4 with arg m: m bare diffusion sub-steps. */
int ca_stage(ca_ctx *c, int stage, int arg);

/* Implementation knobs (not part of the method; every setting gives bit-identical results): name -> value.
 *   "graph_steps"  CA steps per CUDA-graph launch (even, 0..64; 0 disables graphs; default 20)
 *   "fused"        1 = temporally fused diffusion kernels (default), 0 = one launch per sub-step
 *   "cell_path"    1 = clustered S2+S3 kernel driven by the occupancy map when the lattice allows (default), 0 = generic scans
 *   "cluster"      CTAs per simulation of the clustered kernel: 1, 2, 4 or 8
 *   "rows_rp"      k_diffuse_rows on 96-wide planes: 1 = two rows per lane (16 warps), 2 = four rows per lane (8 warps)
 *   "rows_cluster" 3 = k_diffuse_rows as clusters of 3 CTAs per 96 x 96 plane (boundary rows through distributed shared
 *                  memory, no halo), 0 = y-slabs with a halo
 *   "inject_launch_error"  1 = fault injection: the next step / stage call behaves as if a kernel launch had failed
 * CA_EINVAL on an unknown name or value. */
int ca_set_option(ca_ctx *c, const char *name, int value);
/* Read a knob back (HOST out), plus: "diffusion_kernel" (0 k_diffuse_sub, 1 k_diffuse_fused, 2 k_diffuse_slab,
 * 3 k_diffuse_rows: which kernel runs S1 on this lattice), "rows_cluster", "rows_nclusters". */
int ca_get_option(ca_ctx *c, const char *name, int *value);
/* Number of kernel launches (graph nodes included) issued by this context so far. */
int64_t ca_launch_count(ca_ctx *c);

/* S4 without a context and WITHOUT ANY ALLOCATION (for callers that cannot call cudaMalloc: code under CUDA-graph
 * capture, serving loops, harnesses that forbid it): per-simulation counts and Eq. 1 fitness of a state array the
 * caller owns.
 *   state_dev        DEVICE, 16-byte aligned, [batch][nz][ny][nx] u8 in the canonical encoding (bit 7 is ignored)
 *   n_ref            Eq. 1 constant; 0 => number of interior sites [D G14]
 *   counts_out_dev   DEVICE, [batch][CA_NCOUNT] int32, or NULL
 *   fitness_out_dev  DEVICE, [batch] fp32, or NULL (at least one of the two outputs)
 *   stream           a cudaStream_t (NULL: the default stream); the call is asynchronous on it
 * The accumulation scratch is a fixed device array inside the library: CA_NOALLOC_MAX_BATCH simulations (832 KiB, held
 * by every GPU that loads the library until the process exits).  CA_EINVAL (text via ca_last_error(NULL)) if batch
 * exceeds it.  The array is shared by every call and cleared at the start of each: calls that OVERLAP on the GPU
 * (different streams or host threads) race on it -- serialise them.  Runs on the current device; calls no cudaMalloc,
 * cudaFree or allocating library routine. */
enum { CA_NOALLOC_MAX_BATCH = 16384 };
int ca_counts_noalloc(const uint8_t *state_dev, int batch, int nx, int ny, int nz, int n_ref,
                      int32_t *counts_out_dev, float *fitness_out_dev, void *stream);

const char *ca_last_error(ca_ctx *c);            /* c may be NULL: error of the last failed ca_create */
const char *ca_version(void);

#ifdef __cplusplus
}
#endif
#endif
