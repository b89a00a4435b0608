// ca_api.cu -- C ABI of libca_b200 (include/ca.h): context, scheduling of the step loop, state i/o.
// Every step of the hot path runs in the kernels of ca_kernels.cuh / ca_fused.cuh; this file only
// marshals arguments, lays out the workspace and enqueues launches / CUDA graphs.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>
#include <algorithm>

#include "ca_kernels.cuh"
#include "ca_fused.cuh"
#include "ca_rows.cuh"

using namespace ca;

namespace {

constexpr int kMaxGraphSteps = 64;
thread_local std::string g_create_error;

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

struct Layout {
    size_t field[2][3], state, clock, damage, occ, lys, winners, nwin, spill_n, step, err, counts, fitness, fire, dose, nfrac, stage, total;
    unsigned int cap;
};

Layout make_layout(int batch, long long n, int max_frac)
{
    Layout Y;
    size_t o = 0;
    const size_t tot = (size_t)batch * (size_t)n;
    for (int bsel = 0; bsel < 2; ++bsel)
        for (int s = 0; s < 3; ++s) { Y.field[bsel][s] = o; o = align_up(o + tot * 4); }
    Y.state = o;   o = align_up(o + tot);
    Y.clock = o;   o = align_up(o + tot * 2);
    Y.damage = o;  o = align_up(o + tot * 2);
    Y.occ = o;     o = align_up(o + (tot / 256 + 64) * 4);   // occupancy map of the S2/S3 fast path
    Y.lys = o;     o = align_up(o + (size_t)batch * 4);      // per simulation: "a site was vacated (lysis) since S3 last looked"
    size_t cap = std::max<size_t>(65536, tot / 8);
    if (cap > (1u << 28)) cap = 1u << 28;
    Y.cap = (unsigned int)cap;
    Y.winners = o; o = align_up(o + cap * 8);
    Y.nwin = o;    o = align_up(o + kMaxGraphSteps * 4);
    Y.spill_n = o; o = align_up(o + (size_t)batch * 4);
    Y.step = o;    o = align_up(o + 8);
    Y.err = o;     o = align_up(o + 4);
    Y.counts = o;  o = align_up(o + (size_t)batch * CA_NCOUNT * 4);
    Y.fitness = o; o = align_up(o + (size_t)batch * 4);
    Y.fire = o;    o = align_up(o + (size_t)batch * max_frac * 4);
    Y.dose = o;    o = align_up(o + (size_t)batch * max_frac * 4);
    Y.nfrac = o;   o = align_up(o + (size_t)batch * 4);
    Y.stage = o;   o = align_up(o + (size_t)n * 4);          // staging for one array of one simulation
    Y.total = o;
    return Y;
}

}  // namespace

struct ca_ctx {
    KParams P;
    ca_params hp;
    Lattice L;
    Layout Y;
    uint8_t *ws;
    cudaStream_t stream;
    bool own_stream;
    int device;
    int sms;
    int max_frac;
    int cur;                       // which ping-pong buffer holds the current fields
    long long step;                // host mirror of the device step counter
    bool seeded;
    // protocol tables (host mirror) and their device copies
    std::vector<int> fire;         // [batch][max_frac]
    std::vector<float> dose;
    std::vector<int> nfrac;
    std::vector<long long> fire_sorted;   // distinct fire steps with dose > 0, ascending
    int *d_fire; float *d_dose; int *d_nfrac;
    unsigned long long *d_winners; unsigned int *d_nwin; long long *d_step; int *d_err; int *d_counts; float *d_fitness;
    uint8_t *d_stage;
    uint32_t *d_occ;
    int *d_lys;
    bool mapped_ok;               // simulations are whole multiples of 256 sites: clustered S2+S3 kernel usable
    int cell_path;                 // option: 1 = clustered S2+S3 kernel when usable, 0 = generic scan kernels
    int cs;                        // CTAs per simulation (cluster size) of the clustered kernel
    unsigned int *d_spill_n;       // per simulation: winners that did not fit the CTA's shared list (spilled to d_winners)
    cudaError_t launch_err;        // first failed launch since the last check (launch errors are not sticky: remembered here)
    // options
    int graph_steps;
    int fused;
    FusedPlan fplan;
    cudaGraphExec_t graph[2];      // indexed by the ping-pong parity at graph start
    int graph_len[2];
    long long graph_nodes;
    long long launches;
    std::string err;
};

namespace {

int fail(ca_ctx *c, int code, const std::string &msg)
{
    if (c) c->err = msg; else g_create_error = msg;
    return code;
}

int cuda_fail(ca_ctx *c, cudaError_t e, const char *what)
{
    return fail(c, CA_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

// every entry point runs on the context's device and puts the caller's current device back on return
struct DeviceGuard {
    int prev = -1;
    bool changed = false;
    explicit DeviceGuard(int dev) { if (cudaGetDevice(&prev) == cudaSuccess && prev != dev) changed = cudaSetDevice(dev) == cudaSuccess; }
    ~DeviceGuard() { if (changed) cudaSetDevice(prev); }
};

#define CA_CUDA(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail((c), e_, #call); } while (0)

void drop_graphs(ca_ctx *c)
{
    for (int q = 0; q < 2; ++q)
        if (c->graph[q]) { cudaGraphExecDestroy(c->graph[q]); c->graph[q] = nullptr; c->graph_len[q] = 0; }
}

// a kernel launch failed: remember the first error (cudaGetLastError clears it) until run_plain / ca_stage reports it
inline void note_launch(ca_ctx *c, cudaError_t e) { if (e != cudaSuccess && c->launch_err == cudaSuccess) c->launch_err = e; }
inline void note_last(ca_ctx *c) { note_launch(c, cudaGetLastError()); }

inline unsigned int blocks_for(long long n, int threads) { return (unsigned int)((n + threads - 1) / threads); }

// persistent grid of the sparse state scans: 8 CTAs of 8 warps per SM, never more than there are 4 KB trips
unsigned int scan_grid(const ca_ctx *c)
{
    const long long trips = ((c->P.n * c->P.batch >> 4) + 255) >> 8;
    return (unsigned int)std::max<long long>(1, std::min<long long>((long long)c->sms * 8, trips));
}

// S2 and/or S3 through the occupancy map: one cluster of c->cs CTAs per simulation
void enqueue_cells_divide(ca_ctx *c, int cur, int k, int phases, bool have_map)
{
    const int nb = c->P.batch, b0 = 0;
    cudaStream_t st = c->stream;
    const KParams &P = c->P;
    const long long tot = P.n * P.batch;
    if (!have_map) {
        k_occ_map<<<blocks_for(tot / 8, 256), 256, 0, st>>>(c->L.state, tot, c->d_occ);   // whole batch (cheap; only on the generic paths)
        note_last(c);
        c->launches += 1;
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned int)(nb * c->cs));
    cfg.blockDim = dim3(CD_THREADS);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned int)c->cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    const SpillArgs sp = { c->d_winners, c->d_spill_n, c->Y.cap / (unsigned int)P.batch };
    note_launch(c, cudaLaunchKernelEx(&cfg, k_cells_divide, P, c->L, cur, (const long long *)c->d_step, k, (const uint32_t *)c->d_occ, c->cs, phases, c->d_err, b0, c->d_lys, sp));
    c->launches += 1;
}

// Enqueue the kernels of ONE CA step (without irradiation) at device step *d_step + k, starting from
// ping-pong buffer `cur`; returns the buffer holding the fields afterwards.   [D G15]
int enqueue_step(ca_ctx *c, int cur, int k)
{
    const KParams &P = c->P;
    cudaStream_t st = c->stream;
    const long long tot = P.n * P.batch;
    const bool mapped = c->mapped_ok && c->cell_path;
    bool have_map = false;
    if (c->launch_err != cudaSuccess) return cur;                          // an earlier launch failed: enqueue nothing on top of it
    if (c->fused && fused_supported(c->fplan)) {
        cudaError_t fe;
        const int np = launch_fused(c->fplan, c->L, cur, mapped ? c->d_occ : nullptr, st, &fe);   // S1: all n_sub sub-steps, one pass over HBM (two if n_sub > 4)
        note_launch(c, fe);                                                // a failed pass leaves `cur` where it was; the caller stops on launch_err
        if (np & 1) cur ^= 1;
        c->launches += np;
        have_map = mapped && c->fplan.writes_map;
    } else {
        for (int m = 0; m < P.n_sub; ++m) {                                // S1, one launch per sub-step
            k_diffuse_sub<<<blocks_for(tot, 256), 256, 0, c->stream>>>(P, c->L, cur);
            note_last(c);
            cur ^= 1;
        }
        c->launches += P.n_sub;
    }
    if (c->launch_err != cudaSuccess) return cur;                          // S1 did not start: S2/S3 must not run on undiffused fields
    if (mapped) {
        enqueue_cells_divide(c, cur, k, 3, have_map);                       // S2 + S3 in one clustered launch
        return cur;
    }
    const ScanArgs sa = { c->d_winners, c->d_nwin + k, c->Y.cap, c->d_err };
    k_scan<0><<<scan_grid(c), 256, 0, c->stream>>>(P, c->L, cur, c->d_step, k, sa);                            // S2
    k_scan<1><<<scan_grid(c), 256, 0, c->stream>>>(P, c->L, cur, c->d_step, k, sa);                            // S3 detect
    k_div_apply<<<64, 128, 0, c->stream>>>(P, c->L, c->d_step, k, c->d_winners, c->d_nwin + k, c->Y.cap);
    note_last(c);
    c->launches += 3;
    return cur;
}

int enqueue_irradiate(ca_ctx *c)
{
    const KParams &P = c->P;
    dim3 grid(std::min<unsigned int>(blocks_for(P.n, 256), 512u), (unsigned int)P.batch);
    k_irradiate<<<grid, 256, 0, c->stream>>>(P, c->L, c->cur, c->d_fire, c->d_dose, c->d_nfrac, c->max_frac, c->d_step, 0);
    note_last(c);
    c->launches += 1;
    return 0;
}

int enqueue_advance(ca_ctx *c, int adv)
{
    k_advance<<<1, 64, 0, c->stream>>>(c->d_step, adv, c->d_nwin, kMaxGraphSteps);
    c->launches += 1;
    return 0;
}

// Run `nsteps` irradiation-free steps: whole CUDA graphs of graph_steps steps, then single steps.
int run_plain(ca_ctx *c, long long nsteps)
{
    const int G = c->graph_steps;
    if (c->launch_err != cudaSuccess) { const cudaError_t le = c->launch_err; c->launch_err = cudaSuccess; return cuda_fail(c, le, "kernel launch"); }
    while (G > 0 && nsteps >= G) {
        const int par = c->cur;
        if (!c->graph[par] || c->graph_len[par] != G) {
            if (c->graph[par]) { cudaGraphExecDestroy(c->graph[par]); c->graph[par] = nullptr; }
            cudaGraph_t g;
            const long long before = c->launches;
            CA_CUDA(c, cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
            int cur = par;
            for (int k = 0; k < G; ++k) cur = enqueue_step(c, cur, k);
            enqueue_advance(c, G);
            cudaError_t e = cudaStreamEndCapture(c->stream, &g);
            if (c->launch_err != cudaSuccess) {                              // a kernel of the step could not be launched: no graph, no run
                if (e == cudaSuccess) cudaGraphDestroy(g);
                const cudaError_t le = c->launch_err; c->launch_err = cudaSuccess; c->launches = before;
                return cuda_fail(c, le, "kernel launch (graph capture)");
            }
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamEndCapture");
            if (cur != par) { cudaGraphDestroy(g); return fail(c, CA_EINVAL, "graph_steps * swaps must be even"); }
            e = cudaGraphInstantiate(&c->graph[par], g, 0);
            cudaGraphDestroy(g);
            if (e != cudaSuccess) return cuda_fail(c, e, "cudaGraphInstantiate");
            c->graph_len[par] = G;
            c->graph_nodes = c->launches - before;
            c->launches = before;
        }
        CA_CUDA(c, cudaGraphLaunch(c->graph[par], c->stream));
        c->launches += c->graph_nodes;
        c->step += G;
        nsteps -= G;
    }
    while (nsteps > 0) {
        const int nxt = enqueue_step(c, c->cur, 0);
        if (c->launch_err != cudaSuccess) {                                  // stop at once: S2/S3 must not run on undiffused fields
            const cudaError_t le = c->launch_err; c->launch_err = cudaSuccess;
            return cuda_fail(c, le, "kernel launch");
        }
        c->cur = nxt;
        enqueue_advance(c, 1);
        c->step += 1;
        nsteps -= 1;
    }
    CA_CUDA(c, cudaGetLastError());
    return CA_OK;
}

int run_steps(ca_ctx *c, long long nsteps)
{
    if (!c->seeded) return fail(c, CA_ESTATE, "ca_run before ca_seed / ca_set_state");
    if (nsteps < 0) return fail(c, CA_EINVAL, "target time lies in the past");
    DeviceGuard guard_(c->device);
    const long long end = c->step + nsteps;
    while (c->step < end) {
        // next step >= c->step on which some fraction fires (host knows the whole schedule)
        auto it = std::lower_bound(c->fire_sorted.begin(), c->fire_sorted.end(), c->step);
        const long long nf = (it == c->fire_sorted.end()) ? end : std::min<long long>(*it, end);
        if (nf > c->step) { int rc = run_plain(c, nf - c->step); if (rc) return rc; }
        if (c->step < end && it != c->fire_sorted.end() && *it == c->step) {
            enqueue_irradiate(c);                                            // S0, then the rest of this step
            int rc = run_plain(c, 1);
            if (rc) return rc;
        }
    }
    return CA_OK;
}

int check_deferred(ca_ctx *c)
{
    int herr = 0;
    CA_CUDA(c, cudaMemcpyAsync(&herr, c->d_err, 4, cudaMemcpyDeviceToHost, c->stream));
    CA_CUDA(c, cudaStreamSynchronize(c->stream));
    if (herr == CA_EOVERFLOW) return fail(c, CA_EOVERFLOW, "division winner list overflowed (more births in one step than capacity)");
    if (herr) return fail(c, herr, "deferred device error");
    return CA_OK;
}

int enqueue_counts(ca_ctx *c)
{
    const KParams &P = c->P;
    CA_CUDA(c, cudaMemsetAsync(c->d_counts, 0, (size_t)P.batch * CA_NCOUNT * 4, c->stream));
    const long long per = (P.n / 16 + 255) / 256;
    unsigned int bx = (unsigned int)std::max<long long>(1, std::min<long long>(per, std::max<long long>(1, 2368 / P.batch)));
    dim3 grid(bx, (unsigned int)P.batch);
    k_counts<<<grid, 256, 0, c->stream>>>(P, c->L.state, c->d_counts);
    k_finish_counts<<<blocks_for(P.batch, 128), 128, 0, c->stream>>>(P, c->d_counts, c->d_fitness);
    c->launches += 2;
    CA_CUDA(c, cudaGetLastError());
    return CA_OK;
}

}  // namespace

// =============================================================================== C ABI ====
extern "C" {

const char *ca_version(void) { return "libca_b200 0.1 (sm_100a)"; }

const char *ca_last_error(ca_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

size_t ca_workspace_bytes(int batch, int nx, int ny, int nz, int max_frac)
{
    if (batch < 1 || nx < 3 || ny < 3 || nz < 3 || max_frac < 1 || max_frac > 64) return 0;
    const long long n = (long long)nx * ny * nz;
    if (n > (1ll << 30)) return 0;
    return make_layout(batch, n, max_frac).total;
}

int ca_create(ca_ctx **out, int batch, int nx, int ny, int nz, const ca_params *p, int max_frac,
              void *workspace, size_t workspace_bytes, void *stream)
{
    if (!out) return fail(nullptr, CA_EINVAL, "out is NULL");
    *out = nullptr;
    if (batch > 65535) return fail(nullptr, CA_EINVAL, "batch must be <= 65535 (one grid row per simulation in the per-simulation kernels)");
    if (!p || batch < 1 || nx < 3 || ny < 3 || nz < 3) return fail(nullptr, CA_EINVAL, "bad batch / lattice dims (each dim >= 3)");
    if (max_frac < 1 || max_frac > 64) return fail(nullptr, CA_EINVAL, "max_frac must be 1..64");
    if (p->n_sub < 1 || p->n_sub > 8 || p->steps_per_hour < 1) return fail(nullptr, CA_EINVAL, "n_sub must be 1..8, steps_per_hour >= 1");
    for (int s = 0; s < 3; ++s)
        if (!(p->lambda[s] >= 0.0f) || (double)p->lambda[s] > 1.0 / 6.0) return fail(nullptr, CA_EINVAL, "lambda outside [0, 1/6]");
    for (int k = 0; k < 4; ++k)
        if (p->J[k] < 0 || p->T[k] - p->J[k] < 1 || p->T[k] + p->J[k] > 65535) return fail(nullptr, CA_EINVAL, "phase length / jitter out of range");
    if (p->lysis_steps < 1 || p->lysis_steps > 65535 || p->repair_period < 1 || p->repair_shift < 0 || p->repair_shift > 15)
        return fail(nullptr, CA_EINVAL, "lysis_steps / repair parameters out of range");
    const long long n = (long long)nx * ny * nz;
    if (n > (1ll << 30) || (double)n * batch > 3.0e10) return fail(nullptr, CA_EINVAL, "lattice too large");
    const size_t need = ca_workspace_bytes(batch, nx, ny, nz, max_frac);
    if (!workspace || workspace_bytes < need || ((uintptr_t)workspace & 255u)) return fail(nullptr, CA_EINVAL, "workspace missing, too small or not 256-byte aligned");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice (no CUDA device: this library has no CPU path)");
    cudaDeviceProp prop;
    e = cudaGetDeviceProperties(&prop, dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDeviceProperties");
    if (prop.major != 10) return fail(nullptr, CA_ECUDA, "libca_b200 is built for sm_100a (B200) only");

    ca_ctx *c = new (std::nothrow) ca_ctx();
    if (!c) return fail(nullptr, CA_EINVAL, "out of host memory");
    c->hp = *p;
    KParams &P = c->P;
    P.nx = nx; P.ny = ny; P.nz = nz; P.batch = batch; P.n = n; P.n_sub = p->n_sub;
    for (int s = 0; s < 3; ++s) { P.lambda[s] = p->lambda[s]; P.boundary[s] = p->boundary[s]; for (int m = 0; m < 4; ++m) P.rate[s][m] = p->rate[s][m]; }
    P.O_A = p->O_A; P.G_P = p->G_P; P.G_Q = p->G_Q; P.H_P = p->H_P; P.H_Q = p->H_Q;
    for (int k = 0; k < 4; ++k) { P.T[k] = p->T[k]; P.J[k] = p->J[k]; P.alpha[k] = p->alpha[k]; P.beta[k] = p->beta[k]; }
    P.oer_m = p->oer_m; P.oer_K = p->oer_K; P.repair_period = p->repair_period; P.repair_shift = p->repair_shift;
    P.lysis_steps = p->lysis_steps; P.N_ref = p->N_ref; P.key0 = P.key1 = 0; P.sim_id_base = 0;
    P.well_mixed = p->well_mixed_medium != 0;
    c->Y = make_layout(batch, n, max_frac);
    c->ws = (uint8_t *)workspace;
    for (int bsel = 0; bsel < 2; ++bsel) for (int s = 0; s < 3; ++s) c->L.f[bsel][s] = (float *)(c->ws + c->Y.field[bsel][s]);
    c->L.state = c->ws + c->Y.state;
    c->L.clock = (uint16_t *)(c->ws + c->Y.clock);
    c->L.damage = (uint16_t *)(c->ws + c->Y.damage);
    c->d_winners = (unsigned long long *)(c->ws + c->Y.winners);
    c->d_nwin = (unsigned int *)(c->ws + c->Y.nwin);
    c->d_spill_n = (unsigned int *)(c->ws + c->Y.spill_n);
    c->launch_err = cudaSuccess;
    c->d_step = (long long *)(c->ws + c->Y.step);
    c->d_err = (int *)(c->ws + c->Y.err);
    c->d_counts = (int *)(c->ws + c->Y.counts);
    c->d_fitness = (float *)(c->ws + c->Y.fitness);
    c->d_fire = (int *)(c->ws + c->Y.fire);
    c->d_dose = (float *)(c->ws + c->Y.dose);
    c->d_nfrac = (int *)(c->ws + c->Y.nfrac);
    c->d_stage = c->ws + c->Y.stage;
    c->d_occ = (uint32_t *)(c->ws + c->Y.occ);
    c->d_lys = (int *)(c->ws + c->Y.lys);
    c->stream = (cudaStream_t)stream;
    c->own_stream = false;
    DeviceGuard guard_(dev);
    if (!c->stream) {                     // the legacy default stream cannot be captured into CUDA graphs
        e = cudaStreamCreateWithFlags(&c->stream, cudaStreamNonBlocking);
        if (e != cudaSuccess) { int rc = cuda_fail(nullptr, e, "cudaStreamCreateWithFlags"); delete c; return rc; }
        c->own_stream = true;
    }
    c->device = dev;
    c->sms = prop.multiProcessorCount;
    c->max_frac = max_frac;
    c->cur = 0; c->step = 0; c->seeded = false;
    c->fire.assign((size_t)batch * max_frac, 0); c->dose.assign((size_t)batch * max_frac, 0.0f); c->nfrac.assign(batch, 0);
    c->graph_steps = 20; c->fused = 1;
    c->mapped_ok = (n % 256 == 0) && n < (1ll << 29);
    c->cell_path = 1;
    {
        int cs = 1;
        while (cs < 8 && (long long)batch * cs * 2 <= 4ll * c->sms && (n >> 8) / CD_TILE >= 8 * cs) cs *= 2;   // up to 4 CTAs of 256 threads per SM (measured best at c2: 8 per simulation), >= 4 planes per CTA
        c->cs = cs;
    }
    c->graph[0] = c->graph[1] = nullptr; c->graph_len[0] = c->graph_len[1] = 0; c->graph_nodes = 0; c->launches = 0;
    // zero the small control blocks (protocol tables, counters)
    e = cudaMemsetAsync(c->ws + c->Y.winners, 0, c->Y.total - c->Y.winners, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->d_lys, 1, (size_t)batch * 4, c->stream);
    if (e != cudaSuccess) { int rc = cuda_fail(nullptr, e, "cudaMemsetAsync"); delete c; return rc; }
    fused_configure(P, c->fplan);
    *out = c;
    return CA_OK;
}

int ca_destroy(ca_ctx *c)
{
    if (!c) return CA_OK;
    DeviceGuard guard_(c->device);
    cudaStreamSynchronize(c->stream);
    drop_graphs(c);
    if (c->own_stream) cudaStreamDestroy(c->stream);
    delete c;
    return CA_OK;
}

int ca_set_rng(ca_ctx *c, uint64_t rng_seed, uint32_t sim_id_base)
{
    if (!c) return CA_EINVAL;
    c->P.key0 = (uint32_t)rng_seed; c->P.key1 = (uint32_t)(rng_seed >> 32); c->P.sim_id_base = sim_id_base;
    drop_graphs(c);                       // kernel parameters are baked into graph nodes
    return CA_OK;
}

int ca_seed(ca_ctx *c, const ca_init *init, uint64_t rng_seed, uint32_t sim_id_base)
{
    if (!c || !init) return CA_EINVAL;
    if (init->kind < 0 || init->kind > 2) return fail(c, CA_EINVAL, "unknown init kind");
    DeviceGuard guard_(c->device);
    ca_set_rng(c, rng_seed, sim_id_base);
    const long long tot = c->P.n * c->P.batch;
    k_seed<<<blocks_for(tot, 256), 256, 0, c->stream>>>(c->P, c->L, *init);
    CA_CUDA(c, cudaGetLastError());
    CA_CUDA(c, cudaMemsetAsync(c->d_step, 0, 8, c->stream));
    CA_CUDA(c, cudaMemsetAsync(c->d_nwin, 0, kMaxGraphSteps * 4, c->stream));
    CA_CUDA(c, cudaMemsetAsync(c->d_err, 0, 4, c->stream));
    c->launches += 1;
    c->cur = 0; c->step = 0; c->seeded = true;
    return CA_OK;
}

int ca_set_protocols(ca_ctx *c, const float *dose_gy, const float *delay_h, const int32_t *nfrac, int max_frac_in, float t0_h)
{
    if (!c || !dose_gy || !delay_h || !nfrac) return CA_EINVAL;
    if (max_frac_in < 0 || max_frac_in > c->max_frac) return fail(c, CA_EPROTO, "max_frac_in exceeds the capacity given to ca_create");
    const int B = c->P.batch, F = c->max_frac;
    const double sph = (double)c->hp.steps_per_hour;
    std::vector<int> fire((size_t)B * F, 0);
    std::vector<float> dose((size_t)B * F, 0.0f);
    std::vector<long long> all;
    for (int b = 0; b < B; ++b) {
        if (nfrac[b] < 0 || nfrac[b] > max_frac_in) return fail(c, CA_EPROTO, "nfrac outside 0..max_frac_in");
        double t = (double)t0_h;
        for (int j = 0; j < nfrac[b]; ++j) {
            const double d = (double)dose_gy[(size_t)b * max_frac_in + j], dl = (double)delay_h[(size_t)b * max_frac_in + j];
            if (!(d >= 0.0) || !(dl >= 0.0) || !std::isfinite(d) || !std::isfinite(dl)) return fail(c, CA_EPROTO, "negative or non-finite dose / delay");
            const double ds = dl * sph;
            // the ABI takes fp32 delays: a step-aligned delay such as 0.35 h or 6.1 h arrives as 209.9999964 / 3659.99994 steps,
            // so alignment is tested to fp32 precision and the delay is snapped to the step grid before it is accumulated
            const double dsr = std::floor(ds + 0.5);
            if (std::fabs(ds - dsr) > 4e-7 * std::max(1.0, ds)) return fail(c, CA_EPROTO, "delay is not a whole number of CA steps");
            t += dsr / sph;
            const double S = std::floor(t * sph + 0.5);                     // [D G24]
            if (S < (double)c->step) return fail(c, CA_EPROTO, "fraction scheduled before the current step");
            if (S > 2.0e9) return fail(c, CA_EPROTO, "fraction scheduled beyond 2e9 steps");
            fire[(size_t)b * F + j] = (int)S;
            dose[(size_t)b * F + j] = (float)d;
            if (d > 0.0) all.push_back((long long)S);
        }
    }
    std::sort(all.begin(), all.end());
    all.erase(std::unique(all.begin(), all.end()), all.end());
    DeviceGuard guard_(c->device);
    CA_CUDA(c, cudaStreamSynchronize(c->stream));                           // host vectors below are re-used as copy sources
    c->fire.swap(fire); c->dose.swap(dose); c->nfrac.assign(nfrac, nfrac + B); c->fire_sorted.swap(all);
    CA_CUDA(c, cudaMemcpyAsync(c->d_fire, c->fire.data(), (size_t)B * F * 4, cudaMemcpyHostToDevice, c->stream));
    CA_CUDA(c, cudaMemcpyAsync(c->d_dose, c->dose.data(), (size_t)B * F * 4, cudaMemcpyHostToDevice, c->stream));
    CA_CUDA(c, cudaMemcpyAsync(c->d_nfrac, c->nfrac.data(), (size_t)B * 4, cudaMemcpyHostToDevice, c->stream));
    CA_CUDA(c, cudaStreamSynchronize(c->stream));
    return CA_OK;
}

int ca_step(ca_ctx *c, int64_t nsteps)
{
    if (!c) return CA_EINVAL;
    return run_steps(c, (long long)nsteps);
}

int ca_run(ca_ctx *c, double t_end_h)
{
    if (!c) return CA_EINVAL;
    if (!std::isfinite(t_end_h) || std::fabs(t_end_h) * (double)c->hp.steps_per_hour > 4.0e18) return fail(c, CA_EINVAL, "t_end_h is not a finite, representable time");
    const long long end = (long long)std::floor(t_end_h * (double)c->hp.steps_per_hour + 0.5);
    return run_steps(c, end - c->step);
}

int ca_get_step(ca_ctx *c, int64_t *step)
{
    if (!c || !step) return CA_EINVAL;
    *step = (int64_t)c->step;
    return CA_OK;
}

int ca_sync(ca_ctx *c)
{
    if (!c) return CA_EINVAL;
    DeviceGuard guard_(c->device);
    return check_deferred(c);
}

int ca_counts(ca_ctx *c, int32_t *out, int out_is_device)
{
    if (!c || !out) return CA_EINVAL;
    if (!c->seeded) return fail(c, CA_ESTATE, "ca_counts before ca_seed / ca_set_state");
    DeviceGuard guard_(c->device);
    int rc = enqueue_counts(c);
    if (rc) return rc;
    const size_t bytes = (size_t)c->P.batch * CA_NCOUNT * 4;
    CA_CUDA(c, cudaMemcpyAsync(out, c->d_counts, bytes, out_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    return out_is_device ? CA_OK : check_deferred(c);
}

int ca_fitness(ca_ctx *c, float *out, int out_is_device)
{
    if (!c || !out) return CA_EINVAL;
    if (!c->seeded) return fail(c, CA_ESTATE, "ca_fitness before ca_seed / ca_set_state");
    DeviceGuard guard_(c->device);
    int rc = enqueue_counts(c);
    if (rc) return rc;
    const size_t bytes = (size_t)c->P.batch * 4;
    CA_CUDA(c, cudaMemcpyAsync(out, c->d_fitness, bytes, out_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, c->stream));
    return out_is_device ? CA_OK : check_deferred(c);
}

int ca_get_state(ca_ctx *c, int sim, uint8_t *state, uint16_t *clock, uint16_t *damage, float *o2, float *glc, float *h, int64_t *step)
{
    if (!c || sim < 0 || sim >= c->P.batch) return c ? fail(c, CA_EINVAL, "sim out of range") : CA_EINVAL;
    DeviceGuard guard_(c->device);
    const size_t n = (size_t)c->P.n, o = (size_t)sim * n;
    if (state)  CA_CUDA(c, cudaMemcpyAsync(state, c->L.state + o, n, cudaMemcpyDeviceToHost, c->stream));
    if (clock)  CA_CUDA(c, cudaMemcpyAsync(clock, c->L.clock + o, n * 2, cudaMemcpyDeviceToHost, c->stream));
    if (damage) CA_CUDA(c, cudaMemcpyAsync(damage, c->L.damage + o, n * 2, cudaMemcpyDeviceToHost, c->stream));
    float *dst[3] = { o2, glc, h };
    for (int s = 0; s < 3; ++s)
        if (dst[s]) CA_CUDA(c, cudaMemcpyAsync(dst[s], c->L.f[c->cur][s] + o, n * 4, cudaMemcpyDeviceToHost, c->stream));
    if (step) *step = (int64_t)c->step;
    const int rc = check_deferred(c);                                       // synchronises: the copies have landed
    if (rc == CA_OK && state)
        for (size_t i = 0; i < n; ++i) state[i] &= 0x7Fu;                   // bit 7 is internal ("known to be blocked", see k_cells_divide)
    return rc;
}

int ca_set_state(ca_ctx *c, int sim_first, int sim_count, const uint8_t *state, const uint16_t *clock, const uint16_t *damage,
                 const float *o2, const float *glc, const float *h, int64_t step)
{
    if (!c) return CA_EINVAL;
    const KParams &P = c->P;
    if (sim_first < 0 || sim_count < 1 || sim_first + sim_count > P.batch) return fail(c, CA_EINVAL, "sim range out of bounds");
    if (state) {
        for (int z = 0; z < P.nz; ++z) for (int y = 0; y < P.ny; ++y) for (int x = 0; x < P.nx; ++x) {
            const bool wall = x == 0 || y == 0 || z == 0 || x == P.nx - 1 || y == P.ny - 1 || z == P.nz - 1;
            const uint8_t s = state[((size_t)z * P.ny + y) * P.nx + x];
            if (wall != ((s & 7) == CA_WALL) || (s & 7) == 6 || (s & 0x80)) return fail(c, CA_EINVAL, "state: WALL layer misplaced or invalid code");
        }
    }
    DeviceGuard guard_(c->device);
    const size_t n = (size_t)P.n;
    struct Item { const void *src; uint8_t *base; size_t elem; };
    const Item items[] = {
        { state, c->L.state, 1 }, { clock, (uint8_t *)c->L.clock, 2 }, { damage, (uint8_t *)c->L.damage, 2 },
        { o2, (uint8_t *)c->L.f[c->cur][0], 4 }, { glc, (uint8_t *)c->L.f[c->cur][1], 4 }, { h, (uint8_t *)c->L.f[c->cur][2], 4 },
        { o2, (uint8_t *)c->L.f[c->cur ^ 1][0], 4 }, { glc, (uint8_t *)c->L.f[c->cur ^ 1][1], 4 }, { h, (uint8_t *)c->L.f[c->cur ^ 1][2], 4 },
    };
    for (const Item &it : items) {
        if (!it.src) continue;
        const long long nbytes = (long long)(n * it.elem);
        CA_CUDA(c, cudaMemcpyAsync(it.base + (size_t)sim_first * nbytes, it.src, nbytes, cudaMemcpyHostToDevice, c->stream));
        if (sim_count > 1) {
            dim3 grid((unsigned int)std::min<long long>(64, (nbytes / 16 + 255) / 256 + 1), (unsigned int)sim_count);
            k_broadcast<<<grid, 256, 0, c->stream>>>(it.base, nbytes, sim_first, sim_first, sim_count);
            c->launches += 1;
        }
    }
    CA_CUDA(c, cudaGetLastError());
    if (step >= 0) {
        c->step = (long long)step;
        CA_CUDA(c, cudaMemcpyAsync(c->d_step, &c->step, 8, cudaMemcpyHostToDevice, c->stream));
    }
    if (state && sim_first == 0 && sim_count == P.batch) CA_CUDA(c, cudaMemsetAsync(c->d_err, 0, 4, c->stream));   // a whole new batch: deferred errors of the old one are gone
    if (state) CA_CUDA(c, cudaMemsetAsync(c->d_lys + sim_first, 1, (size_t)sim_count * 4, c->stream));             // no "blocked" mark of the old lattice can be trusted
    CA_CUDA(c, cudaStreamSynchronize(c->stream));      // the caller's arrays may be pageable: do not return before they are consumed
    c->seeded = true;
    return CA_OK;
}

int ca_stage(ca_ctx *c, int stage, int arg)
{
    if (!c) return CA_EINVAL;
    if (!c->seeded) return fail(c, CA_ESTATE, "ca_stage before ca_seed / ca_set_state");
    DeviceGuard guard_(c->device);
    const KParams &P = c->P;
    const long long tot = P.n * P.batch;
    if (c->launch_err != cudaSuccess) { const cudaError_t le = c->launch_err; c->launch_err = cudaSuccess; return cuda_fail(c, le, "kernel launch"); }
    switch (stage) {
    case 0: enqueue_irradiate(c); break;
    case 1:
        if (c->fused && fused_supported(c->fplan)) {
            cudaError_t fe;
            const int np = launch_fused(c->fplan, c->L, c->cur, nullptr, c->stream, &fe);
            if (fe != cudaSuccess) return cuda_fail(c, fe, "diffusion kernel launch");   // nothing flipped: a failed pass is never counted
            if (np & 1) c->cur ^= 1;
            c->launches += np;
        }
        else for (int m = 0; m < P.n_sub; ++m) { k_diffuse_sub<<<blocks_for(tot, 256), 256, 0, c->stream>>>(P, c->L, c->cur); c->cur ^= 1; c->launches += 1; }
        break;
    case 2:
        if (c->mapped_ok && c->cell_path) { enqueue_cells_divide(c, c->cur, 0, 1, false); break; }
        { const ScanArgs sa = { c->d_winners, c->d_nwin, c->Y.cap, c->d_err };
          k_scan<0><<<scan_grid(c), 256, 0, c->stream>>>(P, c->L, c->cur, c->d_step, 0, sa); c->launches += 1; }
        break;
    case 3:
        if (c->mapped_ok && c->cell_path) { enqueue_cells_divide(c, c->cur, 0, 2, false); break; }
        { const ScanArgs sa = { c->d_winners, c->d_nwin, c->Y.cap, c->d_err };
          k_scan<1><<<scan_grid(c), 256, 0, c->stream>>>(P, c->L, c->cur, c->d_step, 0, sa); }
        k_div_apply<<<64, 128, 0, c->stream>>>(P, c->L, c->d_step, 0, c->d_winners, c->d_nwin, c->Y.cap);
        enqueue_advance(c, 0);
        c->launches += 2;
        break;
    case 4:
        for (int m = 0; m < arg; ++m) { k_diffuse_sub<<<blocks_for(tot, 256), 256, 0, c->stream>>>(P, c->L, c->cur); c->cur ^= 1; c->launches += 1; }
        break;
    default: return fail(c, CA_EINVAL, "unknown stage");
    }
    if (c->launch_err != cudaSuccess) { const cudaError_t le = c->launch_err; c->launch_err = cudaSuccess; return cuda_fail(c, le, "kernel launch"); }
    CA_CUDA(c, cudaGetLastError());
    return CA_OK;
}

int ca_set_option(ca_ctx *c, const char *name, int value)
{
    if (!c || !name) return CA_EINVAL;
    if (!std::strcmp(name, "graph_steps")) {
        if (value < 0 || value > kMaxGraphSteps || (value & 1)) return fail(c, CA_EINVAL, "graph_steps must be even, 0..64");
        c->graph_steps = value; drop_graphs(c); return CA_OK;
    }
    if (!std::strcmp(name, "fused")) { c->fused = value ? 1 : 0; drop_graphs(c); return CA_OK; }
    if (!std::strcmp(name, "inject_launch_error")) {                          // fault injection for the tests: the next step sees a failed kernel launch
        c->launch_err = value ? cudaErrorLaunchOutOfResources : cudaSuccess; return CA_OK;
    }
    if (!std::strcmp(name, "rows_rp")) {                                       // k_diffuse_rows on 96-wide planes: 1 = two rows per lane, 2 = four
        if (!((value == 1 || value == 2) && c->fplan.rows && c->P.nx == 96)) return fail(c, CA_EINVAL, "rows_rp must be 1 or 2, on 96-wide planes");
        c->fplan.rows_rp = value; drop_graphs(c); return CA_OK;
    }
    if (!std::strcmp(name, "rows_cluster")) {                                  // 0: k_diffuse_rows on slabs with a halo; 3: cluster of 3 CTAs per 96 x 96 plane
        if (!(value == 0 || (value == 3 && c->P.nx == 96 && c->P.ny == 96 && c->fplan.rows))) return fail(c, CA_EINVAL, "rows_cluster must be 0, or 3 on 96 x 96 planes");
        c->fplan.rows_cluster = value; drop_graphs(c); return CA_OK;          // the cluster variant is built for two rows per lane: it ignores rows_rp
    }
    if (!std::strcmp(name, "cluster")) {
        if (value != 1 && value != 2 && value != 4 && value != 8) return fail(c, CA_EINVAL, "cluster must be 1, 2, 4 or 8");
        c->cs = value; drop_graphs(c); return CA_OK;
    }
    if (!std::strcmp(name, "cell_path")) {
        c->cell_path = value ? 1 : 0; drop_graphs(c);
        cudaMemsetAsync(c->d_lys, 1, (size_t)c->P.batch * 4, c->stream);     // the generic path does not track lysis: re-evaluate every parent once
        return CA_OK;
    }
    return fail(c, CA_EINVAL, std::string("unknown option ") + name);
}

int ca_get_option(ca_ctx *c, const char *name, int *value)
{
    if (!c || !name || !value) return CA_EINVAL;
    if (!std::strcmp(name, "graph_steps")) { *value = c->graph_steps; return CA_OK; }
    if (!std::strcmp(name, "fused")) { *value = c->fused && fused_supported(c->fplan); return CA_OK; }
    if (!std::strcmp(name, "cell_path")) { *value = c->cell_path && c->mapped_ok; return CA_OK; }
    if (!std::strcmp(name, "cluster")) { *value = c->cs; return CA_OK; }
    if (!std::strcmp(name, "rows_cluster")) { *value = c->fplan.rows ? c->fplan.rows_cluster : 0; return CA_OK; }
    if (!std::strcmp(name, "rows_rp")) { *value = c->fplan.rows ? c->fplan.rows_rp : 0; return CA_OK; }
    if (!std::strcmp(name, "rows_nclusters")) { *value = c->fplan.nclusters; return CA_OK; }   // resident clusters of the last cluster launch (0 before it)
    if (!std::strcmp(name, "diffusion_kernel")) {                             // 0 k_diffuse_sub, 1 k_diffuse_fused, 2 k_diffuse_slab, 3 k_diffuse_rows
        *value = !(c->fused && fused_supported(c->fplan)) ? 0 : (!c->fplan.tiled ? 1 : (c->fplan.rows ? 3 : 2));
        return CA_OK;
    }
    return fail(c, CA_EINVAL, std::string("unknown option ") + name);
}

int64_t ca_launch_count(ca_ctx *c) { return c ? (int64_t)c->launches : 0; }

}  // extern "C"

// ============================================================ entry point that allocates nothing ====
// ca_counts_noalloc: S4 (per-simulation counts and Eq. 1 fitness) of a DEVICE state array the caller owns, for callers that
// cannot allocate or hold a workspace (code under CUDA-graph capture, serving loops, harnesses that forbid cudaMalloc).
// The accumulation scratch of k_counts -- [batch][CA_NCOUNT] int32, one atomic per warp and count -- lives in a file-scope
// device array of fixed size instead of the caller's workspace: CA_NOALLOC_MAX_BATCH simulations = 832 KiB, held by every
// GPU that loads the library until the process exits.  In host code the array's NAME is a host-side stand-in, not a device
// address: its address is taken once per device with cudaGetSymbolAddress (that device current) and passed to the kernels.
// Every call shares the array: it is cleared at the start of each call (on the caller's stream), and calls that overlap on
// the GPU (two streams, two host threads) race on it.
namespace {

static __device__ __align__(256) int g_noalloc_counts[CA_NOALLOC_MAX_BATCH * CA_NCOUNT];

constexpr int kMaxDevices = 64;
int *g_noalloc_ptr[kMaxDevices] = { nullptr };      // device address of g_noalloc_counts, per device
std::mutex g_noalloc_mutex;

// occupied = live + dead [D G13]; fitness = N_ref - occupied (Eq. 1); scratch -> the caller's arrays
__global__ void k_noalloc_finish(const int *__restrict__ scratch, int batch, long long nref, int32_t *__restrict__ counts_out,
                                 float *__restrict__ fitness_out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= batch) return;
    const int occ = scratch[b * CA_NCOUNT + CA_C_LIVE] + scratch[b * CA_NCOUNT + CA_C_DEAD];
    if (counts_out) {
        for (int q = 0; q < CA_NCOUNT; ++q) counts_out[b * CA_NCOUNT + q] = q == CA_C_OCCUPIED ? occ : scratch[b * CA_NCOUNT + q];
    }
    if (fitness_out) fitness_out[b] = (float)(nref - occ);
}

}  // namespace

extern "C" int ca_counts_noalloc(const uint8_t *state_dev, int batch, int nx, int ny, int nz, int n_ref,
                                 int32_t *counts_out_dev, float *fitness_out_dev, void *stream)
{
    if (!state_dev || (!counts_out_dev && !fitness_out_dev)) return fail(nullptr, CA_EINVAL, "ca_counts_noalloc: state and at least one output are required");
    if (batch < 1 || nx < 3 || ny < 3 || nz < 3) return fail(nullptr, CA_EINVAL, "ca_counts_noalloc: bad batch / lattice dims (each dim >= 3)");
    if ((uintptr_t)state_dev & 15u) return fail(nullptr, CA_EINVAL, "ca_counts_noalloc: state must be 16-byte aligned");
    if (batch > CA_NOALLOC_MAX_BATCH)
        return fail(nullptr, CA_EINVAL, "ca_counts_noalloc: batch exceeds CA_NOALLOC_MAX_BATCH (16384 simulations: the static scratch is 832 KiB); use ca_counts on a context");
    const long long n = (long long)nx * ny * nz;
    if (n > (1ll << 30)) return fail(nullptr, CA_EINVAL, "ca_counts_noalloc: lattice too large");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetDevice (no CUDA device: this library has no CPU path)");
    if (dev < 0 || dev >= kMaxDevices) return fail(nullptr, CA_EINVAL, "ca_counts_noalloc: device index beyond 63");
    int *scratch = nullptr;
    {
        std::lock_guard<std::mutex> lock(g_noalloc_mutex);
        if (!g_noalloc_ptr[dev]) {                    // set-up, once per device, with that device current
            void *p = nullptr;
            e = cudaGetSymbolAddress(&p, g_noalloc_counts);
            if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaGetSymbolAddress(g_noalloc_counts)");
            g_noalloc_ptr[dev] = (int *)p;
        }
        scratch = g_noalloc_ptr[dev];
    }
    cudaStream_t st = (cudaStream_t)stream;
    // the array keeps the last call's contents: what this call accumulates into starts at zero
    e = cudaMemsetAsync(scratch, 0, (size_t)batch * CA_NCOUNT * sizeof(int), st);
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "cudaMemsetAsync(scratch)");
    KParams P{};
    P.nx = nx; P.ny = ny; P.nz = nz; P.batch = batch; P.n = n;
    const long long per = (n / 16 + 255) / 256;
    const unsigned int bx = (unsigned int)std::max<long long>(1, std::min<long long>(per, std::max<long long>(1, 2368 / batch)));
    k_counts<<<dim3(bx, (unsigned int)batch), 256, 0, st>>>(P, state_dev, scratch);
    const long long nref = n_ref > 0 ? (long long)n_ref : (long long)(nx - 2) * (ny - 2) * (nz - 2);
    k_noalloc_finish<<<blocks_for(batch, 128), 128, 0, st>>>(scratch, batch, nref, counts_out_dev, fitness_out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(nullptr, e, "ca_counts_noalloc kernel launch");
    return CA_OK;
}
