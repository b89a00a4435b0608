// ca_kernels.cuh -- per-stage kernels of one CA step over the whole batch (sm_100a).
// Stage numbering follows DESIGN.md section 4: S-SEED, S0 irradiate, S1 diffusion-reaction,
// S2 cell state, S3 division, S4 counts/fitness.
#pragma once
#include "ca_device.cuh"

namespace ca {

// ------------------------------------------------------------------ S-SEED --
// [D S-SEED] BASELINE configs[0]: fields at constant boundary values, WALL layer, cluster at centre,
// phases uniform from the seed.  One thread per site of the whole batch.
__global__ void k_seed(KParams P, Lattice L, ca_init init)
{
    const long long gi = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi >= P.n * P.batch) return;
    const int b = (int)(gi / P.n);
    const uint32_t i = (uint32_t)(gi - (long long)b * P.n);
    const int x = i % P.nx, y = (i / P.nx) % P.ny, z = i / (P.nx * P.ny);
    const bool wall = x == 0 || y == 0 || z == 0 || x == P.nx - 1 || y == P.ny - 1 || z == P.nz - 1;
#pragma unroll
    for (int s = 0; s < 3; ++s) { L.f[0][s][gi] = P.boundary[s]; L.f[1][s][gi] = P.boundary[s]; }
    uint8_t st = wall ? CA_WALL : CA_EMPTY;
    uint16_t ck = 0;
    if (!wall) {
        const int cx = init.cx >= 0 ? init.cx : P.nx / 2;
        const int cy = init.cy >= 0 ? init.cy : P.ny / 2;
        const int cz = init.cz >= 0 ? init.cz : P.nz / 2;
        const int dx = x - cx, dy = y - cy, dz = z - cz;
        const int d2 = dx * dx + dy * dy + dz * dz;
        bool place;
        if (init.kind == 0) place = (d2 == 0);
        else if (init.kind == 1) place = (d2 <= 1);
        else place = ((double)d2 <= (double)init.radius * (double)init.radius);
        if (place) {
            const uint32_t sid = init.shared_init ? 0u : P.sim_id_base + (uint32_t)b;
            const int kind = 1 + (int)uniform_int(rnd(P, i, 0u, sid, P_INIT_PHASE), 4u);
            ck = (uint16_t)(1 + (int)uniform_int(rnd(P, i, 0u, sid, P_INIT_CLOCK), (uint32_t)P.T[kind - 1]));
            int m = decide_mode(P, P.boundary[0], P.boundary[1], P.boundary[2]);
            if (m < 0) m = 3;
            st = (uint8_t)(kind | (m << 3));
        }
    }
    L.state[gi] = st;
    L.clock[gi] = ck;
    L.damage[gi] = 0;
}

// ---------------------------------------------------------------------- S0 --
// [D S0] Irradiation: LQ with incomplete repair, phase- and oxygen-dependent [D G10].  Launched by
// the host only on steps where some simulation has a fraction scheduled; each
// simulation checks its own fire-step table.  fp64 arithmetic: this runs on <= ~100 of 432 000 steps.
// grid = (chunks, batch)
__global__ void k_irradiate(KParams P, Lattice L, int cur, const int *__restrict__ fire, const float *__restrict__ dose,
                            const int *__restrict__ nfrac, int max_frac, const long long *__restrict__ d_step, int k)
{
    const int b = blockIdx.y;
    const long long step = *d_step + k;
    const int nf = nfrac[b];
    const int *fb = fire + (size_t)b * max_frac;
    const float *db = dose + (size_t)b * max_frac;
    bool any = false;
    for (int j = 0; j < nf; ++j) any |= (fb[j] == (int)step && db[j] > 0.0f);
    if (!any) return;
    const uint32_t sid = P.sim_id_base + (uint32_t)b;
    const double m = (double)P.oer_m, K = (double)P.oer_K;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.n; i += (long long)gridDim.x * blockDim.x) {
        const long long gi = (long long)b * P.n + i;
        uint32_t st = L.state[gi];
        if (!is_live(st)) continue;
        const int kind = st & 7;
        const double O = (double)L.f[cur][0][gi];
        const double omf = (m * O + K) / ((O + K) * m);
        const double al = (double)P.alpha[kind - 1], be = (double)P.beta[kind - 1];
        uint32_t D = L.damage[gi];
        for (int j = 0; j < nf; ++j) {
            if (fb[j] != (int)step) continue;
            const double d = (double)db[j];
            if (!(d > 0.0)) continue;
            const double de = d * omf;
            const double Dg = (double)D / 1024.0;
            const double E = al * de + be * de * de + 2.0 * be * de * Dg;
            const double pk = -expm1(-E);
            double t = floor(pk * 4294967296.0);                      // [D G23]
            const uint32_t T = t >= 4294967295.0 ? 4294967295u : (t <= 0.0 ? 0u : (uint32_t)t);
            if (rnd(P, (uint32_t)i, (uint32_t)step, sid, P_IRRADIATE, (uint32_t)j) < T) st |= CA_DOOMED;
            const double nd = (double)D + floor(1024.0 * de + 0.5);  // [D G24]
            D = nd > 65535.0 ? 65535u : (uint32_t)nd;
        }
        L.state[gi] = (uint8_t)st;
        L.damage[gi] = (uint16_t)D;
    }
}

// ---------------------------------------------------------------------- S1 --
// [D S1] ONE explicit 7-point Jacobi sub-step of all three species, plain global loads.
// Reference-grade kernel (the `fused = 0` path): one launch per sub-step, 25 B/site of traffic each.
__global__ void k_diffuse_sub(KParams P, Lattice L, int src)
{
    const long long gi = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (gi >= P.n * P.batch) return;
    const uint32_t i = (uint32_t)(gi % P.n);
    const int x = i % P.nx, y = (i / P.nx) % P.ny, z = i / (P.nx * P.ny);
    const bool wall = x == 0 || y == 0 || z == 0 || x == P.nx - 1 || y == P.ny - 1 || z == P.nz - 1;
    const int dst = src ^ 1;
    if (wall) {
#pragma unroll
        for (int s = 0; s < 3; ++s) L.f[dst][s][gi] = L.f[src][s][gi];
        return;
    }
    const uint32_t st = L.state[gi];
    if (P.well_mixed && (st & 7u) == CA_EMPTY) {                              // well-mixed medium: an EMPTY site is held at the medium values
#pragma unroll
        for (int s = 0; s < 3; ++s) L.f[dst][s][gi] = P.boundary[s];
        return;
    }
    const bool lv = is_live(st);
    const int mode = (st >> 3) & 3;
    const long long sy = P.nx, sz = (long long)P.nx * P.ny;
#pragma unroll
    for (int s = 0; s < 3; ++s) {
        const float *a = L.f[src][s];
        const float r = lv ? P.rate[s][mode] : 0.0f;
        L.f[dst][s][gi] = stencil_point(a[gi], a[gi - 1], a[gi + 1], a[gi - sy], a[gi + sy], a[gi - sz], a[gi + sz],
                                        P.lambda[s], r);
    }
}

// ---------------------------------------------------------------------- S2 --
// [D S2] Per-site cell-state update, in place (a site reads only itself and the post-S1 fields).
__device__ __forceinline__ void cell_update(const KParams &P, uint32_t &st, uint32_t &ck, uint32_t &dm,
                                            float O, float G, float H, uint32_t site, uint32_t step, uint32_t sid)
{
    const int kind = st & 7;
    if (kind == CA_DEAD) {
        ck -= 1;
        if (ck == 0) { st = CA_EMPTY; dm = 0; }
        return;
    }
    const int mode = decide_mode(P, O, G, H);                            // (i) metabolism [D G5]
    if (mode < 0) { st = CA_DEAD; ck = (uint32_t)P.lysis_steps; dm = 0; return; }
    st = (st & ~0x18u) | ((uint32_t)mode << 3);
    if (dm > 0 && (step + 1) % (uint32_t)P.repair_period == 0) {          // (ii) repair [D G11]
        uint32_t dec = dm >> P.repair_shift;
        dm -= dec < 1 ? 1 : dec;
    }
    if (mode < 2 && !(st & CA_READY)) {                                    // (iii) cycle [D G6, G7]
        ck -= 1;
        if (ck == 0) {
            if (kind == CA_G1 || kind == CA_S) {
                st = (st & ~7u) | (uint32_t)(kind + 1);
                ck = draw_clock(P, kind + 1, site, step, sid, P_PHASE_CLOCK);
            } else if (kind == CA_G2) {
                if (st & CA_DOOMED) { st = CA_DEAD; ck = (uint32_t)P.lysis_steps; dm = 0; return; }   // mitotic death [D G10]
                st = (st & ~7u) | CA_M;
                ck = draw_clock(P, CA_M, site, step, sid, P_PHASE_CLOCK);
            } else {
                st |= CA_READY;                                            // M finished: waits for space
            }
        }
    }
}

// S2 for one occupied site
__device__ __forceinline__ uint32_t cells_site(const KParams &P, const Lattice &L, int cur, long long gi, uint32_t st, uint32_t step)
{
    const int b = (int)(gi / P.n);
    const uint32_t i = (uint32_t)(gi - (long long)b * P.n);
    uint32_t ck = L.clock[gi], dm = L.damage[gi];
    const uint32_t st0 = st, ck0 = ck, dm0 = dm;
    cell_update(P, st, ck, dm, L.f[cur][0][gi], L.f[cur][1][gi], L.f[cur][2][gi], i, step, P.sim_id_base + (uint32_t)b);
    if (st != st0) L.state[gi] = (uint8_t)st;
    if (ck != ck0) L.clock[gi] = (uint16_t)ck;
    if (dm != dm0) L.damage[gi] = (uint16_t)dm;
    return st;
}

// Sparse scan of the state array shared by S2 and S3.  A persistent grid walks the flat array in 16-byte
// chunks per lane (4 KB per CTA and trip, the next trip prefetched).  At configs[1] ~99 % of the chunks hold no
// cell and cost a few compares; when a CTA finds sites of interest it compacts them into a shared-memory
// queue and works them off one site per thread, so a dense tumour core is spread over all 256 threads
// instead of serialising inside the lanes that happened to load it.
//   MODE 0: S2, sites holding a cell (kind not EMPTY / WALL);   MODE 1: S3, READY parents.
template <int MODE>
__device__ __forceinline__ uint32_t scan_word_mask(uint32_t w)
{
    uint32_t m = 0;
    if (MODE == 0) {
        if ((((w & 0x07070707u) + 0x01010101u) & 0x06060606u) == 0u) return 0u;   // every byte EMPTY or WALL
#pragma unroll
        for (int r = 0; r < 4; ++r) {
            const uint32_t kind = (w >> (8 * r)) & 7u;
            m |= (kind != CA_EMPTY && kind != CA_WALL) ? (1u << r) : 0u;
        }
    } else {
        if ((w & 0x20202020u) == 0u) return 0u;                                    // no READY byte
#pragma unroll
        for (int r = 0; r < 4; ++r) m |= is_parent((w >> (8 * r)) & 0xFFu) ? (1u << r) : 0u;
    }
    return m;
}

struct ScanArgs {                 // S3 only
    unsigned long long *winners;
    unsigned int *nwin;
    unsigned int cap;
    int *err;
};

__device__ __forceinline__ void detect_site(const KParams &P, const Lattice &L, long long gi, uint32_t step,
                                            unsigned long long *__restrict__ winners, unsigned int *__restrict__ nwin,
                                            unsigned int cap, int *__restrict__ err);

template <int MODE>
__global__ void __launch_bounds__(256) k_scan(KParams P, Lattice L, int cur, const long long *__restrict__ d_step, int k, ScanArgs S)
{
    // one trip of a CTA = 256 lanes x 16 bytes = 4 KB of the state array (one 64x64 plane at configs[1])
    __shared__ uint32_t queue[4096];
    __shared__ uint32_t qn;
    const long long tot = P.n * P.batch;
    const long long nchunk = tot >> 4;
    const uint32_t step = (uint32_t)(*d_step + k);
    const int lane = threadIdx.x & 31;
    const long long ntrip = (nchunk + 255) >> 8;
    if (threadIdx.x == 0) qn = 0;
    __syncthreads();
    long long trip = blockIdx.x;
    uint4 w = make_uint4(0u, 0u, 0u, 0u);
    if (trip < ntrip && trip * 256 + threadIdx.x < nchunk) w = reinterpret_cast<const uint4 *>(L.state)[trip * 256 + threadIdx.x];
    for (; trip < ntrip; trip += gridDim.x) {
        const uint32_t ws[4] = { w.x, w.y, w.z, w.w };
        const long long nxt = trip + gridDim.x;                                     // prefetch the next trip before working on this one
        w = make_uint4(0u, 0u, 0u, 0u);
        if (nxt < ntrip && nxt * 256 + threadIdx.x < nchunk) w = reinterpret_cast<const uint4 *>(L.state)[nxt * 256 + threadIdx.x];
        uint32_t m = 0;
#pragma unroll
        for (int q = 0; q < 4; ++q) m |= scan_word_mask<MODE>(ws[q]) << (4 * q);
        if (!__syncthreads_or(m != 0u)) continue;                                    // nothing of interest in these 4 KB
        // compact the sites of interest of the whole CTA into the queue (order is irrelevant to the result)
        const uint32_t cnt = __popc(m);
        uint32_t pre = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const uint32_t v = __shfl_up_sync(0xFFFFFFFFu, pre, o);
            if (lane >= o) pre += v;
        }
        uint32_t base = 0;
        if (lane == 31 && pre) base = atomicAdd(&qn, pre);
        base = __shfl_sync(0xFFFFFFFFu, base, 31);
        uint32_t pos = base + pre - cnt;
        uint32_t mm = m;
        while (mm) {
            const int bit = __ffs(mm) - 1;
            mm &= mm - 1;
            const uint32_t st = (ws[bit >> 2] >> (8 * (bit & 3))) & 0xFFu;
            queue[pos++] = (uint32_t)(threadIdx.x * 16 + bit) | (st << 16);
        }
        __syncthreads();
        const uint32_t total = qn;
        for (uint32_t r = threadIdx.x; r < total; r += 256) {
            const uint32_t e = queue[r];
            const long long gi = trip * 4096 + (e & 0xFFFFu);
            if (MODE == 0) cells_site(P, L, cur, gi, e >> 16, step);
            else detect_site(P, L, gi, step, S.winners, S.nwin, S.cap, S.err);
        }
        __syncthreads();
        if (threadIdx.x == 0) qn = 0;                                                // ordered before the next use by the __syncthreads_or above
    }
    if (blockIdx.x == 0 && threadIdx.x == 0)                                       // ragged tail of the flat array (tot % 16 sites)
        for (long long gi = nchunk * 16; gi < tot; ++gi) {
            const uint32_t st = L.state[gi];
            const uint32_t kind = st & 7u;
            if (MODE == 0) { if (kind != CA_EMPTY && kind != CA_WALL) cells_site(P, L, cur, gi, st, step); }
            else if (is_parent(st)) detect_site(P, L, gi, step, S.winners, S.nwin, S.cap, S.err);
        }
}

// ---------------------------------------------------------------------- S3 --
// [D S3, G8, G9] Division and placement with deterministic conflict resolution and no racy atomics:
// every decision is a pure function of the post-S2 lattice, so the detect kernel only READS the
// lattice and appends the winners (parent, direction) to a list; the apply kernel then writes them.
//
// choose_dir: the EMPTY face-neighbour of parent p with the smallest (Philox DIR key, dir); -1 if none.
__device__ __forceinline__ uint32_t empty_mask(const uint8_t *__restrict__ sb, uint32_t p, int nx, int nxny)
{
    const uint8_t *q = sb + p;
    // six independent L2 loads (a neighbour may have been written by another SM in S2); offsets in the order of [D G8]
    const uint32_t n0 = __ldcg(q - 1), n1 = __ldcg(q + 1), n2 = __ldcg(q - nx), n3 = __ldcg(q + nx), n4 = __ldcg(q - nxny), n5 = __ldcg(q + nxny);
    return (n0 == CA_EMPTY ? 1u : 0u) | (n1 == CA_EMPTY ? 2u : 0u) | (n2 == CA_EMPTY ? 4u : 0u) | (n3 == CA_EMPTY ? 8u : 0u) |
           (n4 == CA_EMPTY ? 16u : 0u) | (n5 == CA_EMPTY ? 32u : 0u);          // WALL != EMPTY: targets are interior
}

__device__ __forceinline__ int choose_dir_from(const KParams &P, uint32_t em, uint32_t p, uint32_t step, uint32_t sid)
{
    int best = -1;
    uint32_t bk = 0;
#pragma unroll
    for (int d = 0; d < 6; ++d) {
        if (!((em >> d) & 1u)) continue;
        const uint32_t kk = rnd(P, p, step, sid, P_DIR, (uint32_t)d);
        if (best < 0 || kk < bk) { best = d; bk = kk; }                    // ties -> lower dir
    }
    return best;
}

__device__ __forceinline__ int choose_dir(const KParams &P, const uint8_t *__restrict__ sb, uint32_t p,
                                          uint32_t step, uint32_t sid, const int off[6])
{
    return choose_dir_from(P, empty_mask(sb, p, P.nx, P.nx * P.ny), p, step, sid);
}

// Does READY parent p (site index inside its simulation, state array sb) win a target on this step?
// Returns the direction of its daughter, or -1 (blocked, or lost the claim: untouched, retries next step).
__device__ __forceinline__ int detect_decide_from(const KParams &P, const uint8_t *__restrict__ sb, uint32_t p, uint32_t step, uint32_t sid, uint32_t em)
{
    const int off[6] = { -1, 1, -P.nx, P.nx, -P.nx * P.ny, P.nx * P.ny };
    const int dir = choose_dir_from(P, em, p, step, sid);
    if (dir < 0) return -1;                                                // blocked: stays READY, retries
    const uint32_t e = (uint32_t)((int)p + off[dir]);
    const uint32_t mykey = rnd(P, p, step, sid, P_CLAIM);
#pragma unroll 1
    for (int d = 0; d < 6; ++d) {                                          // competitors = other neighbours of e
        const uint32_t q = (uint32_t)((int)e + off[d]);
        if (q == p || !is_parent(__ldcg(sb + q))) continue;
        const int dq = choose_dir(P, sb, q, step, sid, off);
        if (dq < 0 || (uint32_t)((int)q + off[dq]) != e) continue;
        const uint32_t qk = rnd(P, q, step, sid, P_CLAIM);
        if (qk < mykey || (qk == mykey && q < p)) return -1;
    }
    return dir;
}

__device__ __forceinline__ int detect_decide(const KParams &P, const uint8_t *__restrict__ sb, uint32_t p, uint32_t step, uint32_t sid)
{
    return detect_decide_from(P, sb, p, step, sid, empty_mask(sb, p, P.nx, P.nx * P.ny));
}

__device__ __forceinline__ void detect_site(const KParams &P, const Lattice &L, long long gi, uint32_t step,
                                            unsigned long long *__restrict__ winners, unsigned int *__restrict__ nwin,
                                            unsigned int cap, int *__restrict__ err)
{
    const int b = (int)(gi / P.n);
    const uint32_t p = (uint32_t)(gi - (long long)b * P.n);
    const int dir = detect_decide(P, L.state + (long long)b * P.n, p, step, P.sim_id_base + (uint32_t)b);
    if (dir < 0) return;
    const unsigned int slot = atomicAdd(nwin, 1u);                         // list order is irrelevant to the result
    if (slot >= cap) { *err = CA_EOVERFLOW; return; }
    winners[slot] = ((unsigned long long)gi << 3) | (unsigned long long)dir;
}

// [D S3 step 4] write one winner: parent and daughter both restart in G1 with fresh clocks
__device__ __forceinline__ void apply_winner(const KParams &P, const Lattice &L, int b, uint32_t p, int dir, uint32_t step)
{
    const int off[6] = { -1, 1, -P.nx, P.nx, -P.nx * P.ny, P.nx * P.ny };
    const long long gp = (long long)b * P.n + p;
    const uint32_t e = (uint32_t)((int)p + off[dir]);
    const long long ge = gp + off[dir];
    const uint32_t sid = P.sim_id_base + (uint32_t)b;
    const uint32_t keep = L.state[gp] & (0x18u | CA_DOOMED);              // mode and DOOMED carried to both [D G10]
    L.state[gp] = (uint8_t)(CA_G1 | keep);
    L.clock[gp] = draw_clock(P, CA_G1, p, step, sid, P_PARENT_CLOCK);
    L.state[ge] = (uint8_t)(CA_G1 | keep);
    L.clock[ge] = draw_clock(P, CA_G1, e, step, sid, P_DAUGHTER_CLOCK);
    L.damage[ge] = L.damage[gp];
}

__global__ void k_div_apply(KParams P, Lattice L, const long long *__restrict__ d_step, int k,
                            const unsigned long long *__restrict__ winners, const unsigned int *__restrict__ nwin,
                            unsigned int cap)
{
    unsigned int n = *nwin;
    if (n > cap) n = cap;
    const uint32_t step = (uint32_t)(*d_step + k);
    for (unsigned int w = blockIdx.x * blockDim.x + threadIdx.x; w < n; w += gridDim.x * blockDim.x) {
        const unsigned long long ent = winners[w];
        const long long gp = (long long)(ent >> 3);
        const int b = (int)(gp / P.n);
        apply_winner(P, L, b, (uint32_t)(gp - (long long)b * P.n), (int)(ent & 7ull), step);
    }
}

// ------------------------------------------------------------ S2 + S3 fused --
// Fast path for lattices whose simulations are whole multiples of 256 sites.  It works from an occupancy
// map -- one bit per 8 consecutive state bytes, set when a byte holds kind 1..6 -- that the fused diffusion
// kernel produces for free while the state planes pass through its shared memory (k_occ_map builds it
// when that kernel is not in use).  The map is taken before S2 of the same step; S2 never fills an EMPTY
// site and S3's births are applied last, so it covers every site S2 and S3 have to look at.
//
// One thread-block cluster per simulation does S2, S3-detect and S3-apply in ONE launch: S3 needs every
// S2 result of the simulation, which a cluster barrier provides (simulations never interact), and winners
// stay in shared memory.  Work is taken from the map, never from a sweep over the lattice.
__global__ void __launch_bounds__(256) k_occ_map(const uint8_t *__restrict__ state, long long tot, uint32_t *__restrict__ occ)
{
    const long long c8 = (long long)blockIdx.x * blockDim.x + threadIdx.x;          // 8-byte chunk index; tot % 256 == 0
    bool any = false;
    if (c8 * 8 < tot) {
        const unsigned long long w = reinterpret_cast<const unsigned long long *>(state)[c8];
        any = (((w & 0x0707070707070707ull) + 0x0101010101010101ull) & 0x0606060606060606ull) != 0ull;
    }
    const uint32_t ballot = __ballot_sync(0xFFFFFFFFu, any);
    if ((threadIdx.x & 31) == 0 && c8 * 8 < tot) occ[c8 >> 5] = ballot;
}

constexpr int CD_THREADS = 256;
constexpr int CD_WCAP = 2048;     // map words examined per round
constexpr int CD_TILE = 16;       // map words per interleave tile (one 64x64 plane): CTA rank takes tiles rank, rank + cs, ...
constexpr int CD_WINCAP = 2048;   // winners per CTA and step
constexpr int CD_PCAP = 1024;     // READY parents remembered from S2 (more: S3 rescans the map)
constexpr int CD_GWORDS = 128;    // map words whose set bits are expanded into the group list at a time (128 x 32 bits fill it exactly)
constexpr int CD_GCAP = CD_GWORDS * 32;

struct CDShared {
    uint32_t W[CD_WCAP];          // indices of the non-empty map words of this round
    uint32_t win[CD_WINCAP];      // winners: parent site << 3 | direction
    uint32_t Pl[CD_PCAP];         // READY parents after S2 (site index inside the simulation)
    uint32_t G[CD_GCAP];          // occupied groups of 8 sites of the current chunk of map words: word << 5 | bit
    uint32_t nW, nwin, nP, nG;
};

__device__ __forceinline__ void cluster_sync_all()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// winners beyond the CTA's shared list go to the simulation's slice of the global winners array; only when that is full too
// (more than n/8 births of one simulation in one step) a birth is dropped, and then the deferred error says so
struct SpillArgs {
    unsigned long long *list;     // [batch][cap_per_sim]
    unsigned int *n;              // [batch]
    unsigned int cap_per_sim;
};

__device__ __forceinline__ void cd_winner(CDShared &sh, uint32_t site, int dir, int *err, const SpillArgs &sp, int b)
{
    const uint32_t slot = atomicAdd(&sh.nwin, 1u);                                  // order is irrelevant to the result
    if (slot < CD_WINCAP) { sh.win[slot] = (site << 3) | (uint32_t)dir; return; }
    const unsigned int g = atomicAdd(sp.n + b, 1u);
    if (g < sp.cap_per_sim) sp.list[(size_t)b * sp.cap_per_sim + g] = ((unsigned long long)site << 3) | (unsigned long long)dir;
    else *err = CA_EOVERFLOW;
}

// MODE 0: S2 on every cell of simulation b (READY parents are remembered);  MODE 1: S3 detect by rescanning the map.
// CTA `rank` of `cs` takes the 16-word tiles rank, rank + cs, ... of the simulation's map and compacts the non-empty map
// words; the set bits of 128 such words at a time are expanded into a list of occupied GROUPS (one map bit = 8 consecutive
// sites), and every THREAD takes one group: one 8-byte load of its states, one 16-byte load of its clocks, six 16-byte loads
// of its fields, all issued before the first site is worked on, and at most three vector stores back.  (Round 1 gave a
// warp one map word and a lane one bit: on a 3.5k-cell tumour 9 of 32 lanes had a set bit and 4.5 of 32 lanes were active
// per instruction of S2 -- ncu, profiles/r02_ncu_cells_divide_c5_before_regrouping.txt is the capture before this change.)
template <int MODE>
__device__ __forceinline__ void cd_pass(const KParams &P, const Lattice &L, int cur, int b, int rank, int cs, uint32_t step,
                                        const uint32_t *__restrict__ occ_b, uint32_t nblk, CDShared &sh, int *__restrict__ err,
                                        int *__restrict__ lys_b, bool trust, const SpillArgs &sp)
{
    const int tid = threadIdx.x;
    const long long sbase = (long long)b * P.n;
    const uint8_t *sb = L.state + sbase;
    uint8_t *stb = L.state + sbase;
    uint16_t *ckb = L.clock + sbase, *dmb = L.damage + sbase;
    const float *f0 = L.f[cur][0] + sbase, *f1 = L.f[cur][1] + sbase, *f2 = L.f[cur][2] + sbase;
    const bool need_dm = (step + 1u) % (uint32_t)P.repair_period == 0u;      // damage only matters on repair steps [D G11]
    const uint32_t sid = P.sim_id_base + (uint32_t)b;
    for (uint32_t w0 = 0; w0 < nblk; w0 += (uint32_t)(CD_WCAP * cs)) {
        if (tid == 0) sh.nW = 0;
        __syncthreads();
        for (uint32_t idx = tid; idx < CD_WCAP; idx += CD_THREADS) {
            const uint32_t w = w0 + ((idx / CD_TILE) * (uint32_t)cs + (uint32_t)rank) * CD_TILE + (idx % CD_TILE);
            if (w < nblk && occ_b[w] != 0u) sh.W[atomicAdd(&sh.nW, 1u)] = w;
        }
        __syncthreads();
        const uint32_t nW = sh.nW;
        for (uint32_t c0 = 0; c0 < nW; c0 += CD_GWORDS) {
            if (tid == 0) sh.nG = 0;
            __syncthreads();
            {   // two threads per map word expand its set bits (16 each) into the group list; the order is irrelevant to the result
                const uint32_t wi = c0 + ((uint32_t)tid >> 1);
                if (wi < nW) {
                    const uint32_t w = sh.W[wi];
                    uint32_t bits = (occ_b[w] >> (16u * ((uint32_t)tid & 1u))) & 0xFFFFu;
                    if (bits) {
                        uint32_t pos = atomicAdd(&sh.nG, (uint32_t)__popc(bits));
                        while (bits) {
                            const uint32_t bit = (uint32_t)__ffs(bits) - 1u;
                            bits &= bits - 1u;
                            sh.G[pos++] = (w << 5) | (bit + 16u * ((uint32_t)tid & 1u));
                        }
                    }
                }
            }
            __syncthreads();
            const uint32_t nG = sh.nG;
        for (uint32_t gi = tid; gi < nG; gi += CD_THREADS) {
            const uint32_t ge = sh.G[gi];
            const uint32_t site0 = (ge >> 5) * 256u + 8u * (ge & 31u);
            const unsigned long long sv = __ldcg(reinterpret_cast<const unsigned long long *>(sb + site0));
            if (MODE == 0) {
                // Branch-light form of [D S2].  Per step almost every cell only refreshes its mode bits and counts its clock down;
                // starvation, the end of a countdown and repair are rare and go through cell_update, which recomputes the cell
                // from its original values (so the two forms cannot disagree).
                const uint4 cv = *reinterpret_cast<const uint4 *>(ckb + site0);
                uint4 dv = make_uint4(0u, 0u, 0u, 0u);
                if (need_dm) dv = *reinterpret_cast<const uint4 *>(dmb + site0);
                const float4 oa = *reinterpret_cast<const float4 *>(f0 + site0), ob = *reinterpret_cast<const float4 *>(f0 + site0 + 4);
                const float4 ga = *reinterpret_cast<const float4 *>(f1 + site0), gb = *reinterpret_cast<const float4 *>(f1 + site0 + 4);
                const float4 ha = *reinterpret_cast<const float4 *>(f2 + site0), hb = *reinterpret_cast<const float4 *>(f2 + site0 + 4);
                const float fo[8] = { oa.x, oa.y, oa.z, oa.w, ob.x, ob.y, ob.z, ob.w };
                const float fg[8] = { ga.x, ga.y, ga.z, ga.w, gb.x, gb.y, gb.z, gb.w };
                const float fh[8] = { ha.x, ha.y, ha.z, ha.w, hb.x, hb.y, hb.z, hb.w };
                const uint32_t c32[4] = { cv.x, cv.y, cv.z, cv.w }, d32[4] = { dv.x, dv.y, dv.z, dv.w };
                uint32_t cn[4] = { cv.x, cv.y, cv.z, cv.w }, dn[4] = { dv.x, dv.y, dv.z, dv.w };
                unsigned long long sn = sv;
                bool dm_dirty = false;
                uint32_t pmask = 0;                                          // bit k: site k is a READY parent after S2; bit 8 + k: known to be blocked
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    const uint32_t s0 = (uint32_t)(sv >> (8 * k)) & 0xFFu, kind = s0 & 7u;
                    if (kind == CA_EMPTY || kind == CA_WALL) continue;
                    const uint32_t i = site0 + (uint32_t)k;
                    const uint32_t ck0 = (c32[k >> 1] >> (16 * (k & 1))) & 0xFFFFu;
                    const bool dead = kind == CA_DEAD;
                    const bool starved = !dead && (fg[k] < P.G_Q || fh[k] > P.H_Q);
                    const bool prolif = (fg[k] >= P.G_P) && (fh[k] <= P.H_P);
                    const uint32_t mode = 2u * (uint32_t)(!prolif) + (uint32_t)(!(fo[k] >= P.O_A));
                    uint32_t s1 = dead ? s0 : ((s0 & ~0x18u) | (mode << 3));
                    if (!is_parent(s1)) s1 &= ~CA_BLOCKED;                   // "blocked" is only remembered while the cell stays a parent (see S3)
                    const bool tick = dead || (prolif && !(s0 & CA_READY));
                    uint32_t c1 = ck0 - (uint32_t)tick;
                    const uint32_t dm0 = (d32[k >> 1] >> (16 * (k & 1))) & 0xFFFFu;
                    if (starved || (tick && c1 == 0u) || dm0 > 0u) {          // rare: the general state machine (dm0 is 0 off repair steps)
                        uint32_t s2 = s0, c2 = ck0, d2 = need_dm ? dm0 : 1u;   // off repair steps damage can only change to 0 (death, lysis)
                        const uint32_t dref = d2;
                        cell_update(P, s2, c2, d2, fo[k], fg[k], fh[k], i, step, sid);
                        if ((s2 & 7u) == CA_EMPTY) *lys_b = 1;               // a site was vacated: blocked parents must look again
                        if (!is_parent(s2)) s2 &= ~CA_BLOCKED;
                        s1 = s2; c1 = c2;
                        if (d2 != dref) {
                            if (need_dm) { dn[k >> 1] = (dn[k >> 1] & ~(0xFFFFu << (16 * (k & 1)))) | (d2 << (16 * (k & 1))); dm_dirty = true; }
                            else dmb[i] = (uint16_t)d2;                       // the vector was not loaded: single store of the 0
                        }
                    }
                    sn = (sn & ~(0xFFull << (8 * k))) | ((unsigned long long)s1 << (8 * k));
                    cn[k >> 1] = (cn[k >> 1] & ~(0xFFFFu << (16 * (k & 1)))) | ((c1 & 0xFFFFu) << (16 * (k & 1)));
                    if (is_parent(s1)) pmask |= (1u << k) | ((s1 & CA_BLOCKED) << (8 + k - 7));
                }
                // one shared-memory atomic per group, not per parent: the core of a grown tumour is full of blocked READY parents, and
                // a counter that has passed CD_PCAP (S3 then rescans the map) is left alone
                if ((pmask & 0xFFu) && *(volatile uint32_t *)&sh.nP <= (uint32_t)CD_PCAP) {
                    uint32_t slot = atomicAdd(&sh.nP, (uint32_t)__popc(pmask & 0xFFu));
                    for (uint32_t m = pmask & 0xFFu; m; m &= m - 1u, ++slot) {
                        const uint32_t k = (uint32_t)__ffs(m) - 1u;
                        if (slot < CD_PCAP) sh.Pl[slot] = (site0 + k) | (((pmask >> (8 + k)) & 1u) << 31);
                    }
                }
                if (sn != sv) *reinterpret_cast<unsigned long long *>(stb + site0) = sn;
                if (cn[0] != cv.x || cn[1] != cv.y || cn[2] != cv.z || cn[3] != cv.w)
                    *reinterpret_cast<uint4 *>(ckb + site0) = make_uint4(cn[0], cn[1], cn[2], cn[3]);
                if (dm_dirty) *reinterpret_cast<uint4 *>(dmb + site0) = make_uint4(dn[0], dn[1], dn[2], dn[3]);
            } else {
#pragma unroll 1
                for (int k = 0; k < 8; ++k) {
                    const uint32_t st = (uint32_t)(sv >> (8 * k)) & 0xFFu;
                    if (!is_parent(st) || (trust && (st & CA_BLOCKED))) continue;      // most READY parents are blocked, and known to be
                    const uint32_t site = site0 + (uint32_t)k;
                    const uint32_t em = empty_mask(sb, site, P.nx, P.nx * P.ny);
                    const uint32_t nb = em ? (st & ~CA_BLOCKED) : (st | CA_BLOCKED);
                    if (nb != st) stb[site] = (uint8_t)nb;
                    if (!em) continue;
                    const int dir = detect_decide_from(P, sb, site, step, sid, em);
                    if (dir >= 0) cd_winner(sh, site, dir, err, sp, b);
                }
            }
        }
            __syncthreads();                                                  // the group list is rebuilt by the next chunk
        }
        __syncthreads();
    }
}

// grid = batch * cs CTAs in clusters of cs; phases: bit 0 S2, bit 1 S3 (detect + apply)
__global__ void __launch_bounds__(CD_THREADS, 4) k_cells_divide(KParams P, Lattice L, int cur, const long long *__restrict__ d_step, int k,
                                                                const uint32_t *__restrict__ occ, int cs, int phases, int *__restrict__ err, int b0, int *__restrict__ lys,
                                                                const SpillArgs sp)
{
    __shared__ CDShared sh;
    const int b = b0 + blockIdx.x / cs, rank = blockIdx.x % cs;
    const uint32_t step = (uint32_t)(*d_step + k);
    const uint32_t nblk = (uint32_t)(P.n >> 8);
    const uint32_t *occ_b = occ + (size_t)b * nblk;
    if (threadIdx.x == 0) { sh.nwin = 0; sh.nP = (phases & 1) ? 0u : (uint32_t)CD_PCAP + 1u; }
    if (rank == 0 && threadIdx.x == 0 && (phases & 2)) sp.n[b] = 0;             // ordered before the first winner by the barrier below
    if (phases & 1) cd_pass<0>(P, L, cur, b, rank, cs, step, occ_b, nblk, sh, err, lys + b, false, sp);
    if (phases & 2) {
        if (cs > 1) cluster_sync_all(); else __syncthreads();                 // every S2 write of this simulation is visible
        // A READY parent found without an EMPTY neighbour stays blocked until a site of its simulation is vacated, and
        // that only happens by lysis in S2.  Bit 7 of its state byte remembers "blocked" (internal: masked on export); it
        // is trusted on steps on which no lysis happened since it was written, and refreshed otherwise.
        const bool trust = *(volatile int *)(lys + b) == 0;
        const uint32_t nP = sh.nP;
        if (nP <= (uint32_t)CD_PCAP) {                                         // few parents (small tumour): the ones S2 just saw
            const long long sbase = (long long)b * P.n;
            const uint8_t *sb = L.state + sbase;
            for (uint32_t r = threadIdx.x; r < nP; r += CD_THREADS) {
                const uint32_t site = sh.Pl[r] & 0x7FFFFFFFu, was = sh.Pl[r] >> 31;
                if (trust && was) continue;
                const uint32_t em = empty_mask(sb, site, P.nx, P.nx * P.ny);
                if ((em == 0u) != (was != 0u)) L.state[sbase + site] = (uint8_t)(em ? (__ldcg(sb + site) & ~CA_BLOCKED) : (__ldcg(sb + site) | CA_BLOCKED));
                if (!em) continue;
                const int dir = detect_decide_from(P, sb, site, step, P.sim_id_base + (uint32_t)b, em);
                if (dir >= 0) cd_winner(sh, site, dir, err, sp, b);
            }
        } else {
            cd_pass<1>(P, L, cur, b, rank, cs, step, occ_b, nblk, sh, err, lys + b, trust, sp);
        }
        if (cs > 1) cluster_sync_all(); else __syncthreads();                 // every decision is taken: now write
        const uint32_t nw = min(sh.nwin, (uint32_t)CD_WINCAP);
        for (uint32_t w = threadIdx.x; w < nw; w += CD_THREADS) apply_winner(P, L, b, sh.win[w] >> 3, (int)(sh.win[w] & 7u), step);
        if (sh.nwin > (uint32_t)CD_WINCAP || cs > 1) {                            // spilled winners of this simulation: shared out over the cluster
            const uint32_t ns = min(*(volatile unsigned int *)(sp.n + b), sp.cap_per_sim);
            const unsigned long long *sl = sp.list + (size_t)b * sp.cap_per_sim;
            for (uint32_t w = (uint32_t)rank * CD_THREADS + threadIdx.x; w < ns; w += (uint32_t)cs * CD_THREADS) {
                const unsigned long long ent = __ldcg(sl + w);
                apply_winner(P, L, b, (uint32_t)(ent >> 3), (int)(ent & 7ull), step);
            }
        }
        if (rank == 0 && threadIdx.x == 0) lys[b] = 0;                        // every CTA of the cluster read it before the second barrier
    }
}

// end of a group of `adv` steps: advance the device step counter, clear the per-step winner counters
__global__ void k_advance(long long *d_step, int adv, unsigned int *nwin, int nslots)
{
    if (threadIdx.x == 0) *d_step += adv;
    for (int i = threadIdx.x; i < nslots; i += blockDim.x) nwin[i] = 0;
}

// ---------------------------------------------------------------------- S4 --
// [D S4] per-simulation counts by warp-shuffle reduction; grid = (blocks_per_sim, batch).
// Each thread scans 16 state bytes per load; counts go to counts[b][CA_NCOUNT] by one atomic per warp.
__global__ void k_counts(KParams P, const uint8_t *__restrict__ state, int *__restrict__ counts)
{
    const int b = blockIdx.y;
    const uint8_t *sb = state + (long long)b * P.n;
    int c[12];
#pragma unroll
    for (int q = 0; q < 12; ++q) c[q] = 0;
    auto tally = [&](uint32_t st) {
        const uint32_t kind = st & 7u;
        const bool lv = kind >= 1u && kind <= 4u;
        c[CA_C_LIVE] += lv;
        c[CA_C_DOOMED] += lv && (st & CA_DOOMED);
        c[CA_C_READY] += lv && (st & CA_READY);
        c[CA_C_DEAD] += kind == CA_DEAD;
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            c[CA_C_G1 + q] += kind == (uint32_t)(1 + q);
            c[CA_C_PA + q] += lv && (((st >> 3) & 3u) == (uint32_t)q);
        }
    };
    const long long nvec = ((long long)b * P.n % 16 == 0) ? P.n / 16 : 0;   // vector body only when 16B-aligned
    const uint4 *sv = reinterpret_cast<const uint4 *>(sb);
    for (long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x; v < nvec; v += (long long)gridDim.x * blockDim.x) {
        const uint4 w = sv[v];
        const uint32_t ws[4] = { w.x, w.y, w.z, w.w };
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (ws[q] == 0u || ws[q] == 0x07070707u) continue;              // all EMPTY / all WALL
#pragma unroll
            for (int r = 0; r < 4; ++r) tally((ws[q] >> (8 * r)) & 0xFFu);
        }
    }
    for (long long i = nvec * 16 + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.n; i += (long long)gridDim.x * blockDim.x)
        tally(sb[i]);
#pragma unroll
    for (int q = 0; q < 12; ++q) {
        int v = c[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
        if ((threadIdx.x & 31) == 0 && v) atomicAdd(&counts[b * CA_NCOUNT + q], v);   // integer: order-independent
    }
}

// occupied = live + dead [D G13]; fitness = N_ref - occupied (Eq. 1)
__global__ void k_finish_counts(KParams P, int *__restrict__ counts, float *__restrict__ fitness)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= P.batch) return;
    const int occ = counts[b * CA_NCOUNT + CA_C_LIVE] + counts[b * CA_NCOUNT + CA_C_DEAD];
    counts[b * CA_NCOUNT + CA_C_OCCUPIED] = occ;
    const long long nref = P.N_ref > 0 ? (long long)P.N_ref : (long long)(P.nx - 2) * (P.ny - 2) * (P.nz - 2);
    fitness[b] = (float)(nref - occ);
}

// broadcast simulation `src` to simulations [first, first+count) (skipping src itself); bytes per sim = nbytes (16B multiple not required)
__global__ void k_broadcast(uint8_t *base, long long nbytes, int src, int first, int count)
{
    const int b = first + blockIdx.y;
    if (b == src) return;
    const uint8_t *s = base + (long long)src * nbytes;
    uint8_t *d = base + (long long)b * nbytes;
    if (nbytes % 16 == 0) {
        const uint4 *sv = reinterpret_cast<const uint4 *>(s);
        uint4 *dv = reinterpret_cast<uint4 *>(d);
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nbytes / 16; i += (long long)gridDim.x * blockDim.x) dv[i] = sv[i];
    } else {
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < nbytes; i += (long long)gridDim.x * blockDim.x) d[i] = s[i];
    }
}

}  // namespace ca
