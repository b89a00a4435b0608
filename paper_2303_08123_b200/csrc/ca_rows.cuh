// ca_rows.cuh -- temporally fused reaction-diffusion kernel for planes wider than 64 sites (BASELINE configs[2], [3]:
// 96^3, 80^3): NL (<= 4) sub-steps of [D S1] in ONE pass over HBM, like k_diffuse_fused, with a lane layout that covers a
// WHOLE lattice row of width nx = PX * LRP without seams:
//
//   * a lane owns PX consecutive sites (PX = 3 for 96 = 3 * 32 lanes, PX = 5 for 80 = 5 * 16 lanes) of TWO rows (RP = 1) or of
//     FOUR rows (RP = 2: two packed row pairs; the default on 96-wide planes: half the row exchange per site, 8 warps); the packed
//     f32x2 registers pair the two ROWS of one column, so x-neighbours inside a lane are whole registers (one packed add),
//     only the lane's first / last column needs the neighbour lane (two 64-bit shuffles per level), and odd PX is fine;
//   * a CTA holds a y-slab of whole rows (32 rows for 96-wide planes, 44 for 80): contiguous in memory, so a slab of a field
//     plane and of the state plane arrives by ONE 1-D bulk copy each (UBLKCP) into shared-memory rings with mbarrier
//     completion, two planes ahead, and the output rows leave by ONE bulk store (shared -> global) per plane: no per-lane
//     global loads or stores in the march;
//   * slabs carry a halo of F_MAXNL rows towards their neighbour slabs; the first / last loaded row is frozen (lambda = 0:
//     WALL on the lattice face, halo edge at a cut), the error that creates moves inwards one row per sub-step and never
//     reaches the output rows (same argument as for the z-cuts of a segment);
//   * y-neighbours between row pairs go through a double-buffered shared-memory copy of every level's rows (one
//     __syncthreads per plane); z-neighbours and all NL time levels stay in registers, the march loop is unrolled by 3;
//   * the S2/S3 occupancy map is produced from the state slab while it sits in shared memory.
//
// Arithmetic per point is exactly [D S1] (see ca_fused.cuh): sum6 = ((xm+xp)+(ym+yp))+(zm+zp); lap = sum6 - 6*c with the
// product rounded on its own; v = fma(lambda, lap, c); v += r; max(v, 0).  The work split, the pipeline (level k computes
// plane t-k while level 0 loads plane t) and the fast path without source term are those of k_diffuse_fused.
#pragma once
#include "ca_fused.cuh"

namespace ca {

struct RowsSeg {                   // per-segment constants only the producer thread / one lane per warp needs (shared memory)
    const float *src_rows;         // first loaded row of plane 0 of this unit's input field
    const uint8_t *st_rows;
    float *dst_rows;               // first OUTPUT row of plane 0 of this unit's output field
    uint32_t *occ_row;             // occupancy words of this simulation
    uint32_t ld_fbytes, ld_sbytes; // bytes of the slab's rows of a field / state plane
    uint32_t out_off, out_bytes;   // output rows inside the staging slab
    uint32_t occ_w0, occ_soff;     // first occupancy word this slab writes; its byte offset inside the state slot
};

struct RowsGeom {                  // host-computed launch geometry, passed by value
    int nwarps, hrows;             // warps per CTA, rows a CTA holds (the tallest slab fits)
    uint32_t off_lut, off_in, off_st, off_ex, off_out, smem_bytes;
    int start[F_MAXGRID + 1];      // CTA g works on flattened (unit, plane) indices [start[g], start[g+1])
};

struct RowsCtx {
    const float *src;              // input field of this unit at this lane's first site, plane 0 (WALL planes are read directly)
    int nxny, nz;
    int za, zb, t0, nsteps, ld_lo, ld_hi, st_lo, st_hi;
    uint32_t itg, par, flags, slowmask;
    uint32_t bars, in_ring, st_ring, lut, out_ring;
    uint32_t lane_b;               // byte offset of this lane's first site inside a field slab: (row0 * nx + x0) * 4
    uint32_t ex_lane;              // exchange base + lane_b: exchange row r + 1 holds slab row r
    uint32_t st_vote;              // byte offset (inside a state slot) of the 16 bytes of the warp's rows this lane votes on; ~0: none
    uint32_t in_slot, st_slot;     // bytes of one ring slot
    uint32_t ex_lvl;               // bytes of one level of the row exchange
    u64 lamL[2], lamM[2], lamR[2]; // per row pair of the lane: lambda pairs (row 0, row 1) for its first / middle / last column; WALL and frozen rows folded in
    u64 zero2;
    uint32_t occ_nw;               // species 0: occupancy words of a plane this slab writes (else 0)
    // cluster variant: the CTA's first / last row pair also publishes its outer row into the neighbour CTA's exchange
    uint32_t rem;                  // shared::cluster address of that row's slot (buffer 0, level 0) in the neighbour's exchange; 0: none
    bool rem_row1;                 // the row to send: row 1 of the pair (last pair, to the CTA below) or row 0 (first pair, to the CTA above)
};

// cluster helpers (sm_90+): rank inside the cluster, address of a peer CTA's shared memory, cluster-wide barrier
__device__ __forceinline__ uint32_t cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t map_to_rank(uint32_t addr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_f32(uint32_t addr, float v) { asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory"); }
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_barrier()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// CS = 1: y-slabs with a halo (any ny);  CS > 1: a thread-block cluster of CS CTAs holds ny = CS * hrows rows exactly, no halo
// RP: row PAIRS per lane (1: two rows; 2: four rows -- half the row exchange per site, half the warps, twice the registers)
template <int NL, int PX, int LRP, int CS = 1, int RP = 1>
struct Rows {
    static constexpr int NX = PX * LRP;
    static constexpr int RW = 32 / LRP;                                   // row groups (of 2 * RP rows) per warp
    static constexpr int PXR = PX * RP;                                   // packed registers per plane and level: [pair p][column k] at p * PX + k
    static constexpr uint32_t PITCH = (uint32_t)NX * 4u;
    // Row pitch of the EXCHANGE buffer.  A warp with two row groups (LRP = 16) has its half-warps 2 * RP rows apart; at the
    // lattice pitch of 80 words that is a multiple of 32 banks, so lanes l and l + 16 collide on every exchange access (ncu on
    // 96 x 80^3: shared pipe 68 %, short_scoreboard and mio_throttle the top stalls).  88 words put the second half-warp 16
    // banks further: with the lane stride of 5 words the 32 lanes then hit 32 different banks.  The input ring and the staging
    // slab are moved by bulk copies at the lattice pitch and cannot be padded.
    static constexpr uint32_t EXP = (RW > 1 && ((uint32_t)(2 * RP * NX) % 32u) == 0u) ? PITCH + 32u : PITCH;
    static_assert(CS == 1 || RP == 1, "the cluster variant is built for two rows per lane");

    static __device__ __forceinline__ RowsSeg *seg()
    {
        extern __shared__ __align__(128) unsigned char rsm_[];
        return reinterpret_cast<RowsSeg *>(rsm_ + F_SEG_OFF);
    }
    static __device__ __forceinline__ u64 lam(const RowsCtx &c, int p, int k) { return k == 0 ? c.lamL[p] : (k == PX - 1 ? c.lamR[p] : c.lamM[p]); }

    static __device__ __forceinline__ u64 shfl_up64(u64 v)
    {
        float a, b;
        upk(v, a, b);
        return pk(__shfl_up_sync(0xFFFFFFFFu, a, 1, LRP), __shfl_up_sync(0xFFFFFFFFu, b, 1, LRP));
    }
    static __device__ __forceinline__ u64 shfl_down64(u64 v)
    {
        float a, b;
        upk(v, a, b);
        return pk(__shfl_down_sync(0xFFFFFFFFu, a, 1, LRP), __shfl_down_sync(0xFFFFFFFFu, b, 1, LRP));
    }

    // one sub-step of the diffusion part of [D S1] for this lane's PX x 2 points.  C = centre plane, M / P = planes z-1 / z+1,
    // up[k] / dn[k] = the row above / below the pair at column k.
    static __device__ __forceinline__ void level(const u64 (&M)[PXR], const u64 (&C)[PXR], const u64 (&P)[PXR], u64 (&N)[PXR],
                                                 const float (&up)[PX], const float (&dn)[PX], const RowsCtx &c)
    {
        const u64 six2 = pk(6.0f, 6.0f);
#pragma unroll
        for (int p = 0; p < RP; ++p) {
            const u64 left = shfl_up64(C[p * PX + PX - 1]);                  // column x0-1 (own value at the row's first lane: WALL side, lambda = 0)
            const u64 right = shfl_down64(C[p * PX]);                        // column x0+PX
#pragma unroll
            for (int k = 0; k < PX; ++k) {
                const int e = p * PX + k;
                float c0, c1;
                upk(C[e], c0, c1);
                // the row above the pair: the exchange for the lane's first pair, else row 1 of the pair above; likewise below
                float ab = up[k], be = dn[k], t0, t1;
                if (p > 0) { upk(C[(p > 0 ? p - 1 : 0) * PX + k], t0, t1); ab = t1; }
                if (p < RP - 1) { upk(C[(p < RP - 1 ? p + 1 : 0) * PX + k], t0, t1); be = t0; }
                const u64 xs = add2(k == 0 ? left : C[e > 0 ? e - 1 : 0], k == PX - 1 ? right : C[e < PXR - 1 ? e + 1 : 0]);   // xm + xp
                const u64 ys = pk(__fadd_rn(ab, c1), __fadd_rn(c0, be));     // ym + yp: row 0 has (above, row 1), row 1 has (row 0, below)
                const u64 zs = add2(M[e], P[e]);                             // zm + zp
                const u64 s6 = add2(add2(xs, ys), zs);
                const u64 lap = sub2(s6, fma2(six2, C[e], c.zero2));         // 6*c rounded on its own (see Fused::level)
                N[e] = fma2(lam(c, p, k), lap, C[e]);
            }
        }
    }

    // producer (one thread): start the bulk copies of iteration i into field-ring slot i mod 3
    static __device__ __forceinline__ void issue(const RowsCtx &c, int i, int slot)
    {
        const int t = c.t0 + i;
        const uint32_t bar = c.bars + 8u * (uint32_t)slot;
        if (t >= c.ld_lo && t < c.ld_hi) {
            const RowsSeg *sg = seg();
            mbar_expect_tx(bar, sg->ld_fbytes + sg->ld_sbytes);
            bulk_g2s(c.in_ring + (uint32_t)slot * c.in_slot, sg->src_rows + (size_t)t * c.nxny, sg->ld_fbytes, bar);
            bulk_g2s(c.st_ring + ((c.itg + (uint32_t)i) & (F_SRING - 1)) * c.st_slot, sg->st_rows + (size_t)t * c.nxny, sg->ld_sbytes, bar);
        } else {
            mbar_arrive(bar);
        }
    }

    template <int PH, int K, bool STEADY, bool NOCELLS>
    static __device__ __forceinline__ void levels(const int t, const uint32_t q, const uint32_t exr, const uint32_t exw, const uint32_t outw,
                                                  u64 (&h)[NL][3][PXR], RowsCtx &c)
    {
        if constexpr (K <= NL) {
            // cluster variant: every row the neighbours need from this iteration is published once level NL-1 is done; the last
            // level (a quarter of the arithmetic, staging only) runs between the arrive and the wait at the top of the next iteration
            if constexpr (CS > 1 && K == NL) cluster_arrive();
            constexpr int sm = (PH - K - 1 + 12) % 3, sc = (PH - K + 12) % 3, sp = (PH - K + 1 + 12) % 3;
            constexpr int KO = K < NL ? K : 0;
            const int zc = t - K;
            bool compute = true;
            if (!STEADY) compute = zc >= max(1, c.za - (NL - K)) && zc < min(c.nz - 1, c.zb + (NL - K));
            if (compute) {
                // rows above / below my pair at level K-1, written by the previous iteration (slab row r = exchange row r + 1)
                const uint32_t eb = exr + (uint32_t)(K - 1) * c.ex_lvl;
                float up[PX], dn[PX];
#pragma unroll
                for (int k = 0; k < PX; ++k) {
                    up[k] = lds32f(eb + (uint32_t)k * 4u);                    // slab row row0 - 1
                    dn[k] = lds32f(eb + (uint32_t)(2 * RP + 1) * EXP + (uint32_t)k * 4u);     // slab row row0 + 2 * RP
                }
                u64 nloc[PXR];
                u64 (&N)[PXR] = *(K < NL ? &h[KO][sc] : &nloc);
                level(h[K - 1][sm], h[K - 1][sc], h[K - 1][sp], N, up, dn, c);
                if (!NOCELLS && (((c.flags | c.slowmask) >> K) & 1u)) {      // cells in this warp's rows: source term and clamp
                    const uint32_t s = c.st_ring + ((q - (uint32_t)K) & (F_SRING - 1)) * c.st_slot + (c.lane_b >> 2);
#pragma unroll
                    for (int e = 0; e < PXR; ++e) {
                        const uint32_t so = (uint32_t)(2 * (e / PX) * NX + e % PX);
                        uint32_t b0, b1;
                        asm volatile("ld.shared.u8 %0, [%1];" : "=r"(b0) : "r"(s + so));
                        asm volatile("ld.shared.u8 %0, [%1];" : "=r"(b1) : "r"(s + so + (uint32_t)NX));
                        const u64 v = add2(N[e], pk(lds32f(c.lut + (b0 & 31u) * 4u), lds32f(c.lut + (b1 & 31u) * 4u)));
                        float a, b;
                        upk(v, a, b);
                        N[e] = pk(fmaxf(a, 0.0f), fmaxf(b, 0.0f));
                    }
                }
                // publish level K: my first and last row to the exchange for level K+1 of the next iteration (rows in between have
                // their neighbours in this lane), or (last level) every row to the staging slab
                if constexpr (K < NL) {
                    const uint32_t wb = exw + (uint32_t)K * c.ex_lvl + EXP;
#pragma unroll
                    for (int k = 0; k < PX; ++k) {
                        float a, b, a2, b2;
                        upk(N[k], a, b);
                        upk(N[(RP - 1) * PX + k], a2, b2);
                        asm volatile("st.shared.f32 [%0], %1;" ::"r"(wb + (uint32_t)k * 4u), "f"(a) : "memory");
                        asm volatile("st.shared.f32 [%0], %1;" ::"r"(wb + (uint32_t)(2 * RP - 1) * EXP + (uint32_t)k * 4u), "f"(b2) : "memory");
                    }
                } else {
#pragma unroll
                    for (int e = 0; e < PXR; ++e) {
                        float a, b;
                        upk(N[e], a, b);
                        const uint32_t wo = outw + (uint32_t)(2 * (e / PX)) * PITCH + (uint32_t)(e % PX) * 4u;
                        asm volatile("st.shared.f32 [%0], %1;" ::"r"(wo), "f"(a) : "memory");
                        asm volatile("st.shared.f32 [%0], %1;" ::"r"(wo + PITCH), "f"(b) : "memory");
                    }
                }
                if constexpr (CS > 1 && K < NL) {                            // my outer row is the neighbour CTA's halo row of level K
                    if (c.rem != 0u) {
                        const uint32_t ra = c.rem + (exw - c.ex_lane) + (uint32_t)K * c.ex_lvl;
#pragma unroll
                        for (int k = 0; k < PX; ++k) {
                            float a, b;
                            upk(N[k], a, b);
                            st_cluster_f32(ra + (uint32_t)k * 4u, c.rem_row1 ? b : a);
                        }
                    }
                }
            } else if (K < NL && (zc == 0 || zc == c.nz - 1) && zc >= c.za - (NL - K) && zc < c.zb + (NL - K)) {
                // WALL plane: every level equals the input there
                const float *p = c.src + (size_t)zc * c.nxny;
#pragma unroll
                for (int e = 0; e < PXR; ++e) h[KO][sc][e] = pk(p[2 * (e / PX) * NX + e % PX], p[(2 * (e / PX) + 1) * NX + e % PX]);
            }
            levels<PH, K + 1, STEADY, NOCELLS>(t, q, exr, exw, outw, h, c);
        }
    }

    template <int PH, bool STEADY>
    static __device__ __forceinline__ void step(const int i, u64 (&h)[NL][3][PXR], RowsCtx &c)
    {
        // one body per phase: a second copy without the source-term code (as in k_diffuse_fused) costs more in instruction-cache
        // misses than the untaken branches it saves here (measured: 0.806 -> 0.775 ms at 64 x 96^3, 0.659 -> 0.608 ms at 96 x 80^3)
        step_body<PH, STEADY, false>(i, h, c);
    }

    template <int PH, bool STEADY, bool NOCELLS>
    static __device__ __forceinline__ void step_body(const int i, u64 (&h)[NL][3][PXR], RowsCtx &c)
    {
        const int t = c.t0 + i;
        const uint32_t q = c.itg + (uint32_t)i;
        if (threadIdx.x == 0 && i + (F_RING - 1) < c.nsteps) issue(c, i + (F_RING - 1), (PH + F_RING - 1) % 3);
        const uint32_t exb = c.ex_lvl * NL;                                  // bytes of one exchange buffer
        const uint32_t exw = c.ex_lane + ((uint32_t)i & 1u) * exb;           // rows written now, read by the next iteration
        const uint32_t exr = c.ex_lane + exb - ((uint32_t)i & 1u) * exb;     // rows written by the previous iteration
        const uint32_t outw = c.out_ring + (q & 1u) * c.in_slot + c.lane_b;
        if constexpr (CS > 1) cluster_wait();                                // the neighbours' rows of the previous iteration have arrived, and they have read mine
        // ---- level 0: plane t from the ring
        mbar_wait(c.bars + 8u * PH, (c.par >> PH) & 1u);
        c.par ^= 1u << PH;
        bool any = false;
        if (STEADY || (t >= c.ld_lo && t < c.ld_hi)) {
            const uint32_t a = c.in_ring + (uint32_t)PH * c.in_slot + c.lane_b;
#pragma unroll
            for (int e = 0; e < PXR; ++e) {
                const int pp = e / PX, k = e % PX;
                const float v0 = lds32f(a + (uint32_t)(2 * pp) * PITCH + (uint32_t)k * 4u), v1 = lds32f(a + (uint32_t)(2 * pp + 1) * PITCH + (uint32_t)k * 4u);
                h[0][PH][e] = pk(v0, v1);
                if (pp == 0) asm volatile("st.shared.f32 [%0], %1;" ::"r"(exw + EXP + (uint32_t)k * 4u), "f"(v0) : "memory");
                if (pp == RP - 1) asm volatile("st.shared.f32 [%0], %1;" ::"r"(exw + (uint32_t)(2 * RP) * EXP + (uint32_t)k * 4u), "f"(v1) : "memory");
                if constexpr (CS > 1) {
                    if (c.rem != 0u) st_cluster_f32(c.rem + (exw - c.ex_lane) + (uint32_t)k * 4u, c.rem_row1 ? v1 : v0);
                }
            }
            const uint32_t sbase = c.st_ring + (q & (F_SRING - 1)) * c.st_slot;
            // "cells in my warp's rows": the warp's rows are contiguous bytes of the state slab; a byte counts when kind is 1..6
            if (c.st_vote != 0xFFFFFFFFu) {
                uint32_t w0, w1, w2, w3;
                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(w0), "=r"(w1), "=r"(w2), "=r"(w3) : "r"(sbase + c.st_vote));
                const uint32_t m = (((w0 & 0x07070707u) + 0x01010101u) | ((w1 & 0x07070707u) + 0x01010101u) |
                                    ((w2 & 0x07070707u) + 0x01010101u) | ((w3 & 0x07070707u) + 0x01010101u)) & 0x06060606u;
                any = m != 0u;
            }
            // the S2/S3 occupancy map (one bit per 8 consecutive state bytes, one word per 256): this slab's words of the plane
            for (uint32_t w = threadIdx.x >> 5; w < c.occ_nw; w += blockDim.x >> 5) {
                const RowsSeg *sg = seg();
                const u64 v = lds64(sbase + sg->occ_soff + w * 256u + 8u * (threadIdx.x & 31u));
                const uint32_t bal = __ballot_sync(0xFFFFFFFFu, (((v & 0x0707070707070707ull) + 0x0101010101010101ull) & 0x0606060606060606ull) != 0ull);
                if ((threadIdx.x & 31) == 0) sg->occ_row[(size_t)t * (size_t)(c.nxny / 256) + sg->occ_w0 + w] = bal;
            }
        }
        const uint32_t ballot = __ballot_sync(0xFFFFFFFFu, any);
        c.flags = (c.flags << 1) | (ballot ? 1u : 0u);
        // ---- levels 1..NL: level k computes plane t-k from level k-1
        levels<PH, 1, STEADY, NOCELLS>(t, q, exr, exw, outw, h, c);
        // ---- the plane the last level just staged leaves by one bulk store (its rows are contiguous in shared and global memory)
        const int zo = t - NL;
        const bool out_now = STEADY || (zo >= c.za && zo < c.zb);
        // the loads are thread 0's job, the stores thread 32's (bulk groups belong to the thread that commits them): one producer for both is late at every barrier
        if (threadIdx.x == 32) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");  // the store of the previous iteration has read its staging slab: the next iteration may overwrite it
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");        // my staging writes are visible to the bulk-copy engine
        __syncthreads();
        if (threadIdx.x == 32 && out_now) {
            const RowsSeg *sg = seg();
            const uint32_t src = c.out_ring + (q & 1u) * c.in_slot + sg->out_off;
            asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(sg->dst_rows + (size_t)zo * c.nxny), "r"(src), "r"(sg->out_bytes) : "memory");
            asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        }
    }
};

// grid: persistent, one CTA per SM; block = Gm.nwarps warps
template <int NL, int PX, int LRP, int MAXW, int CS, int RP>
__global__ void __launch_bounds__(MAXW * 32, 1) k_diffuse_rows(const FusedArgs A, const RowsGeom Gm)
{
    typedef Rows<NL, PX, LRP, CS, RP> R;
    extern __shared__ __align__(128) unsigned char rsm[];
    constexpr int NX = PX * LRP, RW = 32 / LRP;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lx = lane % LRP, gl = warp * RW + lane / LRP;                 // row pair inside the slab
    const int x0 = PX * lx;
    const uint32_t base = smem_u32(rsm);

    RowsCtx c;
    c.nxny = NX * A.ny; c.nz = A.nz;
    c.bars = base; c.in_ring = base + Gm.off_in; c.st_ring = base + Gm.off_st; c.out_ring = base + Gm.off_out;
    c.in_slot = (uint32_t)(Gm.hrows * NX) * 4u; c.st_slot = (uint32_t)(Gm.hrows * NX);
    c.ex_lvl = (uint32_t)(Gm.hrows + 2) * R::EXP;
    c.itg = 0; c.par = 0;
    c.zero2 = pk(A.zero, A.zero);
    if (tid == 0) {
#pragma unroll
        for (int r = 0; r < F_RING; ++r) mbar_init(c.bars + 8u * r, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int e = tid; e < 96; e += blockDim.x) reinterpret_cast<float *>(rsm + Gm.off_lut)[e] = A.lut[e / 32][e % 32];
    for (uint32_t e = tid; e < (Gm.smem_bytes - Gm.off_ex) / 8u; e += blockDim.x) reinterpret_cast<u64 *>(rsm + Gm.off_ex)[e] = 0ull;   // exchange and staging
    const int rank = CS > 1 ? (int)cluster_rank() : 0;
    c.rem = 0u; c.rem_row1 = false;
    if constexpr (CS > 1) {
        // the CTAs of a cluster hold consecutive ranges of hrows rows; exchange row 0 / hrows + 1 of a CTA is written by its neighbour
        const int pairs = Gm.hrows / 2;
        if (gl == 0 && rank > 0) c.rem = map_to_rank(base + Gm.off_ex + (uint32_t)(Gm.hrows + 1) * R::EXP + (uint32_t)x0 * 4u, (uint32_t)(rank - 1));
        if (gl == pairs - 1 && rank < CS - 1) { c.rem = map_to_rank(base + Gm.off_ex + (uint32_t)x0 * 4u, (uint32_t)(rank + 1)); c.rem_row1 = true; }
        cluster_barrier();                                                   // nobody writes into an exchange that is still being zeroed
        cluster_arrive();                                                    // pairs with the wait at the top of the first iteration
    } else {
        __syncthreads();
    }

    const int nzi = A.nz - 2;
    const int wid = CS > 1 ? (int)blockIdx.x / CS : (int)blockIdx.x;       // the CTAs of a cluster work through the same segments in lockstep
    long long p = Gm.start[wid];
    const long long p_end = Gm.start[wid + 1];
    u64 h[NL][3][PX * RP];
#pragma unroll
    for (int k = 0; k < NL; ++k)
#pragma unroll
        for (int s = 0; s < 3; ++s)
#pragma unroll
            for (int j = 0; j < PX * RP; ++j) h[k][s][j] = 0ull;

    while (p < p_end) {
        const int unit = (int)(p / nzi);
        const int slab = CS > 1 ? rank : unit % A.nslab, us = CS > 1 ? unit : unit / A.nslab;
        const int b = us / 3, sp = us % 3;
        c.za = 1 + (int)(p - (long long)unit * nzi);
        c.zb = (int)min((long long)(A.nz - 1), (long long)c.za + (p_end - p));
        p += c.zb - c.za;
        const int ty0 = A.sy0[slab], ty1 = A.sy1[slab], oy0 = A.so0[slab], oy1 = A.so1[slab];
        const int rows = ty1 - ty0;                                            // a multiple of 2 * RP, >= 2 * RP * RW
        const int row0 = 2 * RP * min(gl, rows / (2 * RP) - 1);                // groups beyond a short slab: duplicates of its last group (same values to the same addresses)
        const size_t ubase = (size_t)b * (size_t)c.nxny * (size_t)A.nz;
        c.lane_b = (uint32_t)(row0 * NX + x0) * 4u;
        c.ex_lane = base + Gm.off_ex + (uint32_t)row0 * R::EXP + (uint32_t)x0 * 4u;
        c.src = A.src[sp] + ubase + (size_t)(ty0 + row0) * NX + x0;
        {   // vote bytes: the warp's 2 * RP * RW rows (clamped into the slab), 16 bytes per lane
            const int vr0 = min(2 * RP * RW * warp, rows - 2 * RP * RW);
            c.st_vote = lane < (2 * RP * RW * NX) / 16 ? (uint32_t)(vr0 * NX + 16 * lane) : 0xFFFFFFFFu;
        }
        c.t0 = c.za - NL;
        c.nsteps = c.zb - c.za + 2 * NL;
        c.ld_lo = max(0, c.za - NL); c.ld_hi = min(A.nz, c.zb + NL);
        c.st_lo = 2 * NL; c.st_hi = min(A.nz, c.zb + NL) - c.t0;
        c.flags = 0; c.slowmask = A.always_slow[sp] ? 0xFFFFFFFFu : 0u;
        c.lut = base + Gm.off_lut + (uint32_t)sp * 128u;
        c.occ_nw = 0;
        if (sp == 0 && A.occ != nullptr) c.occ_nw = (uint32_t)((oy1 * NX + 255) / 256) - (uint32_t)((oy0 * NX + 255) / 256);
        {
            const float l = A.lam[sp];
            // the slab's first / last row is frozen (WALL, or halo edge); in a cluster only the lattice's own first / last row (WALL)
#pragma unroll
            for (int pp = 0; pp < RP; ++pp) {
                const int r0 = row0 + 2 * pp;
                const float m0 = (CS > 1 ? ty0 + r0 > 0 : r0 > 0) ? 1.0f : 0.0f;
                const float m1 = (CS > 1 ? ty0 + r0 + 1 < A.ny - 1 : r0 + 1 < rows - 1) ? 1.0f : 0.0f;
                c.lamM[pp] = pk(l * m0, l * m1);
                c.lamL[pp] = lx == 0 ? pk(0.0f, 0.0f) : c.lamM[pp];            // x = 0 and x = nx-1 are WALL
                c.lamR[pp] = lx == LRP - 1 ? pk(0.0f, 0.0f) : c.lamM[pp];
            }
        }
        // The store of the previous segment's last plane is issued by thread 32 AFTER that segment's last barrier, from the descriptor
        // below (dst_rows, out_off, out_bytes).  Without this barrier thread 0 can overwrite the descriptor first, and the plane goes
        // to the NEXT segment's destination -- another slab, species or simulation.  (Round 2 had that race for a few commits after
        // the stores moved from thread 0 to thread 32: rare, invisible in 60-step parity windows, found when two identical runs of the
        // configs[3] job at batch 512 disagreed; tests/test_gpu_long.py::test_full_batch_runs_are_deterministic_... guards it.)
        __syncthreads();
        if (tid == 0) {
            RowsSeg *sg = R::seg();
            sg->src_rows = A.src[sp] + ubase + (size_t)ty0 * NX;
            sg->st_rows = A.state + ubase + (size_t)ty0 * NX;
            sg->dst_rows = A.dst[sp] + ubase + (size_t)oy0 * NX;
            sg->ld_fbytes = (uint32_t)(rows * NX) * 4u; sg->ld_sbytes = (uint32_t)(rows * NX);
            sg->out_off = (uint32_t)((oy0 - ty0) * NX) * 4u; sg->out_bytes = (uint32_t)((oy1 - oy0) * NX) * 4u;
            // occupancy words of a plane whose first byte lies in this slab's output rows (the halo covers the rest of the word)
            sg->occ_row = A.occ ? A.occ + (size_t)b * (size_t)(c.nxny / 256) * (size_t)A.nz : nullptr;
            sg->occ_w0 = (uint32_t)((oy0 * NX + 255) / 256);
            sg->occ_soff = sg->occ_w0 * 256u - (uint32_t)(ty0 * NX);
        }
        __syncthreads();
        const int i0 = ((c.ld_lo - c.t0) / 3) * 3;                           // iterations before the first loaded plane have nothing to do
        if (tid == 0)
            for (int i = i0; i < i0 + F_RING - 1 && i < c.nsteps; ++i) R::issue(c, i, i - i0);
        for (int i = i0; i < c.nsteps; i += 3) {
            if (i >= c.st_lo && i + 3 <= c.st_hi) {
                R::template step<0, true>(i, h, c);
                R::template step<1, true>(i + 1, h, c);
                R::template step<2, true>(i + 2, h, c);
            } else {
                R::template step<0, false>(i, h, c);
                if (i + 1 < c.nsteps) R::template step<1, false>(i + 1, h, c);
                if (i + 2 < c.nsteps) R::template step<2, false>(i + 2, h, c);
            }
        }
        c.itg += (uint32_t)c.nsteps;
    }
    if (tid == 32) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // the last stores must have left shared memory before the CTA retires
    if constexpr (CS > 1) { cluster_wait(); cluster_barrier(); }              // the last arrive; and no neighbour may still be sending into a CTA that has gone
}

// ------------------------------------------------------------------ host side --
// expitch_words: row pitch of the exchange buffer in words (Rows::EXP / 4)
inline size_t rows_smem(int nx, int nl, int hrows, RowsGeom &G, int expitch_words = 0)
{
    const int exw = expitch_words ? expitch_words : nx;
    size_t o = 128;
    G.hrows = hrows;
    G.off_lut = (uint32_t)o; o += 96 * 4; o = (o + 127) / 128 * 128;
    G.off_in = (uint32_t)o; o += (size_t)F_RING * hrows * nx * 4; o = (o + 127) / 128 * 128;
    G.off_st = (uint32_t)o; o += (size_t)F_SRING * hrows * nx; o = (o + 127) / 128 * 128;
    G.off_ex = (uint32_t)o; o += (size_t)2 * nl * (hrows + 2) * exw * 4; o = (o + 127) / 128 * 128;
    G.off_out = (uint32_t)o; o += (size_t)2 * hrows * nx * 4; o = (o + 127) / 128 * 128;
    G.smem_bytes = (uint32_t)o;
    return o;
}

// lane layouts: 96 = 3 x 32 lanes, 16 warps of one row pair; 80 = 5 x 16 lanes, 11 warps of two row pairs
inline bool rows_shape(int nx, int &px, int &lrp, int &maxw)
{
    if (nx == 96) { px = 3; lrp = 32; maxw = 16; return true; }
    if (nx == 80) { px = 5; lrp = 16; maxw = 11; return true; }   // 11 warps = 44 rows; launch bounds of 12 warps keep ptxas at 168 registers (3 warps per scheduler)
    return false;
}

template <int NL, int PX, int LRP, int MAXW, int RP>
inline cudaError_t rows_launch_t(FusedPlan &F, const FusedArgs &A, int grid, cudaStream_t st)
{
    RowsGeom G{};
    rows_smem(A.nx, NL, A.rga, G, (int)(Rows<NL, PX, LRP, 1, RP>::EXP / 4u));
    G.nwarps = RP == 1 ? F.slab_warps : (F.slab_maxh / (2 * RP) + 32 / LRP - 1) / (32 / LRP);
    const int units = A.batch * 3 * A.nslab;
    if (grid > F_MAXGRID) grid = F_MAXGRID;
    fused_split_cached(F, units, A.nz - 2, NL, grid, G.start);
    bool &done = RP == 1 ? F.attr_done[NL] : F.rp_attr_done[NL];
    if (!done) {
        cudaError_t e = cudaFuncSetAttribute(k_diffuse_rows<NL, PX, LRP, MAXW, 1, RP>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        done = true;
    }
    k_diffuse_rows<NL, PX, LRP, MAXW, 1, RP><<<grid, G.nwarps * 32, G.smem_bytes, st>>>(A, G);
    return cudaGetLastError();
}

// Cluster variant: CS CTAs share a plane (ny = CS * hrows exactly), boundary rows travel through distributed shared memory.
// One cluster per CS SMs, persistent; the (unit, plane) space is split over the clusters.
template <int NL, int PX, int LRP, int MAXW, int CS>
inline cudaError_t rows_launch_cluster_t(FusedPlan &F, const FusedArgs &A0, cudaStream_t st)
{
    FusedArgs A = A0;
    const int hrows = A.ny / CS;
    A.nslab = 1; A.rga = hrows;
    for (int r = 0; r < CS; ++r) { A.sy0[r] = A.so0[r] = (short)(r * hrows); A.sy1[r] = A.so1[r] = (short)((r + 1) * hrows); }
    RowsGeom G{};
    rows_smem(A.nx, NL, hrows, G);
    G.nwarps = (hrows / 2) / (32 / LRP);
    auto kern = k_diffuse_rows<NL, PX, LRP, MAXW, CS, 1>;
    cudaLaunchConfig_t cfg = {};
    cfg.blockDim = dim3((unsigned int)(G.nwarps * 32));
    cfg.dynamicSmemBytes = G.smem_bytes;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = CS; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    if (!F.cluster_attr_done[NL]) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        if (CS > 8) { e = cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1); if (e != cudaSuccess) return e; }
        cfg.gridDim = dim3((unsigned int)(F.sms / CS * CS));
        int nc = 0;
        e = cudaOccupancyMaxActiveClusters(&nc, kern, &cfg);
        if (e != cudaSuccess) return e;
        if (nc < 1) return cudaErrorLaunchOutOfResources;
        F.nclusters = nc;
        F.cluster_attr_done[NL] = true;
    }
    const int units = A.batch * 3;
    const long long total = (long long)units * (A.nz - 2);
    int ncl = (int)std::max<long long>(1, std::min<long long>(std::min(F.nclusters, F_MAXGRID / CS), total / 2 + 1));
    fused_split_cached(F, units, A.nz - 2, NL, ncl, G.start);
    cfg.gridDim = dim3((unsigned int)(ncl * CS));
    return cudaLaunchKernelEx(&cfg, kern, A, G);
}

template <int NL>
inline cudaError_t rows_launch(FusedPlan &F, const FusedArgs &A, int grid, cudaStream_t st)
{
    if (A.nx == 96 && F.rows_cluster == 3) return rows_launch_cluster_t<NL, 3, 32, 16, 3>(F, A, st);   // BASELINE configs[2]: 3 CTAs x 32 rows
    if (A.nx == 96 && F.rows_rp == 2) return rows_launch_t<NL, 3, 32, 8, 2>(F, A, grid, st);   // four rows per lane: 8 warps, up to 255 registers
    if (A.nx == 96) return rows_launch_t<NL, 3, 32, 16, 1>(F, A, grid, st);   // 96-wide planes of any height: slabs with a halo
    return rows_launch_t<NL, 5, 16, 12, 1>(F, A, grid, st);                   // BASELINE configs[3]
}

// Does the rows kernel cover this lattice?  Fills the slab table of F.args (rga = rows a CTA holds).
inline bool rows_configure(const KParams &P, FusedPlan &F)
{
    int px, lrp, maxw;
    if (!rows_shape(P.nx, px, lrp, maxw) || P.ny % F_PY || P.ny < 8) return false;
    const int rw = 32 / lrp, hrows = 2 * rw * maxw;
    F.args.nslab = slab_cuts(P.ny, hrows, F.args.sy0, F.args.sy1, F.args.so0, F.args.so1);
    if (!F.args.nslab) return false;
    int maxh = 0;
    for (int t = 0; t < F.args.nslab; ++t) maxh = std::max(maxh, F.args.sy1[t] - F.args.sy0[t]);
    F.args.rga = hrows;
    F.slab_warps = (maxh / 2 + rw - 1) / rw;
    F.slab_maxh = maxh;
    RowsGeom G{};
    const int exw = (rw > 1 && (2 * P.nx) % 32 == 0) ? P.nx + 8 : P.nx;        // Rows::EXP for two rows per lane (the largest exchange)
    if (rows_smem(P.nx, F_MAXNL, hrows, G, exw) > 227 * 1024) return false;
    F.lrp = lrp;
    // The cluster variant (96 rows = 3 CTAs x 16 warps x one row pair, no halo) is correct and selectable ("rows_cluster" = 3) but
    // OFF by default: measured 0.851 ms against 0.769 ms for the slabs with a halo at 64 x 96^3 (45 clusters = 135 of 148 SMs
    // resident, and an iteration of three SMs in lockstep costs 4075 cycles against 3063), DESIGN.md section 7.
    F.rows_cluster = 0;
    // four rows per lane on 96-wide planes (8 warps, 240 registers): 5.58 against 5.70 ms per launch at 512 x 96^3; the lane
    // layout of 80-wide planes (5 sites per lane) would need more than 255 registers for it
    F.rows_rp = P.nx == 96 ? 2 : 1;
    return true;
}

}  // namespace ca
