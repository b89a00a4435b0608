// ca_fused.cuh -- temporally fused reaction-diffusion kernel: NL (<= 4) sub-steps of [D S1] in ONE pass over HBM.
//
// Why it looks like this: per site and CA step the stencil costs 12 x (8..9) fp32
// operations against 25 bytes, so on B200 the FMA pipe (128 lanes/clk/SM) is as tight as HBM.  The kernel
// therefore (a) reads and writes every field value once per CA step, (b) issues the arithmetic as packed
// f32x2 instructions (same IEEE results as scalar add/mul/fma.rn, half the issue slots), and (c) keeps the
// z-neighbours and all NL time levels of a lane's points in registers:
//
//   * a work unit is (simulation, species, range of z-planes); a persistent grid of one CTA per SM splits
//     the flattened plane space evenly, so the only redundant work is the NL-deep cone at cuts inside a unit;
//   * a CTA covers whole xy-planes (nx, ny <= 64, so no xy halo: the WALL layer closes the plane) and marches
//     along z; a lane owns 2 (x) x 4 (y) points of the plane, a warp a 64 x 4 strip (two 32 x 4 strips
//     when nx <= 32);
//   * input planes and state planes arrive by bulk async copy (TMA 1-D, UBLKCP) into shared-memory rings,
//     completion on mbarriers, 2 planes ahead;
//   * level k (sub-step k) computes plane t-k while level 0 loads plane t: each level keeps 3 planes of its
//     input level in registers (ring of 3, the march loop is unrolled by 3 so that no register is moved);
//   * x-neighbours come from the neighbouring lane by shuffle, y-neighbours across strips through a small
//     double-buffered shared-memory row exchange (one __syncthreads per plane);
//   * the reaction term exists only where cells live (a few % of the lattice at configs[1]): each warp votes per
//     plane on "any cell in my strip" and takes the path without source term and clamp when there is none
//     (bit-identical there: v + 0 = v, and v >= 0 is guaranteed when 6*lambda*(1+2^-23) <= 1).
//
// Arithmetic per point is exactly [D S1]: sum6 = ((xm+xp)+(ym+yp))+(zm+zp); lap = sum6 - 6*c (product rounded
// on its own); v = fma(lambda, lap, c); v += r; max(v, 0).  WALL points use lambda = 0, r = 0, which
// returns c unchanged.
#pragma once
#include <cstdlib>
#include <cstring>
#include "ca_device.cuh"

namespace ca {

typedef unsigned long long u64;

constexpr int F_PY = 4;        // rows per lane
constexpr int F_RING = 3;      // field-plane ring depth = register phase count (prefetch distance 2)
constexpr int F_SRING = 8;     // state-plane ring depth (a plane is used by NL consecutive iterations)
constexpr int F_MAXNL = 4;
constexpr int F_MAXSLAB = 8;
constexpr int F_SLAB_WARPS = 15;  // slab variant: 480 threads, so that a thread may use 136 registers (the seam exchange needs a few more than 128)
constexpr int F_MAXGRID = 640; // persistent CTAs at most (the split table travels as a kernel parameter)

struct FusedArgs {
    const float *src[3];       // current field buffers [batch][nz][ny][nx]
    float *dst[3];             // other ping-pong buffers
    const uint8_t *state;
    int nx, ny, nz, batch;
    float lam[3];
    float lut[3][32];          // source term by (state & 31): rate[s][mode] if kind in 1..4 else 0  [D G4]
    int always_slow[3];        // 1: the clamp cannot be proven idle for this lambda -> always take the full path
    float zero;                // 0.0f, opaque to ptxas (see Fused::level)
    uint32_t *occ;             // occupancy map for S2/S3 (one bit per 8 state bytes), written by the fixed-size kernels; may be NULL
    // slab variant (planes wider or taller than 64 sites): a plane is cut along y into nslab slabs of whole rows; slab s
    // loads rows [sy0, sy1) -- its output rows [so0, so1) plus a halo of F_MAXNL rows towards neighbouring slabs -- and a
    // row is covered by nxb column blocks of 2*LRP sites (rga = row groups of F_PY rows a CTA holds)
    int nslab, nxb, rga;
    short sy0[F_MAXSLAB], sy1[F_MAXSLAB], so0[F_MAXSLAB], so1[F_MAXSLAB];
};

// ---- packed f32x2 arithmetic (Blackwell FADD2/FMUL2/FFMA2); .rn, no ftz: identical to two scalar ops ----
__device__ __forceinline__ u64 pk(float lo, float hi) { u64 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk(u64 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ u64 add2(u64 a, u64 b) { u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 sub2(u64 a, u64 b) { u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 mul2(u64 a, u64 b) { u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) { u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }

// ---- mbarrier / bulk-copy helpers (shared::cta addresses as 32-bit) ----
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) { asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count)); }
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}

__device__ __forceinline__ u64 lds64(uint32_t a) { u64 v; asm volatile("ld.shared.b64 %0, [%1];" : "=l"(v) : "r"(a)); return v; }
__device__ __forceinline__ void sts64(uint32_t a, u64 v) { asm volatile("st.shared.b64 [%0], %1;" ::"r"(a), "l"(v) : "memory"); }
__device__ __forceinline__ uint32_t lds16(uint32_t a) { uint32_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ float lds32f(uint32_t a) { float v; asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(a)); return v; }
__device__ __forceinline__ float4 lds128f(uint32_t a)
{
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(a));
    return v;
}
__device__ __forceinline__ void sts128f(uint32_t a, float x, float y, float z, float w)
{
    asm volatile("st.shared.v4.f32 [%0], {%1, %2, %3, %4};" ::"r"(a), "f"(x), "f"(y), "f"(z), "f"(w) : "memory");
}

struct FusedGeom {             // host-computed launch geometry, passed by value
    int nwarps, ngroups_alloc; // strips of F_PY rows: groups = nwarps * (32 / LRP)
    uint32_t off_lut, off_in, off_st, off_ex, off_xex, off_xdummy, smem_bytes;
    long long total_planes;    // batch * 3 * (nz - 2): the flattened (unit, interior plane) space
    int start[F_MAXGRID + 1];  // CTA g works on flattened planes [start[g], start[g+1]) (cost-balanced on the host)
};

// per-thread view of one segment (unit = simulation x species, planes [za, zb))
struct FusedCtx {
    const float *src;          // field of this unit, already offset to this lane's (x0, y0)
    float *dst;
    const float *src_plane0;   // unit base (for the bulk copies)
    const uint8_t *st_plane0;
    int nx, nxny, nz;          // run-time geometry (ignored by the fixed-size instantiations)
    uint32_t ex_lvl;
    int za, zb, t0, nsteps;
    int ld_lo, ld_hi;          // planes level 0 loads
    int st_lo, st_hi;          // iterations [st_lo, st_hi): every level computes, no WALL plane involved
    uint32_t itg;              // running iteration counter of this CTA (state-ring slots)
    uint32_t par;              // bit r: parity to wait for on field-ring slot r
    uint32_t flags, slowmask;  // bit k: "cells in my strip" for the plane level k works on
    uint32_t bars, in_ring, st_ring, lut;         // shared-memory addresses
    uint32_t in_lane;          // this lane's (x0, y0) inside ring slot 0
    uint32_t st_lane, st_strip;   // this lane's points / this lane's 8 bytes of the warp strip inside state slot 0
    uint32_t ex_self;          // this lane's slot in the "top rows" array of exchange buffer 0, level 0
    u64 lam2[F_PY];
    u64 zero2;                 // (0, 0) that ptxas cannot see through
    uint32_t rowmask;          // bit j: row y0+j exists and this lane's x pair is inside the lattice
    bool strip_ok;
    uint32_t *occ_row;         // species 0 only: occupancy words of this warp's strip, indexed by plane (else NULL)
    // slab variant
    uint32_t in_slot, st_slot;     // bytes of one ring slot (the tallest slab)
    uint32_t yst;                  // bytes of one row of the y-exchange (a whole lattice row)
    uint32_t xs_w, xel;            // x-seam exchange between column blocks: my store slot (buffer 0, level 0), bytes per level
    bool seam_l, seam_r;           // this lane sits on a seam between two column blocks, on the left / right edge of its block
    uint32_t occ_nw;               // species 0: number of occupancy words of a plane this slab is responsible for (else 0)
};

// slab variant: per-segment constants that only the producer thread (bulk copies) or one lane per warp (occupancy words) needs
// live in shared memory, not in registers
struct SlabSeg {
    const float *src_plane0;       // first loaded row of plane 0 of this unit
    const uint8_t *st_plane0;
    uint32_t *occ_row;             // occupancy words of this simulation
    uint32_t ld_fbytes, ld_sbytes; // bytes of this slab's rows of a field / state plane
    uint32_t occ_w0, occ_soff;     // first word this slab writes; its byte offset inside the state slot
};
constexpr uint32_t F_SEG_OFF = 32; // inside the first 128 bytes of shared memory, after the mbarriers

// NX = NY = 0: lattice dims at run time (any even nx <= 2*LRP); otherwise compile-time dims, all address math folds
// SLAB: planes larger than a CTA holds; NX, NY then give the lattice (NX = nxb * 2 * LRP) and the CTA works on y-slabs
template <int NL, int LRP, int NX, int NY, bool SLAB = false>
struct Fused {
    static constexpr bool FIXED = NX != 0;
    static constexpr int RW = 32 / LRP;
    static constexpr int NXB = (SLAB && FIXED) ? NX / (2 * LRP) : 1;                 // column blocks (slab variant with compile-time dims)
    static constexpr int RGA = (SLAB && FIXED) ? (F_SLAB_WARPS * RW) / NXB : 0;      // row groups a CTA of 15 warps holds
    // every lane and row holds valid data: whole fixed-size planes, or a slab (groups beyond a short slab are clamped onto its
    // last row group: they compute duplicates that feed only the frozen last row and are never stored)
    static constexpr bool FULL = SLAB || (FIXED && NX == 2 * LRP && NY % (F_PY * RW) == 0);
    static constexpr uint32_t GRP = LRP * 8u;                                         // bytes one row group exchanges per row
    static constexpr uint32_t EXL = SLAB ? 2u * (uint32_t)(RGA + 2) * (uint32_t)NX * 4u
                                         : (FIXED ? 2u * (((NY + F_PY * RW - 1) / (F_PY * RW)) * RW + 2u) * GRP : 0u);
    static constexpr uint32_t XEL = (uint32_t)(RGA * NXB) * 32u;                      // x-seam exchange, bytes per level

    static __device__ __forceinline__ int nx(const FusedCtx &c) { return FIXED ? NX : c.nx; }
    static __device__ __forceinline__ int nxny(const FusedCtx &c) { return FIXED ? NX * NY : c.nxny; }
    static __device__ __forceinline__ uint32_t exl(const FusedCtx &c) { return FIXED ? EXL : c.ex_lvl; }
    static __device__ __forceinline__ uint32_t xel(const FusedCtx &c) { return FIXED ? XEL : c.xel; }
    static __device__ __forceinline__ uint32_t yst(const FusedCtx &c) { return SLAB ? (FIXED ? (uint32_t)NX * 4u : c.yst) : GRP; }
    static __device__ __forceinline__ bool row(const FusedCtx &c, int j) { return FULL ? true : ((c.rowmask >> j) & 1u) != 0u; }
    // slab variant: only the slab's output rows are stored (and only by the groups that are not clamped duplicates)
    static __device__ __forceinline__ bool srow(const FusedCtx &c, int j) { return SLAB ? ((c.rowmask >> (16 + j)) & 1u) != 0u : row(c, j); }
    static __device__ __forceinline__ uint32_t stpitch(const FusedCtx &c) { return (uint32_t)nx(c); }
    static __device__ __forceinline__ uint32_t stslot(const FusedCtx &c) { return SLAB ? ((FIXED) ? (uint32_t)(RGA * F_PY * NX) : c.st_slot) : (uint32_t)nxny(c); }
    static __device__ __forceinline__ uint32_t inpitch(const FusedCtx &c) { return (uint32_t)nx(c) * 4u; }
    static __device__ __forceinline__ uint32_t inslot(const FusedCtx &c) { return SLAB ? ((FIXED) ? (uint32_t)(RGA * F_PY * NX) * 4u : c.in_slot) : (uint32_t)nxny(c) * 4u; }

    // the diffusion part of one sub-step of [D S1] for this lane's 2 x 4 points; C = centre plane, M/P = planes z-1/z+1
    static __device__ __forceinline__ void level(const u64 (&M)[F_PY], const u64 (&C)[F_PY], const u64 (&P)[F_PY], u64 (&N)[F_PY],
                                                 u64 up, u64 dn, const u64 (&lam2)[F_PY], const u64 zero2,
                                                 const float4 xe, const bool seam_l, const bool seam_r)
    {
        const u64 six2 = pk(6.0f, 6.0f);
        const float xev[F_PY] = { xe.x, xe.y, xe.z, xe.w };
#pragma unroll
        for (int j = 0; j < F_PY; ++j) {
            float c0, c1;
            upk(C[j], c0, c1);
            float xl = __shfl_up_sync(0xFFFFFFFFu, c1, 1, LRP);            // value at x0-1 (own c1 at the strip edge: WALL side, unused)
            float xr = __shfl_down_sync(0xFFFFFFFFu, c0, 1, LRP);          // value at x0+2
            if constexpr (SLAB) {                                           // seam between two column blocks: the neighbour block's edge column
                xl = seam_l ? xev[j] : xl;
                xr = seam_r ? xev[j] : xr;
            }
            const u64 xs = pk(__fadd_rn(xl, c1), __fadd_rn(c0, xr));       // xm + xp
            const u64 ys = add2(j == 0 ? up : C[j > 0 ? j - 1 : 0], j == F_PY - 1 ? dn : C[j < F_PY - 1 ? j + 1 : 0]);   // ym + yp
            const u64 zs = add2(M[j], P[j]);                                 // zm + zp
            const u64 s6 = add2(add2(xs, ys), zs);
            // 6*c must be rounded on its own [D S1].  ptxas contracts mul.rn.f32x2 + sub.rn.f32x2 into one FFMA2 (seen in SASS,
            // CUDA 12.9), so the product is formed as fma(6, c, 0) with a zero the compiler cannot fold: same value, same pipe cost.
            const u64 lap = sub2(s6, fma2(six2, C[j], zero2));
            N[j] = fma2(lam2[j], lap, C[j]);                                 // the source term and the clamp follow in levels()
        }
    }

    // slab variant: a lane on a seam publishes its edge column (F_PY rows) of level K for the neighbouring column block
    static __device__ __forceinline__ void seam_store(const FusedCtx &c, const uint32_t addr, const u64 (&V)[F_PY])
    {
        float e[F_PY];                                                      // no branch: lanes off a seam store into a sink slot
#pragma unroll
        for (int j = 0; j < F_PY; ++j) {
            float a, b;
            upk(V[j], a, b);
            e[j] = c.seam_r ? b : a;
        }
        sts128f(addr, e[0], e[1], e[2], e[3]);
    }

    static __device__ __forceinline__ SlabSeg *slab_seg()
    {
        extern __shared__ __align__(128) unsigned char fsm_[];
        return reinterpret_cast<SlabSeg *>(fsm_ + F_SEG_OFF);
    }

    // producer (one thread): start the bulk copies of iteration i into field-ring slot i mod 3
    static __device__ __forceinline__ void issue(const FusedCtx &c, int i, int slot)
    {
        const int t = c.t0 + i;
        const uint32_t bar = c.bars + 8u * (uint32_t)slot;
        if (t >= c.ld_lo && t < c.ld_hi) {
            uint32_t pb = (uint32_t)nxny(c) * 4u, sb = (uint32_t)nxny(c);
            const float *fsrc = c.src_plane0;
            const uint8_t *ssrc = c.st_plane0;
            if constexpr (SLAB) {                                            // a slab's rows are contiguous; its constants live in shared memory
                const SlabSeg *sg = slab_seg();
                pb = sg->ld_fbytes; sb = sg->ld_sbytes; fsrc = sg->src_plane0; ssrc = sg->st_plane0;
            }
            mbar_expect_tx(bar, pb + sb);
            bulk_g2s(c.in_ring + (uint32_t)slot * inslot(c), fsrc + (size_t)t * nxny(c), pb, bar);
            bulk_g2s(c.st_ring + ((c.itg + (uint32_t)i) & (F_SRING - 1)) * stslot(c), ssrc + (size_t)t * nxny(c), sb, bar);
        } else {
            mbar_arrive(bar);
        }
    }

    // level K (sub-step K) at iteration i: computes plane t-K; outside the steady range it may idle or copy a WALL plane
    template <int PH, int K, bool STEADY, bool NOCELLS>
    static __device__ __forceinline__ void levels(const int t, const uint32_t q, const uint32_t exr, const uint32_t exw,
                                                  const uint32_t xsr, const uint32_t xsw, u64 (&h)[NL][3][F_PY], FusedCtx &c)
    {
        if constexpr (K <= NL) {
            constexpr int sm = (PH - K - 1 + 12) % 3, sc = (PH - K + 12) % 3, sp = (PH - K + 1 + 12) % 3;
            constexpr int KO = K < NL ? K : 0;                              // output level (unused when K == NL)
            const int zc = t - K;
            bool compute = true;
            if (!STEADY) compute = zc >= max(1, c.za - (NL - K)) && zc < min(c.nz - 1, c.zb + (NL - K));
            if (compute) {
                const uint32_t el = exl(c);
                const u64 up = lds64(exr + (uint32_t)(K - 1) * el + (el / 2 - yst(c)));  // bottom row of the strip above
                const u64 dn = lds64(exr + (uint32_t)(K - 1) * el + yst(c));             // top row of the strip below
                float4 xe = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
                if constexpr (SLAB) {
                    xe = lds128f(xsr + (uint32_t)(K - 1) * xel(c));                             // the neighbour block's edge column, written by the previous iteration (lanes off a seam: a sink nobody selects from)
                }
                u64 nloc[F_PY];
                u64 (&N)[F_PY] = *(K < NL ? &h[KO][sc] : &nloc);
                level(h[K - 1][sm], h[K - 1][sc], h[K - 1][sp], N, up, dn, c.lam2, c.zero2, xe, c.seam_l, c.seam_r);
                if (!NOCELLS && (((c.flags | c.slowmask) >> K) & 1u)) {    // cells in this strip: source term and clamp
                    const uint32_t s = c.st_lane + ((q - (uint32_t)K) & (F_SRING - 1)) * stslot(c);
#pragma unroll
                    for (int j = 0; j < F_PY; ++j) {
                        const uint32_t w = row(c, j) ? lds16(s + (uint32_t)j * stpitch(c)) : 0u;
                        const u64 v = add2(N[j], pk(lds32f(c.lut + (w & 31u) * 4u), lds32f(c.lut + ((w >> 8) & 31u) * 4u)));
                        float a, b;
                        upk(v, a, b);
                        N[j] = pk(fmaxf(a, 0.0f), fmaxf(b, 0.0f));
                    }
                }
                if constexpr (K < NL) {
                    sts64(exw + (uint32_t)K * el, N[0]);
                    sts64(exw + (uint32_t)K * el + el / 2, N[F_PY - 1]);
                    if constexpr (SLAB) seam_store(c, xsw + (uint32_t)K * xel(c), N);
                } else {
                    float *o = c.dst + (size_t)zc * nxny(c);
#pragma unroll
                    for (int j = 0; j < F_PY; ++j)
                        if (srow(c, j)) {
                            float a, b;
                            upk(N[j], a, b);
                            *reinterpret_cast<float2 *>(o + j * nx(c)) = make_float2(a, b);
                        }
                }
            } else if (K < NL && (zc == 0 || zc == c.nz - 1) && zc >= c.za - (NL - K) && zc < c.zb + (NL - K)) {
                // WALL plane: every level equals the input there
                const float *p = c.src + (size_t)zc * nxny(c);
#pragma unroll
                for (int j = 0; j < F_PY; ++j) {
                    float2 v = make_float2(0.0f, 0.0f);
                    if (row(c, j)) v = *reinterpret_cast<const float2 *>(p + j * nx(c));
                    h[KO][sc][j] = pk(v.x, v.y);
                }
            }
            levels<PH, K + 1, STEADY, NOCELLS>(t, q, exr, exw, xsr, xsw, h, c);
        }
    }

    // one march iteration; PH = i mod 3 selects the field-ring slot and the register slots
    // (slot of plane z = (z - t0) mod 3 on every level)
    template <int PH, bool STEADY>
    static __device__ __forceinline__ void step(const int i, u64 (&h)[NL][3][F_PY], FusedCtx &c)
    {
        // Round 1 kept a second copy of the steady iteration without any source-term code for strips that hold no cell.  One
        // body per phase is faster (round 2: configs[1] step 130.3 -> 127.9 us on 3k-cell tumours, 210.5 -> 205.0 us on 1.1e5-cell
        // ones): the untaken, warp-uniform branches cost less than the instruction-cache misses of six hot bodies.
        step_body<PH, STEADY, false>(i, h, c);
    }

    template <int PH, bool STEADY, bool NOCELLS>
    static __device__ __forceinline__ void step_body(const int i, u64 (&h)[NL][3][F_PY], FusedCtx &c)
    {
        const int t = c.t0 + i;
        const uint32_t q = c.itg + (uint32_t)i;
        if (threadIdx.x == 0 && i + (F_RING - 1) < c.nsteps) issue(c, i + (F_RING - 1), (PH + F_RING - 1) % 3);
        const uint32_t exb = exl(c) * NL;                                   // bytes of one exchange buffer
        const uint32_t exw = c.ex_self + ((uint32_t)i & 1u) * exb;          // rows written now, read by the next iteration
        const uint32_t exr = c.ex_self + exb - ((uint32_t)i & 1u) * exb;    // rows written by the previous iteration
        uint32_t xsw = 0, xsr = 0;
        if constexpr (SLAB) {                                                // the facing slot of the neighbour block is the next / previous 16 bytes
            const uint32_t xb = xel(c) * NL;
            xsw = c.xs_w + ((uint32_t)i & 1u) * xb;
            xsr = c.xs_w + xb - ((uint32_t)i & 1u) * xb + (c.seam_r ? 16u : 0xFFFFFFF0u);
        }
        // ---- level 0: plane t from the ring
        mbar_wait(c.bars + 8u * PH, (c.par >> PH) & 1u);
        c.par ^= 1u << PH;
        bool any = false;
        if (STEADY || (t >= c.ld_lo && t < c.ld_hi)) {
            const uint32_t a = c.in_lane + (uint32_t)PH * inslot(c);
#pragma unroll
            for (int j = 0; j < F_PY; ++j) h[0][PH][j] = row(c, j) ? lds64(a + (uint32_t)j * inpitch(c)) : 0ull;
            sts64(exw, h[0][PH][0]);
            sts64(exw + exl(c) / 2, h[0][PH][F_PY - 1]);
            if constexpr (SLAB) seam_store(c, xsw, h[0][PH]);
            // "cells in my strip": every lane looks at 8 bytes of the warp's strip of the state plane; a byte counts when kind is 1..6
            if constexpr (SLAB) {                                            // a warp's points are not contiguous bytes: every lane looks at its own 2 x 4 bytes
                // the warp's points are 32 / LRP row groups x F_PY rows x 2 * LRP contiguous bytes: every lane looks at 8 of them
                const u64 wv = lds64(c.st_strip + (q & (F_SRING - 1)) * stslot(c));
                any = (((wv & 0x0707070707070707ull) + 0x0101010101010101ull) & 0x0606060606060606ull) != 0ull;
                // the S2/S3 occupancy map (one bit per 8 consecutive state bytes, one word per 256): this slab's words of the plane,
                // read from the state slab in shared memory, one word per warp and trip
                for (uint32_t w = threadIdx.x >> 5; w < c.occ_nw; w += blockDim.x >> 5) {
                    const SlabSeg *sg = slab_seg();
                    const u64 v = lds64(c.st_ring + (q & (F_SRING - 1)) * stslot(c) + sg->occ_soff + w * 256u + 8u * (threadIdx.x & 31u));
                    const uint32_t bal = __ballot_sync(0xFFFFFFFFu, (((v & 0x0707070707070707ull) + 0x0101010101010101ull) & 0x0606060606060606ull) != 0ull);
                    if ((threadIdx.x & 31) == 0) sg->occ_row[(size_t)t * (size_t)(nxny(c) / 256) + sg->occ_w0 + w] = bal;
                }
            } else {
                const u64 w = c.strip_ok ? lds64(c.st_strip + (q & (F_SRING - 1)) * (uint32_t)nxny(c)) : 0ull;
                any = (((w & 0x0707070707070707ull) + 0x0101010101010101ull) & 0x0606060606060606ull) != 0ull;
            }
        }
        const uint32_t ballot = __ballot_sync(0xFFFFFFFFu, any);
        c.flags = (c.flags << 1) | (ballot ? 1u : 0u);
        if constexpr (FIXED && !SLAB) {                                     // the same vote is the S2/S3 occupancy map: strip = 256 contiguous bytes
            if ((threadIdx.x & 31) == 0 && c.occ_row != nullptr && (STEADY || (t >= c.ld_lo && t < c.ld_hi)))
                c.occ_row[(size_t)t * (NX * NY / 256)] = ballot;
        }
        // ---- levels 1..NL: level k computes plane t-k from level k-1
        levels<PH, 1, STEADY, NOCELLS>(t, q, exr, exw, xsr, xsw, h, c);
        __syncthreads();
    }
};

template <int NL, int LRP, int NX, int NY>
__global__ void __launch_bounds__(512, 1) k_diffuse_fused(const FusedArgs A, const FusedGeom Gm)
{
    typedef Fused<NL, LRP, NX, NY> F;
    extern __shared__ __align__(128) unsigned char fsm[];
    constexpr int RW = 32 / LRP;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lx = lane % LRP, g = warp * RW + lane / LRP;
    const int x0 = 2 * lx, y0 = F_PY * g;
    const uint32_t base = smem_u32(fsm);
    const int nxr = NX ? NX : A.nx, nyr = NY ? NY : A.ny;

    FusedCtx c;
    c.nx = nxr; c.nxny = nxr * nyr; c.nz = A.nz;
    c.bars = base; c.in_ring = base + Gm.off_in; c.st_ring = base + Gm.off_st;
    c.in_lane = c.in_ring + (uint32_t)(y0 * nxr + x0) * 4u;
    c.st_lane = c.st_ring + (uint32_t)(y0 * nxr + x0);
    const int strip_bytes = F_PY * RW * nxr;                                   // the warp's rows are contiguous in the plane
    c.strip_ok = 8 * lane < strip_bytes && (warp * F_PY * RW) * nxr + 8 * lane + 8 <= nxr * nyr;
    c.st_strip = c.st_ring + (uint32_t)((warp * F_PY * RW) * nxr + 8 * lane);
    c.ex_lvl = 2u * (uint32_t)(Gm.ngroups_alloc + 2) * F::GRP;                  // [top rows | bottom rows], each with a zero group at both ends
    c.ex_self = base + Gm.off_ex + (uint32_t)(g + 1) * F::GRP + (uint32_t)lx * 8u;
    c.rowmask = 0;
#pragma unroll
    for (int j = 0; j < F_PY; ++j)
        if (y0 + j < nyr && x0 < nxr) c.rowmask |= 1u << j;
    c.itg = 0; c.par = 0;
    c.zero2 = pk(A.zero, A.zero);

    // one-time shared-memory setup: barriers, source-term tables, zeroed exchange (its end groups stay zero)
    if (tid == 0) {
#pragma unroll
        for (int r = 0; r < F_RING; ++r) mbar_init(c.bars + 8u * r, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int e = tid; e < 96; e += blockDim.x) reinterpret_cast<float *>(fsm + Gm.off_lut)[e] = A.lut[e / 32][e % 32];
    for (uint32_t e = tid; e < 2u * NL * c.ex_lvl / 8u; e += blockDim.x) reinterpret_cast<u64 *>(fsm + Gm.off_ex)[e] = 0ull;
    __syncthreads();

    const int nzi = A.nz - 2;
    long long p = Gm.start[blockIdx.x];
    const long long p_end = Gm.start[blockIdx.x + 1];
    u64 h[NL][3][F_PY];
#pragma unroll
    for (int k = 0; k < NL; ++k)
#pragma unroll
        for (int s = 0; s < 3; ++s)
#pragma unroll
            for (int j = 0; j < F_PY; ++j) h[k][s][j] = 0ull;

    while (p < p_end) {
        const int unit = (int)(p / nzi);
        const int b = unit / 3, sp = unit % 3;
        c.za = 1 + (int)(p - (long long)unit * nzi);
        c.zb = (int)min((long long)(A.nz - 1), (long long)c.za + (p_end - p));
        p += c.zb - c.za;
        const size_t ubase = (size_t)b * (size_t)c.nxny * (size_t)A.nz;
        c.src_plane0 = A.src[sp] + ubase;
        c.st_plane0 = A.state + ubase;
        c.src = c.src_plane0 + (y0 * nxr + x0);
        c.dst = A.dst[sp] + ubase + (y0 * nxr + x0);
        c.t0 = c.za - NL;
        c.nsteps = c.zb - c.za + 2 * NL;
        c.ld_lo = max(0, c.za - NL); c.ld_hi = min(A.nz, c.zb + NL);
        c.st_lo = 2 * NL; c.st_hi = min(A.nz, c.zb + NL) - c.t0;              // za+NL <= t < min(nz, zb+NL)
        c.flags = 0; c.slowmask = A.always_slow[sp] ? 0xFFFFFFFFu : 0u;
        c.lut = base + Gm.off_lut + (uint32_t)sp * 128u;
        c.occ_row = (sp == 0 && A.occ != nullptr && NX != 0) ? A.occ + (size_t)b * (size_t)(c.nxny / 256) * (size_t)A.nz + warp : nullptr;
        const float lam = A.lam[sp];
#pragma unroll
        for (int j = 0; j < F_PY; ++j) {
            const int y = y0 + j;
            const bool rowin = y > 0 && y < nyr - 1;                           // y walls and rows outside the lattice: lambda = 0
            c.lam2[j] = pk(rowin && x0 > 0 && x0 < nxr - 1 ? lam : 0.0f, rowin && x0 + 1 < nxr - 1 ? lam : 0.0f);
        }
        const int i0 = ((c.ld_lo - c.t0) / 3) * 3;                           // iterations before the first loaded plane have nothing to do
        if (tid == 0)
            for (int i = i0; i < i0 + F_RING - 1 && i < c.nsteps; ++i) F::issue(c, i, i - i0);
        for (int i = i0; i < c.nsteps; i += 3) {
            if (i >= c.st_lo && i + 3 <= c.st_hi) {
                F::template step<0, true>(i, h, c);
                F::template step<1, true>(i + 1, h, c);
                F::template step<2, true>(i + 2, h, c);
            } else {
                F::template step<0, false>(i, h, c);
                if (i + 1 < c.nsteps) F::template step<1, false>(i + 1, h, c);
                if (i + 2 < c.nsteps) F::template step<2, false>(i + 2, h, c);
            }
        }
        c.itg += (uint32_t)c.nsteps;
    }
}

// Slab variant for planes a CTA cannot hold whole (BASELINE configs[2], [3]: 96^3, 80^3).  Same march, same levels, same
// bulk-copy rings; a work unit is (simulation, species, y-slab, z-range).  A slab is a range of WHOLE rows of the plane --
// contiguous in memory, so it arrives by the same 1-D bulk copies as a whole plane -- and carries a halo of F_MAXNL rows
// towards its neighbour slabs: its first / last row is frozen (lambda = 0; on the lattice face that is the WALL), the error
// that creates at a cut moves inwards one row per sub-step and never reaches the output rows.  A row is wider than one
// row group of LRP lanes, so it is covered by nxb column blocks side by side; x-neighbours across a seam between two blocks
// go through a small shared-memory exchange (one 16-byte store and load per lane on a seam and level), exactly like the
// y-neighbours across row groups.  The S2/S3 occupancy map is written from the state slab while it is in shared memory.
// NXG, NYG: lattice dims at compile time (all strides fold); 0 = run time.
template <int NL, int LRP, int NXG, int NYG>
__global__ void __launch_bounds__(F_SLAB_WARPS * 32, 1) k_diffuse_slab(const FusedArgs A, const FusedGeom Gm)
{
    typedef Fused<NL, LRP, NXG, NYG, true> F;
    extern __shared__ __align__(128) unsigned char fsm[];
    constexpr int RW = 32 / LRP;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int lx = lane % LRP, gi = warp * RW + lane / LRP;
    const int nxb = NXG ? NXG / (2 * LRP) : A.nxb, rga = NXG ? (F_SLAB_WARPS * RW) / (NXG / (2 * LRP)) : A.rga;
    const int blk = gi % nxb, rg = gi / nxb;                                  // column block, row group inside the slab
    const int nxr = NXG ? NXG : A.nx, nyr = NYG ? NYG : A.ny;
    const int x0 = blk * 2 * LRP + 2 * lx;
    const uint32_t base = smem_u32(fsm);

    FusedCtx c;
    c.nx = nxr; c.nxny = nxr * nyr; c.nz = A.nz;
    c.bars = base; c.in_ring = base + Gm.off_in; c.st_ring = base + Gm.off_st;
    c.in_slot = (uint32_t)(rga * F_PY * nxr) * 4u; c.st_slot = (uint32_t)(rga * F_PY * nxr);
    c.yst = (uint32_t)nxr * 4u;
    c.ex_lvl = 2u * (uint32_t)(rga + 2) * c.yst;                               // [top rows | bottom rows] of rga + 2 lattice rows (a zero row at both ends)
    c.ex_self = base + Gm.off_ex + (uint32_t)(rg + 1) * c.yst + (uint32_t)x0 * 4u;
    c.xel = (uint32_t)(rga * nxb) * 32u;                                       // per level: [row group][block][left edge | right edge] x 16 bytes
    c.seam_r = lx == LRP - 1 && blk < nxb - 1;
    c.seam_l = lx == 0 && blk > 0;
    // slots: [row group][block][left edge | right edge] x 16 bytes, so the facing edge of the neighbour block is the slot before / after mine;
    // lanes off a seam all use the first slot of a sink region of the same shape (written, read, never selected)
    c.xs_w = base + Gm.off_xex + (uint32_t)((rg * nxb + blk) * 2 + (c.seam_r ? 1 : 0)) * 16u;
    if (!c.seam_l && !c.seam_r) c.xs_w = base + Gm.off_xdummy + 16u;
    c.st_strip = 0; c.strip_ok = true; c.src_plane0 = nullptr; c.st_plane0 = nullptr; c.occ_row = nullptr;
    c.itg = 0; c.par = 0;
    c.zero2 = pk(A.zero, A.zero);
    if (tid == 0) {
#pragma unroll
        for (int r = 0; r < F_RING; ++r) mbar_init(c.bars + 8u * r, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int e = tid; e < 96; e += blockDim.x) reinterpret_cast<float *>(fsm + Gm.off_lut)[e] = A.lut[e / 32][e % 32];
    for (uint32_t e = tid; e < (Gm.smem_bytes - Gm.off_ex) / 8u; e += blockDim.x) reinterpret_cast<u64 *>(fsm + Gm.off_ex)[e] = 0ull;   // both exchanges
    __syncthreads();

    const int nzi = A.nz - 2;
    long long p = Gm.start[blockIdx.x];
    const long long p_end = Gm.start[blockIdx.x + 1];
    u64 h[NL][3][F_PY];
#pragma unroll
    for (int k = 0; k < NL; ++k)
#pragma unroll
        for (int s = 0; s < 3; ++s)
#pragma unroll
            for (int j = 0; j < F_PY; ++j) h[k][s][j] = 0ull;

    while (p < p_end) {
        const int unit = (int)(p / nzi);
        const int slab = unit % A.nslab, us = unit / A.nslab;
        const int b = us / 3, sp = us % 3;
        c.za = 1 + (int)(p - (long long)unit * nzi);
        c.zb = (int)min((long long)(A.nz - 1), (long long)c.za + (p_end - p));
        p += c.zb - c.za;
        const int ty0 = A.sy0[slab], ty1 = A.sy1[slab], oy0 = A.so0[slab], oy1 = A.so1[slab];
        const int y0 = ty0 + F_PY * rg;
        const int yc = min(y0, ty1 - F_PY);                                    // groups beyond a short slab: duplicates of its last row group
        const size_t ubase = (size_t)b * (size_t)c.nxny * (size_t)A.nz;
        c.occ_nw = 0;
        if (sp == 0 && A.occ != nullptr) c.occ_nw = (uint32_t)((oy1 * nxr + 255) / 256) - (uint32_t)((oy0 * nxr + 255) / 256);
        if (tid == 0) {                                                        // every reader of the old values is past the last barrier of the previous segment
            SlabSeg *sg = F::slab_seg();
            sg->src_plane0 = A.src[sp] + ubase + (size_t)ty0 * nxr;
            sg->st_plane0 = A.state + ubase + (size_t)ty0 * nxr;
            sg->ld_fbytes = (uint32_t)((ty1 - ty0) * nxr) * 4u; sg->ld_sbytes = (uint32_t)((ty1 - ty0) * nxr);
            // occupancy words of a plane whose first byte lies in this slab's output rows (the halo covers the rest of the word)
            sg->occ_row = A.occ ? A.occ + (size_t)b * (size_t)(c.nxny / 256) * (size_t)A.nz : nullptr;
            sg->occ_w0 = (uint32_t)((oy0 * nxr + 255) / 256);
            sg->occ_soff = sg->occ_w0 * 256u - (uint32_t)(ty0 * nxr);
        }
        __syncthreads();
        c.src = A.src[sp] + ubase + (yc * nxr + x0);
        c.dst = A.dst[sp] + ubase + (yc * nxr + x0);
        c.in_lane = c.in_ring + (uint32_t)((yc - ty0) * nxr + x0) * 4u;
        c.st_lane = c.st_ring + (uint32_t)((yc - ty0) * nxr + x0);
        {   // segment = one row of one row group of this warp: LRP / 4 lanes x 8 bytes
            const int seg = lane / (LRP / 4), sg_g = warp * RW + seg / F_PY, sg_row = seg % F_PY;
            const int sy = min(ty0 + F_PY * (sg_g / nxb), ty1 - F_PY) + sg_row;
            c.st_strip = c.st_ring + (uint32_t)((sy - ty0) * nxr + (sg_g % nxb) * 2 * LRP + (lane % (LRP / 4)) * 8);
        }
        c.t0 = c.za - NL;
        c.nsteps = c.zb - c.za + 2 * NL;
        c.ld_lo = max(0, c.za - NL); c.ld_hi = min(A.nz, c.zb + NL);
        c.st_lo = 2 * NL; c.st_hi = min(A.nz, c.zb + NL) - c.t0;
        c.flags = 0; c.slowmask = A.always_slow[sp] ? 0xFFFFFFFFu : 0u;
        c.lut = base + Gm.off_lut + (uint32_t)sp * 128u;
        const float lam = A.lam[sp];
        c.rowmask = 0;
#pragma unroll
        for (int j = 0; j < F_PY; ++j) {
            const int y = y0 + j;
            if (y0 == yc && y >= oy0 && y < oy1) c.rowmask |= 1u << (16 + j);
            const bool rowin = y > ty0 && y < ty1 - 1;                           // the slab's first / last row is frozen (WALL, or halo edge)
            c.lam2[j] = pk(rowin && x0 > 0 ? lam : 0.0f, rowin && x0 + 1 < nxr - 1 ? lam : 0.0f);
        }
        const int i0 = ((c.ld_lo - c.t0) / 3) * 3;
        if (tid == 0)
            for (int i = i0; i < i0 + F_RING - 1 && i < c.nsteps; ++i) F::issue(c, i, i - i0);
        for (int i = i0; i < c.nsteps; i += 3) {
            if (i >= c.st_lo && i + 3 <= c.st_hi) {
                F::template step<0, true>(i, h, c);
                F::template step<1, true>(i + 1, h, c);
                F::template step<2, true>(i + 2, h, c);
            } else {
                F::template step<0, false>(i, h, c);
                if (i + 1 < c.nsteps) F::template step<1, false>(i + 1, h, c);
                if (i + 2 < c.nsteps) F::template step<2, false>(i + 2, h, c);
            }
        }
        c.itg += (uint32_t)c.nsteps;
    }
}

// ------------------------------------------------------------------ host side --
struct FusedPlan {
    bool ok = false;
    int lrp = 0, sms = 0, fixed = 0;   // fixed: 0 run-time dims, 32 / 64: the cubic fast instantiations
    bool tiled = false;                // planes wider or taller than 64 sites: k_diffuse_slab
    int slab_warps = 0;
    bool rows = false;                 // k_diffuse_rows (ca_rows.cuh) covers this width; else k_diffuse_slab
    int rows_rp = 1;                   // row pairs per lane of k_diffuse_rows on 96-wide planes (1: two rows; 2: four rows)
    int slab_maxh = 0;                 // rows of the tallest slab
    bool rp_attr_done[F_MAXNL + 1] = { false, false, false, false, false };
    int rows_cluster = 0;              // > 0: cluster variant of k_diffuse_rows with that many CTAs per plane
    int nclusters = 0;                 // clusters that can be resident at once (cudaOccupancyMaxActiveClusters)
    bool cluster_attr_done[F_MAXNL + 1] = { false, false, false, false, false };
    bool writes_map = false;           // the kernel writes the S2/S3 occupancy map while the state planes pass through it
    FusedArgs args{};
    int npass = 0, pass_nl[2] = { 0, 0 };
    // per context (= per device and host thread): shared-memory opt-in done, and the last split table, by NL
    bool attr_done[F_MAXNL + 1] = { false, false, false, false, false };
    int split_key[F_MAXNL + 1][3] = { { -1, -1, -1 }, { -1, -1, -1 }, { -1, -1, -1 }, { -1, -1, -1 }, { -1, -1, -1 } };
    int split[F_MAXNL + 1][F_MAXGRID + 1];
};

inline size_t fused_smem(int nx, int ny, int nl, int lrp, FusedGeom &G)
{
    const int rw = 32 / lrp, groups = (ny + F_PY - 1) / F_PY;
    G.nwarps = (groups + rw - 1) / rw;
    G.ngroups_alloc = G.nwarps * rw;
    size_t o = 128;
    G.off_lut = (uint32_t)o; o += 96 * 4; o = (o + 127) / 128 * 128;
    G.off_in = (uint32_t)o; o += (size_t)F_RING * nx * ny * 4; o = (o + 127) / 128 * 128;
    G.off_st = (uint32_t)o; o += (size_t)F_SRING * nx * ny; o = (o + 127) / 128 * 128;
    G.off_ex = (uint32_t)o; o += (size_t)2 * nl * 2 * (G.ngroups_alloc + 2) * lrp * 8;
    G.smem_bytes = (uint32_t)o;
    return o;
}

// Split the flattened (unit, interior plane) space over `grid` CTAs so that every CTA gets the same COST: a segment
// pays for its planes plus the fill of the NL-level pipeline (cheaper when it starts at a WALL plane, where the
// empty lead-in iterations are skipped).  Costs in units of one steady iteration, fitted to the measured kernel.
inline void fused_split(int units, int nzi, int nl, int grid, int *start)
{
    const double f = 0.55;                             // cost of one pipeline-fill iteration relative to a steady one (fitted on the B200)
    const double r_wall = f * (2 * nl - 3), r_cut = f * (2 * nl);
    const long long total = (long long)units * nzi;
    double lo = 0.0, hi = (double)total + (double)(units + grid) * r_cut + 1.0;
    for (int it = 0; it < 60; ++it) {                  // smallest per-CTA budget T that covers everything with `grid` CTAs
        const double T = 0.5 * (lo + hi);
        long long p = 0;
        for (int g = 0; g < grid && p < total; ++g) {
            double used = 0.0;
            while (p < total) {
                const int z = (int)(p % nzi);
                const double r = z == 0 ? r_wall : r_cut;
                const long long room = (long long)(T - used - r);
                if (room < 1) break;
                const long long take = std::min<long long>(room, nzi - z);
                p += take; used += r + (double)take;
            }
        }
        if (p >= total) hi = T; else lo = T;
    }
    long long p = 0;
    for (int g = 0; g < grid; ++g) {
        start[g] = (int)p;
        double used = 0.0;
        while (p < total) {
            const int z = (int)(p % nzi);
            const double r = z == 0 ? r_wall : r_cut;
            const long long room = (long long)(hi - used - r);
            if (room < 1) break;
            const long long take = std::min<long long>(room, nzi - z);
            p += take; used += r + (double)take;
        }
    }
    start[grid] = (int)total;
    for (int g = grid - 1; g >= 0 && start[g] > start[grid]; --g) start[g] = start[grid];
}

// the split depends on (units, planes, NL, grid) only: the plan keeps the last one per NL
inline void fused_split_cached(FusedPlan &F, int units, int nzi, int nl, int grid, int *start)
{
    int *key = F.split_key[nl];
    if (key[0] != units || key[1] != nzi || key[2] != grid) {
        fused_split(units, nzi, nl, grid, F.split[nl]);
        key[0] = units; key[1] = nzi; key[2] = grid;
    }
    memcpy(start, F.split[nl], sizeof(int) * (grid + 1));
}

template <int NL, int LRP, int NX, int NY>
inline cudaError_t fused_launch_t(FusedPlan &F, const FusedArgs &A, int grid, cudaStream_t st)
{
    FusedGeom G{};
    fused_smem(A.nx, A.ny, NL, LRP, G);
    G.total_planes = (long long)A.batch * 3 * (A.nz - 2);
    if (grid > F_MAXGRID) grid = F_MAXGRID;
    fused_split_cached(F, A.batch * 3, A.nz - 2, NL, grid, G.start);
    if (!F.attr_done[NL]) {            // the opt-in is per device: kept per context, not per process
        cudaError_t e = cudaFuncSetAttribute(k_diffuse_fused<NL, LRP, NX, NY>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        F.attr_done[NL] = true;
    }
    k_diffuse_fused<NL, LRP, NX, NY><<<grid, G.nwarps * 32, G.smem_bytes, st>>>(A, G);
    return cudaGetLastError();
}

// shared-memory layout of the slab variant: rings sized for the tallest slab (rga row groups), y-exchange of whole lattice
// rows, x-seam exchange
inline size_t slab_smem(int nx, int nl, int rga, int nxb, FusedGeom &G)
{
    const int H = rga * F_PY;
    size_t o = 128;
    G.off_lut = (uint32_t)o; o += 96 * 4; o = (o + 127) / 128 * 128;
    G.off_in = (uint32_t)o; o += (size_t)F_RING * H * nx * 4; o = (o + 127) / 128 * 128;
    G.off_st = (uint32_t)o; o += (size_t)F_SRING * H * nx; o = (o + 127) / 128 * 128;
    G.off_ex = (uint32_t)o; o += (size_t)2 * nl * 2 * (rga + 2) * nx * 4; o = (o + 127) / 128 * 128;
    G.off_xex = (uint32_t)o; o += (size_t)2 * nl * (rga + 1) * nxb * 32; o = (o + 127) / 128 * 128;
    G.off_xdummy = (uint32_t)o; o += (size_t)2 * nl * (rga + 1) * nxb * 32 + 128;
    G.smem_bytes = (uint32_t)o;
    return o;
}

template <int NL, int LRP, int NXG, int NYG>
inline cudaError_t fused_launch_slab_t(FusedPlan &F, const FusedArgs &A, int grid, cudaStream_t st)
{
    FusedGeom G{};
    slab_smem(A.nx, NL, A.rga, A.nxb, G);
    G.nwarps = F.slab_warps;
    G.ngroups_alloc = A.rga;
    const int units = A.batch * 3 * A.nslab;
    G.total_planes = (long long)units * (A.nz - 2);
    if (grid > F_MAXGRID) grid = F_MAXGRID;
    fused_split_cached(F, units, A.nz - 2, NL, grid, G.start);
    if (!F.attr_done[NL]) {
        cudaError_t e = cudaFuncSetAttribute(k_diffuse_slab<NL, LRP, NXG, NYG>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
        if (e != cudaSuccess) return e;
        F.attr_done[NL] = true;
    }
    k_diffuse_slab<NL, LRP, NXG, NYG><<<grid, G.nwarps * 32, G.smem_bytes, st>>>(A, G);
    return cudaGetLastError();
}

template <int NL>
inline cudaError_t fused_launch_slab(FusedPlan &F, const FusedArgs &A, int grid, cudaStream_t st)
{
    if (A.nx == 96 && A.ny == 96) return fused_launch_slab_t<NL, 16, 96, 96>(F, A, grid, st);    // BASELINE configs[2]
    if (A.nx == 80 && A.ny == 80) return fused_launch_slab_t<NL, 8, 80, 80>(F, A, grid, st);     // BASELINE configs[3]
    if (F.lrp == 32) return fused_launch_slab_t<NL, 32, 0, 0>(F, A, grid, st);
    if (F.lrp == 16) return fused_launch_slab_t<NL, 16, 0, 0>(F, A, grid, st);
    return fused_launch_slab_t<NL, 8, 0, 0>(F, A, grid, st);
}

// cut ny rows into slabs of at most H rows including a halo of F_MAXNL rows towards neighbours; cuts on multiples of F_PY
inline int slab_cuts(int ny, int H, short *y0, short *y1, short *o0, short *o1)
{
    for (int n = 1; n <= F_MAXSLAB; ++n) {
        bool ok = true;
        for (int t = 0; t < n && ok; ++t) {
            const int c0 = t == 0 ? 0 : (ny * t / n) / F_PY * F_PY, c1 = t == n - 1 ? ny : (ny * (t + 1) / n) / F_PY * F_PY;
            y0[t] = (short)(t == 0 ? 0 : c0 - F_MAXNL); y1[t] = (short)(t == n - 1 ? ny : c1 + F_MAXNL);
            o0[t] = (short)c0; o1[t] = (short)c1;
            ok = y1[t] - y0[t] <= H && c1 > c0 && y0[t] >= 0 && y1[t] <= ny && y1[t] - y0[t] >= 2 * F_PY;
        }
        if (ok) return n;
    }
    return 0;
}

template <int NL>
inline cudaError_t rows_launch(FusedPlan &F, const FusedArgs &A, int grid, cudaStream_t st);   // ca_rows.cuh
inline bool rows_configure(const KParams &P, FusedPlan &F);

template <int NL>
inline cudaError_t fused_launch_nl(FusedPlan &F, const FusedArgs &A, int grid, cudaStream_t st)
{
    if (F.tiled && F.rows) return rows_launch<NL>(F, A, grid, st);
    if (F.tiled) return fused_launch_slab<NL>(F, A, grid, st);
    if (F.fixed == 64) return fused_launch_t<NL, 32, 64, 64>(F, A, grid, st);
    if (F.fixed == 32) return fused_launch_t<NL, 16, 32, 32>(F, A, grid, st);
    if (F.lrp == 16) return fused_launch_t<NL, 16, 0, 0>(F, A, grid, st);
    return fused_launch_t<NL, 32, 0, 0>(F, A, grid, st);
}

// Decide whether the fused kernel covers this lattice, and precompute its arguments.
inline void fused_configure(const KParams &P, FusedPlan &F)
{
    F.ok = false;
    F.tiled = (P.nx > 64 || P.ny > 64);
    if (P.nz < 3 || P.n_sub < 1 || P.n_sub > 2 * F_MAXNL || P.nx < 4) return;
    if (P.well_mixed) return;                                     // EMPTY sites pinned at the medium values: the per-sub-step kernel serves that reading
    FusedGeom G{};
    F.rows = F.tiled && rows_configure(P, F);
    if (F.rows) {
        F.fixed = 0;
        F.writes_map = (P.nx * P.ny) % 256 == 0;
    } else if (F.tiled) {
        // rows must be whole 16-byte units of the state array (bulk copies) and whole row groups of 2 * LRP sites
        if (P.nx % 16 || P.ny % F_PY) return;
        F.lrp = P.nx % 64 == 0 ? 32 : (P.nx % 32 == 0 ? 16 : 8);
        const int rw = 32 / F.lrp;
        F.args.nxb = P.nx / (2 * F.lrp);
        F.args.rga = (F_SLAB_WARPS * rw) / F.args.nxb;            // row groups of F_PY rows that 15 warps hold
        if (F.args.rga < 3) return;
        F.args.nslab = slab_cuts(P.ny, F.args.rga * F_PY, F.args.sy0, F.args.sy1, F.args.so0, F.args.so1);
        if (!F.args.nslab) return;
        int maxh = 0;
        for (int t = 0; t < F.args.nslab; ++t) maxh = std::max(maxh, F.args.sy1[t] - F.args.sy0[t]);
        F.slab_warps = ((maxh / F_PY) * F.args.nxb + rw - 1) / rw;   // the tallest slab decides the CTA size (the rings keep their capacity)
        if (slab_smem(P.nx, F_MAXNL, F.args.rga, F.args.nxb, G) > 227 * 1024 || F.slab_warps > F_SLAB_WARPS) return;
        F.fixed = 0;
        F.writes_map = (P.nx * P.ny) % 256 == 0;                  // occupancy words must not straddle planes
    } else {
        if (P.nx % 2 || (P.nx * P.ny) % 16) return;
        F.lrp = P.nx <= 32 ? 16 : 32;
        F.fixed = (P.nx == 64 && P.ny == 64) ? 64 : (P.nx == 32 && P.ny == 32) ? 32 : 0;
        F.writes_map = F.fixed != 0;
        if (fused_smem(P.nx, P.ny, F_MAXNL, F.lrp, G) > 227 * 1024 || G.nwarps > 16) return;
    }
    int dev = 0;
    cudaDeviceProp prop;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return;
    F.sms = prop.multiProcessorCount;
    F.args.zero = 0.0f;
    F.args.nx = P.nx; F.args.ny = P.ny; F.args.nz = P.nz; F.args.batch = P.batch;
    for (int s = 0; s < 3; ++s) {
        F.args.lam[s] = P.lambda[s];
        // without a source term v = c + lambda*(sum6 - RN(6c)) >= c*(1 - 6*lambda*(1 + 2^-24)) >= 0 needs this margin
        F.args.always_slow[s] = !((double)P.lambda[s] * 6.0 * (1.0 + 1.0 / 8388608.0) <= 1.0);
        for (int e = 0; e < 32; ++e) {
            const int kind = e & 7, mode = e >> 3;
            F.args.lut[s][e] = (kind >= 1 && kind <= 4) ? P.rate[s][mode] : 0.0f;
        }
    }
    if (P.n_sub <= F_MAXNL) { F.npass = 1; F.pass_nl[0] = P.n_sub; }
    else { F.npass = 2; F.pass_nl[0] = (P.n_sub + 1) / 2; F.pass_nl[1] = P.n_sub / 2; }
    F.ok = true;
}

inline bool fused_supported(const FusedPlan &F) { return F.ok; }

// Enqueue all n_sub sub-steps starting from ping-pong buffer `cur`; returns the number of passes (= buffer flips).
// A failed launch stops the sequence: *err says why, and the return value counts only the passes that were launched.
inline int launch_fused(FusedPlan &F, const Lattice &L, int cur, uint32_t *occ, cudaStream_t st, cudaError_t *err)
{
    const int nb = F.args.batch;
    const size_t soff = 0;
    *err = cudaSuccess;
    for (int ps = 0; ps < F.npass; ++ps) {
        FusedArgs A = F.args;
        A.batch = nb;
        for (int s = 0; s < 3; ++s) { A.src[s] = L.f[cur][s] + soff; A.dst[s] = L.f[cur ^ 1][s] + soff; }
        A.state = L.state + soff;
        A.occ = (F.writes_map && ps == F.npass - 1 && occ) ? occ + soff / 256 : nullptr;          // the state does not change between passes: write the map once
        FusedGeom G{};
        // CTAs per SM: the 512-thread (nx > 32) kernel fills an SM; smaller lattices use several CTAs per SM
        fused_smem(A.nx, A.ny, F.pass_nl[ps], F.lrp, G);
        const int per_sm = (int)std::max<size_t>(1, std::min<size_t>(std::min<size_t>(4, (227 * 1024) / (G.smem_bytes + 1024)), 512 / (G.nwarps * 32)));
        const long long total = (long long)A.batch * 3 * (A.nz - 2);
        const int grid = (int)std::max<long long>(1, std::min<long long>((long long)F.sms * per_sm, total / 2 + 1));
        cudaError_t e;
        switch (F.pass_nl[ps]) {
#ifndef CA_ONLY_NL4                     // development builds: only the n_sub = 4 instantiations (compile time)
        case 1: e = fused_launch_nl<1>(F, A, grid, st); break;
        case 2: e = fused_launch_nl<2>(F, A, grid, st); break;
        case 3: e = fused_launch_nl<3>(F, A, grid, st); break;
#endif
        case 4: e = fused_launch_nl<4>(F, A, grid, st); break;
        default: e = cudaErrorInvalidValue;
        }
        if (e != cudaSuccess) { *err = e; return ps; }
        cur ^= 1;
    }
    return F.npass;
}

}  // namespace ca
