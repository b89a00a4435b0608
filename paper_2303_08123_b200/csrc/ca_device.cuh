// ca_device.cuh -- device-side building blocks of libca_b200 (sm_100a).
// Product code: shares nothing with oracle/ (the oracle is test infrastructure with its own sources).
// Citations: [D Gn]/[D Sn] = DESIGN.md readings / step algorithm; PAPER.md lines where the paper fixes something.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>
#include "../../include/ca.h"

namespace ca {

// Philox purposes: counter word 3 = purpose | aux << 8  [D "random numbers"]
enum : uint32_t { P_INIT_PHASE = 0, P_INIT_CLOCK = 1, P_PHASE_CLOCK = 2, P_IRRADIATE = 3,
                  P_DIR = 4, P_CLAIM = 5, P_DAUGHTER_CLOCK = 6, P_PARENT_CLOCK = 7 };

// Kernel-side copy of the model parameters plus geometry; passed by value to every kernel.
struct KParams {
    int nx, ny, nz;
    int batch;
    long long n;                 // sites per simulation, WALL layer included
    int n_sub;
    float lambda[3];
    float boundary[3];
    float rate[3][4];
    float O_A, G_P, G_Q, H_P, H_Q;
    int T[4], J[4];
    float alpha[4], beta[4];
    float oer_m, oer_K;
    int repair_period, repair_shift;
    int lysis_steps;
    int N_ref;
    int well_mixed;              // != 0: EMPTY sites are held at the medium values [D G2, alternative reading]
    uint32_t key0, key1;         // Philox key = rng_seed (low, high)
    uint32_t sim_id_base;
};

// Device pointers of one context (SoA, [sim][z][y][x]).
struct Lattice {
    float *f[2][3];              // ping-pong field buffers: [buffer][species O2, glucose, H+]
    uint8_t *state;
    uint16_t *clock;
    uint16_t *damage;
};

// ---- Philox4x32-10 (Salmon et al., SC'11); only output word 0 is used [D "random numbers"] ----
__device__ __forceinline__ uint32_t philox_w0(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    return c0;
}

__device__ __forceinline__ uint32_t rnd(const KParams &P, uint32_t site, uint32_t step, uint32_t sid,
                                        uint32_t purpose, uint32_t aux = 0)
{
    return philox_w0(site, step, sid, purpose | (aux << 8), P.key0, P.key1);
}

// [D G23] uniform integer in [0, m)
__device__ __forceinline__ uint32_t uniform_int(uint32_t x, uint32_t m) { return __umulhi(x, m); }

// [D G7] clock drawn at entry of phase `kind` (1..4): T - J + U{0..2J}
__device__ __forceinline__ uint16_t draw_clock(const KParams &P, int kind, uint32_t site, uint32_t step,
                                               uint32_t sid, uint32_t purpose)
{
    const int T = P.T[kind - 1], J = P.J[kind - 1];
    return (uint16_t)(T - J + (int)uniform_int(rnd(P, site, step, sid, purpose), (uint32_t)(2 * J + 1)));
}

// internal state bit 7 (never exported): READY parent known to have no EMPTY neighbour  (k_cells_divide)
constexpr uint32_t CA_BLOCKED = 0x80u;

__device__ __forceinline__ bool is_live(uint32_t st) { const uint32_t k = st & 7u; return k >= 1u && k <= 4u; }
// READY parent able to divide: kind M, READY, proliferating mode (< 2)  [D S3 step 1]
__device__ __forceinline__ bool is_parent(uint32_t st) { return (st & 0x37u) == (uint32_t)(CA_M | CA_READY); }

// [D S2 (i)] mode decision; returns -1 when starved
__device__ __forceinline__ int decide_mode(const KParams &P, float O, float G, float H)
{
    if (G < P.G_Q || H > P.H_Q) return -1;
    const int prolif = (G >= P.G_P) && (H <= P.H_P);
    const int aerobic = (O >= P.O_A);
    return 2 * (!prolif) + (!aerobic);
}

// [D S1] one sub-step value.  The association of sum6, the un-fused 6*c and the single fma are part
// of the definition: a uniform field is reproduced bit-exactly (pin P5).  Intrinsics stop nvcc from
// contracting or re-associating.
__device__ __forceinline__ float stencil_point(float c, float xm, float xp, float ym, float yp, float zm, float zp,
                                               float lam, float r)
{
    const float sum6 = __fadd_rn(__fadd_rn(__fadd_rn(xm, xp), __fadd_rn(ym, yp)), __fadd_rn(zm, zp));
    const float lap = __fsub_rn(sum6, __fmul_rn(6.0f, c));
    float v = __fmaf_rn(lam, lap, c);
    v = __fadd_rn(v, r);
    return v > 0.0f ? v : 0.0f;
}

}  // namespace ca
