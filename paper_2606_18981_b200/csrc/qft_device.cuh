// qft_device.cuh -- device helpers shared by the pass kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "qft_plan.h"

namespace qftk {

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// exp(-2 pi i * ph / 2^32): the forward-sign phase factor (omega = e^{-2 pi i / N}) of a
// phase held as an exact 32-bit binary fraction of a turn.  Quadrant reduction in integers, then
// Taylor polynomials on |theta| <= pi/4 (truncation error < 2e-9, below fp32 rounding).
__device__ __forceinline__ float2 cis_fwd_u32(uint32_t ph) {
    const uint32_t q = (ph + 0x20000000u) >> 30;  // nearest quarter turn (mod 4)
    const int32_t r = (int32_t)(ph - (q << 30));  // [-2^29, 2^29)
    const float th = (float)r * 1.4629180792671596e-9f;  // 2 pi / 2^32
    const float t2 = th * th;
    float s = fmaf(t2, 2.7557319223985893e-6f, -1.984126984126984e-4f);
    s = fmaf(s, t2, 8.333333333333333e-3f);
    s = fmaf(s, t2, -1.6666666666666666e-1f);
    s = fmaf(s * t2, th, th);
    float c = fmaf(t2, -2.755731922398589e-7f, 2.48015873015873e-5f);
    c = fmaf(c, t2, -1.388888888888889e-3f);
    c = fmaf(c, t2, 4.1666666666666664e-2f);
    c = fmaf(c, t2, -0.5f);
    c = fmaf(c, t2, 1.0f);
    // rotate by q quarter turns, then conjugate (forward sign is minus)
    float re = (q & 1u) ? -s : c;
    float im = (q & 1u) ? c : s;
    if (q & 2u) { re = -re; im = -im; }
    return make_float2(re, -im);
}

// Phase (binary fraction of a turn, 32 bits) of the collapsed controlled-R_m product onto target
// qubit t for an amplitude whose lower logical bits are L (< 2^t):
//   sum_{d=1..min(k,t)} b_{t-d} / 2^{d+1}  =  (L with bits below t-k cleared) / 2^{t+1}.
__device__ __forceinline__ uint32_t cr_phase_u32(uint64_t L, int t, int k) {
    const int cut = t - k;
    if (cut > 0) L &= ~((1ull << cut) - 1ull);
    return (t <= 31) ? (uint32_t)(L << (31 - t)) : (uint32_t)(L >> (t - 31));
}

// v * exp(-2 pi i M / 32), M compile-time in [0, 16): the constant twiddles inside a register group.
template <int M>
__device__ __forceinline__ float2 mul_w32(float2 v) {
    constexpr float C[16] = {1.0f,
                             0.9807852804032304f,
                             0.9238795325112867f,
                             0.8314696123025452f,
                             0.7071067811865476f,
                             0.5555702330196023f,
                             0.38268343236508984f,
                             0.19509032201612833f,
                             0.0f,
                             -0.1950903220161282f,
                             -0.3826834323650897f,
                             -0.555570233019602f,
                             -0.7071067811865475f,
                             -0.8314696123025453f,
                             -0.9238795325112867f,
                             -0.9807852804032304f};
    constexpr float S[16] = {0.0f,
                             0.19509032201612825f,
                             0.3826834323650898f,
                             0.5555702330196022f,
                             0.7071067811865475f,
                             0.8314696123025452f,
                             0.9238795325112867f,
                             0.9807852804032304f,
                             1.0f,
                             0.9807852804032304f,
                             0.9238795325112867f,
                             0.8314696123025455f,
                             0.7071067811865476f,
                             0.5555702330196022f,
                             0.3826834323650899f,
                             0.1950903220161286f};
    if constexpr (M == 0) {
        return v;
    } else if constexpr (M == 8) {  // -i
        return make_float2(v.y, -v.x);
    } else if constexpr (M == 4) {  // (1 - i)/sqrt 2
        return make_float2(0.70710678118654752f * (v.x + v.y), 0.70710678118654752f * (v.y - v.x));
    } else if constexpr (M == 12) {  // (-1 - i)/sqrt 2
        return make_float2(0.70710678118654752f * (v.y - v.x), -0.70710678118654752f * (v.x + v.y));
    } else {
        // (x + i y)(c - i s) = (x c + y s) + i (y c - x s)
        return make_float2(fmaf(v.x, C[M], v.y * S[M]), fmaf(v.y, C[M], -v.x * S[M]));
    }
}

// Table of exp(-2 pi i m / 32), m < 16, for the general (small-k) in-group path.
__constant__ float2 c_w32[16] = {
    {1.0f, -0.0f},
    {0.9807852804032304f, -0.19509032201612825f},
    {0.9238795325112867f, -0.3826834323650898f},
    {0.8314696123025452f, -0.5555702330196022f},
    {0.7071067811865476f, -0.7071067811865475f},
    {0.5555702330196023f, -0.8314696123025452f},
    {0.38268343236508984f, -0.9238795325112867f},
    {0.19509032201612833f, -0.9807852804032304f},
    {0.0f, -1.0f},
    {-0.1950903220161282f, -0.9807852804032304f},
    {-0.3826834323650897f, -0.9238795325112867f},
    {-0.555570233019602f, -0.8314696123025455f},
    {-0.7071067811865475f, -0.7071067811865476f},
    {-0.8314696123025453f, -0.5555702330196022f},
    {-0.9238795325112867f, -0.3826834323650899f},
    {-0.9807852804032304f, -0.1950903220161286f},
};

// One decimation-in-frequency stage of a register group: the Hadamard on the group's qubit at
// register-index bit POS (unnormalised butterfly, Eq. 1) followed by the controlled
// rotations from the group's lower qubits onto it (the constant twiddles).
template <int R, int POS, int U, bool FAST>
struct DifStage {
    static __device__ __forceinline__ void run(float2 (&x)[1 << R], int k) {
        if constexpr (U < (1 << R)) {
            if constexpr ((U & (1 << POS)) == 0) {
                constexpr int V = U | (1 << POS);
                constexpr int LOW = U & ((1 << POS) - 1);
                const float2 a = x[U], b = x[V];
                x[U] = cadd(a, b);
                const float2 d = csub(a, b);
                if constexpr (FAST) {
                    x[V] = mul_w32<(LOW << (4 - POS))>(d);
                } else {
                    const int cut = POS - k;
                    const int lowm = cut > 0 ? (LOW & ~((1 << cut) - 1)) : LOW;
                    x[V] = cmul(d, c_w32[lowm << (4 - POS)]);
                }
            }
            DifStage<R, POS, U + 1, FAST>::run(x, k);
        }
    }
};

template <int R, int POS, bool FAST>
struct DifAll {
    static __device__ __forceinline__ void run(float2 (&x)[1 << R], int k) {
        DifStage<R, POS, 0, FAST>::run(x, k);
        if constexpr (POS > 0) DifAll<R, POS - 1, FAST>::run(x, k);
    }
};

// All R qubits of a group, highest first: after this, register-index bit POS holds the frequency bit
// of the group's qubit on that bit (no reordering: qubits stay on their wires).
template <int R, bool FAST>
__device__ __forceinline__ void dif_group(float2 (&x)[1 << R], int k) {
    DifAll<R, R - 1, FAST>::run(x, k);
}

// Decode the tile(s) a CTA works on.  Without pairing the tile index is the block index.  With p
// swapped tile-index bit pairs, tile (x, y, z) stores into tile (y, x, z); CTAs 2c and 2c+1 form a
// cluster that holds either a tile and its partner, or (x = y) two self-paired tiles.
__device__ __forceinline__ void decode_tile(uint32_t bid, int p, uint32_t* mload, uint32_t* mstore) {
    if (p == 0) {
        *mload = bid;
        *mstore = bid;
        return;
    }
    const uint32_t rho = bid & 1u;
    const uint32_t cid = bid >> 1;
    const uint32_t z = cid >> (2 * p - 1);
    const uint32_t c = cid & ((1u << (2 * p - 1)) - 1u);
    const uint32_t dd = c >> (p - 1);
    const uint32_t xc = c & ((1u << (p - 1)) - 1u);
    uint32_t x, y;
    if (dd == 0) {
        x = y = 2u * xc + rho;
    } else {
        const int h = 31 - __clz(dd);
        const uint32_t x0 = ((xc >> h) << (h + 1)) | (xc & ((1u << h) - 1u));
        x = rho ? (x0 ^ dd) : x0;
        y = rho ? x0 : (x0 ^ dd);
    }
    *mload = x | (y << p) | (z << (2 * p));
    *mstore = y | (x << p) | (z << (2 * p));
}

// Streaming 8-byte global load: every amplitude is read exactly once per pass, so do not allocate
// in L1.  (Plain ld.global, not the non-coherent path: the same kernel later writes these addresses.)
__device__ __forceinline__ float2 ld_stream(const float2* p) {
    float2 v;
    asm volatile("ld.global.L1::no_allocate.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "l"(p));
    return v;
}

// Relaxed arrive for the TMA kernels: the arriving CTA only announces "my tile is on chip" (it has
// observed its own mbarrier), it publishes no writes, so the release fence (a MEMBAR that waits for
// the previous tile's stores to drain) is not needed.
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

}  // namespace qftk
