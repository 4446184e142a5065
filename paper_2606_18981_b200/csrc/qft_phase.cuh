// qft_phase.cuh -- the phase arithmetic every pass kernel shares (sm_100a): the collapsed controlled-R_m
// phase as an exact 32-bit fraction of a turn, its evaluation, and the 32nd roots of unity
// (exp(-2 pi i m / 32) = (kC32[m], -kS32[m]): the constant twiddles inside a register group,
// R_m = diag(1, exp(-2 pi i / 2^m)), m <= 5).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qftc {

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
    float re = (q & 1u) ? -s : c;
    float im = (q & 1u) ? c : s;
    if (q & 2u) { re = -re; im = -im; }
    return make_float2(re, -im);
}

// Phase (binary fraction of a turn, 32 bits) of the collapsed controlled-R_m product onto target
// qubit t for an amplitude whose lower logical bits are L (< 2^t):
//   sum_{d=1..min(k,t)} b_{t-d} / 2^{d+1}  =  (L with bits below t-k cleared) / 2^{t+1}.
// Linear in L over disjoint bit sets (mod one turn), which is what lets a pass split it into a part
// from the tile's own bits and a part from the tile index.
__device__ __forceinline__ uint32_t cr_phase_u32(uint64_t L, int t, int k) {
    const int cut = t - k;
    if (cut > 0) L &= ~((1ull << cut) - 1ull);
    return (t <= 31) ? (uint32_t)(L << (31 - t)) : (uint32_t)(L >> (t - 31));
}

__device__ constexpr float kC32[16] = {1.0f,
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
__device__ constexpr float kS32[16] = {0.0f,
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

}  // namespace qftc
