// qft_packed.cuh -- complex arithmetic on packed FP32 pairs (sm_100a FADD2 / FMUL2 / FFMA2).
//
// Blackwell issues add/mul/fma on two FP32 lanes of a 64-bit register pair in one instruction
// (PTX add/sub/mul/fma .f32x2).  An amplitude (re, im) is exactly such a pair, so
//   complex add/sub            = 1 instruction  (FADD2),
//   complex * complex          = 2 instructions (FMUL2 with the swapped, half-negated operand that
//                                SASS encodes as an operand modifier, then FFMA2),
//   multiplication by -i       = 0 instructions (operand modifier of the consumer).
// The pass kernels are bound by instruction issue before they are bound by HBM (profiles/r01_fused2_v1),
// so halving the FP32 instruction count is what moves them towards the HBM roofline.
//
// The gate arithmetic itself is the paper's: H = [[1,1],[1,-1]] (Eq. 1, the 1/sqrt2 of
// :138 is applied once per pass as a scale), R_m = diag(1, exp(-2 pi i / 2^m)).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace qftp {

__device__ __forceinline__ float2 padd(float2 a, float2 b) {
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; add.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 psub(float2 a, float2 b) {
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; sub.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 pmul(float2 a, float2 b) {
    float2 r;
    asm("{.reg .b64 ra, rb, rc; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; mul.rn.f32x2 rc, ra, rb; mov.b64 {%0,%1}, rc;}"
        : "=f"(r.x), "=f"(r.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y));
    return r;
}
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c) {
    float2 r;
    asm("{.reg .b64 ra, rb, rc, rd; mov.b64 ra,{%2,%3}; mov.b64 rb,{%4,%5}; mov.b64 rc,{%6,%7}; "
        "fma.rn.f32x2 rd, ra, rb, rc; mov.b64 {%0,%1}, rd;}"
        : "=f"(r.x), "=f"(r.y)
        : "f"(a.x), "f"(a.y), "f"(b.x), "f"(b.y), "f"(c.x), "f"(c.y));
    return r;
}

// a * w = (a.x w.x - a.y w.y, a.y w.x + a.x w.y)
__device__ __forceinline__ float2 cmul(float2 a, float2 w) {
    const float2 t = pmul(make_float2(a.y, a.x), make_float2(-w.y, w.y));
    return pfma(a, make_float2(w.x, w.x), t);
}
__device__ __forceinline__ float2 cscale(float2 a, float s) { return pmul(a, make_float2(s, s)); }
__device__ __forceinline__ float2 mul_negi(float2 v) { return make_float2(v.y, -v.x); }

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

// v * exp(-2 pi i M / 32), M compile-time in [0, 16)
template <int M>
__device__ __forceinline__ float2 mul_w32(float2 v) {
    if constexpr (M == 0) return v;
    else if constexpr (M == 8) return mul_negi(v);
    else return cmul(v, make_float2(kC32[M], -kS32[M]));
}

// One decimation-in-frequency stage over 2^NB registers: the Hadamard on the qubit at register-index
// bit POS (unnormalised butterfly) followed by the controlled rotations onto it from the qubits on
// register bits below POS (constant twiddles).  KC = min(k, 4) truncates them for the AQFT: only
// controls at distance <= KC are kept.  Register bits >= R are batch bits: several
// independent groups side by side.
template <int NB, int POS, int U, int KC>
struct DifStage {
    static __device__ __forceinline__ void run(float2 (&x)[1 << NB]) {
        if constexpr (U < (1 << NB)) {
            if constexpr ((U & (1 << POS)) == 0) {
                constexpr int V = U | (1 << POS);
                constexpr int LOW = U & ((1 << POS) - 1);
                constexpr int CUT = POS - KC;
                constexpr int LOWM = CUT > 0 ? (LOW & ~((1 << CUT) - 1)) : LOW;
                const float2 a = x[U], b = x[V];
                x[U] = padd(a, b);
                x[V] = mul_w32<(LOWM << (4 - POS))>(psub(a, b));
            }
            DifStage<NB, POS, U + 1, KC>::run(x);
        }
    }
};
template <int NB, int POS, int KC>
struct DifAll {
    static __device__ __forceinline__ void run(float2 (&x)[1 << NB]) {
        DifStage<NB, POS, 0, KC>::run(x);
        if constexpr (POS > 0) DifAll<NB, POS - 1, KC>::run(x);
    }
};
// R qubits on register bits [0, R), highest first; 2^(NB-R) groups in the 2^NB registers.
template <int NB, int R, int KC>
__device__ __forceinline__ void dif_group(float2 (&x)[1 << NB]) {
    DifAll<NB, R - 1, KC>::run(x);
}

// x[BASE + u] *= p * prod_{i : bit i of u set} W[i], u < 2^R, walking the subset tree so that every
// product is formed once: 2^R - 1 - R multiplications to build, 2^R - 1 to apply (HASP adds R + 1).
template <int NB, int BASE, int BIT, int U, bool HASP, int NW>
struct TwTree {
    static __device__ __forceinline__ void run(float2 (&x)[1 << NB], const float2 (&W)[NW], float2 p) {
        if constexpr (BIT < 0) {
            if constexpr (HASP) x[BASE + U] = cmul(x[BASE + U], p);
        } else {
            TwTree<NB, BASE, BIT - 1, U, HASP, NW>::run(x, W, p);
            if constexpr (HASP) TwTree<NB, BASE, BIT - 1, U | (1 << BIT), true, NW>::run(x, W, cmul(p, W[BIT]));
            else TwTree<NB, BASE, BIT - 1, U | (1 << BIT), true, NW>::run(x, W, W[BIT]);
        }
    }
};

}  // namespace qftp
