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

#include "qft_phase.cuh"

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

using qftc::cis_fwd_u32;
using qftc::cr_phase_u32;
using qftc::kC32;
using qftc::kS32;

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
