// qft_device.cuh -- device helpers shared by the pass kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "qft_phase.cuh"
#include "qft_plan.h"

namespace qftk {

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

using qftc::cis_fwd_u32;
using qftc::cr_phase_u32;

// v * exp(-2 pi i M / 32), M compile-time in [0, 16): the constant twiddles inside a register group.
template <int M>
__device__ __forceinline__ float2 mul_w32(float2 v) {
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
        return make_float2(fmaf(v.x, qftc::kC32[M], v.y * qftc::kS32[M]), fmaf(v.y, qftc::kC32[M], -v.x * qftc::kS32[M]));
    }
}

// exp(-2 pi i m / 32), m < 16 at run time, for the general (small-k) in-group path.
__device__ __forceinline__ float2 w32(int m) { return make_float2(qftc::kC32[m], -qftc::kS32[m]); }

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
                    x[V] = cmul(d, w32(lowm << (4 - POS)));
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
