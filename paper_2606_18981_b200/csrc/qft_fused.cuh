// qft_fused.cuh -- the fused two-step pass kernel (QFT_KERNEL_FUSED2), sm_100a.
//
// One CTA per tile.  Data flow per amplitude: HBM -> registers -> shared memory -> registers -> HBM,
// i.e. exactly one shared-memory round trip and one 8 B read + one 8 B write of HBM per pass.
//   step 1: each thread reads the 2^R1 amplitudes of one radix-2^R1 butterfly straight from HBM
//           (lanes run along the hub, so each warp request covers whole 64-byte granules), applies
//           H and every controlled-R_m onto the R1 highest qubits of the window, writes them to
//           shared memory through a conflict-free XOR swizzle;
//   step 2: each thread gathers the 2^R2 amplitudes of a butterfly over the window's remaining
//           qubits from shared memory, applies their gates, and writes them straight to HBM at the
//           addresses the layout adapter dictates (in-tile bit permutation; partner tile after a
//           cluster barrier for pair passes).
#pragma once
#include "qft_device.cuh"

namespace qftk {

// x[u] *= prod over set bits of u of W[R-1-pos]  (W[i] belongs to the group's i-th qubit, highest
// first, which sits on register-index bit R-1-i).  Built as (low 3 bits table) x (high bits table)
// to keep the multiplication count near the minimum without a 2^R-entry table.
template <int R>
__device__ __forceinline__ void apply_group_twiddles(float2 (&x)[1 << R], const float2 (&W)[R]) {
    constexpr int LB = R < 3 ? R : 3;
    constexpr int HB = R - LB;
    float2 tlo[1 << LB];
    tlo[0] = make_float2(1.f, 0.f);
#pragma unroll
    for (int pos = 0; pos < LB; ++pos) {
#pragma unroll
        for (int v = (1 << pos); v < (2 << pos); ++v)
            tlo[v] = (v == (1 << pos)) ? W[R - 1 - pos] : cmul(tlo[v - (1 << pos)], W[R - 1 - pos]);
    }
    float2 thi[1 << HB];
    thi[0] = make_float2(1.f, 0.f);
#pragma unroll
    for (int pos = 0; pos < HB; ++pos) {
#pragma unroll
        for (int v = (1 << pos); v < (2 << pos); ++v)
            thi[v] = (v == (1 << pos)) ? W[R - 1 - (LB + pos)] : cmul(thi[v - (1 << pos)], W[R - 1 - (LB + pos)]);
    }
#pragma unroll
    for (int u = 1; u < (1 << R); ++u) {
        if ((u & ((1 << LB) - 1)) != 0) x[u] = cmul(x[u], tlo[u & ((1 << LB) - 1)]);
        if ((u >> LB) != 0) x[u] = cmul(x[u], thi[u >> LB]);
    }
}

// The R index-bit phase factors of one register group for an amplitude whose lower logical bits are L.
template <int R>
__device__ __forceinline__ void group_twiddle_bases(float2 (&W)[R], uint64_t L, int t_hi, int k) {
#pragma unroll
    for (int i = 0; i < R; ++i) W[i] = cis_fwd_u32(cr_phase_u32(L, t_hi - i, k));
}

template <int R1, int R2, bool FAST>
__global__ void __launch_bounds__(256, 2) qft_pass_fused2(float2* __restrict__ state,
                                                          const __grid_constant__ QftPassDesc d) {
    extern __shared__ float2 tile[];
    const uint32_t tid = threadIdx.x;
    const int f = d.f;

    uint32_t mload, mstore;
    decode_tile(blockIdx.x + (uint32_t)d.unit_lo * (d.npair ? 2u : 1u), d.npair, &mload, &mstore);
    uint64_t base_ld = 0, base_st = 0, Ltile = 0;
    for (int i = 0; i < d.ntile; ++i) {
        if ((mload >> i) & 1u) {
            base_ld |= 1ull << d.tile_addr[i];
            Ltile |= 1ull << d.log_tile[i];
        }
        if ((mstore >> i) & 1u) base_st |= 1ull << d.tile_addr[i];
    }

    // ------------------------------ step 1: HBM -> registers -> smem ------------------------------
    {
        const int a = d.steps[0].a;
        const int t_hi = d.steps[0].t_hi;
        const int t_lo = t_hi - R1 + 1;
        const uint64_t lmask = (t_lo > 0) ? ((1ull << t_lo) - 1ull) : 0ull;
        uint64_t rs[R1];  // element stride of each register bit
        uint32_t rp[R1];  // swizzled smem index contribution of each register bit
#pragma unroll
        for (int b = 0; b < R1; ++b) {
            rs[b] = 1ull << d.r1_addr[b];
            const int c = a + b;
            rp[b] = (c < 4) ? (1u << c) : ((1u << c) ^ d.swz_col[c]);
        }
        const uint32_t nb = 1u << (f - R1);
        for (uint32_t u = tid; u < nb; u += blockDim.x) {
            uint64_t off = base_ld;
            uint32_t can = 0, pcan = 0;
            for (int j = 0; j < f - R1; ++j) {
                if ((u >> j) & 1u) {
                    const int c = d.t1_canon[j];
                    off |= 1ull << d.t1_addr[j];
                    can |= 1u << c;
                    pcan ^= (c < 4) ? (1u << c) : ((1u << c) ^ d.swz_col[c]);
                }
            }
            const float2* __restrict__ src = state + off;
            float2 x[1 << R1];
#pragma unroll
            for (int B = 0; B < (1 << R1); ++B) {
                uint64_t o = 0;
#pragma unroll
                for (int b = 0; b < R1; ++b)
                    if (B & (1 << b)) o += rs[b];
                x[B] = ld_stream(src + o);
            }
            if (d.conj) {
#pragma unroll
                for (int B = 0; B < (1 << R1); ++B) x[B].y = -x[B].y;
            }
            dif_group<R1, FAST>(x, d.k);
            if (t_lo > 0) {
                uint64_t L = Ltile;
                for (int b = 0; b < a; ++b)
                    if ((can >> b) & 1u) L |= 1ull << d.log_canon[b];
                L &= lmask;
                float2 W[R1];
                group_twiddle_bases<R1>(W, L, t_hi, d.k);
                apply_group_twiddles<R1>(x, W);
            }
#pragma unroll
            for (int B = 0; B < (1 << R1); ++B) {
                uint32_t p = pcan;
#pragma unroll
                for (int b = 0; b < R1; ++b)
                    if (B & (1 << b)) p ^= rp[b];
                tile[p] = x[B];
            }
        }
    }
    __syncthreads();
    if (d.npair) cluster_arrive();  // this CTA's tile is entirely on chip

    // ------------------------------ step 2: smem -> registers -> HBM ------------------------------
    {
        const int a = d.steps[1].a;
        const int t_hi = d.steps[1].t_hi;
        const int t_lo = t_hi - R2 + 1;
        const uint64_t lmask = (t_lo > 0) ? ((1ull << t_lo) - 1ull) : 0ull;
        uint64_t rs[R2];
        uint32_t rp[R2];
#pragma unroll
        for (int b = 0; b < R2; ++b) {
            rs[b] = 1ull << d.r2_addr[b];
            const int c = a + b;
            rp[b] = (c < 4) ? (1u << c) : ((1u << c) ^ d.swz_col[c]);
        }
        const uint32_t nb = 1u << (f - R2);
        bool waited = false;
        for (uint32_t u = tid; u < nb; u += blockDim.x) {
            uint64_t off = base_st;
            uint32_t can = 0, pcan = 0;
            for (int j = 0; j < f - R2; ++j) {
                if ((u >> j) & 1u) {
                    const int c = d.t2_canon[j];
                    off |= 1ull << d.t2_addr[j];
                    can |= 1u << c;
                    pcan ^= (c < 4) ? (1u << c) : ((1u << c) ^ d.swz_col[c]);
                }
            }
            float2 x[1 << R2];
#pragma unroll
            for (int B = 0; B < (1 << R2); ++B) {
                uint32_t p = pcan;
#pragma unroll
                for (int b = 0; b < R2; ++b)
                    if (B & (1 << b)) p ^= rp[b];
                x[B] = tile[p];
            }
            dif_group<R2, FAST>(x, d.k);
            if (t_lo > 0) {
                uint64_t L = Ltile;
                for (int b = 0; b < a; ++b)
                    if ((can >> b) & 1u) L |= 1ull << d.log_canon[b];
                L &= lmask;
                float2 W[R2];
                group_twiddle_bases<R2>(W, L, t_hi, d.k);
                apply_group_twiddles<R2>(x, W);
            }
            if (d.do_scale) {
                const float sc = d.scale;
#pragma unroll
                for (int B = 0; B < (1 << R2); ++B) { x[B].x *= sc; x[B].y *= sc; }
            }
            if (d.conj) {
#pragma unroll
                for (int B = 0; B < (1 << R2); ++B) x[B].y = -x[B].y;
            }
            if (d.npair && !waited) {  // the partner tile has been read by its CTA
                cluster_wait();
                waited = true;
            }
            float2* __restrict__ dst = state + off;
#pragma unroll
            for (int B = 0; B < (1 << R2); ++B) {
                uint64_t o = 0;
#pragma unroll
                for (int b = 0; b < R2; ++b)
                    if (B & (1 << b)) o += rs[b];
                dst[o] = x[B];
            }
        }
    }
}

}  // namespace qftk
