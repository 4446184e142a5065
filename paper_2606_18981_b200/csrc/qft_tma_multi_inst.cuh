// qft_tma_multi_inst.cuh -- kernel-pointer tables of the single-launch kernel qft_multi_tma2 per register-group shape
// (passes 1 and 3: A1 + A2, mid pass: B1 + B2) and in-group truncation KC, for one thread count.
#pragma once
#include "qft_tma_inst.cuh"

typedef void (*tma2_multi_kernel_t)(float2*, const CUtensorMap, const CUtensorMap, const CUtensorMap, const QftPassDesc,
                                    const QftPassDesc, const QftPassDesc, unsigned*);

template <int A1, int A2, int B1, int B2, int LT>
static tma2_multi_kernel_t pick_kc(int kc) {
    switch (kc) {
        case 0: return qftk::qft_multi_tma2<A1, A2, B1, B2, 0, LT>;
        case 1: return qftk::qft_multi_tma2<A1, A2, B1, B2, 1, LT>;
        case 2: return qftk::qft_multi_tma2<A1, A2, B1, B2, 2, LT>;
        case 3: return qftk::qft_multi_tma2<A1, A2, B1, B2, 3, LT>;
        default: return qftk::qft_multi_tma2<A1, A2, B1, B2, 4, LT>;
    }
}

template <int LT>
static tma2_multi_kernel_t pick_shape(int a1, int a2, int b1, int b2, int kc) {
    if (a1 == 4 && a2 == 3 && b1 == 3 && b2 == 3) return pick_kc<4, 3, 3, 3, LT>(kc);
    if (a1 == 4 && a2 == 3 && b1 == 4 && b2 == 3) return pick_kc<4, 3, 4, 3, LT>(kc);
    if (a1 == 4 && a2 == 4 && b1 == 3 && b2 == 3) return pick_kc<4, 4, 3, 3, LT>(kc);
    if (a1 == 4 && a2 == 4 && b1 == 4 && b2 == 3) return pick_kc<4, 4, 4, 3, LT>(kc);
    if (a1 == 4 && a2 == 4 && b1 == 4 && b2 == 4) return pick_kc<4, 4, 4, 4, LT>(kc);
    return nullptr;
}

