// qft_tma_inst.cuh -- kernel-pointer tables of qft_pass_tma2 per (R1, R2, KC) for one thread count.
#pragma once
#include "qft_tma.cuh"

typedef void (*tma2_kernel_t)(float2*, const CUtensorMap, const QftPassDesc);

template <int R1, int R2, int LT, int XT, int ES = 0>
static tma2_kernel_t qft_pick_tma2_kc(int kc) {
    switch (kc) {
        case 0: return qftk::qft_pass_tma2<R1, R2, 0, LT, XT, ES>;
        case 1: return qftk::qft_pass_tma2<R1, R2, 1, LT, XT, ES>;
        case 2: return qftk::qft_pass_tma2<R1, R2, 2, LT, XT, ES>;
        case 3: return qftk::qft_pass_tma2<R1, R2, 3, LT, XT, ES>;
        default: return qftk::qft_pass_tma2<R1, R2, 4, LT, XT, ES>;
    }
}

// split end table (more than QFT_TMA2_EB_DIRECT in-tile qubits below the window): windows of 2 ... 6 qubits
#define QFT_TMA2_DEFINE_PICK_ES(LT)                                             \
    tma2_kernel_t qft_pick_tma2_es##LT(int r1, int r2, int kc) {                \
        if (r1 == 3 && r2 == 3) return qft_pick_tma2_kc<3, 3, LT, 0, 1>(kc);    \
        if (r1 == 3 && r2 == 2) return qft_pick_tma2_kc<3, 2, LT, 0, 1>(kc);    \
        if (r1 == 2 && r2 == 2) return qft_pick_tma2_kc<2, 2, LT, 0, 1>(kc);    \
        if (r1 == 2 && r2 == 1) return qft_pick_tma2_kc<2, 1, LT, 0, 1>(kc);    \
        if (r1 == 1 && r2 == 1) return qft_pick_tma2_kc<1, 1, LT, 0, 1>(kc);    \
        return nullptr;                                                         \
    }

#define QFT_TMA2_DEFINE_PICK(LT)                                             \
    tma2_kernel_t qft_pick_tma2_lt##LT(int r1, int r2, int kc) {             \
        if (r1 == 5 && r2 == 5) return qft_pick_tma2_kc<5, 5, LT, 0>(kc);    \
        if (r1 == 5 && r2 == 4) return qft_pick_tma2_kc<5, 4, LT, 0>(kc);    \
        if (r1 == 4 && r2 == 4) return qft_pick_tma2_kc<4, 4, LT, 0>(kc);    \
        if (r1 == 4 && r2 == 3) return qft_pick_tma2_kc<4, 3, LT, 0>(kc);    \
        if (r1 == 3 && r2 == 3) return qft_pick_tma2_kc<3, 3, LT, 0>(kc);    \
        if (r1 == 3 && r2 == 2) return qft_pick_tma2_kc<3, 2, LT, 0>(kc);    \
        if (r1 == 2 && r2 == 2) return qft_pick_tma2_kc<2, 2, LT, 0>(kc);    \
        if (r1 == 2 && r2 == 1) return qft_pick_tma2_kc<2, 1, LT, 0>(kc);    \
        if (r1 == 1 && r2 == 1) return qft_pick_tma2_kc<1, 1, LT, 0>(kc);    \
        return nullptr;                                                      \
    }
