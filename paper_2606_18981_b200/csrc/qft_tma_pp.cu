// qft_tma_pp.cu -- instantiations of the ping-pong TMA pass kernel (2^14-amplitude tiles, 512 threads).
#include "qft_tma_pp.cuh"

typedef void (*tma2_kernel_t)(float2*, const CUtensorMap, const QftPassDesc);

template <int R1, int R2>
static tma2_kernel_t pick_kc(int kc) {
    switch (kc) {
        case 0: return qftk::qft_pass_tma2pp<R1, R2, 0>;
        case 1: return qftk::qft_pass_tma2pp<R1, R2, 1>;
        case 2: return qftk::qft_pass_tma2pp<R1, R2, 2>;
        case 3: return qftk::qft_pass_tma2pp<R1, R2, 3>;
        default: return qftk::qft_pass_tma2pp<R1, R2, 4>;
    }
}

tma2_kernel_t qft_pick_tma2pp(int r1, int r2, int kc) {
    if (r1 == 5 && r2 == 5) return pick_kc<5, 5>(kc);
    if (r1 == 5 && r2 == 4) return pick_kc<5, 4>(kc);
    if (r1 == 4 && r2 == 4) return pick_kc<4, 4>(kc);
    if (r1 == 4 && r2 == 3) return pick_kc<4, 3>(kc);
    return nullptr;
}
