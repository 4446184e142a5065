// qft_tma_xt.cu -- instantiations of the TMA-staged pass kernel with the tensor-memory extended tile
// (2^9 threads, two 2^14-amplitude halves per tile): windows of 9, 10 and 11 qubits.
#include "qft_tma_inst.cuh"
tma2_kernel_t qft_pick_tma2_xt(int r1, int r2, int kc) {
    if (r1 == 5 && r2 == 5) return qft_pick_tma2_kc<5, 5, 9, 1>(kc);
    if (r1 == 5 && r2 == 4) return qft_pick_tma2_kc<5, 4, 9, 1>(kc);
    if (r1 == 4 && r2 == 4) return qft_pick_tma2_kc<4, 4, 9, 1>(kc);
    return nullptr;
}
