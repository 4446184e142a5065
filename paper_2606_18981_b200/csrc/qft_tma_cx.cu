// qft_tma_cx.cu -- instantiations of the TMA-staged pass kernel with the cluster-extended tile (two CTAs of a cluster
// share a tile of 2^16 amplitudes: 2^9 threads each, two 2^14-amplitude halves per CTA through tensor memory, the
// last qubit across the CTAs through distributed shared memory): windows of 10 and 11 qubits.
#include "qft_tma_inst.cuh"
tma2_kernel_t qft_pick_tma2_cx(int r1, int r2, int kc) {
    if (r1 == 5 && r2 == 4) return qft_pick_tma2_kc<5, 4, 9, 1, 0, 1>(kc);
    if (r1 == 4 && r2 == 4) return qft_pick_tma2_kc<4, 4, 9, 1, 0, 1>(kc);
    return nullptr;
}
