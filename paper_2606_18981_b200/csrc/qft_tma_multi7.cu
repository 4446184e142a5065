// qft_tma_multi7.cu -- instantiations of the single-launch kernel (three passes, grid-wide barriers between them)
// for the register-group shapes of n = 20 ... 24 on 2^12 tiles (2^7 threads).
#include "qft_tma_multi_inst.cuh"
tma2_multi_kernel_t qft_pick_tma2_multi7(int a1, int a2, int b1, int b2, int kc) { return pick_shape<7>(a1, a2, b1, b2, kc); }
