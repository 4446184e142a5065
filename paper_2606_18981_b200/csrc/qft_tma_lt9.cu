// qft_tma_lt9.cu -- instantiations of the TMA-staged pass kernel for 2^9 threads (tile of 2^14 amplitudes).
// One translation unit per thread count so that the build compiles them in parallel.
#include "qft_tma_inst.cuh"
QFT_TMA2_DEFINE_PICK(9)
