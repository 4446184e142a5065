// qft_tma_lt8.cu -- instantiations of the TMA-staged pass kernel for 2^8 threads (tile of 2^13 amplitudes).
// One translation unit per thread count so that the build compiles them in parallel.
#include "qft_tma_inst.cuh"
QFT_TMA2_DEFINE_PICK(8)
