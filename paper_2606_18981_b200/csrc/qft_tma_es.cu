// qft_tma_es.cu -- instantiations of the TMA-staged pass kernel with the split end table (small windows high up
// in a large tile: more than QFT_TMA2_EB_DIRECT in-tile qubits below the window), 2^7 / 2^8 / 2^9 threads.
#include "qft_tma_inst.cuh"
QFT_TMA2_DEFINE_PICK_ES(7)
QFT_TMA2_DEFINE_PICK_ES(8)
QFT_TMA2_DEFINE_PICK_ES(9)
