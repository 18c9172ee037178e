// tma_inst.cu -- one translation unit per (digit length, bundle width, pipeline depth) of the TMA column
// kernels (tma_col.cuh): compiled with -DDOP_INST_TMA_L=<L> -DDOP_INST_TMA_NB=<NB> -DDOP_INST_TMA_NST=<NST>.
#include "tma_col.cuh"

#if !defined(DOP_INST_TMA_L) || !defined(DOP_INST_TMA_NB) || !defined(DOP_INST_TMA_NST)
#error "compile with -DDOP_INST_TMA_L=<digit length> -DDOP_INST_TMA_NB=<16|32> -DDOP_INST_TMA_NST=<stages>"
#endif

namespace dop {
template cudaError_t launch_tma<DOP_INST_TMA_L, DOP_INST_TMA_NB, DOP_INST_TMA_NST>(const PassDesc&, int, int, cudaStream_t);
} // namespace dop
