// pow2_inst.cu -- one translation unit per (tile type, digit length): compiled once for every
// -DDOP_INST_COL=<0|1> -DDOP_INST_L=<length> pair listed in build.py, in parallel, so the ~120
// kernel instantiations of pow2_impl.cuh do not serialise in one nvcc process.
#include "pow2_impl.cuh"

#ifndef DOP_INST_L
#error "compile with -DDOP_INST_COL=<0|1> -DDOP_INST_L=<digit length>"
#endif

namespace dop {
template cudaError_t launch_L<DOP_INST_L, (DOP_INST_COL != 0)>(const PassDesc&, int, int, cudaStream_t);
} // namespace dop
