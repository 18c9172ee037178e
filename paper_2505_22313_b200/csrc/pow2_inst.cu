// pow2_inst.cu -- one translation unit per (tile type, digit length): compiled once for every
// -DDOP_INST_COL=<0|1> -DDOP_INST_L=<length> pair listed in build.py, in parallel, so the ~120
// kernel instantiations of pow2_impl.cuh do not serialise in one nvcc process.
#include "pow2_impl.cuh"

#if !defined(DOP_INST_L) && !defined(DOP_INST_X3)
#error "compile with -DDOP_INST_COL=<0|1> -DDOP_INST_L=<digit length>, or -DDOP_INST_X3=<LP> for digits 3*LP"
#endif

namespace dop {
#ifdef DOP_INST_X3
template cudaError_t launch_x3<DOP_INST_X3>(const PassDesc&, int, int, cudaStream_t);
#else
template cudaError_t launch_L<DOP_INST_L, (DOP_INST_COL != 0)>(const PassDesc&, int, int, cudaStream_t);
#endif
} // namespace dop
