// cluster_inst.cu -- one translation unit per cluster row geometry (M = local transform length,
// S = lines per CTA, cluster size 16 / S): compiled with -DDOP_INST_CLUSTER_M=<M> -DDOP_INST_CLUSTER_S=<S>.
#include "cluster_row.cuh"

#if !defined(DOP_INST_CLUSTER_M) || !defined(DOP_INST_CLUSTER_S)
#error "compile with -DDOP_INST_CLUSTER_M=<1024|2048|4096> -DDOP_INST_CLUSTER_S=<8|4|2>"
#endif

namespace dop {
template cudaError_t launch_cluster<DOP_INST_CLUSTER_M, DOP_INST_CLUSTER_S>(const PassDesc&, int, cudaStream_t);
} // namespace dop
