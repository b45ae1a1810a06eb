// qmc_sweep_cluster_f32.cu -- FP32C instantiations of the cluster sweep kernel (qmc_sweep_cluster.cuh).
#include "qmc_sweep_cluster.cuh"

namespace qmc {

#define XC(T, J, V) QMC_CLUSTER_ENTRY(float, T, J, V, 1)
static const ClusterShape kClusterF32[] = {
    XC(64, 4, 4) XC(128, 4, 4) XC(128, 8, 4) XC(128, 16, 4) XC(256, 8, 4) XC(256, 12, 4) XC(256, 16, 4) XC(256, 20, 4)
    XC(512, 8, 4) XC(512, 12, 4) XC(512, 16, 4) XC(512, 20, 4) XC(1024, 8, 4) XC(1024, 10, 2)
};
#undef XC

const ClusterShape *cluster_shapes_f32(int *n) { *n = (int)(sizeof(kClusterF32) / sizeof(kClusterF32[0])); return kClusterF32; }

}  // namespace qmc
