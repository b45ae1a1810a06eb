// qmc_sweep_cluster_f64.cu -- FP64 instantiations of the cluster sweep kernel (qmc_sweep_cluster.cuh).
#include "qmc_sweep_cluster.cuh"

namespace qmc {

#define XC(T, J, V) QMC_CLUSTER_ENTRY(double, T, J, V, 0)
static const ClusterShape kClusterF64[] = {
    XC(64, 4, 2) XC(128, 4, 2) XC(128, 8, 2) XC(128, 16, 2) XC(256, 8, 2) XC(256, 16, 2) XC(512, 4, 2) XC(512, 8, 2)
    XC(1024, 4, 2) XC(1024, 6, 2)
};
#undef XC

const ClusterShape *cluster_shapes_f64(int *n) { *n = (int)(sizeof(kClusterF64) / sizeof(kClusterF64[0])); return kClusterF64; }

}  // namespace qmc
