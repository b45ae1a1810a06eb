// qmc_sweep_f64.cu -- FP64 instantiations of the sweep kernel (qmc_sweep_impl.cuh).
// V = 2 shapes read 16-byte coordinate packs; padding is NaN per element, so any N works with any V
// as long as the rows stay 16-byte aligned (N even for V = 2).
#include "qmc_sweep_impl.cuh"

namespace qmc {

#define X(T, J, V) QMC_SHAPE_ENTRY(double, T, J, V, 0)
static const SweepShape kShapesF64[] = {
    X(64, 1, 1) X(64, 2, 1) X(64, 4, 1) X(128, 1, 1) X(128, 2, 1) X(128, 4, 1) X(256, 1, 1) X(256, 2, 1) X(64, 2, 2) X(256, 2, 2)
    X(32, 1, 1) X(32, 2, 1) X(32, 4, 1) X(32, 8, 1) X(64, 8, 1) X(128, 8, 1) X(256, 8, 1) X(512, 8, 1) X(1024, 6, 1)
    X(32, 2, 2) X(32, 4, 2) X(32, 8, 2) X(32, 16, 2) X(64, 4, 2) X(64, 8, 2) X(64, 16, 2)
    X(128, 2, 2) X(128, 4, 2) X(128, 8, 2) X(128, 16, 2) X(256, 4, 2) X(256, 8, 2) X(512, 4, 2) X(512, 8, 2) X(1024, 4, 2) X(1024, 6, 2)
};
#undef X

const SweepShape *sweep_shapes_f64(int *n) { *n = (int)(sizeof(kShapesF64) / sizeof(kShapesF64[0])); return kShapesF64; }

}  // namespace qmc
