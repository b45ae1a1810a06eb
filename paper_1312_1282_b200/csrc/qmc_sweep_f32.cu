// qmc_sweep_f32.cu -- FP32C instantiations of the sweep kernel (qmc_sweep_impl.cuh).
// V = 4 shapes need N % 4 == 0, V = 2 shapes N % 2 == 0 (whole packs are real or padding); V = 1 serves any N.
#include "qmc_sweep_impl.cuh"

namespace qmc {

#define X(T, J, V) QMC_SHAPE_ENTRY(float, T, J, V, 0)
#define XP(T, J, V) QMC_SHAPE_ENTRY(float, T, J, V, 1)
static const SweepShape kShapesF32[] = {
    XP(32, 4, 4) XP(32, 8, 4) XP(32, 16, 4) XP(32, 32, 4) XP(64, 4, 4) XP(64, 8, 4) XP(64, 16, 4) XP(64, 32, 4)
    XP(128, 4, 4) XP(128, 8, 4) XP(128, 16, 4) XP(256, 4, 4) XP(256, 8, 4) XP(512, 4, 4) XP(512, 8, 4)
    XP(1024, 8, 4) XP(512, 20, 4) XP(1024, 10, 2)
    X(32, 1, 1) X(32, 2, 1) X(32, 4, 1) X(32, 8, 1) X(64, 8, 1) X(128, 8, 1) X(256, 8, 1) X(512, 8, 1) X(1024, 8, 1) X(1024, 10, 1)
    X(32, 4, 4) X(32, 8, 4) X(32, 16, 4) X(32, 32, 4) X(64, 8, 4) X(64, 16, 4) X(64, 32, 4)
    X(128, 4, 4) X(128, 8, 4) X(128, 16, 4) X(256, 4, 4) X(256, 8, 4) X(512, 4, 4) X(512, 8, 4) X(1024, 8, 4)
    X(512, 20, 4) X(1024, 10, 2)
};
#undef X
#undef XP

const SweepShape *sweep_shapes_f32(int *n) { *n = (int)(sizeof(kShapesF32) / sizeof(kShapesF32[0])); return kShapesF32; }

}  // namespace qmc
