// inst_penta_f32.cu -- instantiations of sweep_kernel for KIND_PENTA, f32 (all vector widths / rows).
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_penta_f32(int vec, int rows, int single, int tma, int ws, int fuse)
{
    return pick_f32<KIND_PENTA>(vec, rows, single, tma, ws, fuse);
}
}  // namespace btps
