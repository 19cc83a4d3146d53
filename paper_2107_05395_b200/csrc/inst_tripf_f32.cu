// inst_tripf_f32.cu -- instantiations of sweep_kernel for KIND_TRIPF (periodic, Sherman-Morrison finish in the carry scan), f32.
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_tripf_f32(int vec, int rows, int single, int tma, int ws, int fuse)
{
    return pick_f32<KIND_TRIPF>(vec, rows, single, tma, ws, fuse);
}
}  // namespace btps
