// inst_pentapf_f32.cu -- instantiations of sweep_kernel for KIND_PENTAPF (periodic, cyclic correction in the carry scan), f32.
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_pentapf_f32(int vec, int rows, int single, int tma, int ws, int fuse)
{
    return pick_f32<KIND_PENTAPF>(vec, rows, single, tma, ws, fuse);
}
}  // namespace btps
