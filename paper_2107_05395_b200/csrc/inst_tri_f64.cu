// inst_tri_f64.cu -- instantiations of sweep_kernel for KIND_TRI, f64 (all vector widths / rows).
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_tri_f64(int vec, int rows, int single, int tma, int ws, int fuse)
{
    return pick_f64<KIND_TRI>(vec, rows, single, tma, ws, fuse);
}
}  // namespace btps
