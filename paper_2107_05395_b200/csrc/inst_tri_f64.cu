// inst_tri_f64.cu -- instantiations of sweep_kernel for KIND_TRI, f64 (all vector widths / rows).
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_tri_f64(int vec, int rows, int single, int tma, int ws, int fuse)
{
    return pick_f64<KIND_TRI>(vec, rows, single, tma, ws, fuse);
}
SweepEntry find_sweep_cl_tri_f64(int fuse) { return pick_cl<double, 2, KIND_TRI>(fuse); }
}  // namespace btps
