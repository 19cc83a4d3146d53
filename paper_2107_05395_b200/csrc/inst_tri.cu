// inst_tri.cu -- instantiations of sweep_kernel for KIND_TRI (all dtypes / vector widths / rows).
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_tri(int elem_bytes, int vec, int rows, int single)
{
    return pick_all<KIND_TRI>(elem_bytes, vec, rows, single);
}
}  // namespace btps
