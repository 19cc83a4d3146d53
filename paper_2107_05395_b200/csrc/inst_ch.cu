// inst_ch.cu -- instantiations of sweep_kernel for KIND_CH (all dtypes / vector widths / rows).
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_ch(int elem_bytes, int vec, int rows, int single)
{
    return pick_all<KIND_CH>(elem_bytes, vec, rows, single);
}
}  // namespace btps
