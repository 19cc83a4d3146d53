// inst_penta.cu -- instantiations of sweep_kernel for KIND_PENTA (all dtypes / vector widths / rows).
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_penta(int elem_bytes, int vec, int rows, int single)
{
    return pick_all<KIND_PENTA>(elem_bytes, vec, rows, single);
}
}  // namespace btps
