// inst_ch_f64.cu -- instantiations of sweep_kernel for KIND_CH, f64 (all vector widths / rows).
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_ch_f64(int vec, int rows, int single, int tma, int ws, int fuse)
{
    return pick_f64<KIND_CH>(vec, rows, single, tma, ws, fuse);
}
}  // namespace btps
