// inst_tricnpf_f64.cu -- instantiations of sweep_kernel for KIND_TRICNPF (periodic, Sherman-Morrison finish in the carry scan), f64.
#include "inst_common.cuh"

namespace btps {
SweepEntry find_sweep_tricnpf_f64(int vec, int rows, int single, int tma, int ws, int fuse)
{
    return pick_f64<KIND_TRICNPF>(vec, rows, single, tma, ws, fuse);
}
}  // namespace btps
