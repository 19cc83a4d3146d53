// inst_f32s.cu -- instantiations of sweep_kernel for fp32 storage with fp64 arithmetic (the *_f32s calls):
// KIND_TRI / KIND_PENTA, 32 rows per thread, one or two systems per thread, single-step launches; also on clusters.
#include "inst_common.cuh"

namespace btps {

template <int V, int MR, int KIND>
static SweepEntry pick_f32s(int single, int tma, int ws)
{
    if (single) return tma ? make_entry<double, V, MR, true, KIND, true, false, false, false, float>()
                           : make_entry<double, V, MR, true, KIND, false, false, false, false, float>();
    if constexpr (MR == 32) {
        if (ws) return tma ? make_entry<double, V, 32, false, KIND, true, true, false, false, float>()
                           : make_entry<double, V, 32, false, KIND, false, true, false, false, float>();
    }
    return SweepEntry{nullptr, nullptr, 0};
}

template <int V, int KIND>
static SweepEntry pick_f32s_rows(int rows, int single, int tma, int ws)
{
    // 8 / 16 rows per thread: the single-partition plans of very short systems (n <= 16)
    if (rows == 8) return pick_f32s<V, 8, KIND>(single, tma, ws);
    if (rows == 16) return pick_f32s<V, 16, KIND>(single, tma, ws);
    if (rows == 32) return pick_f32s<V, 32, KIND>(single, tma, ws);
    return SweepEntry{nullptr, nullptr, 0};
}

// kind in {TRI, PENTA}; vec in {1, 2}; partitioned plans need the warp scan (N <= 1024)
SweepEntry find_sweep_f32s(int kind, int vec, int rows, int single, int tma, int ws)
{
    if (kind == KIND_TRI)
        return vec == 2 ? pick_f32s_rows<2, KIND_TRI>(rows, single, tma, ws) : pick_f32s_rows<1, KIND_TRI>(rows, single, tma, ws);
    if (kind == KIND_PENTA)
        return vec == 2 ? pick_f32s_rows<2, KIND_PENTA>(rows, single, tma, ws) : pick_f32s_rows<1, KIND_PENTA>(rows, single, tma, ws);
    return SweepEntry{nullptr, nullptr, 0};
}

// cluster-split variants (rows of a tile over 2 ... 8 CTAs): two systems per thread, 16 lanes = 128-byte row segments of floats
SweepEntry find_sweep_cl_f32s(int kind)
{
    if (kind == KIND_TRI) return make_entry<double, 2, 32, false, KIND_TRI, true, true, false, true, float>();
    if (kind == KIND_PENTA) return make_entry<double, 2, 32, false, KIND_PENTA, true, true, false, true, float>();
    return SweepEntry{nullptr, nullptr, 0};
}

}  // namespace btps
