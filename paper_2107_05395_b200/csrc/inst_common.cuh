// inst_common.cuh -- explicit-instantiation helper shared by the inst_*.cu units (one unit per
// kind so that nvcc compiles them in parallel).
#pragma once
#include "sweep.cuh"

namespace btps {

template <typename T, int V, int MR, bool SINGLE, int KIND>
static SweepEntry make_entry()
{
    SweepEntry e;
    e.launch = &launch_sweep<T, V, MR, SINGLE, KIND>;
    e.func = reinterpret_cast<const void *>(&sweep_kernel<T, V, MR, SINGLE, KIND>);
    return e;
}

template <typename T, int V, int KIND>
static SweepEntry pick_rows(int rows, int single)
{
    switch (rows) {
        case 8: return single ? make_entry<T, V, 8, true, KIND>() : make_entry<T, V, 8, false, KIND>();
        case 16: return single ? make_entry<T, V, 16, true, KIND>() : make_entry<T, V, 16, false, KIND>();
        case 32: return single ? make_entry<T, V, 32, true, KIND>() : make_entry<T, V, 32, false, KIND>();
        default: break;
    }
    SweepEntry none = {nullptr, nullptr};
    return none;
}

template <int KIND>
static SweepEntry pick_all(int elem_bytes, int vec, int rows, int single)
{
    if (elem_bytes == 8) {
        if (vec == 1) return pick_rows<double, 1, KIND>(rows, single);
        if (vec == 2) return pick_rows<double, 2, KIND>(rows, single);
    } else if (elem_bytes == 4) {
        if (vec == 1) return pick_rows<float, 1, KIND>(rows, single);
        if (vec == 2) return pick_rows<float, 2, KIND>(rows, single);
    }
    SweepEntry none = {nullptr, nullptr};
    return none;
}

SweepEntry find_sweep_tri(int elem_bytes, int vec, int rows, int single);
SweepEntry find_sweep_penta(int elem_bytes, int vec, int rows, int single);
SweepEntry find_sweep_ch(int elem_bytes, int vec, int rows, int single);

}  // namespace btps
