// inst_common.cuh -- explicit-instantiation helper shared by the inst_*.cu units (one unit per
// kind and element type so that nvcc compiles them in parallel).
#pragma once
#include "sweep.cuh"
#include <cstdio>

namespace btps {

template <typename T, int V, int MR, bool SINGLE, int KIND, bool TMA, bool WS, bool FUSE = false, bool CL = false, typename S = T>
static SweepEntry make_entry()
{
    SweepEntry e;
    e.launch = &launch_sweep<T, V, MR, SINGLE, KIND, TMA, WS, FUSE, CL, S>;
    e.func = reinterpret_cast<const void *>(&sweep_kernel<T, V, MR, SINGLE, KIND, TMA, WS, FUSE, CL, S>);
    e.max_threads = CtaShape<T, V, MR>::MAX_THREADS;
    static char tag[72];
    static const int once = snprintf(tag, sizeof(tag), "%s, %d, %d, %d, %d, %d, %d, %d, %d, %s", sizeof(T) == 8 ? "double" : "float", V,
                                     MR, (int)SINGLE, KIND, (int)TMA, (int)WS, (int)FUSE, (int)CL, sizeof(S) == 8 ? "double" : "float");
    (void)once;
    e.tag = tag;
    return e;
}

template <typename T, int V, int MR, int KIND>
static SweepEntry pick_variant_general(int single, int tma, int ws, int fuse);

// variants: single partition (no carries) with / without TMA; partitioned with the warp scan
// (with / without TMA) or with the serial carry walk (direct loads only); the fused multi-step
// form exists for the TMA variants
template <typename T, int V, int MR, int KIND>
static SweepEntry pick_variant(int single, int tma, int ws, int fuse)
{
    if constexpr (RecLayout<KIND>::WOODF || RecLayout<KIND>::PERTF) {
        // cyclic correction folded into the warp scan: partitioned, warp-scan variants only
        if (single || !ws) return SweepEntry{nullptr, nullptr, 0};
        if (fuse) return tma ? make_entry<T, V, MR, false, KIND, true, true, true>() : SweepEntry{nullptr, nullptr, 0};
        return tma ? make_entry<T, V, MR, false, KIND, true, true>() : make_entry<T, V, MR, false, KIND, false, true>();
    } else {
        return pick_variant_general<T, V, MR, KIND>(single, tma, ws, fuse);
    }
}

template <typename T, int V, int MR, int KIND>
static SweepEntry pick_variant_general(int single, int tma, int ws, int fuse)
{
    if (fuse) {
        if (!tma) return SweepEntry{nullptr, nullptr, 0};
        if (single) return make_entry<T, V, MR, true, KIND, true, false, true>();
        if (ws) return make_entry<T, V, MR, false, KIND, true, true, true>();
        return SweepEntry{nullptr, nullptr, 0};
    }
    if (single) return tma ? make_entry<T, V, MR, true, KIND, true, false>() : make_entry<T, V, MR, true, KIND, false, false>();
    if (ws) return tma ? make_entry<T, V, MR, false, KIND, true, true>() : make_entry<T, V, MR, false, KIND, false, true>();
    if (!tma) return make_entry<T, V, MR, false, KIND, false, false>();
    SweepEntry none = {nullptr, nullptr, 0};
    return none;
}

template <typename T, int V, int KIND>
static SweepEntry pick_rows(int rows, int single, int tma, int ws, int fuse)
{
    // the base kinds exist for 8, 16 and 32 rows per thread (small n, tuning); the periodic and
    // Crank-Nicolson kinds only for 32 (other plans run their two-pass form)
    if constexpr (KIND == KIND_TRI || KIND == KIND_PENTA || KIND == KIND_CH) {
#ifdef BTPS_TUNING_VARIANTS
        // tuning builds (BTPS_TUNING_VARIANTS=1 python -m paper_2107_05395_b200.build): partitioned plans with 8 / 16 rows per thread
        switch (rows) {
            case 8: return pick_variant<T, V, 8, KIND>(single, tma, ws, fuse);
            case 16: return pick_variant<T, V, 16, KIND>(single, tma, ws, fuse);
            default: break;
        }
#else
        // default build: 8 / 16 rows per thread only as the single-partition plans of very short systems (n <= 16)
        if (single && rows == 8)
            return fuse ? (tma ? make_entry<T, V, 8, true, KIND, true, false, true>() : SweepEntry{nullptr, nullptr, 0})
                        : (tma ? make_entry<T, V, 8, true, KIND, true, false>() : make_entry<T, V, 8, true, KIND, false, false>());
        if (single && rows == 16)
            return fuse ? (tma ? make_entry<T, V, 16, true, KIND, true, false, true>() : SweepEntry{nullptr, nullptr, 0})
                        : (tma ? make_entry<T, V, 16, true, KIND, true, false>() : make_entry<T, V, 16, true, KIND, false, false>());
        if (rows == 8 || rows == 16) return SweepEntry{nullptr, nullptr, 0};
#endif
    }
    if (rows == 32) return pick_variant<T, V, 32, KIND>(single, tma, ws, fuse);
    SweepEntry none = {nullptr, nullptr, 0};
    return none;
}

template <int KIND>
static SweepEntry pick_f64(int vec, int rows, int single, int tma, int ws, int fuse)
{
    if (vec == 1) return pick_rows<double, 1, KIND>(rows, single, tma, ws, fuse);
    if (vec == 2) return pick_rows<double, 2, KIND>(rows, single, tma, ws, fuse);
    SweepEntry none = {nullptr, nullptr, 0};
    return none;
}

template <int KIND>
static SweepEntry pick_f32(int vec, int rows, int single, int tma, int ws, int fuse)
{
    if (vec == 1) return pick_rows<float, 1, KIND>(rows, single, tma, ws, fuse);
#ifdef BTPS_TUNING_VARIANTS
    if (vec == 2) return pick_rows<float, 2, KIND>(rows, single, tma, ws, fuse);  // (plans use 4, or 1 for ragged batches)
#endif
    if (vec == 4) return pick_rows<float, 4, KIND>(rows, single, tma, ws, fuse);
    SweepEntry none = {nullptr, nullptr, 0};
    return none;
}

// cluster-split variants (rows of a tile over two CTAs): plain solves, 32 rows per thread, 16 bytes per thread
template <typename T, int V, int KIND>
static SweepEntry pick_cl(int fuse)
{
    return fuse ? make_entry<T, V, 32, false, KIND, true, true, true, true>()
                : make_entry<T, V, 32, false, KIND, true, true, false, true>();
}
SweepEntry find_sweep_cl(int kind, int elem_bytes, int fuse);
SweepEntry find_sweep_f32s(int kind, int vec, int rows, int single, int tma, int ws);
SweepEntry find_sweep_cl_f32s(int kind);
SweepEntry find_sweep_cl_tri_f64(int fuse);
SweepEntry find_sweep_cl_tri_f32(int fuse);
SweepEntry find_sweep_cl_penta_f64(int fuse);
SweepEntry find_sweep_cl_penta_f32(int fuse);

// kind in {TRI, PENTA, CH}; elem_bytes 8: vec in {1, 2}; 4: vec in {1, 2, 4}; rows in {8, 16, 32}
SweepEntry find_sweep(int kind, int elem_bytes, int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_tri_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_tri_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_penta_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_penta_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_ch_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_ch_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_trip_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_trip_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_pentap_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_pentap_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_chp_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_chp_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_tricn_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_tricnp_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_pentacn_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_pentacnp_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_pentapf_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_pentapf_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_chpf_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_pentacnpf_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_tripf_f64(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_tripf_f32(int vec, int rows, int single, int tma, int ws, int fuse);
SweepEntry find_sweep_tricnpf_f64(int vec, int rows, int single, int tma, int ws, int fuse);

}  // namespace btps
