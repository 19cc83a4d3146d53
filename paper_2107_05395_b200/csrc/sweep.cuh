// sweep.cuh -- register-resident partitioned sweep kernels (sm_100a).
//
// What is computed (per system, shared LHS):
//   tri   : forward  g_i = (d_i - a_i g_{i-1}) / b^_i         PAPER.md:95-99  (eq. 3-4), Alg. 2
//           backward x_i = g_i - c^_i x_{i+1}                  PAPER.md:101-108 (eq. 5-6), Alg. 2
//   penta : forward  g_i = (f_i - eps_i g_{i-2} - beta_i g_{i-1}) / alpha_i
//           backward x_i = g_i - gamma_i x_{i+1} - delta_i x_{i+2}            PAPER.md:268-278, Alg. 4
//   periodic tri : A = A' + u (x) v (Sherman-Morrison, eq. 12-15): y = A'^{-1} d by the
//           sweeps above, then x = y - (v.y)/(1 + v.z) z with z = A'^{-1} u from the factor tables
//   ch    : f_i = c_i + alpha_x (w_{i-1} - 2 w_i + w_{i+1}), w = c^3 - c, then the penta sweeps
//           PAPER.md:365-392 (eq. 24, 25a, 26c), truncated stencil (C-18, C-21).
//
// How: the paper gives one thread a whole system and writes g to global
// memory between the sweeps (2 reads + 2 writes per element).  Here a tile of W adjacent systems
// is owned by a GROUP of P*lanes threads: thread (part, lane) keeps rows [part*MR, part*MR+MR) of
// V adjacent systems in registers, so HBM sees one read and one write per element.  Both
// recurrences are linear, so each partition sweeps locally with zero incoming carries; the true
// carries across the P partitions follow from an affine scan  G_{q+1} = g^last_q + Phi_q G_q
// (and its mirror image for the back substitution).  Because A is shared, Phi_q and all products
// of Phi's depend on the LHS only: the scan is run as a log2(P)-step Kogge-Stone scan over the
// lanes of one warp (__shfl) with multipliers precomputed at factor time, and the per-row
// response vectors (chi, psi) that turn the carries into the final correction are part of the
// factor tables ("blob") staged into shared memory once per CTA.  Divisions are replaced by
// factor-time reciprocals and the elimination multipliers are pre-negated so that each row
// costs one multiply and FMAs (C-16).
//
// Data movement: the NEXT tile of a group is fetched by TMA (cp.async.bulk.tensor.2d, one box of
// [rows x W systems] per 256 rows, completion on an mbarrier) into a shared-memory ring while the
// current tile is swept in registers; results are stored straight from registers (coalesced).
// When the batch pitch or base pointer is not 16-byte aligned the same kernel body runs with
// direct (non-prefetched) global loads instead.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace btps {

// TRIP / PENTAP / CHP: the periodic (cyclic) forms of TRI / PENTA / CH
// TRICN / TRICNP: Crank-Nicolson step (explicit three-point half + tri solve), truncated / periodic
enum Kind {
    KIND_TRI = 0, KIND_PENTA = 1, KIND_CH = 2, KIND_TRIP = 3, KIND_PENTAP = 4, KIND_CHP = 5, KIND_TRICN = 6, KIND_TRICNP = 7,
    KIND_PENTACN = 8, KIND_PENTACNP = 9,  // Crank-Nicolson hyperdiffusion step (explicit five-point half + penta solve)
    // PENTAP / CHP / PENTACNP with the cyclic correction folded into the carry scan (whole partitions, P >= 2)
    KIND_PENTAPF = 10, KIND_CHPF = 11, KIND_PENTACNPF = 12,
    KIND_TRIPF = 13, KIND_TRICNPF = 14  // TRIP / TRICNP with the Sherman-Morrison finish folded into the carry scan
};

constexpr int SCAN_STEPS = 5;   // Kogge-Stone steps held in the tables (scan width <= 32)
constexpr int SCAN_LANES = 32;
constexpr int MAX_PARTS = 128;  // partitions of the largest on-chip plan (8 CTAs x 16)

struct SweepArgs {
    void *rhs;             // device, n*batch elements, interleaved
    const void *blob;      // device coefficient image, 16-B aligned, blob_bytes long
    long long batch;
    long long num_tiles;   // ceil(batch / (lanes*V))
    double alpha_x;        // CH only: dt/dx^2
    double per_vN;         // periodic tri: last entry of v, eq. 13a (-a_1/b_1)
    double per_invden;     // periodic tri: 1 / (1 + v.z), eq. 15
    int last_part, last_k; // periodic tri: partition and local row of row n-1
    double ex[5];          // Crank-Nicolson steps: explicit stencil, 3 (eq. 9) or 5 values (eq. 18)
    double per_H[16];      // periodic penta: (I + V^T Z)^{-1}, row-major (Woodbury)
    double per_w6[6];      // periodic penta: wrap-around entries e_0, a_0, e_1, f_{n-2}, c_{n-1}, f_{n-1}
    int wrow_part[4], wrow_k[4];  // periodic penta: partition / local row of rows 0, 1, n-2, n-1
    int xstride;           // elements of exchange area per group
    int xper;              // element offset (inside a group's area) of the 4 x W periodic-penta values
    double per_ngl;        // periodic penta, correction in the scan: -gamma at row n-2
    double *stat;          // CH, fused kernels: device array, stat[ks] += stat_scale * sum over this launch's runs of
                           // 1 / (1 - <C^2>) after step ks (eq. 30); nullptr: no statistic
    double stat_scale;     // 1 / batch
    int n;                 // true number of rows
    int P;                 // partitions per system (rows padded to P*MR with all-zero table rows)
    int lanes;             // threads side by side on adjacent systems (power of two <= 32)
    int lanes_log2;
    int tpc;               // tile groups per CTA (each walks its own tiles)
    int reverse;           // 1: walk the tiles from the last to the first
    int hold_stores;       // 1: a tile's stores wait until the next tile's TMA load has landed
    int scan_log2;         // warp scan: log2 of the scan width (smallest power of two >= P)
    int tq;                // partitions per scan-table row (max(32, P))
    int ksteps;            // time steps advanced per tile while it is on chip (>= 1)
    int xvals;             // values per (partition, system) in the exchange area: 2*NC (+2 halo rows, CH)
    unsigned blob_bytes;   // multiple of 16
    unsigned offT;         // byte offset of the scan tables inside the blob (row records start at 0)
    unsigned offTl;        // byte offset of the scan tables in shared memory (= offT unless the rows are split, CL)
    unsigned offX;         // byte offset of the exchange area in shared memory
    unsigned offM;         // byte offset of the per-group mbarriers (TMA kernels)
    unsigned offR;         // byte offset of the prefetch ring (TMA kernels), 128-B aligned
    unsigned box_rows;     // rows per TMA box (<= 256)
    unsigned nboxes;       // boxes per tile = ceil(P*MR / box_rows)
    // cluster-split kernels (CL): the rows of a tile over `csz` CTAs of one thread-block cluster
    int csz;               // CTAs per cluster (2, 4 or 8); each keeps P / csz partitions
    int scan_log2_cl;      // log2 of the scan width inside one CTA (smallest power of two >= P / csz)
    unsigned tab_bytes_cl; // bytes of one CTA's scan-table block (csz blocks back to back at offT in the blob)
    unsigned offIn;        // byte offset (shared memory) of the carry inboxes: [forward | backward][NC][W]
    int blk;               // elements between the coefficient blocks of successive partitions (ELEMS * MR + padding)
    // coefficient blocks shared between partitions: shared memory holds nuniq blocks, partition p reads block pmap[p]
    int nuniq;
    int cl_own;            // CL: 1 = nothing shared, this CTA stages its own P / csz blocks and indexes them locally
    unsigned char pmap[MAX_PARTS];
};

template <typename T, int N>
struct alignas((sizeof(T) * N) <= 16 ? (sizeof(T) * N) : 16) Tup {
    T v[N];
};

// ---- access to V adjacent systems (global or shared) ------------------------------------------
// S = storage type of the batch (global memory / prefetch ring), T = type of the registers and of all arithmetic:
// the same, or S = float with T = double (fp32 in HBM, fp64 sweeps: the *_f32s calls)
template <typename T, int V, typename S>
__device__ __forceinline__ void ld_sys(T (&d)[V], const S *p)
{
    if constexpr (V == 1) {
        d[0] = (T)*p;
    } else {
        const Tup<S, V> t = *reinterpret_cast<const Tup<S, V> *>(p);
#pragma unroll
        for (int e = 0; e < V; ++e) d[e] = (T)t.v[e];
    }
}

template <typename T, int V, typename S>
__device__ __forceinline__ void st_sys(S *p, const T (&s)[V])
{
    if constexpr (V == 1) {
        *p = (S)s[0];
    } else {
        Tup<S, V> t;
#pragma unroll
        for (int e = 0; e < V; ++e) t.v[e] = (S)s[e];
        *reinterpret_cast<Tup<S, V> *>(p) = t;
    }
}

template <typename T>
__device__ __forceinline__ T fma_t(T a, T b, T c);
template <>
__device__ __forceinline__ double fma_t<double>(double a, double b, double c) { return fma(a, b, c); }
template <>
__device__ __forceinline__ float fma_t<float>(float a, float b, float c) { return fmaf(a, b, c); }

// w(c) = c^3 - c  (the explicit nonlinear term of eq. 24)
template <typename T>
__device__ __forceinline__ T ch_w(T c) { return fma_t<T>(c * c, c, -c); }

// Coefficient image ("blob"), all in element type T, rows padded to Np = P*MR with all-zero rows (a padding row solves to exactly 0).
// One block per partition (MR rows), inside it a structure of arrays with one entry per row, pairs
// {T,T} where one phase of a row needs two values (one LDS.128 in fp64), so that a thread addresses
// everything as one base + compile-time offsets; element offsets of the arrays in units of MR:
//   tri   (5 MR): 0: {inv, nl}   2: nch    3: {chi, psi}
//           inv = 1/b^_i, nl = -a_i/b^_i, nch = -c^_i; chi/psi = response of the finished local
//           sweeps to the incoming forward / backward carry
//   periodic tri, finish in the scan (6 MR): as tri, plus 5: zl, the local (zero-carry) solve of u in the first and
//           last partition (zero elsewhere); scan table slots 10: GZ_q, 11: XZ_q, the carries of A' z = u
//   periodic tri (6 MR): as tri, plus 5: z = A'^{-1} u of the Sherman-Morrison splitting
//   periodic penta (13 MR): as penta, plus 9: {z0, z1}  11: {z2, z3}, the rows of Z = A'^{-1} U (Woodbury)
//   periodic penta, correction in the scan (11 MR): as penta, plus 9: {zl0, zl1}, the local (zero-carry) solves of the
//           unit vectors at rows 0, 1 (first partition) / n-2, n-1 (last partition), zero elsewhere; scan table slots
//           10-11: GZ_q, 12-13: XZ_q (2 x 4 each): the carries of A' z = e_r for r = 0, 1, n-2, n-1
//   penta (9 MR): 0: {inv, nle}  2: nlb    3: {ngam, ndel}   5: {chi1, chi2}   7: {psi1, psi2}
//           inv = 1/alpha_i, nle = -eps_i/alpha_i, nlb = -beta_i/alpha_i, ngam = -gamma_i, ndel = -delta_i
// followed at offT by the carry-scan tables, indexed [slot][m][q] with q = partition (tq entries),
// m = entry of the NC x NC matrix (row-major), NC = 1 (tri) or 2 (penta):
//   slot 2*s     : forward  multiplier of Kogge-Stone step s < 4, A^(s)_q = Phi_q Phi_{q-1} ... (2^s factors),
//                  zero where q < 2^s
//   slot 2*s + 1 : backward multiplier of step s < 4, B^(s)_q = Psi_q Psi_{q+1} ..., zero where q + 2^s >= P
//   slot 8       : step 4, both directions: A^(4)_q at q >= 16, B^(4)_q at q < 16 (each is zero on the
//                  other half, so they share the slot and the reader masks)
//   slot 9       : chi at the partition's first NC rows (turns the forward carry into the local
//                  back-substitution's value at those rows)
// (the serial carry walk keeps only slots 0 and 1, holding Phi_q and Psi_q themselves, and takes chi
// from the row arrays).
template <int KIND>
struct RecLayout {
    static constexpr bool PERTF = (KIND == KIND_TRIPF || KIND == KIND_TRICNPF);  // Sherman-Morrison finish in the scan
    static constexpr bool TRI = (KIND == KIND_TRI || KIND == KIND_TRIP || KIND == KIND_TRICN || KIND == KIND_TRICNP || PERTF);
    static constexpr bool PERT = (KIND == KIND_TRIP || KIND == KIND_TRICNP);  // Sherman-Morrison finish
    static constexpr bool WOOD = (KIND == KIND_PENTAP || KIND == KIND_CHP || KIND == KIND_PENTACNP);  // rank-4 Woodbury correction
    // the same correction folded into the carries
    static constexpr bool WOODF = (KIND == KIND_PENTAPF || KIND == KIND_CHPF || KIND == KIND_PENTACNPF);
    static constexpr int ELEMS = TRI ? ((PERT || PERTF) ? 6 : 5) : (WOOD ? 13 : (WOODF ? 11 : 9));  // values per row
    static constexpr int NC = TRI ? 1 : 2;                     // carries per direction
};

// ---- TMA / mbarrier primitives (PTX) -------------------------------------------------------------
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

// A shared-memory pointer passed through an opaque 32-bit register: the compiler recomputes what it derives from it where
// it is used (hoisted out of the tile / step loops those addresses spill) and still knows the result to be shared memory
// (LDS / STS; through a 64-bit generic register it would emit generic LD / ST).
template <typename P>
__device__ __forceinline__ P *opaque_shared(P *p)
{
    unsigned a32 = smem_u32(p);
    asm volatile("" : "+r"(a32));
    return reinterpret_cast<P *>(__cvta_shared_to_generic((size_t)a32));
}

__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_load(unsigned dst, const void *src, unsigned bytes, unsigned bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_2d(unsigned dst, const CUtensorMap *tm, int c0, int c1, unsigned bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar) : "memory");
}

// ---- thread-block cluster primitives (CL kernels) ---------------------------------------------------
__device__ __forceinline__ unsigned cluster_ctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared-memory address of the same variable in CTA `rank` of the cluster
__device__ __forceinline__ unsigned cluster_map(unsigned local_addr, unsigned rank)
{
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ unsigned cluster_nctarank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
    return r;
}
// wait on a local mbarrier whose arrivals come from another CTA (acquire at cluster scope).  A neighbour that never
// arrives would otherwise hang the device: after ~4 s without progress the kernel traps (the launch then fails with
// an error instead of spinning forever).
__device__ __forceinline__ void mbar_wait_cluster(unsigned bar, unsigned parity)
{
    unsigned done = 0;
    unsigned long long t0 = 0;
    for (unsigned spin = 0;; ++spin) {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(bar), "r"(parity) : "memory");
        if (done) return;
        if ((spin & 1023u) == 1023u) {
            unsigned long long now;
            asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(now));
            if (t0 == 0) t0 = now;
            else if (now - t0 > 4000000000ull) __trap();
        }
    }
}
// Store into another CTA's shared memory that signals the receiver's mbarrier itself (complete_tx of its own bytes): no
// arrive and so no release fence on the sender.  (A separate mbarrier.arrive.release.cluster compiles to MEMBAR.ALL + ERRBAR,
// which also waits for the sender's global stores of the previous tile: 18 % of all stall samples of the cluster kernels.)
__device__ __forceinline__ void st_async_cluster(unsigned addr, double v, unsigned remote_bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f64 [%0], %1, [%2];" ::"r"(addr), "d"(v), "r"(remote_bar) : "memory");
}
__device__ __forceinline__ void st_async_cluster(unsigned addr, float v, unsigned remote_bar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.f32 [%0], %1, [%2];" ::"r"(addr), "f"(v), "r"(remote_bar) : "memory");
}
// the V adjacent values of one owner thread as one 16-byte store where they are 16 bytes (V = 2 doubles / 4 floats)
template <typename T, int V>
__device__ __forceinline__ void st_async_cluster_vec(unsigned addr, const T (&v)[V], unsigned remote_bar)
{
    if constexpr (sizeof(T) == 8 && V == 2) {
        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(addr), "d"(v[0]),
                     "d"(v[1]), "r"(remote_bar) : "memory");
    } else if constexpr (sizeof(T) == 4 && V == 4) {
        asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v4.f32 [%0], {%1, %2, %3, %4}, [%5];" ::"r"(addr),
                     "f"(v[0]), "f"(v[1]), "f"(v[2]), "f"(v[3]), "r"(remote_bar) : "memory");
    } else {
#pragma unroll
        for (int e = 0; e < V; ++e) st_async_cluster(addr + (unsigned)(e * (int)sizeof(T)), v[e], remote_bar);
    }
}

// Barrier over the threads of one tile group.  A CTA hosts `tpc` groups that walk their tiles
// independently of one another (so one group's arithmetic overlaps another group's waits); a
// group of one warp synchronises with __syncwarp, one group per CTA with the CTA barrier, and
// otherwise each group owns the named barrier 1 + sub.
__device__ __forceinline__ void group_sync(int tpc, int sub, int count)
{
    if (count == 32) __syncwarp();
    else if (tpc == 1) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(sub + 1), "r"(count) : "memory");
}

// threads per CTA the kernel is compiled for: 128 registers per thread (512 threads) while the
// tile rows of a thread fit in 64 registers, else 255 registers (256 threads)
template <typename T, int V, int MR>
struct CtaShape {
    static constexpr bool WIDE = (sizeof(T) * V * MR > 256);
    static constexpr int MAX_THREADS = WIDE ? 256 : 512;
};

// Loop over the Kogge-Stone steps.  Measured with ptxas -v, per family, what keeps the 255-register variants from spilling
// their tile rows and what is fastest in the fused time loops: fp32 keeps the loop rolled (MODE 1); the fp64 tridiagonal kinds
// unroll it with a compile-time step index (MODE 2: 26.1 -> 25.8 us per fused step at N = 512, 65536 systems); the fp64
// pentadiagonal kinds leave it to the compiler (MODE 0: unrolled, the fused Cahn-Hilliard step loses 2 %).
template <int MODE, typename F>
__device__ __forceinline__ void scan_steps(int n, F &&f)
{
    if constexpr (MODE == 1) {
#pragma unroll 1
        for (int st = 0; st < n; ++st) f(st);
    } else if constexpr (MODE == 2) {
        // unrolled with a compile-time step index (table slots become immediate offsets, the step-4 masks fold away);
        // steps beyond the scan width are skipped by a warp-uniform branch
#pragma unroll
        for (int st = 0; st < SCAN_STEPS; ++st)
            if (st < n) f(st);
    } else {
        for (int st = 0; st < n; ++st) f(st);
    }
}

// -----------------------------------------------------------------------------------------------
// sweep_kernel<T, V, MR, SINGLE, KIND, TMA, WS>
//   V      systems per thread (adjacent, one vector access)
//   MR     rows per thread (= rows per partition)
//   SINGLE P == 1: no carries to exchange
//   TMA    next tile prefetched by TMA into the shared-memory ring (else direct global loads)
//   WS     carries by the warp-shuffle scan (needs P <= 32 and whole-warp groups); else each
//          thread walks the partitions before / after it serially (any P)
//   CL     the tile's rows are split over a cluster of two CTAs (two SMs): CTA r keeps partitions
//          [r*P/2, (r+1)*P/2) -- twice the systems per tile for long systems (wider row segments in HBM);
//          carries cross the CTAs through distributed shared memory, cluster barriers order them
//   FUSE   a.ksteps time steps per tile (separate instantiation: the step loop costs registers, so
//          single-step launches run the FUSE = false kernel)
// -----------------------------------------------------------------------------------------------
template <typename T, int V, int MR, bool SINGLE, int KIND, bool TMA, bool WS, bool FUSE, bool CL = false, typename S = T>
__global__ void __launch_bounds__(CtaShape<T, V, MR>::MAX_THREADS, 1)
sweep_kernel(const SweepArgs a, const __grid_constant__ CUtensorMap tmap)
{
    constexpr bool TRI = RecLayout<KIND>::TRI;
    constexpr bool ISCH = (KIND == KIND_CH || KIND == KIND_CHP || KIND == KIND_CHPF);  // explicit Cahn-Hilliard half fused in
    constexpr bool ISCN = (KIND == KIND_TRICN || KIND == KIND_TRICNP || KIND == KIND_TRICNPF);  // explicit three-point half (eq. 9) fused in
    constexpr bool ISCN5 = (KIND == KIND_PENTACN || KIND == KIND_PENTACNP || KIND == KIND_PENTACNPF);  // explicit five-point half (eq. 18)
    constexpr bool HALO2 = ISCN5;                                 // needs two rows on each side
    constexpr bool HALO1 = ISCH || ISCN || HALO2;                 // needs the rows r0-1 and r0+MR
    constexpr int NHALO = HALO2 ? 4 : (HALO1 ? 2 : 0);            // exchange values for the fused steps' halos
    constexpr bool WRAP = (KIND == KIND_CHP || KIND == KIND_TRICNP || KIND == KIND_PENTACNP || KIND == KIND_CHPF ||
                           KIND == KIND_PENTACNPF || KIND == KIND_TRICNPF);  // periodic differences
    constexpr bool PERTF = RecLayout<KIND>::PERTF;
    constexpr bool WOODF = RecLayout<KIND>::WOODF;
    constexpr bool PERT = RecLayout<KIND>::PERT;
    constexpr bool WOOD = RecLayout<KIND>::WOOD;
    constexpr int NC = RecLayout<KIND>::NC;
    [[maybe_unused]] constexpr int SCAN_MODE = sizeof(T) == 4 ? 1 : ((TRI && !PERTF) ? 2 : 0);
    using Pair = Tup<T, 2>;
    extern __shared__ __align__(128) unsigned char smem[];

    static_assert(!CL || (!SINGLE && TMA && WS && (KIND == KIND_TRI || KIND == KIND_PENTA)), "cluster split: plain solves only");
    const int W = a.lanes * V;
    [[maybe_unused]] const unsigned crank = CL ? cluster_ctarank() : 0u;  // which block of the rows this CTA keeps
    [[maybe_unused]] const int csz = CL ? a.csz : 1;                      // CTAs that share a tile
    const int PL = CL ? (a.P / a.csz) : a.P;                              // partitions kept by this CTA
    const int tpt = PL * a.lanes;  // threads per tile group (SINGLE: P == 1)
    const int sub = SINGLE ? (threadIdx.x >> a.lanes_log2) : (threadIdx.x / tpt);
    const int lt = SINGLE ? (threadIdx.x & (a.lanes - 1)) : (threadIdx.x - sub * tpt);
    const int plidx = SINGLE ? 0 : (lt >> a.lanes_log2);                  // partition index inside this CTA
    const int part = plidx + (int)crank * PL;                             // partition index inside the system
    const int sl = lt & (a.lanes - 1);
    const int r0 = part * MR;
    const long long batch = a.batch;

    // ---- stage the coefficient image once per CTA: one asynchronous bulk copy ---------------------
    // mbarrier slots at offM: 0..15 = the groups' prefetch rings, 16 = the coefficient image,
    // CL: 17 + job / 33 + job = carry inbox of scan job `job` (a column of owner threads, 16 per CTA) on even / odd
    // exchanges, filled by the other CTAs of the cluster.  One barrier per job: a warp that runs two jobs per tile step must
    // not need its second job's carries from a CTA that is still waiting for this warp's first job.  Two sets (and two
    // inbox buffers) used in turn: a CTA that runs ahead arrives for exchange t + 1 on the other set, and cannot reach
    // exchange t + 2 before this CTA has sent its values of t + 1, i.e. has consumed exchange t.
    [[maybe_unused]] const unsigned mbar = smem_u32(smem + a.offM) + 8u * sub;
    const unsigned bbar = smem_u32(smem + a.offM) + 8u * 16u;
    [[maybe_unused]] const unsigned fin_bar = smem_u32(smem + a.offM) + 8u * 17u;
    [[maybe_unused]] const unsigned bin_bar = smem_u32(smem + a.offM) + 8u * 33u;
    if (threadIdx.x == 0) {
        mbar_init(bbar, 1);
        if constexpr (CL) {  // per exchange one local arrival that states the bytes to expect (F and B from every other CTA)
            for (int jb = 0; jb < a.lanes; ++jb) {
                mbar_init(fin_bar + 8u * jb, 1);
                mbar_init(bin_bar + 8u * jb, 1);
            }
        }
    }
    if constexpr (TMA) {
        if (lt == 0) mbar_init(mbar, 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    if constexpr (CL) cluster_sync();  // the peer CTA is resident (its shared memory may be written) from here on
    else __syncthreads();
    if (threadIdx.x == 0) {
        if constexpr (CL) {
            // this CTA's partitions' coefficient blocks, then its own scan-table block behind them
            const unsigned rows_bytes = (unsigned)((a.cl_own ? PL : a.nuniq) * a.blk) * (unsigned)sizeof(T);
            mbar_expect_tx(bbar, rows_bytes + a.tab_bytes_cl);
            bulk_load(smem_u32(smem), reinterpret_cast<const unsigned char *>(a.blob) + (a.cl_own ? (size_t)crank * rows_bytes : 0),
                      rows_bytes, bbar);
            bulk_load(smem_u32(smem + a.offTl),
                      reinterpret_cast<const unsigned char *>(a.blob) + a.offT + (size_t)crank * a.tab_bytes_cl,
                      a.tab_bytes_cl, bbar);
        } else {
            mbar_expect_tx(bbar, a.blob_bytes);
            bulk_load(smem_u32(smem), a.blob, a.blob_bytes, bbar);
        }
    }
    // Programmatic dependent launch (time-step loops): everything above overlaps the tail of the
    // previous launch on the stream; the batch itself is only touched after the wait.  Both
    // instructions are no-ops for a launch without the attribute.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");

    // rows of this partition that exist
    int nrow_part = a.n - r0;
    nrow_part = nrow_part < 0 ? 0 : (nrow_part > MR ? MR : nrow_part);

    // coefficient arrays of this partition's rows (RecLayout): one base address, the arrays at
    // compile-time offsets from it
    const T *const cb = reinterpret_cast<const T *>(smem) + (size_t)((CL && a.cl_own) ? plidx : (int)a.pmap[part]) * a.blk;
    const Pair *const RA = reinterpret_cast<const Pair *>(cb);                             // {inv, nl | nle}
    const T *const RB1 = cb + 2 * MR;                                                      // nch | nlb
    [[maybe_unused]] const Pair *const RBW = reinterpret_cast<const Pair *>(cb + 3 * MR);  // {chi, psi} | {ngam, ndel}
    [[maybe_unused]] const Pair *const RC0 = reinterpret_cast<const Pair *>(cb + 5 * MR);  // penta {chi1, chi2}
    [[maybe_unused]] const Pair *const RC1 = reinterpret_cast<const Pair *>(cb + 7 * MR);  // penta {psi1, psi2}
    [[maybe_unused]] const T *const TAB = reinterpret_cast<const T *>(smem + a.offTl);
    // exchange area of this group: [2*NC values][P][W], columns XOR-swizzled with the partition index
    [[maybe_unused]] T *const xb = reinterpret_cast<T *>(smem + a.offX) + (size_t)sub * a.xstride;
    // prefetch ring of this group: [P*MR rows][W]
    [[maybe_unused]] const unsigned ring_bytes = (unsigned)(PL * MR * W) * (unsigned)sizeof(S);
    [[maybe_unused]] const int rbase = (int)crank * PL * MR;  // first row kept by this CTA
    // carry inboxes of this CTA (CL): [forward | backward][sending CTA: 8 slots][NC][W], written by the other CTAs of the
    // cluster through distributed shared memory
    [[maybe_unused]] T *const inbox = reinterpret_cast<T *>(smem + a.offIn);
    [[maybe_unused]] const unsigned inbox_u32 = smem_u32(smem + a.offIn);
    [[maybe_unused]] unsigned cstep = 0;  // exchanges done: set = cstep & 1, barrier parity = (cstep >> 1) & 1
    [[maybe_unused]] S *const ring = reinterpret_cast<S *>(smem + a.offR + (size_t)sub * ring_bytes);

    const int ntiles = (int)a.num_tiles;
    const int stride_tiles = CL ? (int)(gridDim.x / (unsigned)csz) : (int)(gridDim.x * a.tpc);
    S *const rhs0 = reinterpret_cast<S *>(a.rhs) + (long long)r0 * batch + (long long)sl * V;

    // one thread of the group asks the TMA unit for tile `t` (walking order); columns beyond the
    // batch and rows beyond n are zero-filled by the unit
    auto tma_issue = [&](int t) {
        const int tile = a.reverse ? ntiles - 1 - t : t;
        mbar_expect_tx(mbar, ring_bytes);
        const unsigned dst = smem_u32(ring);
        const unsigned box_bytes = a.box_rows * (unsigned)W * (unsigned)sizeof(S);
        for (unsigned b = 0; b < a.nboxes; ++b)
            tma_load_2d(dst + b * box_bytes, &tmap, tile * W, (int)(b * a.box_rows) + rbase, mbar);
    };

    // group-major tile order: consecutive tiles go to different CTAs, so a small batch spreads over all SMs
    // before any CTA runs a second group
    int t = CL ? (int)(blockIdx.x / (unsigned)csz) : (int)(blockIdx.x + sub * gridDim.x);
    [[maybe_unused]] unsigned phase = 0;
    if constexpr (TMA) {
        if (lt == 0 && t < ntiles) tma_issue(t);
    }
    mbar_wait(bbar, 0);  // coefficient image has landed
    for (; t < ntiles; t += stride_tiles) {
        const int tile = a.reverse ? ntiles - 1 - t : t;
        const long long j = (long long)tile * W + (long long)sl * V;
        const bool act = (j < batch);  // V > 1 requires batch % V == 0
        const int nrow = act ? nrow_part : 0;  // rows stored by this thread
        S *const p0 = rhs0 + (long long)tile * W;

        T v[MR][V];
        [[maybe_unused]] T cm[V], cp[V];    // halo rows r0-1 and r0+MR (c^n)
        [[maybe_unused]] T cm2[V], cp2[V];  // five-point stencil: rows r0-2 and r0+MR+1
        if constexpr (TMA) {
            // ---- take the prefetched tile out of the ring, then have it refilled ---------------
            mbar_wait(mbar, phase);
            phase ^= 1u;
            // (the address goes through an opaque 32-bit register so that the MR row addresses are recomputed per tile
            //  -- hoisted out of the loop they spill -- and comes back as a pointer the compiler still knows to be shared
            //  memory: LDS, not generic LD)
            const S *rp = opaque_shared(ring + ((r0 - rbase) * W + sl * V));
#pragma unroll
            for (int k = 0; k < MR; ++k) ld_sys<T, V>(v[k], rp + k * W);
            if constexpr (HALO1) {
#pragma unroll
                for (int e = 0; e < V; ++e) cm[e] = cp[e] = T(0);
                if constexpr (HALO2) {
#pragma unroll
                    for (int e = 0; e < V; ++e) cm2[e] = cp2[e] = T(0);
                }
                if constexpr (!SINGLE) {
                    // periodic form (n a multiple of MR): row -1 is row n-1, row n is row 0
                    if (part > 0) ld_sys<T, V>(cm, rp - W);
                    else if (WRAP) ld_sys<T, V>(cm, ring + ((a.n - 1) * W + sl * V));
                    if (part + 1 < a.P) ld_sys<T, V>(cp, rp + MR * W);
                    else if (WRAP) ld_sys<T, V>(cp, ring + sl * V);
                    if constexpr (HALO2) {
                        if (part > 0) ld_sys<T, V>(cm2, rp - 2 * W);
                        else if (WRAP) ld_sys<T, V>(cm2, ring + ((a.n - 2) * W + sl * V));
                        if (part + 1 < a.P) ld_sys<T, V>(cp2, rp + (MR + 1) * W);
                        else if (WRAP) ld_sys<T, V>(cp2, ring + (W + sl * V));
                    }
                }
            }
            // The ring is about to be overwritten by the TMA unit (async proxy) while these loads went through the generic
            // proxy: every thread orders its own reads before that write with a proxy fence, then the group meets.  Without
            // it a one-warp group (__syncwarp does not wait for outstanding shared-memory loads) could have loads of this
            // tile still queued behind seven other groups' when the next tile arrived from L2: wrong tiles now and then on
            // L2-resident batches with eight groups per CTA (N = 64, found by the randomised sweep against the oracle).
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            group_sync(a.tpc, sub, tpt);  // every thread has drained the ring
            if (lt == 0 && t + stride_tiles < ntiles) tma_issue(t + stride_tiles);
        } else {
            // ---- load: all MR rows issued back to back (independent of the recurrence) ---------
            // (one running row pointer: keeping MR separate 64-bit addresses alive would cost 2*MR registers)
            const S *pl = p0;
#pragma unroll
            for (int k = 0; k < MR; ++k) {
                if (k < nrow) {
                    ld_sys<T, V>(v[k], pl);
                } else {
#pragma unroll
                    for (int e = 0; e < V; ++e) v[k][e] = T(0);
                }
                pl += batch;
            }
            if constexpr (HALO1) {
                // halo rows come from the neighbouring partitions' rows in global memory (still
                // c^n: nobody stores before the barriers below).
#pragma unroll
                for (int e = 0; e < V; ++e) cm[e] = cp[e] = T(0);
                // (r0 <= n: partitions that lie wholly beyond row n -- plans padded to whole cluster CTAs -- have no row r0-1)
                if (act && r0 > 0 && r0 <= a.n) ld_sys<T, V>(cm, p0 - batch);
                else if (WRAP && act) ld_sys<T, V>(cm, p0 + (long long)(a.n - 1) * batch);   // r0 == 0: row n-1
                if (act && (r0 + MR < a.n)) ld_sys<T, V>(cp, p0 + (long long)MR * batch);
                else if (WRAP && act) ld_sys<T, V>(cp, p0 - (long long)r0 * batch);          // row 0
                if constexpr (HALO2) {
#pragma unroll
                    for (int e = 0; e < V; ++e) cm2[e] = cp2[e] = T(0);
                    if (act && r0 > 1 && r0 <= a.n + 1) ld_sys<T, V>(cm2, p0 - 2 * batch);
                    else if (WRAP && act) ld_sys<T, V>(cm2, p0 + (long long)(a.n - 2) * batch);      // r0 == 0: row n-2
                    if (act && (r0 + MR + 1 < a.n)) ld_sys<T, V>(cp2, p0 + (long long)(MR + 1) * batch);
                    else if (WRAP && act) ld_sys<T, V>(cp2, p0 - (long long)(r0 - 1) * batch);       // row 1
                }
            }
        }

        // ---- ksteps time steps on the tile while it is on chip (RHS = previous solution) ----
        const int nks = FUSE ? a.ksteps : 1;
        for (int ks = 0; ks < nks; ++ks) {
        if constexpr (HALO1 && !SINGLE) {
            if (ks > 0) {
                // halo rows of c^{n+ks}: the neighbouring partitions' first / last rows, published to
                // exchange values 2NC (first row) and 2NC+1 (last row) at the end of the previous step
                group_sync(a.tpc, sub, tpt);
                const int hv = a.P * W, hm = W - 1;
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    const int pm = (part > 0) ? part - 1 : (WRAP ? a.P - 1 : -1);
                    const int pp = (part + 1 < a.P) ? part + 1 : (WRAP ? 0 : -1);
                    cm[e] = (pm >= 0) ? xb[(2 * NC + 1) * hv + pm * W + ((sl * V + e) ^ (pm & hm))] : T(0);
                    cp[e] = (pp >= 0) ? xb[2 * NC * hv + pp * W + ((sl * V + e) ^ (pp & hm))] : T(0);
                    if constexpr (HALO2) {  // values 2NC+2 / 2NC+3: second row / last-but-one row
                        cm2[e] = (pm >= 0) ? xb[(2 * NC + 3) * hv + pm * W + ((sl * V + e) ^ (pm & hm))] : T(0);
                        cp2[e] = (pp >= 0) ? xb[(2 * NC + 2) * hv + pp * W + ((sl * V + e) ^ (pp & hm))] : T(0);
                    }
                }
            }
        }
        [[maybe_unused]] T glast2[V];  // penta: g at the partition's last-but-one row (overwritten by the backward sweep)
        if constexpr (TRI) {
            // ---- local forward sweep, zero incoming carry ---------------------------------
            T gp[V];
#pragma unroll
            for (int e = 0; e < V; ++e) gp[e] = T(0);
            if constexpr (ISCN) {
                // explicit half of Crank-Nicolson (eq. 9): f_k = xa c_{k-1} + xb c_k + xc c_{k+1}, in registers
                const T xa = (T)a.ex[0], xb = (T)a.ex[1], xc = (T)a.ex[2];
                T cprev[V];
#pragma unroll
                for (int e = 0; e < V; ++e) cprev[e] = cm[e];
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    // (padding rows need no masking: their table rows have inv = nl = 0, so whatever f holds there,
                    //  g and x of a padding row come out as exact zeros)
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T cn = (k + 1 < MR) ? v[(k + 1 < MR) ? k + 1 : k][e] : cp[e];
                        const T f = fma_t<T>(xa, cprev[e], fma_t<T>(xc, cn, xb * v[k][e]));
                        cprev[e] = v[k][e];
                        v[k][e] = f;
                    }
                }
            }
#pragma unroll
            for (int k = 0; k < MR; ++k) {
                const Pair cf = RA[k];
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    v[k][e] = fma_t<T>(cf.v[1], gp[e], cf.v[0] * v[k][e]);
                    gp[e] = v[k][e];
                }
            }
            // ---- local backward sweep, zero incoming carry --------------------------------
#pragma unroll
            for (int e = 0; e < V; ++e) gp[e] = T(0);
#pragma unroll
            for (int k = MR - 1; k >= 0; --k) {
                const T nch = RB1[k];
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    v[k][e] = fma_t<T>(nch, gp[e], v[k][e]);
                    gp[e] = v[k][e];
                }
            }
        } else {
            T g1[V], g2[V];  // g_{k-1}, g_{k-2}
#pragma unroll
            for (int e = 0; e < V; ++e) g1[e] = g2[e] = T(0);
            if constexpr (ISCN5) {
                // explicit half of the Crank-Nicolson hyperdiffusion step (eq. 18), in registers:
                // f_k = x0 c_{k-2} + x1 c_{k-1} + x2 c_k + x3 c_{k+1} + x4 c_{k+2}
                const T x0 = (T)a.ex[0], x1 = (T)a.ex[1], x2 = (T)a.ex[2], x3 = (T)a.ex[3], x4 = (T)a.ex[4];
                T c1[V], c2[V];
#pragma unroll
                for (int e = 0; e < V; ++e) { c1[e] = cm[e]; c2[e] = cm2[e]; }
#pragma unroll
                for (int k = 0; k < MR; ++k) {
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T n1 = (k + 1 < MR) ? v[(k + 1 < MR) ? k + 1 : k][e] : cp[e];
                        const T n2 = (k + 2 < MR) ? v[(k + 2 < MR) ? k + 2 : k][e] : ((k + 2 == MR) ? cp[e] : cp2[e]);
                        T f = fma_t<T>(x1, c1[e], x0 * c2[e]);
                        f = fma_t<T>(x2, v[k][e], f);
                        f = fma_t<T>(x3, n1, f);
                        f = fma_t<T>(x4, n2, f);
                        c2[e] = c1[e];
                        c1[e] = v[k][e];
                        v[k][e] = f;  // (padding rows: inv = 0 in their table rows, see above)
                    }
                }
            }
            if constexpr (ISCH) {
                // explicit half: f_k = c_k + alpha_x (w_{k-1} - 2 w_k + w_{k+1}); cm / cp are the
                // halo rows r0-1 and r0+MR fetched above (zero outside the system).
                const T ax = (T)a.alpha_x;
                T wm[V], wc[V];
#pragma unroll
                for (int e = 0; e < V; ++e) { wm[e] = ch_w<T>(cm[e]); wc[e] = ch_w<T>(v[0][e]); }
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    const Pair cf = RA[k];
                    const T nlb = RB1[k];
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T wn = ch_w<T>((k + 1 < MR) ? v[(k + 1 < MR) ? k + 1 : k][e] : cp[e]);
                        T s = wm[e] + wn;
                        s = fma_t<T>(T(-2), wc[e], s);
                        const T f = fma_t<T>(ax, s, v[k][e]);  // (padding rows: inv = 0 in their table rows, see above)
                        wm[e] = wc[e];
                        wc[e] = wn;
                        const T t2 = fma_t<T>(cf.v[1], g2[e], cf.v[0] * f);
                        const T g = fma_t<T>(nlb, g1[e], t2);
                        v[k][e] = g;
                        g2[e] = g1[e];
                        g1[e] = g;
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    const Pair cf = RA[k];
                    const T nlb = RB1[k];
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T t2 = fma_t<T>(cf.v[1], g2[e], cf.v[0] * v[k][e]);
                        const T g = fma_t<T>(nlb, g1[e], t2);
                        v[k][e] = g;
                        g2[e] = g1[e];
                        g1[e] = g;
                    }
                }
            }
#pragma unroll
            for (int e = 0; e < V; ++e) glast2[e] = g2[e];  // = g at row MR-2
            // backward
#pragma unroll
            for (int e = 0; e < V; ++e) g1[e] = g2[e] = T(0);  // x_{k+1}, x_{k+2}
#pragma unroll
            for (int k = MR - 1; k >= 0; --k) {
                const Pair cbw = RBW[k];
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    const T t2 = fma_t<T>(cbw.v[1], g2[e], v[k][e]);
                    const T x = fma_t<T>(cbw.v[0], g1[e], t2);
                    v[k][e] = x;
                    g2[e] = g1[e];
                    g1[e] = x;
                }
            }
        }

        // ---- carries across the partitions ----------------------------------------------------------
        // exchange area xb[value][partition][column], value 0..NC-1: forward (g at the partition's
        // last NC rows), NC..2NC-1: backward (x^ at its first NC rows); the scan overwrites them
        // with the incoming carries G (forward) and X (backward) of that partition.
        if constexpr (!SINGLE) {
            // partitions that exchange carries inside this CTA (CL: the CTA's own block of the system's partitions; the
            // carries across the CTAs of the cluster travel through the inboxes, see the scan below)
            const int P = CL ? PL : a.P;
            const int tq = a.tq;
            const int wm = W - 1;
            // this thread's columns of its partition: element e lives at xc[XI(e)]
            T *xc = xb + (size_t)(CL ? plidx : part) * W;
            if constexpr (FUSE) xc = opaque_shared(xc);
            const int xsw = (CL ? plidx : part) & wm;
#define XI(e) (((sl * V + (e)) ^ xsw))
            const int vstr = P * W;  // elements between successive values
            [[maybe_unused]] T G[NC][V], X[NC][V];
            if constexpr (WS) {
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    if constexpr (TRI) {
                        xc[XI(e)] = v[MR - 1][e];
                        xc[vstr + XI(e)] = v[0][e];
                    } else {
                        xc[XI(e)] = v[MR - 1][e];
                        xc[vstr + XI(e)] = glast2[e];
                        xc[2 * vstr + XI(e)] = v[0][e];
                        xc[3 * vstr + XI(e)] = v[1][e];
                    }
                }
                group_sync(a.tpc, sub, tpt);
                {
                    // lane q of a `width`-lane segment holds partition q
                    const int slog = CL ? a.scan_log2_cl : a.scan_log2;
                    const int lane = lt & 31;
                    const int wd = 1 << slog;
                    const int q = lane & (wd - 1);
                    const int spw = 32 >> slog;  // jobs per warp pass
                    const T *tb = TAB + q;
                    if constexpr (FUSE) tb = opaque_shared(tb);
                    // (warp-scan plans have at most 32 partitions, so their table rows always hold SCAN_LANES entries:
                    //  compile-time strides turn the table addressing into immediate offsets)
                    constexpr int mstr = SCAN_LANES;            // elements between matrix entries
                    constexpr int sstr = NC * NC * SCAN_LANES;  // elements between table slots
                    // multipliers of step st: slots 2st (forward) / 2st+1 (backward); step 4 shares
                    // slot 8: its forward entries are nonzero only at q >= 16, its backward ones only
                    // at q < 16, and each reader masks the other half
                    auto fwm = [&](int st, int m) -> T {
                        const T val = tb[(st < 4 ? 2 * st : 8) * sstr + m * mstr];
                        return (st < 4 || q >= 16) ? val : T(0);
                    };
                    auto bwm = [&](int st, int m) -> T {
                        const T val = tb[(st < 4 ? 2 * st + 1 : 8) * sstr + m * mstr];
                        return (st < 4 || q < 16) ? val : T(0);
                    };
                    // job = the V systems of one owner thread column sg: V independent chains per lane
                    const int job0 = 0;
                    const int job1 = a.lanes;
                    for (int s0 = job0 + (lt >> 5) * spw; s0 < job1; s0 += (tpt >> 5) * spw) {
                        const int sg = s0 + (lane >> slog);
                        const bool ok = (q < P) && (sg < job1);
                        T *xs = xb + (size_t)q * W;
                        if constexpr (FUSE) xs = opaque_shared(xs);  // (as for rp: hoisted out of the step loop it spills)
                        const int qsw = q & wm;
                        T fb[NC][V], bb[NC][V];  // forward / backward scan state (then the carries G / X)
#pragma unroll
                        for (int c = 0; c < NC; ++c)
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                const int ix = (sg * V + e) ^ qsw;
                                fb[c][e] = ok ? xs[c * vstr + ix] : T(0);
                                bb[c][e] = ok ? xs[(NC + c) * vstr + ix] : T(0);
                            }
                        scan_steps<SCAN_MODE>(slog, [&](int st) {
                            T m[NC * NC];
#pragma unroll
                            for (int i = 0; i < NC * NC; ++i) m[i] = fwm(st, i);
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                T o[NC];
#pragma unroll
                                for (int c = 0; c < NC; ++c) o[c] = __shfl_up_sync(0xffffffffu, fb[c][e], 1 << st, wd);
                                if constexpr (TRI) {
                                    fb[0][e] = fma_t<T>(m[0], o[0], fb[0][e]);
                                } else {
                                    fb[0][e] = fma_t<T>(m[1], o[1], fma_t<T>(m[0], o[0], fb[0][e]));
                                    fb[1][e] = fma_t<T>(m[3], o[1], fma_t<T>(m[2], o[0], fb[1][e]));
                                }
                            }
                        });
                        // CL: fb is the inclusive scan of this CTA's partitions with zero carry-in; its last value F is this
                        // CTA's forward contribution to the cluster-level recurrence (exchanged below, once, together with B)
                        [[maybe_unused]] T Fown[NC][V];
                        if constexpr (CL) {
#pragma unroll
                            for (int c = 0; c < NC; ++c)
#pragma unroll
                                for (int e = 0; e < V; ++e) Fown[c][e] = __shfl_sync(0xffffffffu, fb[c][e], P - 1, wd);
                        }
                        [[maybe_unused]] T yn1[V], yn2[V];  // cyclic forms: y at rows n-1, n-2 (true g at the last rows)
                        if constexpr (PERTF) {
#pragma unroll
                            for (int e = 0; e < V; ++e) yn1[e] = __shfl_sync(0xffffffffu, fb[0][e], P - 1, wd);  // y_N = g_N
                        }
                        if constexpr (WOODF) {
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                const T i0 = __shfl_sync(0xffffffffu, fb[0][e], P - 1, wd);
                                const T i1 = __shfl_sync(0xffffffffu, fb[1][e], P - 1, wd);
                                yn1[e] = i0;                                  // x_{n-1} = g_{n-1}
                                yn2[e] = fma_t<T>((T)a.per_ngl, i0, i1);      // x_{n-2} = g_{n-2} - gamma_{n-2} x_{n-1}
                            }
                        }
                        {
                            // carry INTO partition q = inclusive result of partition q-1; then the local
                            // back-substitution's first rows given that carry: u = x^_first + chi G
                            T ch[NC * NC];
#pragma unroll
                            for (int i = 0; i < NC * NC; ++i) ch[i] = tb[9 * sstr + i * mstr];
#pragma unroll
                            for (int e = 0; e < V; ++e) {
#pragma unroll
                                for (int c = 0; c < NC; ++c) {
                                    const T g = __shfl_up_sync(0xffffffffu, fb[c][e], 1, wd);
                                    fb[c][e] = (q == 0) ? T(0) : g;
                                }
                                if constexpr (TRI) {
                                    bb[0][e] = fma_t<T>(ch[0], fb[0][e], bb[0][e]);
                                } else {
                                    bb[0][e] = fma_t<T>(ch[1], fb[1][e], fma_t<T>(ch[0], fb[0][e], bb[0][e]));
                                    bb[1][e] = fma_t<T>(ch[3], fb[1][e], fma_t<T>(ch[2], fb[0][e], bb[1][e]));
                                }
                            }
                        }
                        scan_steps<SCAN_MODE>(slog, [&](int st) {
                            T m[NC * NC];
#pragma unroll
                            for (int i = 0; i < NC * NC; ++i) m[i] = bwm(st, i);
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                T o[NC];
#pragma unroll
                                for (int c = 0; c < NC; ++c) o[c] = __shfl_down_sync(0xffffffffu, bb[c][e], 1 << st, wd);
                                if constexpr (TRI) {
                                    bb[0][e] = fma_t<T>(m[0], o[0], bb[0][e]);
                                } else {
                                    bb[0][e] = fma_t<T>(m[1], o[1], fma_t<T>(m[0], o[0], bb[0][e]));
                                    bb[1][e] = fma_t<T>(m[3], o[1], fma_t<T>(m[2], o[0], bb[1][e]));
                                }
                            }
                        });
                        // CL: the carries across the CTAs of the cluster, ONE exchange per tile step whatever the cluster size.  So
                        // far this CTA's block of partitions was solved on its own: F = its forward carry out, B = bb at its first
                        // partition = its backward carry out, both for zero carries in.  Every CTA sends (F, B) to all the others,
                        // and forms its own carries in from them with the LHS-only matrices of table slot 12 (put_scan_tables in
                        // btps.cu: the cluster-level recurrences unrolled):  Gin = sum_{s<r} C_s F_s,  Xin = sum_{s>r} D_s B_s +
                        // sum_t E_t F_t.  They then reach partition q through slots 10 (Pin_q), 13 (Th_{q+1}) and 11 (Sf_{q+1}).
                        [[maybe_unused]] T gin[NC][V], xin[NC][V];
                        if constexpr (CL) {
                            const unsigned set = cstep & 1u;
                            const unsigned xbar = (set ? bin_bar : fin_bar) + 8u * (unsigned)sg;
                            const int ibuf = (int)set * (2 * 8 * NC * W);  // this exchange's inbox buffer (elements)
                            if (ok && (q == P - 1 || q == 0)) {
                                // lane 0 arms this CTA's barrier for the bytes the others will send (its own arrival; it has waited
                                // for this barrier's previous phase itself), then lane P-1 sends F (slot crank) and lane 0 sends B
                                // (slot 8 + crank): every store completes its own bytes on the receiver's barrier
                                if (q == 0) mbar_expect_tx(xbar, (unsigned)((csz - 1) * 2 * NC * V) * (unsigned)sizeof(T));
                                const int slot = (q == 0) ? 8 + (int)crank : (int)crank;
                                for (int r = 0; r < csz; ++r) {
                                    if (r == (int)crank) continue;
                                    const unsigned rin = cluster_map(inbox_u32, (unsigned)r);
                                    const unsigned rbar = cluster_map(xbar, (unsigned)r);
#pragma unroll
                                    for (int c = 0; c < NC; ++c) {
                                        T pay[V];
#pragma unroll
                                        for (int e = 0; e < V; ++e) pay[e] = (q == 0) ? bb[c][e] : Fown[c][e];
                                        st_async_cluster_vec<T, V>(rin + (unsigned)((ibuf + (slot * NC + c) * W + sg * V) * (int)sizeof(T)), pay, rbar);
                                    }
                                }
                            }
#pragma unroll
                            for (int c = 0; c < NC; ++c)
#pragma unroll
                                for (int e = 0; e < V; ++e) {
                                    gin[c][e] = T(0);
                                    xin[c][e] = T(0);
                                }
                            if (sg < job1) {
                                mbar_wait_cluster(xbar, (cstep >> 1) & 1u);
                                const T *const ib = inbox + ibuf;
                                const T *const t12 = TAB + 12 * sstr;
                                // Gin = sum_{s<r} C_s F_s;  Xin = sum_{s>r} D_s B_s + sum_t E_t F_t  (entries s, 8 + s, 16 + t of slot 12)
                                for (int cc = 0; cc < csz; ++cc) {
                                    T cm_[NC * NC], dm_[NC * NC], em_[NC * NC];
#pragma unroll
                                    for (int i = 0; i < NC * NC; ++i) {
                                        cm_[i] = t12[i * mstr + cc];        // zero for cc >= r (never written)
                                        dm_[i] = t12[i * mstr + 8 + cc];    // zero for cc <= r
                                        em_[i] = t12[i * mstr + 16 + cc];
                                    }
                                    const bool own = cc == (int)crank;
#pragma unroll
                                    for (int e = 0; e < V; ++e) {
                                        T f[NC], b[NC];
#pragma unroll
                                        for (int c = 0; c < NC; ++c) {
                                            f[c] = own ? Fown[c][e] : (ok ? ib[(cc * NC + c) * W + sg * V + e] : T(0));
                                            b[c] = own ? T(0) : (ok ? ib[((8 + cc) * NC + c) * W + sg * V + e] : T(0));
                                        }
                                        if constexpr (TRI) {
                                            gin[0][e] = fma_t<T>(cm_[0], f[0], gin[0][e]);
                                            xin[0][e] = fma_t<T>(em_[0], f[0], fma_t<T>(dm_[0], b[0], xin[0][e]));
                                        } else {
                                            gin[0][e] = fma_t<T>(cm_[1], f[1], fma_t<T>(cm_[0], f[0], gin[0][e]));
                                            gin[1][e] = fma_t<T>(cm_[3], f[1], fma_t<T>(cm_[2], f[0], gin[1][e]));
                                            xin[0][e] = fma_t<T>(dm_[1], b[1], fma_t<T>(dm_[0], b[0], xin[0][e]));
                                            xin[1][e] = fma_t<T>(dm_[3], b[1], fma_t<T>(dm_[2], b[0], xin[1][e]));
                                            xin[0][e] = fma_t<T>(em_[1], f[1], fma_t<T>(em_[0], f[0], xin[0][e]));
                                            xin[1][e] = fma_t<T>(em_[3], f[1], fma_t<T>(em_[2], f[0], xin[1][e]));
                                        }
                                    }
                                }
                            }
                        }
                        // Cyclic correction in the scan: x = y - Z w with w = H V^T y.  Column m of Z = A'^{-1} e_r is
                        // itself "local solve + chi GZ^m + psi XZ^m", so -Z w only shifts the carries,
                        // G_q += GZ_q nw, X_q += XZ_q nw (nw = -w), plus the local solves in the two end partitions.
                        [[maybe_unused]] T nw[4][V];
                        if constexpr (PERTF) {
                            // Sherman-Morrison in the scan: x = y + nfac z, nfac = -(y_1 + v_N y_N)/(1 + v.z), and z is
                            // itself "local solve + chi GZ + psi XZ": G_q += GZ_q nfac, X_q += XZ_q nfac
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                const T y0 = __shfl_sync(0xffffffffu, bb[0][e], 0, wd);
                                nw[0][e] = -(fma_t<T>((T)a.per_vN, yn1[e], y0) * (T)a.per_invden);
                            }
                        }
                        if constexpr (WOODF) {
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                const T y0 = __shfl_sync(0xffffffffu, bb[0][e], 0, wd);  // true x at rows 0, 1
                                const T y1 = __shfl_sync(0xffffffffu, bb[1][e], 0, wd);
                                const T t0 = fma_t<T>((T)a.per_w6[1], yn1[e], (T)a.per_w6[0] * yn2[e]);
                                const T t1 = (T)a.per_w6[2] * yn1[e];
                                const T t2 = (T)a.per_w6[3] * y0;
                                const T t3 = fma_t<T>((T)a.per_w6[5], y1, (T)a.per_w6[4] * y0);
#pragma unroll
                                for (int m = 0; m < 4; ++m)
                                    nw[m][e] = -fma_t<T>((T)a.per_H[m * 4 + 3], t3, fma_t<T>((T)a.per_H[m * 4 + 2], t2,
                                                          fma_t<T>((T)a.per_H[m * 4 + 1], t1, (T)a.per_H[m * 4] * t0)));
                            }
                        }
#pragma unroll
                        for (int c = 0; c < NC; ++c)
#pragma unroll
                            for (int e = 0; e < V; ++e) {
                                T x = __shfl_down_sync(0xffffffffu, bb[c][e], 1, wd);
                                const int ix = (sg * V + e) ^ qsw;
                                x = (q + 1 < P) ? x : T(0);
                                if constexpr (CL) {
                                    // G_q = G0_q + Pin_q Gin;  X_q = X0_q + Th_{q+1} Gin + Sf_{q+1} Xin  (row c of each matrix)
                                    if constexpr (TRI) {
                                        fb[c][e] = fma_t<T>(tb[10 * sstr], gin[0][e], fb[c][e]);
                                        x = fma_t<T>(tb[11 * sstr], xin[0][e], fma_t<T>(tb[13 * sstr], gin[0][e], x));
                                    } else {
                                        fb[c][e] = fma_t<T>(tb[10 * sstr + (2 * c + 1) * mstr], gin[1][e],
                                                            fma_t<T>(tb[10 * sstr + (2 * c) * mstr], gin[0][e], fb[c][e]));
                                        x = fma_t<T>(tb[13 * sstr + (2 * c + 1) * mstr], gin[1][e],
                                                     fma_t<T>(tb[13 * sstr + (2 * c) * mstr], gin[0][e], x));
                                        x = fma_t<T>(tb[11 * sstr + (2 * c + 1) * mstr], xin[1][e],
                                                     fma_t<T>(tb[11 * sstr + (2 * c) * mstr], xin[0][e], x));
                                    }
                                }
                                if constexpr (PERTF) {
                                    fb[c][e] = fma_t<T>(tb[10 * sstr], nw[0][e], fb[c][e]);
                                    x = fma_t<T>(tb[11 * sstr], nw[0][e], x);
                                    if (ok && (q == 0 || q == P - 1)) xs[(2 * NC + NHALO) * vstr + ix] = nw[0][e];
                                }
                                if constexpr (WOODF) {
                                    const T *const gz = tb + (40 + c * 4) * mstr;  // slots 10-11: GZ_q, row c
                                    const T *const xz = tb + (48 + c * 4) * mstr;  // slots 12-13: XZ_q, row c
#pragma unroll
                                    for (int m = 0; m < 4; ++m) {
                                        fb[c][e] = fma_t<T>(gz[m * mstr], nw[m][e], fb[c][e]);
                                        x = fma_t<T>(xz[m * mstr], nw[m][e], x);
                                    }
                                    // the end partitions also need nw itself: (nw0, nw1) for partition 0, (nw2, nw3) for P-1
                                    // (selected, not indexed: a run-time index would put nw into local memory)
                                    if (ok && (q == 0 || q == P - 1))
                                        xs[(2 * NC + NHALO + c) * vstr + ix] = (q == 0) ? nw[c][e] : nw[2 + c][e];
                                }
                                if (ok) {
                                    xs[c * vstr + ix] = fb[c][e];
                                    xs[(NC + c) * vstr + ix] = x;
                                }
                            }
                    }
                }
                if constexpr (CL) ++cstep;
                group_sync(a.tpc, sub, tpt);
#pragma unroll
                for (int e = 0; e < V; ++e) {
#pragma unroll
                    for (int c = 0; c < NC; ++c) {
                        G[c][e] = xc[c * vstr + XI(e)];
                        X[c][e] = xc[(NC + c) * vstr + XI(e)];
                    }
                }
            } else {
                // ---- serial form (any P): every thread walks the partitions before / after it ------
                const T *const tb = TAB;
                const int sstr = NC * NC * tq;
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    xc[XI(e)] = v[MR - 1][e];
                    if constexpr (!TRI) xc[vstr + XI(e)] = glast2[e];
                }
                group_sync(a.tpc, sub, tpt);
#pragma unroll
                for (int e = 0; e < V; ++e)
#pragma unroll
                    for (int c = 0; c < NC; ++c) G[c][e] = X[c][e] = T(0);
                for (int q = 0; q < part; ++q) {
                    const T *const xq = xb + (size_t)q * W;
                    const int qsw = q & wm;
                    if constexpr (TRI) {
                        const T ph = tb[q];
#pragma unroll
                        for (int e = 0; e < V; ++e) G[0][e] = fma_t<T>(ph, G[0][e], xq[(sl * V + e) ^ qsw]);
                    } else {
                        const T m0 = tb[q], m1 = tb[tq + q], m2 = tb[2 * tq + q], m3 = tb[3 * tq + q];
#pragma unroll
                        for (int e = 0; e < V; ++e) {
                            const T n1 = fma_t<T>(m1, G[1][e], fma_t<T>(m0, G[0][e], xq[(sl * V + e) ^ qsw]));
                            const T n2 = fma_t<T>(m3, G[1][e], fma_t<T>(m2, G[0][e], xq[vstr + ((sl * V + e) ^ qsw)]));
                            G[0][e] = n1;
                            G[1][e] = n2;
                        }
                    }
                }
                {
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        if constexpr (TRI) {
                            xc[vstr + XI(e)] = fma_t<T>(RBW[0].v[0], G[0][e], v[0][e]);
                        } else {
                            const Pair ch0 = RC0[0], ch1 = RC0[1];  // chi at this partition's first two rows
                            xc[2 * vstr + XI(e)] = fma_t<T>(ch0.v[1], G[1][e], fma_t<T>(ch0.v[0], G[0][e], v[0][e]));
                            xc[3 * vstr + XI(e)] = fma_t<T>(ch1.v[1], G[1][e], fma_t<T>(ch1.v[0], G[0][e], v[1][e]));
                        }
                    }
                }
                group_sync(a.tpc, sub, tpt);
                for (int q = P - 1; q > part; --q) {
                    const T *const xq = xb + (size_t)q * W + NC * vstr;
                    const int qsw = q & wm;
                    const T *const m = tb + sstr + q;
                    if constexpr (TRI) {
                        const T ps = m[0];
#pragma unroll
                        for (int e = 0; e < V; ++e) X[0][e] = fma_t<T>(ps, X[0][e], xq[(sl * V + e) ^ qsw]);
                    } else {
                        const T m0 = m[0], m1 = m[tq], m2 = m[2 * tq], m3 = m[3 * tq];
#pragma unroll
                        for (int e = 0; e < V; ++e) {
                            const T n1 = fma_t<T>(m1, X[1][e], fma_t<T>(m0, X[0][e], xq[(sl * V + e) ^ qsw]));
                            const T n2 = fma_t<T>(m3, X[1][e], fma_t<T>(m2, X[0][e], xq[vstr + ((sl * V + e) ^ qsw)]));
                            X[0][e] = n1;
                            X[1][e] = n2;
                        }
                    }
                }
            }
            // ---- correction: x_k = x^_k + chi_k . G + psi_k . X ------------------------------------
#pragma unroll
            for (int k = 0; k < MR; ++k) {
                if constexpr (TRI) {
                    const Pair cc = RBW[k];
#pragma unroll
                    for (int e = 0; e < V; ++e)
                        v[k][e] = fma_t<T>(X[0][e], cc.v[1], fma_t<T>(G[0][e], cc.v[0], v[k][e]));
                } else {
                    const Pair cc = RC0[k], cs = RC1[k];
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        T x = fma_t<T>(G[0][e], cc.v[0], v[k][e]);
                        x = fma_t<T>(G[1][e], cc.v[1], x);
                        x = fma_t<T>(X[0][e], cs.v[0], x);
                        v[k][e] = fma_t<T>(X[1][e], cs.v[1], x);
                    }
                }
            }
            if constexpr (PERTF) {
                if (part == 0 || part == P - 1) {  // local solve of u in the end partitions
                    const T *const RZ = cb + 5 * MR;
                    T nf[V];
#pragma unroll
                    for (int e = 0; e < V; ++e) nf[e] = xc[(2 * NC + NHALO) * vstr + XI(e)];
#pragma unroll
                    for (int k = 0; k < MR; ++k) {
                        const T zk = RZ[k];
#pragma unroll
                        for (int e = 0; e < V; ++e) v[k][e] = fma_t<T>(nf[e], zk, v[k][e]);
                    }
                }
            }
            if constexpr (WOODF) {
                if (part == 0 || part == P - 1) {  // local solves of the unit vectors at the system's ends
                    T wl0[V], wl1[V];
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        wl0[e] = xc[(2 * NC + NHALO) * vstr + XI(e)];
                        wl1[e] = xc[(2 * NC + NHALO + 1) * vstr + XI(e)];
                    }
                    const Pair *const RZL = reinterpret_cast<const Pair *>(cb + 9 * MR);
#pragma unroll
                    for (int k = 0; k < MR; ++k) {
                        const Pair zl = RZL[k];
#pragma unroll
                        for (int e = 0; e < V; ++e) v[k][e] = fma_t<T>(wl1[e], zl.v[1], fma_t<T>(wl0[e], zl.v[0], v[k][e]));
                    }
                }
            }
#undef XI
        }
        if constexpr (PERT) {
            // ---- eq. 15: x = y - (v.y)/(1 + v.z) z,  v.y = y_1 + v_N y_N ------------------------------
            T y0[V], yN[V];
#pragma unroll
            for (int e = 0; e < V; ++e) { y0[e] = v[0][e]; yN[e] = T(0); }
#pragma unroll
            for (int k = 0; k < MR; ++k)
                if (k == a.last_k) {
#pragma unroll
                    for (int e = 0; e < V; ++e) yN[e] = v[k][e];
                }
            if constexpr (!SINGLE) {
                // y_1 lives in partition 0, y_N in partition last_part: two more exchange planes
                T *const pz = xb + (size_t)(2 * NC + NHALO) * a.P * W + sl * V;
                if (part == 0) {
#pragma unroll
                    for (int e = 0; e < V; ++e) pz[e] = y0[e];
                }
                if (part == a.last_part) {
#pragma unroll
                    for (int e = 0; e < V; ++e) pz[a.P * W + e] = yN[e];
                }
                group_sync(a.tpc, sub, tpt);
#pragma unroll
                for (int e = 0; e < V; ++e) { y0[e] = pz[e]; yN[e] = pz[a.P * W + e]; }
            }
            const T vN = (T)a.per_vN, invden = (T)a.per_invden;
            T nfac[V];
#pragma unroll
            for (int e = 0; e < V; ++e) nfac[e] = -(fma_t<T>(vN, yN[e], y0[e]) * invden);
            const T *const RZ = cb + 5 * MR;
#pragma unroll
            for (int k = 0; k < MR; ++k) {
                const T zk = RZ[k];
#pragma unroll
                for (int e = 0; e < V; ++e) v[k][e] = fma_t<T>(nfac[e], zk, v[k][e]);
            }
        }
        if constexpr (WOOD) {
            // ---- cyclic pentadiagonal: x = y - Z H (V^T y)  (Woodbury; C-31) ------------------
            // V^T y needs y at rows 0, 1, n-2, n-1; their owners publish them to 4 x W exchange values
            T yr[4][V];
#pragma unroll
            for (int m = 0; m < 4; ++m) {
#pragma unroll
                for (int e = 0; e < V; ++e) yr[m][e] = T(0);
                if (SINGLE || part == a.wrow_part[m]) {
#pragma unroll
                    for (int k = 0; k < MR; ++k)
                        if (k == a.wrow_k[m]) {
#pragma unroll
                            for (int e = 0; e < V; ++e) yr[m][e] = v[k][e];
                        }
                }
            }
            if constexpr (!SINGLE) {
                T *const pw = xb + a.xper + sl * V;
#pragma unroll
                for (int m = 0; m < 4; ++m)
                    if (part == a.wrow_part[m]) {
#pragma unroll
                        for (int e = 0; e < V; ++e) pw[m * W + e] = yr[m][e];
                    }
                group_sync(a.tpc, sub, tpt);
#pragma unroll
                for (int m = 0; m < 4; ++m)
#pragma unroll
                    for (int e = 0; e < V; ++e) yr[m][e] = pw[m * W + e];
            }
            T nw[4][V];
#pragma unroll
            for (int e = 0; e < V; ++e) {
                const T t0 = fma_t<T>((T)a.per_w6[1], yr[3][e], (T)a.per_w6[0] * yr[2][e]);
                const T t1 = (T)a.per_w6[2] * yr[3][e];
                const T t2 = (T)a.per_w6[3] * yr[0][e];
                const T t3 = fma_t<T>((T)a.per_w6[5], yr[1][e], (T)a.per_w6[4] * yr[0][e]);
#pragma unroll
                for (int m = 0; m < 4; ++m)
                    nw[m][e] = -fma_t<T>((T)a.per_H[m * 4 + 3], t3, fma_t<T>((T)a.per_H[m * 4 + 2], t2,
                                          fma_t<T>((T)a.per_H[m * 4 + 1], t1, (T)a.per_H[m * 4] * t0)));
            }
            const Pair *const Z01 = reinterpret_cast<const Pair *>(cb + 9 * MR);
            const Pair *const Z23 = reinterpret_cast<const Pair *>(cb + 11 * MR);
#pragma unroll
            for (int k = 0; k < MR; ++k) {
                const Pair za = Z01[k], zb = Z23[k];
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    T x = fma_t<T>(nw[0][e], za.v[0], v[k][e]);
                    x = fma_t<T>(nw[1][e], za.v[1], x);
                    x = fma_t<T>(nw[2][e], zb.v[0], x);
                    v[k][e] = fma_t<T>(nw[3][e], zb.v[1], x);
                }
            }
        }
        if constexpr (ISCH && FUSE) {
            if (a.stat != nullptr) {
                // ---- eq. 30: l = 1 / (1 - <C^2>) of every run after this step, summed over the tile ------
                T s2[V];
#pragma unroll
                for (int e = 0; e < V; ++e) s2[e] = T(0);
#pragma unroll
                for (int k = 0; k < MR; ++k)
#pragma unroll
                    for (int e = 0; e < V; ++e) s2[e] = fma_t<T>(v[k][e], v[k][e], s2[e]);  // padding rows are zero
                double lsum = 0.0;
                const double invn = 1.0 / (double)a.n;
                if constexpr (SINGLE) {
#pragma unroll
                    for (int e = 0; e < V; ++e)
                        if (j + e < batch) lsum += 1.0 / (1.0 - (double)s2[e] * invn);
                } else {
                    // partial sums of the partitions through exchange value 0 (its carries have been consumed)
                    const int hx = part & (W - 1);
#pragma unroll
                    for (int e = 0; e < V; ++e) xb[part * W + ((sl * V + e) ^ hx)] = s2[e];
                    group_sync(a.tpc, sub, tpt);
                    if (part == 0) {
#pragma unroll
                        for (int e = 0; e < V; ++e) {
                            T tot = T(0);
                            for (int q = 0; q < a.P; ++q) tot += xb[q * W + ((sl * V + e) ^ (q & (W - 1)))];
                            if (j + e < batch) lsum += 1.0 / (1.0 - (double)tot * invn);
                        }
                    }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) lsum += __shfl_xor_sync(0xffffffffu, lsum, o);
                if ((threadIdx.x & 31) == 0 && lsum != 0.0) atomicAdd(a.stat + ks, lsum * a.stat_scale);
            }
        }
        if constexpr (HALO1 && !SINGLE) {
            if (ks + 1 < nks) {  // publish this partition's first / last rows: the neighbours' halo of the next step
                const int hv = a.P * W, hx = part & (W - 1);
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    xb[2 * NC * hv + part * W + ((sl * V + e) ^ hx)] = v[0][e];
                    xb[(2 * NC + 1) * hv + part * W + ((sl * V + e) ^ hx)] = v[MR - 1][e];
                    if constexpr (HALO2) {
                        xb[(2 * NC + 2) * hv + part * W + ((sl * V + e) ^ hx)] = v[1][e];
                        xb[(2 * NC + 3) * hv + part * W + ((sl * V + e) ^ hx)] = v[MR - 2][e];
                    }
                }
            }
        }
        }  // ksteps

        // ---- store ---------------------------------------------------------------------------
        if constexpr (TMA) {
            // Kinds with little arithmetic reach the stores while the next tile's load is still streaming in, and the
            // two then slow each other down (measured: tri fp64 N=512, 2^20 systems 0.85 -> 0.93 of the peak with the
            // stores held back; the pentadiagonal kinds arrive later by themselves and lose 0-4 %): wait for the
            // ring's barrier first (the same wait the next iteration starts with; it does not consume the phase).
            if (a.hold_stores && t + stride_tiles < ntiles) mbar_wait(mbar, phase);
        }
        {
            S *ps = p0;
            asm volatile("" : "+l"(ps));  // keep the store addresses from being shared with the loads
            if (nrow == MR) {  // the common case (whole partition, live columns): no per-row predicate
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    st_sys<T, V>(ps, v[k]);
                    ps += batch;
                }
            } else {
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    if (k < nrow) st_sys<T, V>(ps, v[k]);
                    ps += batch;
                }
            }
        }
    }
    if constexpr (CL) cluster_sync();  // no CTA of the pair leaves while the other may still write into it
}
// -----------------------------------------------------------------------------------------------
// Two-pass kernel in the paper's own form (Alg. 2 / Alg. 4: one thread per system, g written to
// global memory by the forward loop and re-read by the backward loop).  Used only when n is too
// large for the register-resident plan, and as the A/B baseline for the ncu comparison
// ("force_two_pass").  Coefficients: SoA arrays of length n in global memory, read through the
// read-only path (every thread reads the same entry).
//   tri   : co[0..n) inv, co[n..2n) nl, co[2n..3n) nch
//   penta : inv, nle, nlb, ngam, ndel
// -----------------------------------------------------------------------------------------------
struct PerPenta {  // scalars of the cyclic pentadiagonal (Woodbury) correction and of the CN explicit half
    double ex[5];  // Crank-Nicolson: explicit stencil, 3 (eq. 9) or 5 values (eq. 18)
    double H[16];  // (I + V^T Z)^{-1}, row-major
    double w6[6];  // wrap-around entries e_0, a_0, e_1, f_{n-2}, c_{n-1}, f_{n-1}
};

// Rows streamed through a thread in a fixed order, a block of 8 rows at a time (16 in fp32 when a row needs at most two coefficients): the loads of the NEXT block are
// issued first (fetch(k) must not depend on a store body() makes for an earlier k), then the coefficients of this
// block (coef(k): read-only path), then body(k, value, coefficients) runs the recurrence and stores.  The compiler
// cannot move a load of rhs above an earlier store to rhs by itself, so without this every row waits for its own
// load; the arithmetic and its order are unchanged.
template <typename T, int NCF>
struct RowCoef {
    T c[NCF];
};
template <typename T, int NCF, typename Fetch, typename Coef, typename Body>
__device__ __forceinline__ void pipelined_rows(int count, Fetch fetch, Coef coef, Body body)
{
    constexpr int TP_U = (sizeof(T) == 4 && NCF < 3) ? 16 : 8;  // (measured: 16 loses with three coefficients per row)
    T cur[TP_U], nxt[TP_U];
#pragma unroll
    for (int u = 0; u < TP_U; ++u) cur[u] = (u < count) ? fetch(u) : T(0);
    for (int k0 = 0; k0 < count; k0 += TP_U) {
#pragma unroll
        for (int u = 0; u < TP_U; ++u) nxt[u] = (k0 + TP_U + u < count) ? fetch(k0 + TP_U + u) : T(0);
        RowCoef<T, NCF> cf[TP_U];
#pragma unroll
        for (int u = 0; u < TP_U; ++u)
            if (k0 + u < count) cf[u] = coef(k0 + u);
#pragma unroll
        for (int u = 0; u < TP_U; ++u)
            if (k0 + u < count) body(k0 + u, cur[u], cf[u]);
#pragma unroll
        for (int u = 0; u < TP_U; ++u) cur[u] = nxt[u];
    }
}

template <typename T, int KIND>
__global__ void __launch_bounds__(128) two_pass_kernel(const T *__restrict__ co, T *rhs, long long batch,
                                                       int n, double alpha_x, double alpha_y, const PerPenta pp)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= batch) return;
    T *p = rhs + j;
    auto row = [&](int r) -> T { return p[(long long)r * batch]; };
    if constexpr (RecLayout<KIND>::TRI) {
        const T *inv = co, *nl = co + n, *nch = co + 2 * (size_t)n;
        T g = T(0);
        if constexpr (KIND == KIND_TRICN || KIND == KIND_TRICNP) {
            // Crank-Nicolson step: explicit three-point half (eq. 9) formed on the fly (row i+1 is still c^n)
            constexpr bool WRAPS = (KIND == KIND_TRICNP);
            const T xa = (T)pp.ex[0], xb = (T)pp.ex[1], xc = (T)pp.ex[2];
            const T c_first = p[0];
            T cprev = WRAPS ? p[(long long)(n - 1) * batch] : T(0), cc = c_first;
            pipelined_rows<T, 2>(n, [&](int k) -> T { return (k + 1 < n) ? row(k + 1) : (WRAPS ? c_first : T(0)); },
                              [&](int i) { return RowCoef<T, 2>{{__ldg(nl + i), __ldg(inv + i)}}; },
                              [&](int i, T cn, const RowCoef<T, 2> &cf) {
                                  const T f = fma_t<T>(xa, cprev, fma_t<T>(xc, cn, xb * cc));
                                  g = fma_t<T>(cf.c[0], g, cf.c[1] * f);
                                  p[(long long)i * batch] = g;
                                  cprev = cc;
                                  cc = cn;
                              });
        } else {
            pipelined_rows<T, 2>(n, row, [&](int i) { return RowCoef<T, 2>{{__ldg(nl + i), __ldg(inv + i)}}; },
                                 [&](int i, T d, const RowCoef<T, 2> &cf) {
                                     g = fma_t<T>(cf.c[0], g, cf.c[1] * d);
                                     p[(long long)i * batch] = g;
                                 });
        }
        T x = g;
        pipelined_rows<T, 1>(n - 1, [&](int k) -> T { return row(n - 2 - k); },
                             [&](int k) { return RowCoef<T, 1>{{__ldg(nch + (n - 2 - k))}}; },
                             [&](int k, T d, const RowCoef<T, 1> &cf) {
                                 x = fma_t<T>(cf.c[0], x, d);
                                 p[(long long)(n - 2 - k) * batch] = x;
                             });
        if constexpr (RecLayout<KIND>::PERT) {
            // eq. 15: alpha_x carries v_N, alpha_y 1/(1 + v.z); z follows nch in co
            const T *z = co + 3 * (size_t)n;
            const T nfac = -(fma_t<T>((T)alpha_x, g, x) * (T)alpha_y);  // x = y_1, g = y_N here
            pipelined_rows<T, 1>(n, row, [&](int i) { return RowCoef<T, 1>{{__ldg(z + i)}}; },
                                 [&](int i, T y, const RowCoef<T, 1> &cf) { p[(long long)i * batch] = fma_t<T>(nfac, cf.c[0], y); });
        }
    } else {
        const T *inv = co, *nle = co + n, *nlb = co + 2 * (size_t)n, *ngam = co + 3 * (size_t)n,
                *ndel = co + 4 * (size_t)n;
        T g1 = T(0), g2 = T(0);
        if constexpr (KIND == KIND_CH || KIND == KIND_CHP) {
            constexpr bool WRAPS = (KIND == KIND_CHP);  // periodic differences: row -1 = row n-1, row n = row 0
            const T ax = (T)alpha_x;
            const T c_first = p[0];
            T wm = WRAPS ? ch_w<T>(p[(long long)(n - 1) * batch]) : T(0), cc = c_first, wc = ch_w<T>(cc);
            pipelined_rows<T, 3>(n, [&](int k) -> T { return (k + 1 < n) ? row(k + 1) : (WRAPS ? c_first : T(0)); },
                              [&](int i) { return RowCoef<T, 3>{{__ldg(nle + i), __ldg(inv + i), __ldg(nlb + i)}}; },
                              [&](int i, T cn, const RowCoef<T, 3> &cf) {
                                  const T wn = ch_w<T>(cn);
                                  T s = wm + wn;
                                  s = fma_t<T>(T(-2), wc, s);
                                  const T f = fma_t<T>(ax, s, cc);
                                  const T t = fma_t<T>(cf.c[0], g2, cf.c[1] * f);
                                  const T g = fma_t<T>(cf.c[2], g1, t);
                                  p[(long long)i * batch] = g;
                                  g2 = g1; g1 = g;
                                  wm = wc; wc = wn; cc = cn;
                              });
        } else if constexpr (KIND == KIND_PENTACN || KIND == KIND_PENTACNP) {
            // Crank-Nicolson hyperdiffusion: explicit five-point half (eq. 18) on the fly (rows i+1, i+2 still c^n)
            constexpr bool WRAPS = (KIND == KIND_PENTACNP);
            const T x0 = (T)pp.ex[0], x1 = (T)pp.ex[1], x2 = (T)pp.ex[2], x3 = (T)pp.ex[3], x4 = (T)pp.ex[4];
            const T c_0 = p[0], c_1 = (n > 1) ? p[batch] : T(0);
            T c2 = WRAPS ? p[(long long)(n - 2) * batch] : T(0), c1 = WRAPS ? p[(long long)(n - 1) * batch] : T(0);
            T cc = c_0, cn1 = c_1;
            pipelined_rows<T, 3>(n, [&](int k) -> T {
                                  const int i2 = k + 2;
                                  return (i2 < n) ? row(i2) : (WRAPS ? (i2 == n ? c_0 : c_1) : T(0));
                              },
                              [&](int i) { return RowCoef<T, 3>{{__ldg(nle + i), __ldg(inv + i), __ldg(nlb + i)}}; },
                              [&](int i, T cn2, const RowCoef<T, 3> &cf) {
                                  T f = fma_t<T>(x1, c1, x0 * c2);
                                  f = fma_t<T>(x2, cc, f);
                                  f = fma_t<T>(x3, cn1, f);
                                  f = fma_t<T>(x4, cn2, f);
                                  const T t = fma_t<T>(cf.c[0], g2, cf.c[1] * f);
                                  const T g = fma_t<T>(cf.c[2], g1, t);
                                  p[(long long)i * batch] = g;
                                  g2 = g1; g1 = g;
                                  c2 = c1; c1 = cc; cc = cn1; cn1 = cn2;
                              });
        } else {
            pipelined_rows<T, 3>(n, row, [&](int i) { return RowCoef<T, 3>{{__ldg(nle + i), __ldg(inv + i), __ldg(nlb + i)}}; },
                                 [&](int i, T d, const RowCoef<T, 3> &cf) {
                                     const T t = fma_t<T>(cf.c[0], g2, cf.c[1] * d);
                                     const T g = fma_t<T>(cf.c[2], g1, t);
                                     p[(long long)i * batch] = g;
                                     g2 = g1; g1 = g;
                                 });
        }
        T x1 = g1, x2 = T(0);
        pipelined_rows<T, 2>(n - 1, [&](int k) -> T { return row(n - 2 - k); },
                             [&](int k) { return RowCoef<T, 2>{{__ldg(ndel + (n - 2 - k)), __ldg(ngam + (n - 2 - k))}}; },
                             [&](int k, T d, const RowCoef<T, 2> &cf) {
                                 const T t = fma_t<T>(cf.c[0], x2, d);
                                 const T x = fma_t<T>(cf.c[1], x1, t);
                                 p[(long long)(n - 2 - k) * batch] = x;
                                 x2 = x1; x1 = x;
                             });
        if constexpr (RecLayout<KIND>::WOOD) {
            // cyclic matrix: x = y - Z H (V^T y) (Woodbury, C-31); Z's four columns follow ndel in co
            const T y0 = p[0], y1 = p[batch], yn2 = p[(long long)(n - 2) * batch], yn1 = p[(long long)(n - 1) * batch];
            const T t0 = fma_t<T>((T)pp.w6[1], yn1, (T)pp.w6[0] * yn2), t1 = (T)pp.w6[2] * yn1, t2 = (T)pp.w6[3] * y0;
            const T t3 = fma_t<T>((T)pp.w6[5], y1, (T)pp.w6[4] * y0);
            T nw[4];
            for (int m = 0; m < 4; ++m)
                nw[m] = -fma_t<T>((T)pp.H[m * 4 + 3], t3, fma_t<T>((T)pp.H[m * 4 + 2], t2,
                                  fma_t<T>((T)pp.H[m * 4 + 1], t1, (T)pp.H[m * 4] * t0)));
            const T *z0 = co + 5 * (size_t)n, *z1 = co + 6 * (size_t)n, *z2 = co + 7 * (size_t)n, *z3 = co + 8 * (size_t)n;
            pipelined_rows<T, 4>(n, row, [&](int i) { return RowCoef<T, 4>{{__ldg(z0 + i), __ldg(z1 + i), __ldg(z2 + i), __ldg(z3 + i)}}; },
                                 [&](int i, T y, const RowCoef<T, 4> &cf) {
                                     T x = fma_t<T>(nw[0], cf.c[0], y);
                                     x = fma_t<T>(nw[1], cf.c[1], x);
                                     x = fma_t<T>(nw[2], cf.c[2], x);
                                     p[(long long)i * batch] = fma_t<T>(nw[3], cf.c[3], x);
                                 });
        }
    }
}

// Coarsening statistic from the state in global memory (one extra read pass; used where no fused CH
// kernel runs: misaligned batches, two-pass plans): stat[0] += scale * sum_j 1 / (1 - mean_i c_ij^2).
template <typename T>
__global__ void __launch_bounds__(128) lbar_kernel(const T *__restrict__ c, long long batch, int n, double *stat,
                                                   double scale)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double l = 0.0;
    if (j < batch) {
        T s2 = T(0);
        for (int i = 0; i < n; ++i) {
            const T x = c[(long long)i * batch + j];
            s2 = fma_t<T>(x, x, s2);
        }
        l = 1.0 / (1.0 - (double)s2 / (double)n);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) l += __shfl_xor_sync(0xffffffffu, l, o);
    if ((threadIdx.x & 31) == 0 && l != 0.0) atomicAdd(stat, l * scale);
}

// launcher table entry (defined by the instantiation units)
typedef cudaError_t (*sweep_launch_fn)(const SweepArgs &, const CUtensorMap &, int grid, int block, size_t smem,
                                       cudaStream_t, int pdl);

struct SweepEntry {
    sweep_launch_fn launch;
    const void *func;  // for cudaFuncSetAttribute / occupancy queries
    int max_threads;   // threads per CTA the kernel was compiled for
    const char *tag;   // the template arguments as profilers print them: "double, 2, 32, 0, 0, 1, 1, 0, 0"
};

template <typename T, int V, int MR, bool SINGLE, int KIND, bool TMA, bool WS, bool FUSE, bool CL = false, typename S = T>
cudaError_t launch_sweep(const SweepArgs &a, const CUtensorMap &tm, int grid, int block, size_t smem,
                         cudaStream_t st, int pdl)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)grid);
    cfg.blockDim = dim3((unsigned)block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute attr[2];
    int na = 0;
    if (CL) {  // a.csz CTAs (SMs) share a tile: grid is a multiple of a.csz
        attr[na].id = cudaLaunchAttributeClusterDimension;
        attr[na].val.clusterDim.x = (unsigned)a.csz;
        attr[na].val.clusterDim.y = 1;
        attr[na].val.clusterDim.z = 1;
        ++na;
    }
    if (pdl) {
        attr[na].id = cudaLaunchAttributeProgrammaticStreamSerialization;
        attr[na].val.programmaticStreamSerializationAllowed = 1;
        ++na;
    }
    cfg.attrs = attr;
    cfg.numAttrs = na;
    return cudaLaunchKernelEx(&cfg, sweep_kernel<T, V, MR, SINGLE, KIND, TMA, WS, FUSE, CL, S>, a, tm);
}

}  // namespace btps
