// sweep.cuh -- register-resident partitioned sweep kernels (sm_100a).
//
// What is computed (per system, shared LHS):
//   tri   : forward  g_i = (d_i - a_i g_{i-1}) / b^_i         PAPER.md:95-99  (eq. 3-4), Alg. 2
//           backward x_i = g_i - c^_i x_{i+1}                  PAPER.md:101-108 (eq. 5-6), Alg. 2
//   penta : forward  g_i = (f_i - eps_i g_{i-2} - beta_i g_{i-1}) / alpha_i
//           backward x_i = g_i - gamma_i x_{i+1} - delta_i x_{i+2}            PAPER.md:268-278, Alg. 4
//   ch    : f_i = c_i + alpha_x (w_{i-1} - 2 w_i + w_{i+1}), w = c^3 - c, then the penta sweeps
//           PAPER.md:365-392 (eq. 24, 25a, 26c), truncated stencil (C-18, C-21).
//
// How: the paper gives one thread a whole system and writes
// g to global memory between the sweeps (2 reads + 2 writes per element).  Here a tile of W
// adjacent systems is owned by P*lanes threads: thread (part, lane) keeps rows
// [part*MR, part*MR+MR) of V adjacent systems in registers, so HBM sees one read and one
// write per element.  Both recurrences are linear, so each partition sweeps locally with zero
// incoming carries and the true carries are recovered by a short scan over partitions through
// shared memory; because A is shared, the partition response vectors (Phi, chi, Psi) depend
// on the LHS only and are part of the factor tables ("blob") staged into shared memory once
// per CTA.  Divisions are replaced by factor-time reciprocals and the elimination multipliers
// are pre-negated so that each row costs one multiply and FMAs (C-16).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace btps {

enum Kind { KIND_TRI = 0, KIND_PENTA = 1, KIND_CH = 2 };

struct SweepArgs {
    void *rhs;             // device, n*batch elements, interleaved
    const void *blob;      // device coefficient image, 16-B aligned, blob_bytes long
    long long batch;
    long long num_tiles;   // ceil(batch / (lanes*V))
    double alpha_x;        // CH only: dt/dx^2
    int n;                 // true number of rows
    int P;                 // partitions per system (rows padded to P*MR with identity rows)
    int lanes;             // threads side by side on adjacent systems (power of two <= 32)
    int lanes_log2;
    int tpc;               // tiles processed concurrently by one CTA
    int reverse;           // 1: walk the tiles from the last to the first
    unsigned blob_bytes;   // multiple of 16
    unsigned offS;         // byte offset of the per-partition table inside the blob (row records start at 0)
    unsigned offX;         // byte offset of the exchange area in shared memory (after the blob)
};

template <typename T, int N>
struct alignas((sizeof(T) * N) <= 16 ? (sizeof(T) * N) : 16) Tup {
    T v[N];
};

// ---- global memory access for V adjacent systems -------------------------------------------
template <typename T, int V>
__device__ __forceinline__ void ld_sys(T (&d)[V], const T *p)
{
    if constexpr (V == 1) {
        d[0] = *p;
    } else {
        const Tup<T, V> t = *reinterpret_cast<const Tup<T, V> *>(p);
#pragma unroll
        for (int e = 0; e < V; ++e) d[e] = t.v[e];
    }
}

template <typename T, int V>
__device__ __forceinline__ void st_sys(T *p, const T (&s)[V])
{
    if constexpr (V == 1) {
        *p = s[0];
    } else {
        Tup<T, V> t;
#pragma unroll
        for (int e = 0; e < V; ++e) t.v[e] = s[e];
        *reinterpret_cast<Tup<T, V> *>(p) = t;
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

// Coefficient image ("blob"), all in element type T, rows padded to Np = P*MR with identity rows.
// One record per row, made of pairs {T,T} so that one LDS fetches what one phase of a row needs:
//   tri   record = 3 pairs: {inv, nl} {nch, 0} {chi, psi}
//           inv = 1/b^_i, nl = -a_i/b^_i, nch = -c^_i; chi/psi = response of the finished local
//           sweeps to the incoming forward / backward carry
//   penta record = 5 pairs: {inv, nle} {nlb, 0} {ngam, ndel} {chi1, chi2} {psi1, psi2}
//           inv = 1/alpha_i, nle = -eps_i/alpha_i, nlb = -beta_i/alpha_i, ngam = -gamma_i, ndel = -delta_i
// followed at offS by one entry per partition (forward response at the partition's last rows):
//   tri   {phi_last, 0};   penta {phi1_last, phi2_last} {phi1_prev, phi2_prev}
template <int KIND>
struct RecLayout {
    static constexpr int PAIRS = (KIND == KIND_TRI) ? 3 : 5;   // pairs per row record
    static constexpr int SPAIRS = (KIND == KIND_TRI) ? 1 : 2;  // pairs per partition entry
};

template <typename T, int V, int MR, bool SINGLE, int KIND>
__global__ void __launch_bounds__(512, 1) sweep_kernel(const SweepArgs a)
{
    constexpr bool TRI = (KIND == KIND_TRI);
    constexpr int NC = TRI ? 1 : 2;  // carries per direction
    constexpr int RP = RecLayout<KIND>::PAIRS;
    constexpr int SP = RecLayout<KIND>::SPAIRS;
    using Pair = Tup<T, 2>;
    extern __shared__ __align__(16) unsigned char smem[];

    // ---- stage the coefficient image once per CTA ------------------------------------------
    {
        const uint4 *src = reinterpret_cast<const uint4 *>(a.blob);
        uint4 *dst = reinterpret_cast<uint4 *>(smem);
        const unsigned nvec = a.blob_bytes >> 4;
        for (unsigned i = threadIdx.x; i < nvec; i += blockDim.x) dst[i] = __ldg(src + i);
    }
    __syncthreads();

    const int W = a.lanes * V;
    const int tpt = a.P * a.lanes;  // threads per tile
    const int sub = SINGLE ? (threadIdx.x >> a.lanes_log2) : (threadIdx.x / tpt);
    const int lt = SINGLE ? (threadIdx.x & (a.lanes - 1)) : (threadIdx.x - sub * tpt);
    const int part = SINGLE ? 0 : (lt >> a.lanes_log2);
    const int sl = lt & (a.lanes - 1);
    const int r0 = part * MR;
    const long long batch = a.batch;

    const Pair *const Rall = reinterpret_cast<const Pair *>(smem);   // all row records
    const Pair *const R = Rall + (size_t)r0 * RP;                    // this partition's records
    const Pair *const S = reinterpret_cast<const Pair *>(smem + a.offS);
    // exchange area: [tpc][2 (g-last | u-first)][P][NC][W]; this thread's column inside it
    T *const xg = reinterpret_cast<T *>(smem + a.offX) + (size_t)sub * 2 * a.P * NC * W + sl * V;
    const int xu_off = a.P * NC * W;

    const int ntiles = (int)a.num_tiles;
    const int stride_tiles = gridDim.x * a.tpc;
    for (int base = blockIdx.x * a.tpc; base < ntiles; base += stride_tiles) {
        int tile = base + sub;
        const bool tile_ok = tile < ntiles;
        if (a.reverse) tile = ntiles - 1 - tile;
        const long long j = (long long)tile * W + (long long)sl * V;
        const bool act = tile_ok && (j < batch);  // V > 1 requires batch % V == 0
        // rows of this partition that exist and are touched by this thread
        int nrow = a.n - r0;
        nrow = nrow < 0 ? 0 : (nrow > MR ? MR : nrow);
        if (!act) nrow = 0;
        T *const p0 = reinterpret_cast<T *>(a.rhs) + (long long)r0 * batch + j;

        // ---- load: all MR rows issued back to back (independent of the recurrence) ---------
        // (one running row pointer: keeping MR separate 64-bit addresses alive would cost 2*MR registers)
        T v[MR][V];
        {
            const T *pl = p0;
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
        }

        T glast2[V];  // penta: g at the partition's last-but-one row (overwritten by the backward sweep)
        if constexpr (TRI) {
            // ---- local forward sweep, zero incoming carry ---------------------------------
            T gp[V];
#pragma unroll
            for (int e = 0; e < V; ++e) gp[e] = T(0);
#pragma unroll
            for (int k = 0; k < MR; ++k) {
                const Pair cf = R[k * RP + 0];
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
                const T nch = R[k * RP + 1].v[0];
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
            if constexpr (KIND == KIND_CH) {
                // explicit half: f_k = c_k + alpha_x (w_{k-1} - 2 w_k + w_{k+1}); halo rows come
                // from the neighbouring partitions' rows in global memory (still c^n: nobody
                // stores before the barriers below).
                const T ax = (T)a.alpha_x;
                T cm[V], cp[V], wm[V], wc[V];
                if (act && r0 > 0) ld_sys<T, V>(cm, p0 - batch);
                else {
#pragma unroll
                    for (int e = 0; e < V; ++e) cm[e] = T(0);
                }
                if (act && (r0 + MR < a.n)) ld_sys<T, V>(cp, p0 + (long long)MR * batch);
                else {
#pragma unroll
                    for (int e = 0; e < V; ++e) cp[e] = T(0);
                }
#pragma unroll
                for (int e = 0; e < V; ++e) { wm[e] = ch_w<T>(cm[e]); wc[e] = ch_w<T>(v[0][e]); }
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    const Pair cf = R[k * RP + 0];
                    const T nlb = R[k * RP + 1].v[0];
                    const bool row_ok = (k < nrow);
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T wn = ch_w<T>((k + 1 < MR) ? v[(k + 1 < MR) ? k + 1 : k][e] : cp[e]);
                        T s = wm[e] + wn;
                        s = fma_t<T>(T(-2), wc[e], s);
                        T f = fma_t<T>(ax, s, v[k][e]);
                        f = row_ok ? f : T(0);
                        wm[e] = wc[e];
                        wc[e] = wn;
                        const T t = fma_t<T>(cf.v[1], g2[e], cf.v[0] * f);
                        const T g = fma_t<T>(nlb, g1[e], t);
                        v[k][e] = g;
                        g2[e] = g1[e];
                        g1[e] = g;
                    }
                }
            } else {
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    const Pair cf = R[k * RP + 0];
                    const T nlb = R[k * RP + 1].v[0];
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T t = fma_t<T>(cf.v[1], g2[e], cf.v[0] * v[k][e]);
                        const T g = fma_t<T>(nlb, g1[e], t);
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
                const Pair cb = R[k * RP + 2];
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    const T t = fma_t<T>(cb.v[1], g2[e], v[k][e]);
                    const T x = fma_t<T>(cb.v[0], g1[e], t);
                    v[k][e] = x;
                    g2[e] = g1[e];
                    g1[e] = x;
                }
            }
        }

        if constexpr (!SINGLE) {
            const int P = a.P;
            T *const xu = xg + xu_off;
            // ---- publish the local forward result at the partition's end -------------------
            if constexpr (TRI) {
#pragma unroll
                for (int e = 0; e < V; ++e) xg[part * W + e] = v[MR - 1][e];
            } else {
#pragma unroll
                for (int e = 0; e < V; ++e) {
                    xg[(part * 2 + 0) * W + e] = v[MR - 1][e];  // g_{last}  (x^ = g^ there)
                    xg[(part * 2 + 1) * W + e] = glast2[e];     // g_{last-1}
                }
            }
            __syncthreads();
            if constexpr (TRI) {
                // ---- forward carry scan: G_{q+1} = g^last_q + phi_last_q G_q ----------------
                T G[V], X[V];
#pragma unroll
                for (int e = 0; e < V; ++e) G[e] = T(0);
                for (int q = 0; q < part; ++q) {
                    const T ph = S[q].v[0];
#pragma unroll
                    for (int e = 0; e < V; ++e) G[e] = fma_t<T>(ph, G[e], xg[q * W + e]);
                }
                {
                    const T chi0 = R[2].v[0];
#pragma unroll
                    for (int e = 0; e < V; ++e) xu[part * W + e] = fma_t<T>(G[e], chi0, v[0][e]);
                }
                __syncthreads();
                // ---- backward carry scan: X_{q-1} = u_q + psi_first_q X_q -------------------
#pragma unroll
                for (int e = 0; e < V; ++e) X[e] = T(0);
                for (int q = P - 1; q > part; --q) {
                    const T ps = Rall[(size_t)q * MR * RP + 2].v[1];
#pragma unroll
                    for (int e = 0; e < V; ++e) X[e] = fma_t<T>(ps, X[e], xu[q * W + e]);
                }
                // ---- correction ------------------------------------------------------------
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    const Pair cc = R[k * RP + 2];
#pragma unroll
                    for (int e = 0; e < V; ++e)
                        v[k][e] = fma_t<T>(X[e], cc.v[1], fma_t<T>(G[e], cc.v[0], v[k][e]));
                }
            } else {
                T G1[V], G2[V], X1[V], X2[V];
#pragma unroll
                for (int e = 0; e < V; ++e) G1[e] = G2[e] = T(0);
                for (int q = 0; q < part; ++q) {
                    const Pair s0 = S[q * SP + 0], s1 = S[q * SP + 1];
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T a1 = xg[(q * 2 + 0) * W + e];
                        const T a2 = xg[(q * 2 + 1) * W + e];
                        const T n1 = fma_t<T>(s0.v[1], G2[e], fma_t<T>(s0.v[0], G1[e], a1));
                        const T n2 = fma_t<T>(s1.v[1], G2[e], fma_t<T>(s1.v[0], G1[e], a2));
                        G1[e] = n1;
                        G2[e] = n2;
                    }
                }
                {
                    const Pair c0 = R[3], c1 = R[RP + 3];  // chi pairs of the partition's rows 0, 1
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        xu[(part * 2 + 0) * W + e] = fma_t<T>(G2[e], c0.v[1], fma_t<T>(G1[e], c0.v[0], v[0][e]));
                        xu[(part * 2 + 1) * W + e] = fma_t<T>(G2[e], c1.v[1], fma_t<T>(G1[e], c1.v[0], v[1][e]));
                    }
                }
                __syncthreads();
#pragma unroll
                for (int e = 0; e < V; ++e) X1[e] = X2[e] = T(0);
                for (int q = P - 1; q > part; --q) {
                    const Pair p0q = Rall[(size_t)q * MR * RP + 4];        // psi pair, row 0 of partition q
                    const Pair p1q = Rall[(size_t)q * MR * RP + RP + 4];   // psi pair, row 1
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        const T u1 = xu[(q * 2 + 0) * W + e];
                        const T u2 = xu[(q * 2 + 1) * W + e];
                        const T n1 = fma_t<T>(X2[e], p0q.v[1], fma_t<T>(X1[e], p0q.v[0], u1));
                        const T n2 = fma_t<T>(X2[e], p1q.v[1], fma_t<T>(X1[e], p1q.v[0], u2));
                        X1[e] = n1;
                        X2[e] = n2;
                    }
                }
#pragma unroll
                for (int k = 0; k < MR; ++k) {
                    const Pair cc = R[k * RP + 3], cs = R[k * RP + 4];
#pragma unroll
                    for (int e = 0; e < V; ++e) {
                        T x = fma_t<T>(G1[e], cc.v[0], v[k][e]);
                        x = fma_t<T>(G2[e], cc.v[1], x);
                        x = fma_t<T>(X1[e], cs.v[0], x);
                        v[k][e] = fma_t<T>(X2[e], cs.v[1], x);
                    }
                }
            }
        }

        // ---- store ---------------------------------------------------------------------------
        {
            T *ps = p0;
            asm volatile("" : "+l"(ps));  // keep the store addresses from being shared with the loads
#pragma unroll
            for (int k = 0; k < MR; ++k) {
                if (k < nrow) st_sys<T, V>(ps, v[k]);
                ps += batch;
            }
        }
    }
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
template <typename T, int KIND>
__global__ void __launch_bounds__(128) two_pass_kernel(const T *__restrict__ co, T *rhs, long long batch,
                                                       int n, double alpha_x)
{
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= batch) return;
    T *p = rhs + j;
    if constexpr (KIND == KIND_TRI) {
        const T *inv = co, *nl = co + n, *nch = co + 2 * (size_t)n;
        T g = T(0);
        for (int i = 0; i < n; ++i) {
            g = fma_t<T>(__ldg(nl + i), g, __ldg(inv + i) * p[(long long)i * batch]);
            p[(long long)i * batch] = g;
        }
        T x = g;
        for (int i = n - 2; i >= 0; --i) {
            x = fma_t<T>(__ldg(nch + i), x, p[(long long)i * batch]);
            p[(long long)i * batch] = x;
        }
    } else {
        const T *inv = co, *nle = co + n, *nlb = co + 2 * (size_t)n, *ngam = co + 3 * (size_t)n,
                *ndel = co + 4 * (size_t)n;
        T g1 = T(0), g2 = T(0);
        if constexpr (KIND == KIND_CH) {
            const T ax = (T)alpha_x;
            T wm = T(0), cc = p[0], wc = ch_w<T>(cc);
            for (int i = 0; i < n; ++i) {
                const T cn = (i + 1 < n) ? p[(long long)(i + 1) * batch] : T(0);
                const T wn = ch_w<T>(cn);
                T s = wm + wn;
                s = fma_t<T>(T(-2), wc, s);
                const T f = fma_t<T>(ax, s, cc);
                const T t = fma_t<T>(__ldg(nle + i), g2, __ldg(inv + i) * f);
                const T g = fma_t<T>(__ldg(nlb + i), g1, t);
                p[(long long)i * batch] = g;
                g2 = g1; g1 = g;
                wm = wc; wc = wn; cc = cn;
            }
        } else {
            for (int i = 0; i < n; ++i) {
                const T t = fma_t<T>(__ldg(nle + i), g2, __ldg(inv + i) * p[(long long)i * batch]);
                const T g = fma_t<T>(__ldg(nlb + i), g1, t);
                p[(long long)i * batch] = g;
                g2 = g1; g1 = g;
            }
        }
        T x1 = g1, x2 = T(0);
        for (int i = n - 2; i >= 0; --i) {
            const T t = fma_t<T>(__ldg(ndel + i), x2, p[(long long)i * batch]);
            const T x = fma_t<T>(__ldg(ngam + i), x1, t);
            p[(long long)i * batch] = x;
            x2 = x1; x1 = x;
        }
    }
}

// launcher table entry (defined by the instantiation units)
typedef cudaError_t (*sweep_launch_fn)(const SweepArgs &, int grid, int block, size_t smem, cudaStream_t);
typedef const void *(*sweep_func_ptr)(void);

struct SweepEntry {
    sweep_launch_fn launch;
    const void *func;  // for cudaFuncSetAttribute / occupancy queries
};

// kind in {TRI, PENTA, CH}, elem_bytes in {8, 4}, vec in {1, 2}, rows in {8, 16, 32}, single in {0,1}
SweepEntry find_sweep(int kind, int elem_bytes, int vec, int rows, int single);

template <typename T, int V, int MR, bool SINGLE, int KIND>
cudaError_t launch_sweep(const SweepArgs &a, int grid, int block, size_t smem, cudaStream_t st)
{
    sweep_kernel<T, V, MR, SINGLE, KIND><<<grid, block, smem, st>>>(a);
    return cudaGetLastError();
}

}  // namespace btps
