/*
 * btps.h -- C-ABI of the B200-native batched shared-LHS tridiagonal / pentadiagonal solver
 * (the hot path of arxiv/paper_2107_05395, "A Batched GPU Methodology for Numerical Solutions
 * of PDEs").  One LHS matrix A is factored once on the host; every right-hand side of a huge
 * batch then runs one forward-elimination and one back-substitution sweep, in place.
 *
 * Citations are PAPER.md:<line> (+ section / equation / algorithm).  Readings of garbled or
 * silent passages are listed in DESIGN.md ("Readings", items C-n).
 *
 * Conventions shared by every call
 * --------------------------------
 *  - Layout (Sec. 2; Alg. 2 "rowID +- M"): a batch is ONE array of
 *    n*batch values; element i (0-based row) of system j lives at  rhs[i*batch + j]
 *    ("interleaved").  The solution overwrites the right-hand side.
 *  - "host" pointers are ordinary CPU memory, "device" pointers are CUDA global memory of the
 *    current device.  All pointers are borrowed for the duration of the call only.
 *  - The `stream` argument is a cudaStream_t passed as void* (0 = legacy default stream), e.g.
 *    torch.cuda.current_stream().cuda_stream.  Device-buffer calls only enqueue work on it:
 *    no host synchronisation, no allocation, no host<->device copy.
 *  - Handles are immutable after creation, own their device-side coefficient tables, may be
 *    used from several streams at once, and must be destroyed by the matching *_destroy.
 *    A handle belongs to the CUDA device that was current when it was factored (one process
 *    per GPU sets its device first); using it while another device is current fails with
 *    BTPS_E_DEVICE.
 *  - Status codes: 0 = success, negative = BTPS_E_* below.  The failing call also records the
 *    code (and, for factor failures, the 1-based row of the bad pivot) per host thread; read
 *    it with btps_last_error().
 *  - No pivoting (the paper has none): a zero or non-finite pivot makes the
 *    factor call fail with BTPS_E_PIVOT.
 *  - There is no CPU fallback anywhere: every call that touches a batch needs a CUDA device.
 *  - Numerical behaviour: the kernels evaluate the paper's LU solve (no pivoting) partition-wise -- 32 rows per
 *    thread, carries across partitions by a scan whose multipliers are products of up to 32 elimination multipliers
 *    l_i = a_i / b^_i.  For diagonally dominant A (every benchmark of the paper) |l_i| < 1.  For valid but
 *    non-dominant A those products grow as the rounding error of Alg. 2's own recurrence does; results then agree
 *    with the sequential algorithm to rounding times cond(A), not to the last bits (C-33).
 *  - btps_tune is process-global and not synchronised: set it before the threads that factor and solve start.
 */
#ifndef BTPS_H_
#define BTPS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define BTPS_API __attribute__((visibility("default")))
#else
#define BTPS_API
#endif

#define BTPS_OK 0
#define BTPS_E_ARG (-1)     /* null pointer, n < 1, batch < 1, nsteps < 0, bad handle            */
#define BTPS_E_PIVOT (-2)   /* zero / non-finite pivot in the factorisation (row reported)        */
#define BTPS_E_CUDA (-3)    /* a CUDA runtime call failed (cudaGetLastError text via btps_error_string) */
#define BTPS_E_ALIGN (-4)   /* device pointer not aligned to sizeof(element)                      */
#define BTPS_E_DEVICE (-5)  /* handle used while another CUDA device is current than at its creation */
#define BTPS_E_TOO_LARGE (-6) /* tri_solve_batched_host_static: n * batch * 8 > BTPS_STATIC_SCRATCH_BYTES      */

typedef struct btps_tri_s *tri_handle_t;
typedef struct btps_penta_s *penta_handle_t;

/* ------------------------------------------------------------------------------------------
 * (a1) Tridiagonal factor.  PAPER.md:87-93 (eq. 1-2), 555-566 (Alg. 1), run once on the host
 * (PAPER.md:73).  Row i (0-based):  a[i]*x[i-1] + b[i]*x[i] + c[i]*x[i+1] = rhs[i]
 * (paper's a, b, c).  a, b, c: host, length n; a[0] and c[n-1] are never read.
 * Computes  c^_0 = c_0/b_0;  b^_i = b_i - a_i c^_{i-1};  c^_i = c_i/b^_i  in fp64, derives the
 * sweep tables (reciprocal pivots, l_i = a_i/b^_i, partition response vectors -- DESIGN.md
 * "Partitioned sweep") for fp64 and fp32, and uploads them once.
 * Returns NULL on failure (see btps_last_error).
 * ---------------------------------------------------------------------------------------- */
BTPS_API tri_handle_t tri_factor(int n, const double *a, const double *b, const double *c);
BTPS_API void tri_destroy(tri_handle_t h);

/* ------------------------------------------------------------------------------------------
 * Periodic (cyclic) tridiagonal factor.  PAPER.md:140-164 (Sec. 3.3, eq. 12-15): the matrix of
 * tri_factor plus the two corner entries a[0] (row 0, column n-1) and c[n-1] (row n-1, column 0),
 * i.e. row i is  a[i]*x[(i-1) mod n] + b[i]*x[i] + c[i]*x[(i+1) mod n] = rhs[i].  n >= 3.
 * Sherman-Morrison: A = A' + u (x) v with u = (-b_0, 0, ..., c_{n-1})^T, v = (1, 0, ..., -a_0/b_0)^T;
 * A' (diagonal ends 2 b_0 and b_{n-1} + a_0 c_{n-1} / b_0) is factored as in tri_factor and
 * z = A'^{-1} u is solved once on the host.  The returned handle is used with the same
 * tri_solve_batched[_f32] / tri_solve_steps / tri_solve_batched_host calls: each solve runs the sweeps
 * for A' y = rhs and finishes in the same kernel with x = y - (v.y)/(1 + v.z) z (eq. 15), so HBM still
 * sees one read and one write per element.  Fails with BTPS_E_PIVOT if b_0, a pivot of A' or 1 + v.z
 * is zero / non-finite.
 * ---------------------------------------------------------------------------------------- */
BTPS_API tri_handle_t tri_factor_periodic(int n, const double *a, const double *b, const double *c);

/* ------------------------------------------------------------------------------------------
 * (a3) Pentadiagonal factor A = L R.  PAPER.md:206-256 (Sec. 4.1 steps 1-14), 601-637 (Alg. 3).
 * Row i:  e[i]*x[i-2] + a[i]*x[i-1] + d[i]*x[i] + c[i]*x[i+1] + f[i]*x[i+2] = rhs[i].
 * NOTE the naming: BASELINE.json's (e,a,d,c,f) = the paper's (a,b,c,d,e) of PAPER.md:204.
 * Host arrays of length n; never read: e[0], e[1], a[0], c[n-1], f[n-2], f[n-1].
 * Computes (eps, beta, alpha, gamma, delta) in fp64 by the general-row form of step 8
 * (identical to steps 1-14 for n >= 4, extends to n = 1..3; C-13).
 * ---------------------------------------------------------------------------------------- */
BTPS_API penta_handle_t penta_factor(int n, const double *e, const double *a, const double *d,
                            const double *c, const double *f);
BTPS_API void penta_destroy(penta_handle_t h);

/* ------------------------------------------------------------------------------------------
 * Periodic (cyclic) pentadiagonal factor (eq. 26a): the matrix of penta_factor plus
 * its six wrap-around entries, i.e. row i is  e[i]*x[i-2] + a[i]*x[i-1] + d[i]*x[i] + c[i]*x[i+1] +
 * f[i]*x[i+2]  with indices mod n (e[0], e[1], a[0], c[n-1], f[n-2], f[n-1] ARE read here).  n >= 5.
 * The paper cites [24,4,25] for the method; this library uses the Woodbury identity on the pattern of
 * its Sec. 3.3 (C-31): A = A' + U V^T, Z = A'^{-1} U (4 columns) and H = (I + V^T Z)^{-1}
 * computed once on the host; every solve runs the sweeps for A' y = rhs and finishes in the same kernel
 * with x = y - Z H (V^T y).  The handle is used with penta_solve_batched[_f32], penta_solve_steps,
 * penta_solve_batched_host and with ch_step_batched / ch_step_batched_host, where the explicit half then
 * uses periodic differences too (the paper's own Cahn-Hilliard setting; total mass is
 * conserved, eq. 21-22).
 * ---------------------------------------------------------------------------------------- */
BTPS_API penta_handle_t penta_factor_periodic(int n, const double *e, const double *a, const double *d,
                                     const double *c, const double *f);

/* ------------------------------------------------------------------------------------------
 * (a2)/(a4) Batched sweeps.  Tri: PAPER.md:95-108 (eq. 3-6), 568-597 (Alg. 2).
 * Penta: PAPER.md:258-278 (Sec. 4.1 "g" steps + back-substitution), 639-676 (Alg. 4).
 * d_rhs: DEVICE, n*batch elements, interleaved, solved in place.  Any batch >= 1.
 * Asynchronous on `stream`.  HBM sees one read and one write per element (sweep intermediates
 * stay in registers) unless n exceeds the on-chip plan limit (see btps_plan_info), in which
 * case a two-pass kernel in the paper's own form (2 reads + 2 writes) is used.
 * The *_f32 variants take float data and use the fp32-rounded tables of the same handle.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int tri_solve_batched(tri_handle_t h, double *d_rhs, int64_t batch, void *stream);
BTPS_API int tri_solve_batched_f32(tri_handle_t h, float *d_rhs, int64_t batch, void *stream);
BTPS_API int penta_solve_batched(penta_handle_t h, double *d_rhs, int64_t batch, void *stream);
BTPS_API int penta_solve_batched_f32(penta_handle_t h, float *d_rhs, int64_t batch, void *stream);

/* ------------------------------------------------------------------------------------------
 * The same solves with the batch STORED in fp32 and every sweep COMPUTED in fp64 (storage type /=
 * compute type).  d_rhs: DEVICE, n*batch floats, interleaved, solved in place: each element is read once as a float,
 * widened to double, carried through the forward elimination, back-substitution and carry correction in fp64 registers
 * with the handle's fp64 tables (eq. 3-6 / Sec. 4.1 as above), and rounded to float once when it is stored.  HBM moves
 * half the bytes of the fp64 calls; the result is the fp64 solution of the (exactly representable) float right-hand
 * side, rounded to nearest float -- about 6e-8 relative to each entry, against ~1e-6 for the all-fp32 *_f32 calls.
 * Non-periodic handles with n <= 4096 (the register-resident plans; above 1024 rows, on thread-block clusters, the batch needs
 * 16-byte aligned rows: batch a multiple of 4 and a 16-byte aligned pointer); other handles fail with BTPS_E_ARG.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int tri_solve_batched_f32s(tri_handle_t h, float *d_rhs, int64_t batch, void *stream);
BTPS_API int penta_solve_batched_f32s(penta_handle_t h, float *d_rhs, int64_t batch, void *stream);

/* ------------------------------------------------------------------------------------------
 * (a6) Time-step driver: nsteps successive solves with RHS = previous solution (the paper
 * times "just the time-stepping sections"; implicit diffusion / hyperdiffusion
 * loops PAPER.md:120-136, 288-296, in BASELINE.json's backward-Euler form, C-22).
 * Same arguments as the single solve; nsteps >= 0 launches are enqueued back to back on
 * `stream` with no host synchronisation.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int tri_solve_steps(tri_handle_t h, double *d_rhs, int64_t batch, int nsteps, void *stream);
BTPS_API int penta_solve_steps(penta_handle_t h, double *d_rhs, int64_t batch, int nsteps, void *stream);

/* ------------------------------------------------------------------------------------------
 * Fused Crank-Nicolson diffusion step.  PAPER.md:120-136 (eq. 9-11): per step the right-hand side
 *   f_i = xa*u[i-1] + xb*u[i] + xc*u[i+1]      (eq. 9: xa = xc = sigma_x, xb = 1 - 2*sigma_x)
 * is built in registers and the tridiagonal system of `h` (eq. 11: a = c = -sigma_x, b = 1 + 2*sigma_x,
 * factored by the caller) is solved in the same kernel; nsteps steps, in place, fp64.  With a
 * tri_factor_periodic handle both the stencil and the solve are periodic (the paper's benchmark of
 * Table 1); with a tri_factor handle ghost values are zero.  Same conventions as ch_step_batched.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int tri_cn_step_batched(tri_handle_t h, double *d_u, int64_t batch, double xa, double xb, double xc,
                        int nsteps, void *stream);

/* ------------------------------------------------------------------------------------------
 * Fused Crank-Nicolson hyperdiffusion step.  PAPER.md:284-296 (eq. 17-19): per step
 *   f_i = x5[0]*u[i-2] + x5[1]*u[i-1] + x5[2]*u[i] + x5[3]*u[i+1] + x5[4]*u[i+2]
 * (eq. 18: x5 = (-s, 4s, 1-6s, 4s, -s), s = sigma_x; x5: HOST, 5 doubles) is built in registers and the
 * pentadiagonal system of `h` (s, -4s, 1+6s, -4s, s) solved in the same kernel; nsteps steps, in place,
 * fp64.  Periodic stencil and solve with a penta_factor_periodic handle (the paper's Table 2 benchmark),
 * ghost values zero with a penta_factor handle.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int penta_cn_step_batched(penta_handle_t h, double *d_u, int64_t batch, const double *x5, int nsteps,
                          void *stream);

/* ------------------------------------------------------------------------------------------
 * (a5) Fused semi-implicit Cahn-Hilliard step.  PAPER.md:365-392 (eq. 24, 25a, 26a-c):
 *   (I + sigma*D4) c^{n+1} = c^n + alpha * D2( (c^n)^3 - c^n ),   alpha = dt/dx^2,
 * `h` is the caller's factor of I + sigma*D4; d_c: DEVICE, n*batch fp64, interleaved, advanced nsteps
 * steps in place.  With a penta_factor handle both stencils are truncated (non-periodic), ghost values
 * zero (BASELINE.json config 5; C-18, C-21); with a penta_factor_periodic handle the explicit
 * D2 and the implicit D4 both wrap around (the paper's own setting: total mass is
 * conserved, eq. 21-22).  The RHS is built in registers and swept in the same kernel, up to 64 steps per
 * launch while a tile is on chip (btps_tune "fuse_steps"); nothing but c^n in / c^{n+k} out crosses HBM.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int ch_step_batched(penta_handle_t h, double *d_c, int64_t batch, double alpha, int nsteps,
                    void *stream);

/* ------------------------------------------------------------------------------------------
 * The same steps, recording the coarsening statistic of PAPER.md:433-439 (eq. 30) after every step:
 *   d_lbar[s] = (1/batch) * sum over the runs j of  1 / (1 - <C_j^2>),  <C_j^2> = (1/n) sum_i c[i*batch+j]^2
 * for s = 0 .. nsteps-1 ("captured for each simulation at every time-step and then averaged across
 * simulations").  d_lbar: DEVICE, nsteps doubles, overwritten (zeroed on the stream, then accumulated
 * with atomic adds: the summation order over the runs is not fixed, results agree to rounding).  The sums
 * are formed inside the fused step kernels from the registers that hold c^{n+1}; where no fused kernel
 * runs (unaligned batches, two-pass plans) a separate read pass computes them.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int ch_step_batched_stat(penta_handle_t h, double *d_c, int64_t batch, double alpha, int nsteps,
                         double *d_lbar, void *stream);

/* ------------------------------------------------------------------------------------------
 * End-to-end variants on HOST buffers (the call a user without device code makes).
 * h_rhs / h_c: HOST, n*batch elements, interleaved; pinned memory is used at full speed,
 * pageable memory works but copies slower.  The batch is cut into column chunks; each chunk
 * is copied to the device (strided 2-D copy into its own interleaved buffer), advanced
 * nsteps steps, and copied back, with copies and kernels of different chunks overlapped on
 * internal streams.  Synchronous: returns when h_rhs holds the result.
 * ---------------------------------------------------------------------------------------- */
BTPS_API int tri_solve_batched_host(tri_handle_t h, double *h_rhs, int64_t batch, int nsteps);
BTPS_API int penta_solve_batched_host(penta_handle_t h, double *h_rhs, int64_t batch, int nsteps);
BTPS_API int ch_step_batched_host(penta_handle_t h, double *h_c, int64_t batch, double alpha, int nsteps);

/* ------------------------------------------------------------------------------------------
 * The same solve for callers that must not allocate (code under CUDA graph capture set-up, tight serving loops,
 * harnesses that forbid cudaMalloc): tri_solve_batched_host stages the batch in device buffers it allocates on
 * first use; this variant stages it in a fixed array of BTPS_STATIC_SCRATCH_BYTES bytes that is part of the library
 * image (file-scope `static __device__` in btps.cu; every GPU that loads the library holds those 32 MiB until the
 * process exits).  It calls no cudaMalloc, cudaFree or other allocating routine.
 *   h      : tridiagonal handle (plain or periodic) factored earlier on the current device (the factor call allocates;
 *            this call does not);
 *   h_rhs  : HOST, n*batch doubles, interleaved rhs[i*batch + j]; in: right-hand sides, out: the state after nsteps
 *            solves (RHS = previous solution), exactly what tri_solve_steps gives on a device buffer.
 *            Pinned memory copies at full speed; pageable memory works;
 *   stream : cudaStream_t the copies and kernels are issued on (NULL = default stream).
 * Limit: n * batch * 8 <= BTPS_STATIC_SCRATCH_BYTES (e.g. n = 512: batch <= 8192); larger problems are rejected with
 * BTPS_E_TOO_LARGE before anything is issued (btps_error_string names the sizes).  Synchronous: returns when h_rhs
 * holds the result.  Every call on a device shares the one array, which keeps the previous call's contents: nothing
 * in it has to start at zero (the copy in overwrites all n*batch elements the kernels read), but two calls that
 * overlap on the same GPU -- from two host threads or two processes' worth of streams in one process -- race on it.
 * Serialise them.
 * ---------------------------------------------------------------------------------------- */
#define BTPS_STATIC_SCRATCH_BYTES (32ll << 20)
BTPS_API int tri_solve_batched_host_static(tri_handle_t h, double *h_rhs, int64_t batch, int nsteps, void *stream);

/* ------------------------------------------------------------------------------------------
 * Introspection / tuning (used by tests, bench.py and ncu A/B runs; not needed by callers).
 * ---------------------------------------------------------------------------------------- */

/* Last status recorded on this host thread; *row (may be NULL) = 1-based pivot row or 0. */
BTPS_API int btps_last_error(int *row);
BTPS_API const char *btps_error_string(int code);

/* Kernel plan of a handle for element size `elem_bytes` (8 or 4).  Writes 10 ints to out:
 *   out[0] rows per thread (0 = two-pass kernel), out[1] partitions per system,
 *   out[2] lanes (threads side by side on adjacent systems), out[3] systems per thread,
 *   out[4] tile groups per CTA, out[5] threads per CTA, out[6] dynamic shared memory bytes,
 *   out[7] coefficient table bytes resident on the device for this plan,
 *   out[8] 1 if aligned batches are prefetched by TMA, out[9] 1 if carries use the warp scan.
 * kind: 0 = tri handle, 1 = penta handle (solve kernels), 2 = penta handle (fused CH step kernels),
 * 3 = tri handle (fused Crank-Nicolson step kernels), 4 = penta handle (fused Crank-Nicolson step kernels). */
BTPS_API int btps_plan_info(int kind, const void *handle, int elem_bytes, int *out);

/* Override the plan chosen at factor time (call BEFORE tri_factor / penta_factor; process
 * global).  key is one of "rows" (rows per thread: 32; 8 and 16 only in a library built with BTPS_TUNING_VARIANTS=1,
 * otherwise BTPS_E_ARG), "lanes" (32, 16, 8, 4),
 * "vec" (systems per thread: 1, 2, 4), "tiles_per_cta", "force_two_pass" (0/1), "prefetch"
 * (0: never use the TMA prefetch variant), "warp_scan" (0: serial carry walk), "pdl" (1 / 0: launch with / without the
 * programmatic-dependent-launch attribute; default: with it for batches of at most 128 MiB, where hiding the launch
 * latency gains 3-17 %; larger ones are indifferent or lose), "fuse_steps" (time steps advanced per launch while a tile
 * is on chip in *_solve_steps / ch_step_batched: default and maximum 64, 1 = one launch per step), "grid" (cap on
 * the number of CTAs), "cyclic_in_scan" (0: periodic pentadiagonal handles apply the cyclic correction row by row
 * instead of folding it into the carry scan), "cluster" (1: run every eligible plain solve of 17..32 partitions on clusters of two CTAs
 * that split the rows of a tile, 0: never use cluster kernels -- systems longer than 1024 rows then run the serial carry walk or the
 * two-pass form; default: by the length of a row of the batch in bytes -- tridiagonal with 32 partitions from 512 KiB, 24-31
 * partitions from 4 MiB, 18-23 from 32 MiB; pentadiagonal with 31-32 partitions from 8 MiB; always above 1024 rows; calls that
 * advance 3 or more time steps keep up to 32 partitions on one CTA, which is the faster one per step once the tile stays on chip), "reverse"
 * (0/1: alternate the tile order on successive steps of *_solve_steps / ch_step_batched so a
 * step starts on the data the previous one left in L2), "one_step_fused" (1: one-step calls run the multi-step
 * instantiation of their kernel, 0: the single-step one; default: whichever keeps the smaller local-memory frame),
 * "narrow_loops" (0: fused time loops never switch to half-width tiles; default: launches of 4 or more steps of the plain
 * tridiagonal loop and of the Crank-Nicolson steps with 8-16 partitions and of the Cahn-Hilliard step with 8-12 partitions do, when
 * the partitions share their coefficient blocks -- 2-11 % faster per step, bitwise the same results),
 * "host_chunk_kib" (size in KiB of the column chunks the *_host calls pipeline through the device; default 32768:
 * measured best on B200 / PCIe Gen5, 43.5 GB/s in each direction at once).
 * "hold_stores" (1: a tile's stores wait until the next tile's prefetch has landed, 0: never; default: the kinds
 * and tile sizes where that was measured to win -- tridiagonal kinds and the plain fp64 pentadiagonal solve on full tiles).
 * "blk_pad" (bytes of padding behind every partition's coefficient block in shared memory, a multiple of 16: moves the
 * coefficient reads of the partitions that share a warp onto different banks).
 * "dedupe" (0: every partition keeps its own coefficient block in shared memory; 1: partitions whose blocks are bitwise
 * equal -- all interior partitions of a constant-coefficient LHS -- share one, also for the single-step plain pentadiagonal
 * solve at 32 partitions, which by default keeps an unshared image of its own because it was measured to lose there;
 * default: share.  Results are bitwise identical either way).
 * value < 0 restores the default.  "pdl", "fuse_steps", "grid", "cluster", "reverse", "one_step_fused",
 * "host_chunk_kib" and "hold_stores" are read at launch time, the others ("dedupe" too) when a handle is built. */
BTPS_API int btps_tune(const char *key, int value);

/* Number of kernel launches issued by this library in this process (bench.py's gpu_launches). */
BTPS_API int64_t btps_launch_count(void);

/* Which kernel a call would launch, without launching it: writes into buf (len bytes, NUL-terminated) the template
 * arguments of sweep_kernel<...> exactly as profilers print them ("double, 2, 32, 0, 1, 1, 1, 0, 0, double" = arithmetic
 * type, systems per thread, rows per thread, single partition, kind, TMA prefetch, warp scan, fused steps, cluster
 * split, storage type), or "two_pass_kernel" for the 2R + 2W form.  kind as in btps_plan_info; elem_bytes 8, 4, or 12
 * for the *_f32s calls (4-byte storage, 8-byte arithmetic); batch and nsteps as in the call asked about
 * (the choice depends on the batch's alignment and size and on nsteps > 1); an allocation-aligned base pointer is
 * assumed.  bench.py uses it to check that a committed ncu capture (profiles/) is of the kernels it has just timed. */
BTPS_API int btps_kernel_tag(int kind, const void *handle, int elem_bytes, int64_t batch, int nsteps, char *buf, int len);

/* Identifier of this build of the library: a hash of the kernel sources (csrc/) and compile flags, set by the build script. */
BTPS_API const char *btps_build_id(void);

#ifdef __cplusplus
}
#endif
#endif /* BTPS_H_ */
