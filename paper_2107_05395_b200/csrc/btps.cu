// btps.cu -- C-ABI (include/btps.h): host factorisation, factor tables, plan selection, kernel
// dispatch, time-step driver and the host-buffer (end-to-end) path.
//
// The host factor routines below are this library's own restatement of the paper's
// pre-factorisation (eq. 1-2 / Alg. 1; Sec. 4.1 / Alg. 3); they
// share no code with oracle/ (the test oracle), which is never linked or loaded from here.
#include "../../include/btps.h"
#include "inst_common.cuh"

#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <vector>

using namespace btps;

namespace {

// ------------------------------------------------------------------------------------------------
// error state
// ------------------------------------------------------------------------------------------------
thread_local int tl_err = BTPS_OK;
thread_local int tl_err_row = 0;
thread_local char tl_cuda_msg[256] = {0};

int set_err(int code, int row = 0)
{
    tl_err = code;
    tl_err_row = row;
    return code;
}

int cuda_fail(cudaError_t e, const char *what)
{
    snprintf(tl_cuda_msg, sizeof(tl_cuda_msg), "%s: %s", what, cudaGetErrorString(e));
    return set_err(BTPS_E_CUDA);
}

#define CU_TRY(call)                                        \
    do {                                                    \
        cudaError_t e__ = (call);                           \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)

std::atomic<long long> g_launches{0};

// ------------------------------------------------------------------------------------------------
// tuning knobs (btps_tune)
// ------------------------------------------------------------------------------------------------
struct Tune {
    int rows = -1, lanes = -1, vec = -1, tpc = -1, force_two_pass = -1, reverse = -1;
};
Tune g_tune;

// ------------------------------------------------------------------------------------------------
// plans
// ------------------------------------------------------------------------------------------------
struct KernelSlot {
    SweepEntry ent = {nullptr, nullptr};
    int vec = 1;
    size_t smem = 0;
    int max_grid = 0;  // occupancy * SM count, resolved at first launch
};

struct DtypePlan {
    int elem = 8;
    int rows = 0, P = 0, lanes = 0, lanes_log2 = 0, vec = 1, tpc = 1, threads = 0;
    bool two_pass = false;
    void *d_blob = nullptr;  // partitioned-sweep coefficient image
    unsigned blob_bytes = 0, offS = 0;
    void *d_soa = nullptr;   // two-pass coefficient arrays
    size_t soa_bytes = 0;
    // [kind slot][0 = vectorised, 1 = scalar tail-safe]; kind slot 0 = solve, 1 = CH (penta only)
    KernelSlot k[2][2];
};

constexpr int MAGIC_TRI = 0x74726931;    // "tri1"
constexpr int MAGIC_PENTA = 0x70656e31;  // "pen1"

struct Handle {
    int magic;
    int kind;  // KIND_TRI / KIND_PENTA
    int n;
    int device;
    DtypePlan plan[2];  // 0: fp64, 1: fp32
    std::mutex mu;      // guards lazy occupancy resolution
};

int ilog2(int v)
{
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

void choose_plan(int n, int elem, DtypePlan &pl)
{
    pl.elem = elem;
    int rows = g_tune.rows > 0 ? g_tune.rows : (n <= 8 ? 8 : (n <= 16 ? 16 : 32));
    if (rows != 8 && rows != 16 && rows != 32) rows = 32;
    int P = (n + rows - 1) / rows;
    int lanes = g_tune.lanes > 0 ? g_tune.lanes : 32;
    if (lanes != 32 && lanes != 16 && lanes != 8 && lanes != 4) lanes = 32;
    while (P * lanes > 512 && lanes > 4) lanes >>= 1;
    pl.two_pass = (P * lanes > 512) || (g_tune.force_two_pass > 0);
    int vec = g_tune.vec > 0 ? g_tune.vec : (elem == 4 ? 2 : 1);
    if (vec != 1 && vec != 2) vec = 1;
    if (rows * vec * elem > 256) vec = 1;  // at most 64 data registers per thread
    int tpc = g_tune.tpc > 0 ? g_tune.tpc : 256 / (P * lanes);
    if (tpc < 1) tpc = 1;
    while (tpc > 1 && tpc * P * lanes > 512) --tpc;
    pl.rows = rows;
    pl.P = P;
    pl.lanes = lanes;
    pl.lanes_log2 = ilog2(lanes);
    pl.vec = vec;
    pl.tpc = tpc;
    pl.threads = tpc * P * lanes;
}

template <typename T>
void put(std::vector<unsigned char> &blob, size_t off, double v)
{
    T t = (T)v;
    memcpy(blob.data() + off, &t, sizeof(T));
}

size_t align16(size_t v) { return (v + 15) & ~(size_t)15; }

// ------------------------------------------------------------------------------------------------
// (a1) tridiagonal factor, PAPER.md:87-93 (eq. 1-2), Alg. 1.  Outputs the sweep multipliers:
//   inv_i = 1/b^_i,  nl_i = -a_i/b^_i  (nl_0 = 0),  nch_i = -c^_i  (nch_{n-1} = 0).
// ------------------------------------------------------------------------------------------------
int factor_tri_host(int n, const double *a, const double *b, const double *c, std::vector<double> &inv,
                    std::vector<double> &nl, std::vector<double> &nch, int *bad_row)
{
    inv.assign(n, 1.0);
    nl.assign(n, 0.0);
    nch.assign(n, 0.0);
    double chat_prev = 0.0;
    for (int i = 0; i < n; ++i) {
        const double bh = (i == 0) ? b[0] : b[i] - a[i] * chat_prev;  // eq. 2
        if (bh == 0.0 || !std::isfinite(bh)) {
            *bad_row = i + 1;
            return BTPS_E_PIVOT;
        }
        inv[i] = 1.0 / bh;
        nl[i] = (i == 0) ? 0.0 : -(a[i] / bh);
        const double chat = (i < n - 1) ? c[i] / bh : 0.0;  // eq. 1-2; c^_N is never used
        nch[i] = -chat;
        chat_prev = chat;
    }
    return BTPS_OK;
}

// ------------------------------------------------------------------------------------------------
// (a3) pentadiagonal factor A = L R, PAPER.md:219-256 (steps 1-14) in general-row form
// (out-of-range gamma, delta are zero; C-13).  API names (e,a,d,c,f) = paper (a,b,c,d,e).
// Outputs: inv = 1/alpha, nle = -eps/alpha, nlb = -beta/alpha, ngam = -gamma, ndel = -delta.
// ------------------------------------------------------------------------------------------------
int factor_penta_host(int n, const double *e, const double *a, const double *d, const double *c,
                      const double *f, std::vector<double> &inv, std::vector<double> &nle,
                      std::vector<double> &nlb, std::vector<double> &ngam, std::vector<double> &ndel,
                      int *bad_row)
{
    inv.assign(n, 1.0);
    nle.assign(n, 0.0);
    nlb.assign(n, 0.0);
    ngam.assign(n, 0.0);
    ndel.assign(n, 0.0);
    std::vector<double> gam(n, 0.0), del(n, 0.0);
    for (int i = 0; i < n; ++i) {
        const double gm1 = (i >= 1) ? gam[i - 1] : 0.0, gm2 = (i >= 2) ? gam[i - 2] : 0.0;
        const double dm1 = (i >= 1) ? del[i - 1] : 0.0, dm2 = (i >= 2) ? del[i - 2] : 0.0;
        const double eps = (i >= 2) ? e[i] : 0.0;                    // step 14
        const double beta = (i >= 1) ? a[i] - eps * gm2 : 0.0;       // steps 4, 8a, 9, 12
        const double alpha = d[i] - eps * dm2 - beta * gm1;          // steps 1, 5, 8b, 10, 13
        if (alpha == 0.0 || !std::isfinite(alpha)) {
            *bad_row = i + 1;
            return BTPS_E_PIVOT;
        }
        gam[i] = (i <= n - 2) ? (c[i] - beta * dm1) / alpha : 0.0;   // steps 2, 6, 8c, 11
        del[i] = (i <= n - 3) ? f[i] / alpha : 0.0;                  // steps 3, 7, 8d
        inv[i] = 1.0 / alpha;
        nle[i] = -(eps / alpha);
        nlb[i] = -(beta / alpha);
        ngam[i] = -gam[i];
        ndel[i] = -del[i];
    }
    return BTPS_OK;
}

// ------------------------------------------------------------------------------------------------
// factor tables for the partitioned sweep; fp64 host arithmetic,
// rounded to T when written into the blob.  Rows are padded to Np = P*rows with identity rows.
// ------------------------------------------------------------------------------------------------
template <typename T>
void build_blob_tri(int n, DtypePlan &pl, const std::vector<double> &inv, const std::vector<double> &nl,
                    const std::vector<double> &nch, std::vector<unsigned char> &blob)
{
    const int MR = pl.rows, P = pl.P, Np = P * MR;
    constexpr int RT = 2 * RecLayout<KIND_TRI>::PAIRS;   // elements per row record
    constexpr int STN = 2 * RecLayout<KIND_TRI>::SPAIRS;  // elements per partition entry
    auto at = [&](const std::vector<double> &v, int i, double pad) { return i < n ? v[i] : pad; };
    pl.offS = (unsigned)align16((size_t)Np * RT * sizeof(T));
    pl.blob_bytes = (unsigned)align16(pl.offS + (size_t)P * STN * sizeof(T));
    blob.assign(pl.blob_bytes, 0);
    std::vector<double> phi(MR), chi(MR), psi(MR);
    for (int p = 0; p < P; ++p) {
        const int r0 = p * MR;
        double prev = 1.0;  // forward response to a unit incoming carry g_{r0-1} = 1
        for (int k = 0; k < MR; ++k) {
            phi[k] = at(nl, r0 + k, 0.0) * prev;
            prev = phi[k];
        }
        double nxt = 1.0, cx = 0.0;  // backward response to x_{r1} = 1; local backward sweep of phi
        for (int k = MR - 1; k >= 0; --k) {
            const double h = at(nch, r0 + k, 0.0);
            psi[k] = h * nxt;
            nxt = psi[k];
            chi[k] = phi[k] + h * cx;
            cx = chi[k];
        }
        for (int k = 0; k < MR; ++k) {
            const int i = r0 + k;
            const size_t r = (size_t)i * RT * sizeof(T);
            put<T>(blob, r + 0 * sizeof(T), at(inv, i, 1.0));
            put<T>(blob, r + 1 * sizeof(T), at(nl, i, 0.0));
            put<T>(blob, r + 2 * sizeof(T), at(nch, i, 0.0));
            put<T>(blob, r + 3 * sizeof(T), 0.0);
            put<T>(blob, r + 4 * sizeof(T), chi[k]);
            put<T>(blob, r + 5 * sizeof(T), psi[k]);
        }
        put<T>(blob, pl.offS + ((size_t)p * STN + 0) * sizeof(T), phi[MR - 1]);
        put<T>(blob, pl.offS + ((size_t)p * STN + 1) * sizeof(T), 0.0);
    }
}

template <typename T>
void build_blob_penta(int n, DtypePlan &pl, const std::vector<double> &inv, const std::vector<double> &nle,
                      const std::vector<double> &nlb, const std::vector<double> &ngam,
                      const std::vector<double> &ndel, std::vector<unsigned char> &blob)
{
    const int MR = pl.rows, P = pl.P, Np = P * MR;
    constexpr int RT = 2 * RecLayout<KIND_PENTA>::PAIRS;
    constexpr int STN = 2 * RecLayout<KIND_PENTA>::SPAIRS;
    auto at = [&](const std::vector<double> &v, int i, double pad) { return i < n ? v[i] : pad; };
    pl.offS = (unsigned)align16((size_t)Np * RT * sizeof(T));
    pl.blob_bytes = (unsigned)align16(pl.offS + (size_t)P * STN * sizeof(T));
    blob.assign(pl.blob_bytes, 0);
    std::vector<double> phi[2], chi[2], psi[2];
    for (int t = 0; t < 2; ++t) {
        phi[t].resize(MR);
        chi[t].resize(MR);
        psi[t].resize(MR);
    }
    for (int p = 0; p < P; ++p) {
        const int r0 = p * MR;
        for (int t = 0; t < 2; ++t) {
            // forward response to a unit carry: t = 0: g_{r0-1} = 1; t = 1: g_{r0-2} = 1
            double p1 = (t == 0) ? 1.0 : 0.0, p2 = (t == 0) ? 0.0 : 1.0;
            for (int k = 0; k < MR; ++k) {
                const double g = at(nlb, r0 + k, 0.0) * p1 + at(nle, r0 + k, 0.0) * p2;
                phi[t][k] = g;
                p2 = p1;
                p1 = g;
            }
            // backward response to a unit carry: t = 0: x_{r1} = 1; t = 1: x_{r1+1} = 1
            double n1 = (t == 0) ? 1.0 : 0.0, n2 = (t == 0) ? 0.0 : 1.0;
            double c1 = 0.0, c2 = 0.0;
            for (int k = MR - 1; k >= 0; --k) {
                const double gm = at(ngam, r0 + k, 0.0), dl = at(ndel, r0 + k, 0.0);
                const double x = gm * n1 + dl * n2;
                psi[t][k] = x;
                n2 = n1;
                n1 = x;
                const double cx = phi[t][k] + gm * c1 + dl * c2;  // local backward sweep of phi
                chi[t][k] = cx;
                c2 = c1;
                c1 = cx;
            }
        }
        for (int k = 0; k < MR; ++k) {
            const int i = r0 + k;
            const size_t r = (size_t)i * RT * sizeof(T);
            put<T>(blob, r + 0 * sizeof(T), at(inv, i, 1.0));
            put<T>(blob, r + 1 * sizeof(T), at(nle, i, 0.0));
            put<T>(blob, r + 2 * sizeof(T), at(nlb, i, 0.0));
            put<T>(blob, r + 3 * sizeof(T), 0.0);
            put<T>(blob, r + 4 * sizeof(T), at(ngam, i, 0.0));
            put<T>(blob, r + 5 * sizeof(T), at(ndel, i, 0.0));
            put<T>(blob, r + 6 * sizeof(T), chi[0][k]);
            put<T>(blob, r + 7 * sizeof(T), chi[1][k]);
            put<T>(blob, r + 8 * sizeof(T), psi[0][k]);
            put<T>(blob, r + 9 * sizeof(T), psi[1][k]);
        }
        const size_t sOff = pl.offS + (size_t)p * STN * sizeof(T);
        put<T>(blob, sOff + 0 * sizeof(T), phi[0][MR - 1]);
        put<T>(blob, sOff + 1 * sizeof(T), phi[1][MR - 1]);
        put<T>(blob, sOff + 2 * sizeof(T), phi[0][MR - 2]);
        put<T>(blob, sOff + 3 * sizeof(T), phi[1][MR - 2]);
    }
}

template <typename T>
void build_soa(const std::vector<const std::vector<double> *> &arrs, int n, std::vector<unsigned char> &out)
{
    out.assign(arrs.size() * (size_t)n * sizeof(T), 0);
    for (size_t k = 0; k < arrs.size(); ++k)
        for (int i = 0; i < n; ++i) put<T>(out, (k * (size_t)n + i) * sizeof(T), (*arrs[k])[i]);
}

int upload(const std::vector<unsigned char> &src, void **dst)
{
    *dst = nullptr;
    CU_TRY(cudaMalloc(dst, src.size() ? src.size() : 16));
    CU_TRY(cudaMemcpy(*dst, src.data(), src.size(), cudaMemcpyHostToDevice));
    return BTPS_OK;
}

void free_handle(Handle *h)
{
    if (!h) return;
    for (int t = 0; t < 2; ++t) {
        if (h->plan[t].d_blob) cudaFree(h->plan[t].d_blob);
        if (h->plan[t].d_soa) cudaFree(h->plan[t].d_soa);
    }
    h->magic = 0;
    delete h;
}

size_t slot_smem(const DtypePlan &pl, int kind, int vec)
{
    const int NC = (kind == KIND_TRI) ? 1 : 2;
    const size_t W = (size_t)pl.lanes * vec;
    const size_t xch = (pl.P > 1) ? (size_t)pl.tpc * 2 * pl.P * NC * W * pl.elem : 0;
    return (size_t)pl.blob_bytes + xch;
}

// The partitioned plan keeps the whole coefficient image plus the exchange area in shared memory;
// beyond the per-CTA limit of sm_100a (227 KB) the handle falls back to the two-pass kernel.
constexpr size_t SMEM_LIMIT = 227 * 1024;

void fit_plan(DtypePlan &pl, int handle_kind)
{
    if (pl.two_pass) return;
    if (slot_smem(pl, handle_kind, pl.vec) > SMEM_LIMIT) pl.vec = 1;
    if (slot_smem(pl, handle_kind, pl.vec) > SMEM_LIMIT) pl.two_pass = true;
}

void fill_slots(Handle *h)
{
    for (int t = 0; t < 2; ++t) {
        DtypePlan &pl = h->plan[t];
        if (pl.two_pass) continue;
        const int single = (pl.P == 1) ? 1 : 0;
        for (int ks = 0; ks < 2; ++ks) {
            int kind;
            if (h->kind == KIND_TRI) {
                if (ks == 1) continue;
                kind = KIND_TRI;
            } else {
                kind = (ks == 0) ? KIND_PENTA : KIND_CH;
            }
            for (int s = 0; s < 2; ++s) {
                const int vec = (s == 0) ? pl.vec : 1;
                KernelSlot &sl = pl.k[ks][s];
                sl.vec = vec;
                if (kind == KIND_TRI) sl.ent = find_sweep_tri(pl.elem, vec, pl.rows, single);
                else if (kind == KIND_PENTA) sl.ent = find_sweep_penta(pl.elem, vec, pl.rows, single);
                else sl.ent = find_sweep_ch(pl.elem, vec, pl.rows, single);
                sl.smem = slot_smem(pl, kind, vec);
                sl.max_grid = 0;
            }
        }
    }
}

int resolve_slot(Handle *h, const DtypePlan &pl, KernelSlot &sl)
{
    std::lock_guard<std::mutex> lk(h->mu);
    if (sl.max_grid > 0) return BTPS_OK;
    if (!sl.ent.func) return set_err(BTPS_E_ARG);
    if (sl.smem > 48 * 1024)
        CU_TRY(cudaFuncSetAttribute(sl.ent.func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sl.smem));
    int occ = 0, sms = 0, dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sl.ent.func, pl.threads, sl.smem));
    if (occ < 1) {
        snprintf(tl_cuda_msg, sizeof(tl_cuda_msg), "kernel does not fit: %d threads, %zu B smem", pl.threads,
                 sl.smem);
        return set_err(BTPS_E_CUDA);
    }
    sl.max_grid = occ * sms;
    return BTPS_OK;
}

// one sweep launch (kind = KIND_TRI / KIND_PENTA / KIND_CH) on a device buffer
template <typename T>
int launch_one(Handle *h, int kind, T *d_rhs, long long batch, double alpha_x, int reverse, cudaStream_t st)
{
    DtypePlan &pl = h->plan[sizeof(T) == 8 ? 0 : 1];
    if (pl.two_pass) {
        const int block = 128;
        const long long grid = (batch + block - 1) / block;
        if (kind == KIND_TRI)
            two_pass_kernel<T, KIND_TRI><<<(unsigned)grid, block, 0, st>>>((const T *)pl.d_soa, d_rhs, batch, h->n, 0.0);
        else if (kind == KIND_PENTA)
            two_pass_kernel<T, KIND_PENTA><<<(unsigned)grid, block, 0, st>>>((const T *)pl.d_soa, d_rhs, batch, h->n, 0.0);
        else
            two_pass_kernel<T, KIND_CH><<<(unsigned)grid, block, 0, st>>>((const T *)pl.d_soa, d_rhs, batch, h->n, alpha_x);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        CU_TRY(cudaGetLastError());
        return BTPS_OK;
    }
    const int ks = (kind == KIND_CH) ? 1 : 0;
    // the vectorised kernel needs whole vectors: batch % vec == 0 and an aligned base pointer
    int s = 0;
    if (pl.vec > 1) {
        const bool ok = (batch % pl.vec == 0) && (((uintptr_t)d_rhs % (sizeof(T) * pl.vec)) == 0);
        if (!ok) s = 1;
    }
    KernelSlot &sl = pl.k[ks][s];
    if (sl.max_grid == 0) {
        const int rc = resolve_slot(h, pl, sl);
        if (rc != BTPS_OK) return rc;
    }
    SweepArgs a;
    a.rhs = d_rhs;
    a.blob = pl.d_blob;
    a.batch = batch;
    const long long W = (long long)pl.lanes * sl.vec;
    a.num_tiles = (batch + W - 1) / W;
    a.alpha_x = alpha_x;
    a.n = h->n;
    a.P = pl.P;
    a.lanes = pl.lanes;
    a.lanes_log2 = pl.lanes_log2;
    a.tpc = pl.tpc;
    a.reverse = reverse;
    a.blob_bytes = pl.blob_bytes;
    a.offS = pl.offS;
    a.offX = pl.blob_bytes;
    long long grid = (a.num_tiles + pl.tpc - 1) / pl.tpc;
    if (grid > sl.max_grid) grid = sl.max_grid;
    const cudaError_t e = sl.ent.launch(a, (int)grid, pl.threads, sl.smem, st);
    g_launches.fetch_add(1, std::memory_order_relaxed);
    if (e != cudaSuccess) return cuda_fail(e, "sweep launch");
    return BTPS_OK;
}

Handle *check(const void *hv, int magic)
{
    Handle *h = (Handle *)hv;
    if (!h || h->magic != magic) return nullptr;
    return h;
}

template <typename T>
int solve_steps(const void *hv, int magic, int kind, T *d_rhs, int64_t batch, double alpha_x, int nsteps,
                void *stream)
{
    Handle *h = check(hv, magic);
    if (!h || !d_rhs || batch < 1 || nsteps < 0) return set_err(BTPS_E_ARG);
    if ((uintptr_t)d_rhs % sizeof(T)) return set_err(BTPS_E_ALIGN);
    const bool rev = g_tune.reverse > 0;
    for (int s = 0; s < nsteps; ++s) {
        const int rc = launch_one<T>(h, kind, d_rhs, batch, alpha_x, rev ? (s & 1) : 0, (cudaStream_t)stream);
        if (rc != BTPS_OK) return rc;
    }
    return set_err(BTPS_OK);
}

// ------------------------------------------------------------------------------------------------
// host-buffer path: column chunks, 3 streams, strided 2-D copies in and out
// ------------------------------------------------------------------------------------------------
struct HostPipe {
    std::mutex mu;
    static constexpr int NBUF = 3;
    cudaStream_t st[NBUF] = {nullptr, nullptr, nullptr};
    void *buf[NBUF] = {nullptr, nullptr, nullptr};
    size_t cap = 0;
    bool ready = false;
};
HostPipe g_pipe;

int pipe_prepare(size_t bytes)
{
    if (!g_pipe.ready) {
        for (int i = 0; i < HostPipe::NBUF; ++i) CU_TRY(cudaStreamCreateWithFlags(&g_pipe.st[i], cudaStreamNonBlocking));
        g_pipe.ready = true;
    }
    if (bytes > g_pipe.cap) {
        for (int i = 0; i < HostPipe::NBUF; ++i) {
            if (g_pipe.buf[i]) CU_TRY(cudaFree(g_pipe.buf[i]));
            g_pipe.buf[i] = nullptr;
        }
        g_pipe.cap = 0;
        for (int i = 0; i < HostPipe::NBUF; ++i) CU_TRY(cudaMalloc(&g_pipe.buf[i], bytes));
        g_pipe.cap = bytes;
    }
    return BTPS_OK;
}

template <typename T>
int solve_host(const void *hv, int magic, int kind, T *h_rhs, int64_t batch, double alpha_x, int nsteps)
{
    Handle *h = check(hv, magic);
    if (!h || !h_rhs || batch < 1 || nsteps < 0) return set_err(BTPS_E_ARG);
    std::lock_guard<std::mutex> lk(g_pipe.mu);
    const int n = h->n;
    // chunk width: about 32 MiB per chunk, a multiple of 256 systems, at least 4 chunks when possible
    long long wc = (long long)((32ull << 20) / ((size_t)n * sizeof(T)));
    wc = (wc / 256) * 256;
    if (wc < 256) wc = 256;
    if (wc > batch) wc = batch;
    const size_t chunk_bytes = (size_t)n * wc * sizeof(T);
    int rc = pipe_prepare(chunk_bytes);
    if (rc != BTPS_OK) return rc;
    const bool rev = g_tune.reverse > 0;
    int ci = 0;
    for (long long j0 = 0; j0 < batch; j0 += wc, ++ci) {
        const long long w = (batch - j0 < wc) ? (batch - j0) : wc;
        const int b = ci % HostPipe::NBUF;
        cudaStream_t st = g_pipe.st[b];
        T *d = (T *)g_pipe.buf[b];
        CU_TRY(cudaMemcpy2DAsync(d, (size_t)w * sizeof(T), h_rhs + j0, (size_t)batch * sizeof(T),
                                 (size_t)w * sizeof(T), (size_t)n, cudaMemcpyHostToDevice, st));
        for (int s = 0; s < nsteps; ++s) {
            rc = launch_one<T>(h, kind, d, w, alpha_x, rev ? (s & 1) : 0, st);
            if (rc != BTPS_OK) return rc;
        }
        CU_TRY(cudaMemcpy2DAsync(h_rhs + j0, (size_t)batch * sizeof(T), d, (size_t)w * sizeof(T),
                                 (size_t)w * sizeof(T), (size_t)n, cudaMemcpyDeviceToHost, st));
    }
    for (int i = 0; i < HostPipe::NBUF; ++i) CU_TRY(cudaStreamSynchronize(g_pipe.st[i]));
    return set_err(BTPS_OK);
}

}  // namespace

// ================================================================================================
// exported C-ABI
// ================================================================================================
extern "C" {

tri_handle_t tri_factor(int n, const double *a, const double *b, const double *c)
{
    if (n < 1 || !a || !b || !c) {
        set_err(BTPS_E_ARG);
        return nullptr;
    }
    std::vector<double> inv, nl, nch;
    int row = 0;
    if (factor_tri_host(n, a, b, c, inv, nl, nch, &row) != BTPS_OK) {
        set_err(BTPS_E_PIVOT, row);
        return nullptr;
    }
    Handle *h = new Handle();
    h->magic = MAGIC_TRI;
    h->kind = KIND_TRI;
    h->n = n;
    h->device = 0;
    for (int t = 0; t < 2; ++t) {
        DtypePlan &pl = h->plan[t];
        choose_plan(n, t == 0 ? 8 : 4, pl);
        std::vector<unsigned char> blob, soa;
        if (t == 0) {
            build_blob_tri<double>(n, pl, inv, nl, nch, blob);
            build_soa<double>({&inv, &nl, &nch}, n, soa);
        } else {
            build_blob_tri<float>(n, pl, inv, nl, nch, blob);
            build_soa<float>({&inv, &nl, &nch}, n, soa);
        }
        pl.soa_bytes = soa.size();
        fit_plan(pl, h->kind);
        if (upload(blob, &pl.d_blob) != BTPS_OK || upload(soa, &pl.d_soa) != BTPS_OK) {
            free_handle(h);
            return nullptr;
        }
    }
    fill_slots(h);
    set_err(BTPS_OK);
    return (tri_handle_t)h;
}

void tri_destroy(tri_handle_t hv)
{
    Handle *h = check(hv, MAGIC_TRI);
    if (h) free_handle(h);
}

penta_handle_t penta_factor(int n, const double *e, const double *a, const double *d, const double *c,
                            const double *f)
{
    if (n < 1 || !e || !a || !d || !c || !f) {
        set_err(BTPS_E_ARG);
        return nullptr;
    }
    std::vector<double> inv, nle, nlb, ngam, ndel;
    int row = 0;
    if (factor_penta_host(n, e, a, d, c, f, inv, nle, nlb, ngam, ndel, &row) != BTPS_OK) {
        set_err(BTPS_E_PIVOT, row);
        return nullptr;
    }
    Handle *h = new Handle();
    h->magic = MAGIC_PENTA;
    h->kind = KIND_PENTA;
    h->n = n;
    h->device = 0;
    for (int t = 0; t < 2; ++t) {
        DtypePlan &pl = h->plan[t];
        choose_plan(n, t == 0 ? 8 : 4, pl);
        std::vector<unsigned char> blob, soa;
        if (t == 0) {
            build_blob_penta<double>(n, pl, inv, nle, nlb, ngam, ndel, blob);
            build_soa<double>({&inv, &nle, &nlb, &ngam, &ndel}, n, soa);
        } else {
            build_blob_penta<float>(n, pl, inv, nle, nlb, ngam, ndel, blob);
            build_soa<float>({&inv, &nle, &nlb, &ngam, &ndel}, n, soa);
        }
        pl.soa_bytes = soa.size();
        fit_plan(pl, h->kind);
        if (upload(blob, &pl.d_blob) != BTPS_OK || upload(soa, &pl.d_soa) != BTPS_OK) {
            free_handle(h);
            return nullptr;
        }
    }
    fill_slots(h);
    set_err(BTPS_OK);
    return (penta_handle_t)h;
}

void penta_destroy(penta_handle_t hv)
{
    Handle *h = check(hv, MAGIC_PENTA);
    if (h) free_handle(h);
}

int tri_solve_batched(tri_handle_t h, double *d_rhs, int64_t batch, void *stream)
{
    return solve_steps<double>(h, MAGIC_TRI, KIND_TRI, d_rhs, batch, 0.0, 1, stream);
}
int tri_solve_batched_f32(tri_handle_t h, float *d_rhs, int64_t batch, void *stream)
{
    return solve_steps<float>(h, MAGIC_TRI, KIND_TRI, d_rhs, batch, 0.0, 1, stream);
}
int penta_solve_batched(penta_handle_t h, double *d_rhs, int64_t batch, void *stream)
{
    return solve_steps<double>(h, MAGIC_PENTA, KIND_PENTA, d_rhs, batch, 0.0, 1, stream);
}
int penta_solve_batched_f32(penta_handle_t h, float *d_rhs, int64_t batch, void *stream)
{
    return solve_steps<float>(h, MAGIC_PENTA, KIND_PENTA, d_rhs, batch, 0.0, 1, stream);
}
int tri_solve_steps(tri_handle_t h, double *d_rhs, int64_t batch, int nsteps, void *stream)
{
    return solve_steps<double>(h, MAGIC_TRI, KIND_TRI, d_rhs, batch, 0.0, nsteps, stream);
}
int penta_solve_steps(penta_handle_t h, double *d_rhs, int64_t batch, int nsteps, void *stream)
{
    return solve_steps<double>(h, MAGIC_PENTA, KIND_PENTA, d_rhs, batch, 0.0, nsteps, stream);
}
int ch_step_batched(penta_handle_t h, double *d_c, int64_t batch, double alpha, int nsteps, void *stream)
{
    return solve_steps<double>(h, MAGIC_PENTA, KIND_CH, d_c, batch, alpha, nsteps, stream);
}

int tri_solve_batched_host(tri_handle_t h, double *h_rhs, int64_t batch, int nsteps)
{
    return solve_host<double>(h, MAGIC_TRI, KIND_TRI, h_rhs, batch, 0.0, nsteps);
}
int penta_solve_batched_host(penta_handle_t h, double *h_rhs, int64_t batch, int nsteps)
{
    return solve_host<double>(h, MAGIC_PENTA, KIND_PENTA, h_rhs, batch, 0.0, nsteps);
}
int ch_step_batched_host(penta_handle_t h, double *h_c, int64_t batch, double alpha, int nsteps)
{
    return solve_host<double>(h, MAGIC_PENTA, KIND_CH, h_c, batch, alpha, nsteps);
}

int btps_last_error(int *row)
{
    if (row) *row = tl_err_row;
    return tl_err;
}

const char *btps_error_string(int code)
{
    switch (code) {
        case BTPS_OK: return "ok";
        case BTPS_E_ARG: return "bad argument (null pointer, n < 1, batch < 1, nsteps < 0 or bad handle)";
        case BTPS_E_PIVOT: return "zero or non-finite pivot (no pivoting; see btps_last_error row)";
        case BTPS_E_CUDA: return tl_cuda_msg[0] ? tl_cuda_msg : "CUDA runtime failure";
        case BTPS_E_ALIGN: return "device pointer not aligned to the element size";
        default: return "unknown";
    }
}

int btps_plan_info(int kind, const void *handle, int elem_bytes, int *out)
{
    Handle *h = check(handle, kind == 0 ? MAGIC_TRI : MAGIC_PENTA);
    if (!h || !out || (elem_bytes != 8 && elem_bytes != 4)) return set_err(BTPS_E_ARG);
    const DtypePlan &pl = h->plan[elem_bytes == 8 ? 0 : 1];
    out[0] = pl.two_pass ? 0 : pl.rows;
    out[1] = pl.two_pass ? 1 : pl.P;
    out[2] = pl.two_pass ? 128 : pl.lanes;
    out[3] = pl.two_pass ? 1 : pl.vec;
    out[4] = pl.two_pass ? 1 : pl.tpc;
    out[5] = pl.two_pass ? 128 : pl.threads;
    out[6] = pl.two_pass ? 0 : (int)pl.k[0][0].smem;
    out[7] = pl.two_pass ? (int)pl.soa_bytes : (int)pl.blob_bytes;
    return set_err(BTPS_OK);
}

int btps_tune(const char *key, int value)
{
    if (!key) return set_err(BTPS_E_ARG);
    if (!strcmp(key, "rows")) g_tune.rows = value;
    else if (!strcmp(key, "lanes")) g_tune.lanes = value;
    else if (!strcmp(key, "vec")) g_tune.vec = value;
    else if (!strcmp(key, "tiles_per_cta")) g_tune.tpc = value;
    else if (!strcmp(key, "force_two_pass")) g_tune.force_two_pass = value;
    else if (!strcmp(key, "reverse")) g_tune.reverse = value;
    else return set_err(BTPS_E_ARG);
    return set_err(BTPS_OK);
}

int64_t btps_launch_count(void) { return (int64_t)g_launches.load(std::memory_order_relaxed); }

}  // extern "C"
