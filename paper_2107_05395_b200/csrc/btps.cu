// btps.cu -- C-ABI (include/btps.h): host factorisation, factor tables, plan selection, kernel
// dispatch, time-step driver and the host-buffer (end-to-end) path.
//
// The host factor routines below are this library's own restatement of the paper's
// pre-factorisation (eq. 1-2 / Alg. 1; Sec. 4.1 / Alg. 3); they
// share no code with oracle/ (the test oracle), which is never linked or loaded from here.
#include "../../include/btps.h"
#include "inst_common.cuh"

#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <map>
#include <mutex>
#include <type_traits>
#include <vector>

using namespace btps;

namespace {

// ------------------------------------------------------------------------------------------------
// error state
// ------------------------------------------------------------------------------------------------
thread_local int tl_err = BTPS_OK;
thread_local int tl_err_row = 0;
thread_local char tl_cuda_msg[256] = {0};
thread_local char tl_size_msg[320] = {0};

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
    int rows = -1, lanes = -1, vec = -1, tpc = -1, force_two_pass = -1, reverse = -1, prefetch = -1, pdl = -1,
        warp_scan = -1, grid = -1, fuse = -1, cluster = -1, blk_pad = -1, cyclic_scan = -1, one_step_fused = -1, host_chunk_kib = -1, hold_stores = -1, dedupe = -1, narrow = -1;
};
Tune g_tune;

// ------------------------------------------------------------------------------------------------
// plans
// ------------------------------------------------------------------------------------------------
struct KernelSlot {
    SweepEntry ent = {nullptr, nullptr, 0};
    SweepEntry fused = {nullptr, nullptr, 0};  // multi-step form of the same variant (TMA variants)
    int prefer_fused = 0;  // the fused instantiation spills less than the single-step one: use it for one step too
    int vec = 1;
    int tma = 0;       // 1: the TMA-prefetch variant (needs the ring in shared memory)
    int xvals = 2;     // exchange values per (partition, system)
    int xstride = 0, xper = 0;  // exchange elements per group; offset of the periodic-penta values in it
    size_t smem = 0;
    unsigned offX = 0, offM = 0, offR = 0, offTl = 0, offIn = 0;
    unsigned box_rows = 0, nboxes = 0;
    int max_grid = 0;  // occupancy * SM count, resolved at first launch
};

// how one kernel family (solve / CH step) lays a tile over the threads of a CTA
struct Shape {
    int lanes = 32, lanes_log2 = 5, vec = 1, tpc = 1, threads = 0;
};

struct DtypePlan {
    int elem = 8;
    int rows = 0, P = 0;
    Shape shape[3];     // [0] solve, [1] fused CH step (penta) / CN diffusion step (tri), [2] CN hyperdiffusion step (penta)
    int ws = 0;         // carries by the warp-shuffle scan
    int wfast = 0;      // periodic penta handle: the cyclic correction is folded into the scan (KIND_*F kernels)
    int scan_log2 = 0;  // log2 of the scan width
    int tq = 32;        // partitions per scan-table row
    bool two_pass = false;
    void *d_blob = nullptr;  // partitioned-sweep coefficient image
    unsigned blob_bytes = 0, offT = 0;
    void *d_soa = nullptr;   // two-pass coefficient arrays
    size_t soa_bytes = 0;
    // [kind slot][vector mode: 0 = plan.vec, 1 = scalar tail-safe][0 = TMA prefetch, 1 = direct loads]
    // kind slot 0 = solve, 1 = CH (penta handles only)
    KernelSlot k[3][2][2];
    // fp64 plan only: the plain solve on fp32 storage (the *_f32s calls): [vector mode][0 = TMA prefetch, 1 = direct loads]
    KernelSlot ks32[2][2];
    // plain solves of long systems (P > 16): the tile's rows split over a thread-block cluster of csz CTAs (two, four
    // or eight SMs), each keeping PLc partitions; carries cross the CTAs as a chain through distributed shared memory
    int csz = 0, PLc = 0, scan_log2_cl = 0;
    unsigned offTc = 0;         // byte offset in the blob of the csz per-CTA scan-table blocks
    unsigned tab_bytes_cl = 0;  // bytes of one such block
    unsigned blob_total = 0;    // blob bytes on the device (blob_bytes = what the single-CTA kernels stage)
    int blk_pad = 0;            // bytes of padding behind every partition's coefficient block (blk_stride)
    // coefficient blocks shared between partitions (dedupe_blocks): the blob holds nuniq distinct blocks, partition p
    // reads block pmap[p].  nuniq == P: nothing shared, pmap is the identity.
    int nuniq = 0;
    unsigned char pmap[MAX_PARTS] = {0};
    Shape cshape;
    KernelSlot ck;
    // long fused time loops of plans whose partitions share coefficient blocks (fp64): half-width tiles (8 lanes), so that a
    // CTA hosts two or four tile groups whose phases overlap (fill_slots, launch_one); kn[ks].fused.func == nullptr: none
    Shape nshape[3];
    KernelSlot kn[3];
    KernelSlot ck32;  // fp64 plan only: the cluster kernels on fp32 storage (the *_f32s calls); same shape, a ring of floats
};

constexpr int MAGIC_TRI = 0x74726931;    // "tri1"
constexpr int MAGIC_PENTA = 0x70656e31;  // "pen1"

struct Handle {
    int magic;
    int kind;  // KIND_TRI / KIND_PENTA
    bool periodic = false;                    // tri: cyclic matrix solved by Sherman-Morrison (KIND_TRIP kernels)
    double per_vN = 0.0, per_invden = 0.0;    // eq. 13a / 15 scalars of the periodic solve
    PerPenta pp = {};                         // periodic penta: Woodbury scalars (H, wrap-around entries)
    double per_ngl = 0.0;                     // periodic penta: -gamma at row n-2
    int n;
    int device;
    DtypePlan plan[2];  // 0: fp64, 1: fp32
    // plain pentadiagonal handles of 32 partitions (N = 993 ... 1024): a second plan whose blob keeps every partition's
    // own coefficient block, used by the single-step plain solve only (make_penta_handle says why)
    bool has_alt = false;
    DtypePlan alt[2];
    std::mutex mu;      // guards lazy occupancy resolution
};

int blk_stride(const DtypePlan &pl, int RT) { return RT * pl.rows + pl.blk_pad / pl.elem; }

int ilog2(int v)
{
    int l = 0;
    while ((1 << l) < v) ++l;
    return l;
}

// Plan of the partitioned sweep: rows per thread, partitions, and per kernel
// family the lanes, systems per thread and tile groups per CTA.  A thread keeps rows*vec elements
// in registers: up to 64 registers' worth the kernels run 512 threads per CTA, above that 256.
int thread_cap(int rows, int vec, int elem) { return (rows * vec * elem > 256) ? 256 : 512; }

void choose_shape(int kind, int elem, int rows, int P, Shape &sh)
{
    // 16 bytes per thread and row (one LDS.128 / ST.128)
    int vec = g_tune.vec > 0 ? g_tune.vec : 16 / elem;
    if (vec != 1 && vec != 2 && vec != 4) vec = 1;
    if (vec * elem > 16) vec = 16 / elem;  // one vector access is at most 16 bytes
    const int cap = thread_cap(rows, vec, elem);
    int lanes = g_tune.lanes > 0 ? g_tune.lanes : ((P > 1 && (vec * elem == 16 || P >= 16)) ? 16 : 32);
    if (lanes != 32 && lanes != 16 && lanes != 8 && lanes != 4) lanes = 32;
    while (P * lanes > cap && lanes > 4) lanes >>= 1;
    sh.lanes = lanes;
    sh.lanes_log2 = ilog2(lanes);
    sh.vec = vec;
}

void finish_shape(int elem, int rows, int P, Shape &sh)
{
    const int cap = thread_cap(rows, sh.vec, elem);
    const int tpt = P * sh.lanes;
    int tpc = g_tune.tpc > 0 ? g_tune.tpc : cap / tpt;
    if (tpc < 1) tpc = 1;
    while (tpc > 1 && tpc * tpt > cap) --tpc;
    if (tpt % 32 != 0) tpc = 1;             // groups synchronise on whole warps
    if (tpt != 32 && tpc > 15) tpc = 15;    // named barriers 1..15
    if (tpc > 16) tpc = 16;                 // one mbarrier per group, 16 slots
    sh.tpc = tpc;
    sh.threads = tpc * tpt;
}

void choose_plan(int n, int elem, int handle_kind, DtypePlan &pl)
{
    pl.elem = elem;
    int rows = g_tune.rows > 0 ? g_tune.rows : (n <= 8 ? 8 : (n <= 16 ? 16 : 32));
    if (rows != 8 && rows != 16 && rows != 32) rows = 32;
    int P = (n + rows - 1) / rows;
    const int nshape = 3;  // [0] solves, [1] CH (penta) / CN diffusion (tri) steps, [2] CN hyperdiffusion steps (penta)
    for (int k = 0; k < nshape; ++k)
        choose_shape(k == 0 ? handle_kind : (handle_kind == KIND_TRI ? KIND_TRICN : (k == 1 ? KIND_CH : KIND_PENTACN)), elem,
                     rows, P, pl.shape[k]);
    // the warp scan wants whole warps per group and at most 32 partitions: pad P with identity
    // partitions where that makes every family's group a whole number of warps
    int ws = (P > 1 && P <= 32 && g_tune.warp_scan != 0) ? 1 : 0;
    if (ws) {
        int Pp = P;
        auto fits = [&](int q) {
            for (int k = 0; k < nshape; ++k) {
                const Shape &sh = pl.shape[k];
                if ((q * sh.lanes) % 32 != 0 || q * sh.lanes > thread_cap(rows, sh.vec, elem)) return false;
            }
            return true;
        };
        while (Pp <= 32 && !fits(Pp)) ++Pp;
        if (Pp <= 32) P = Pp;
        else ws = 0;
    }
    // cluster-chain plan (sweep.cuh, CL): csz = 2 / 4 / 8 CTAs with at most 16 partitions each (16 lanes x 16 bytes =
    // 256-byte row segments); whole warps per CTA want an even number of partitions per CTA
    pl.csz = pl.PLc = 0;
    if (rows == 32 && P > 16 && g_tune.cluster != 0 && g_tune.prefetch != 0) {
        const int k = P <= 32 ? 2 : (P + 15) / 16;  // as few CTAs as 16 partitions each allow; at most 8 (portable cluster size)
        if (k <= 8) {
            int PLc = (P + k - 1) / k;
            PLc += (PLc & 1);
            if (PLc <= 16 && (k * PLc == P || P > 32)) {
                pl.csz = k;
                pl.PLc = PLc;
                pl.scan_log2_cl = ilog2(PLc);
                if (P > 32) P = k * PLc;  // no warp-scan plan of one CTA exists: pad to whole CTAs (identity partitions)
            }
        }
    }
    pl.two_pass = (g_tune.force_two_pass > 0);
    for (int k = 0; k < nshape; ++k) {
        finish_shape(elem, rows, P, pl.shape[k]);
        if (P * pl.shape[k].lanes > thread_cap(rows, pl.shape[k].vec, elem)) pl.two_pass = true;
    }
    pl.blk_pad = g_tune.blk_pad >= 0 ? (g_tune.blk_pad / 16) * 16 : 0;
    pl.rows = rows;
    pl.P = P;
    pl.ws = ws;
    pl.scan_log2 = ilog2(P);
    pl.tq = P > SCAN_LANES ? P : SCAN_LANES;
}

// Elements between the coefficient blocks of successive partitions: the block itself (RT arrays of `rows` entries) plus
// padding.  The threads of one partition read the same coefficient (a broadcast); the 2 or 4 partitions that share a warp
// read theirs one block apart, and an unpadded block (5 or 9 arrays x 32 rows x 8 bytes) is a multiple of 128 bytes, which
// puts them all on the same banks.  pl.blk_pad bytes of padding (a multiple of 16) walk them onto different banks.
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
// factor tables for the partitioned sweep; fp64 host arithmetic, rounded to
// T when written into the blob.  Rows are padded to Np = P*rows with all-zero rows (inv = 0: a padding row solves to exactly 0).
// ------------------------------------------------------------------------------------------------

// Carry-scan tables (sweep.cuh, RecLayout): slot 0 / 1 = forward / backward carry matrices of each
// partition (Phi_q, Psi_q), slot 2 = chi at the partition's first rows, and for the warp scan the
// Kogge-Stone multipliers of steps s >= 1 at slots 1+2s (forward) and 2+2s (backward):
//   A^(s+1)_q = A^(s)_q A^(s)_{q-2^s}  (zero where q < 2^s),
//   B^(s+1)_q = B^(s)_q B^(s)_{q+2^s}  (zero where q + 2^s >= P).
// Matrices are NC x NC, row-major, stored [slot][entry][q] with tq partitions per row.
struct Mat {
    double m[4] = {0, 0, 0, 0};
};

Mat matmul(const Mat &x, const Mat &y, int nc)
{
    Mat r;
    if (nc == 1) {
        r.m[0] = x.m[0] * y.m[0];
    } else {
        r.m[0] = x.m[0] * y.m[0] + x.m[1] * y.m[2];
        r.m[1] = x.m[0] * y.m[1] + x.m[1] * y.m[3];
        r.m[2] = x.m[2] * y.m[0] + x.m[3] * y.m[2];
        r.m[3] = x.m[2] * y.m[1] + x.m[3] * y.m[3];
    }
    return r;
}

// scan-table slots of the partitions [q0, q0 + P) at byte offset `base` of the blob, tq entries per table row
template <typename T>
void put_scan_slots(std::vector<unsigned char> &blob, size_t base, int q0, int P, int tq, int nc, bool ws, bool chain,
                    const std::vector<Mat> &PhiAll, const std::vector<Mat> &PsiAll, const std::vector<Mat> &Chi0All)
{
    const int ne = nc * nc;
    const std::vector<Mat> Phi(PhiAll.begin() + q0, PhiAll.begin() + q0 + P), Psi(PsiAll.begin() + q0, PsiAll.begin() + q0 + P),
        Chi0(Chi0All.begin() + q0, Chi0All.begin() + q0 + P);
    auto put_slot = [&](int slot, const std::vector<Mat> &v) {
        for (int q = 0; q < P; ++q)
            for (int m = 0; m < ne; ++m)
                put<T>(blob, base + (((size_t)slot * ne + m) * tq + q) * sizeof(T), v[q].m[m]);
    };
    put_slot(0, Phi);
    put_slot(1, Psi);
    if (!ws) return;
    if (chain) {
        // cluster kernels (sweep.cuh, CL): how the carries that enter this CTA's block of partitions -- Gin from the CTA below
        // into its first partition, Xin from the CTA above into its last -- reach partition q.  With G0 / X0 the carries of the
        // block solved on its own (Gin = Xin = 0):
        //   carry into q from below  G_q = G0_q + Pin_q Gin,            Pin_q = Phi_{q-1} ... Phi_first      (slot 10; I at q = 0)
        //   carry into q from above  X_q = X0_q + Th_{q+1} Gin + Sf_{q+1} Xin   (slots 13 and 11; 0 and I at the last partition)
        // where Sf_q = Psi_q ... Psi_last and Th_q = Chi0_q Pin_q + Psi_q Th_{q+1} is what Gin adds to the backward sweep's
        // inclusive value at q through u = x^_first + Chi0 G.
        const Mat zero;
        Mat ident;
        ident.m[0] = 1.0;
        if (nc == 2) ident.m[3] = 1.0;
        std::vector<Mat> Pin(P), SfIn(P), ThIn(P);
        Pin[0] = ident;
        for (int q = 1; q < P; ++q) Pin[q] = matmul(Phi[q - 1], Pin[q - 1], nc);
        Mat sf = ident, th = zero;  // Sf_{q+1}, Th_{q+1}
        for (int q = P - 1; q >= 0; --q) {
            SfIn[q] = sf;
            ThIn[q] = th;
            const Mat cp = matmul(Chi0[q], Pin[q], nc), pt = matmul(Psi[q], th, nc);
            for (int m = 0; m < ne; ++m) th.m[m] = cp.m[m] + pt.m[m];
            sf = matmul(Psi[q], sf, nc);
        }
        put_slot(10, Pin);
        put_slot(11, SfIn);
        put_slot(13, ThIn);
    }
    std::vector<Mat> A = Phi, B = Psi;
    const Mat zero;
    // step 0 multipliers: no partner below / above the ends
    A[0] = zero;
    B[P - 1] = zero;
    put_slot(0, A);
    put_slot(1, B);
    for (int st = 0; st + 1 < SCAN_STEPS; ++st) {
        const int d = 1 << st;
        std::vector<Mat> A2(P), B2(P);
        for (int q = 0; q < P; ++q) {
            A2[q] = (q >= 2 * d) ? matmul(A[q], A[q - d], nc) : zero;
            B2[q] = (q + 2 * d < P) ? matmul(B[q], B[q + d], nc) : zero;
        }
        A.swap(A2);
        B.swap(B2);
        if (st + 1 < 4) {
            put_slot(2 * (st + 1), A);
            put_slot(2 * (st + 1) + 1, B);
        } else {
            // step 4: forward entries (q >= 16) and backward entries (q < 16) share slot 8
            std::vector<Mat> AB(P);
            for (int q = 0; q < P; ++q) AB[q] = (q >= 16) ? A[q] : B[q];
            put_slot(8, AB);
        }
    }
    put_slot(9, Chi0);
}

template <typename T>
void put_scan_tables(std::vector<unsigned char> &blob, DtypePlan &pl, int nc, const std::vector<Mat> &Phi,
                     const std::vector<Mat> &Psi, const std::vector<Mat> &Chi0)
{
    put_scan_slots<T>(blob, pl.offT, 0, pl.P, pl.tq, nc, pl.ws != 0, false, Phi, Psi, Chi0);
    pl.blob_total = pl.blob_bytes;
    if (pl.csz) {
        // one table block per CTA of the cluster chain, behind everything the single-CTA kernels stage
        pl.offTc = pl.blob_bytes;
        pl.tab_bytes_cl = (unsigned)align16((size_t)14 * nc * nc * SCAN_LANES * sizeof(T));
        pl.blob_total = pl.offTc + (unsigned)pl.csz * pl.tab_bytes_cl;
        blob.resize(pl.blob_total, 0);
        const int k = pl.csz, PL = pl.PLc, ne = nc * nc;
        for (int r = 0; r < k; ++r)
            put_scan_slots<T>(blob, pl.offTc + (size_t)r * pl.tab_bytes_cl, r * PL, PL, SCAN_LANES, nc, true, true, Phi, Psi, Chi0);
        // slot 12 of CTA r's block: how the other CTAs' local carries reach it.  With PhiT_c = Phi_last ... Phi_first,
        // PsiT_c = Psi_first ... Psi_last and ThT_c = Th_first of CTA c's block (put_scan_slots), the cluster-level recurrences
        //   Gin_0 = 0, Gin_{c+1} = F_c + PhiT_c Gin_c;   Xin_last = 0, Xin_{c-1} = B_c + ThT_c Gin_c + PsiT_c Xin_c
        // unroll to  Gin_r = sum_{s<r} C_{r,s} F_s,   Xin_r = sum_{s>r} D_{r,s} B_s + sum_t E_{r,t} F_t  with
        //   C_{r,s} = PhiT_{r-1} ... PhiT_{s+1}  (entry s;      identity for s = r - 1),
        //   D_{r,s} = PsiT_{r+1} ... PsiT_{s-1}  (entry 8 + s;  identity for s = r + 1),
        //   E_{r,t} = sum_{s > max(r,t)} D_{r,s} ThT_s C_{s,t}  (entry 16 + t),
        // all LHS-only, so every CTA finishes its carries after ONE exchange of (F, B).
        std::vector<Mat> PhiT(k), PsiT(k), ThT(k);
        Mat ident;
        ident.m[0] = 1.0;
        if (nc == 2) ident.m[3] = 1.0;
        for (int c = 0; c < k; ++c) {
            Mat f = Phi[c * PL], b = Psi[c * PL + PL - 1];
            for (int q = 1; q < PL; ++q) f = matmul(Phi[c * PL + q], f, nc);
            for (int q = PL - 2; q >= 0; --q) b = matmul(Psi[c * PL + q], b, nc);
            std::vector<Mat> pins(PL);
            pins[0] = ident;
            for (int q = 1; q < PL; ++q) pins[q] = matmul(Phi[c * PL + q - 1], pins[q - 1], nc);
            Mat th;
            for (int q = PL - 1; q >= 0; --q) {
                const Mat cp = matmul(Chi0[c * PL + q], pins[q], nc), pt = matmul(Psi[c * PL + q], th, nc);
                for (int m = 0; m < ne; ++m) th.m[m] = cp.m[m] + pt.m[m];
            }
            PhiT[c] = f;
            PsiT[c] = b;
            ThT[c] = th;
        }
        // C[r][s], s < r and D[r][s], s > r
        std::vector<std::vector<Mat>> C(k, std::vector<Mat>(k)), D(k, std::vector<Mat>(k));
        for (int r = 0; r < k; ++r) {
            Mat c = ident;
            for (int sb = r - 1; sb >= 0; --sb) {
                if (sb < r - 1) c = matmul(c, PhiT[sb + 1], nc);
                C[r][sb] = c;
            }
            Mat d = ident;
            for (int sb = r + 1; sb < k; ++sb) {
                if (sb > r + 1) d = matmul(d, PsiT[sb - 1], nc);
                D[r][sb] = d;
            }
        }
        for (int r = 0; r < k; ++r) {
            const size_t base = pl.offTc + (size_t)r * pl.tab_bytes_cl + (size_t)12 * ne * SCAN_LANES * sizeof(T);
            for (int sb = 0; sb < k; ++sb) {
                if (sb < r)
                    for (int m = 0; m < ne; ++m) put<T>(blob, base + ((size_t)m * SCAN_LANES + sb) * sizeof(T), C[r][sb].m[m]);
                if (sb > r)
                    for (int m = 0; m < ne; ++m) put<T>(blob, base + ((size_t)m * SCAN_LANES + 8 + sb) * sizeof(T), D[r][sb].m[m]);
            }
            for (int t = 0; t < k; ++t) {
                Mat e;
                for (int sb = (r > t ? r : t) + 1; sb < k; ++sb) {
                    const Mat x = matmul(matmul(D[r][sb], ThT[sb], nc), C[sb][t], nc);
                    for (int m = 0; m < ne; ++m) e.m[m] += x.m[m];
                }
                for (int m = 0; m < ne; ++m) put<T>(blob, base + ((size_t)m * SCAN_LANES + 16 + t) * sizeof(T), e.m[m]);
            }
        }
    }
}

// Partitions whose coefficient blocks are bitwise equal share one block.  The factor coefficients of a constant-
// coefficient LHS (every LHS of the paper: PAPER.md:126, 172, 306, 380) converge to their limit bitwise within 13-28
// rows, and the per-partition responses (chi, psi) are functions of the block's own rows only, so every interior
// partition of such a matrix has the same block: N = 1024 keeps 2-3 blocks of 32 (penta fp64: 74 KB -> 7 KB of shared
// memory).  A general LHS has P distinct blocks and nothing changes.  Called at the very end of build_blob_*: the blob
// becomes [distinct blocks][everything behind the row records, moved down]; offT / blob_bytes / offTc / blob_total follow.
// Cluster plans (a CTA stages only its own partitions' blocks) share blocks only when all the distinct ones fit the
// space of one CTA's share (nuniq <= PLc); otherwise the blob stays whole and each CTA stages its own PLc blocks.
void dedupe_blocks(DtypePlan &pl, std::vector<unsigned char> &blob, int RT, bool allow)
{
    const int P = pl.P;
    const size_t bb = (size_t)blk_stride(pl, RT) * pl.elem;
    pl.nuniq = P;
    for (int p = 0; p < P && p < MAX_PARTS; ++p) pl.pmap[p] = (unsigned char)p;
    if (!allow || P < 2 || P > MAX_PARTS) return;
    std::vector<int> first;  // partition index of each distinct block, in order of appearance
    std::vector<unsigned char> map(P);
    for (int p = 0; p < P; ++p) {
        int u = -1;
        for (size_t k = 0; k < first.size() && u < 0; ++k)
            if (!memcmp(&blob[(size_t)first[k] * bb], &blob[(size_t)p * bb], bb)) u = (int)k;
        if (u < 0) {
            u = (int)first.size();
            first.push_back(p);
        }
        map[p] = (unsigned char)u;
    }
    const int U = (int)first.size();
    if (U == P || (pl.csz && U > pl.PLc)) return;
    std::vector<unsigned char> out;
    out.reserve(blob.size());
    for (int u = 0; u < U; ++u) out.insert(out.end(), blob.begin() + (size_t)first[u] * bb, blob.begin() + (size_t)(first[u] + 1) * bb);
    const unsigned new_offT = (unsigned)align16((size_t)U * bb);
    out.resize(new_offT, 0);
    out.insert(out.end(), blob.begin() + pl.offT, blob.end());
    const unsigned delta = pl.offT - new_offT;
    pl.offT = new_offT;
    pl.blob_bytes -= delta;
    pl.blob_total -= delta;
    if (pl.csz) pl.offTc -= delta;
    blob.swap(out);
    pl.nuniq = U;
    for (int p = 0; p < P; ++p) pl.pmap[p] = map[p];
}

// mode: 1 / 0 = share blocks or not, -1 = as btps_tune("dedupe") says (default: share)
bool dedupe_wanted(int mode)
{
    if (mode >= 0) return mode > 0;
    return g_tune.dedupe != 0;
}

size_t scan_table_bytes(const DtypePlan &pl, int nc, size_t elem)
{
    int slots = pl.ws ? 2 * SCAN_STEPS : 2;  // ws: 8 step slots + merged step 4 + chi
    if (pl.wfast) slots += (nc == 2) ? 4 : 2;  // GZ / XZ: carries of A' z = e_r (penta: slots 10-13) or A' z = u (tri: 10, 11)
    return (size_t)slots * nc * nc * pl.tq * elem;
}

template <typename T>
void build_blob_tri(int n, DtypePlan &pl, const std::vector<double> &inv, const std::vector<double> &nl,
                    const std::vector<double> &nch, std::vector<unsigned char> &blob,
                    const std::vector<double> *z = nullptr, const std::vector<double> *zfwd = nullptr, double u0 = 0.0,
                    double uN = 0.0, int dedupe_mode = -1)
{
    const int MR = pl.rows, P = pl.P, Np = P * MR;
    // coefficient values per row: the periodic form carries z = A'^{-1} u as a sixth array
    const int RT = z ? RecLayout<KIND_TRIP>::ELEMS : RecLayout<KIND_TRI>::ELEMS;
    auto at = [&](const std::vector<double> &v, int i, double pad) { return i < n ? v[i] : pad; };
    pl.offT = (unsigned)align16((size_t)P * blk_stride(pl, RT) * sizeof(T));
    pl.blob_bytes = (unsigned)align16(pl.offT + scan_table_bytes(pl, 1, sizeof(T)));
    blob.assign(pl.blob_bytes, 0);
    std::vector<double> phi(MR), chi(MR), psi(MR);
    std::vector<Mat> Phi(P), Psi(P), Chi0(P);
    auto putv = [&](int arr, int i, int j, double v) {  // partition block, array at offset arr*MR, row i, value j
        const size_t blk = (size_t)(i / MR) * blk_stride(pl, RT);
        put<T>(blob, (blk + (size_t)arr * MR + (size_t)(i % MR) * (arr == 2 ? 1 : 2) + j) * sizeof(T), v);
    };
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
            putv(0, i, 0, at(inv, i, 0.0));  // padding rows: g = 0 * f, whatever the explicit half put there
            putv(0, i, 1, at(nl, i, 0.0));
            putv(2, i, 0, at(nch, i, 0.0));
            putv(3, i, 0, chi[k]);
            putv(3, i, 1, psi[k]);
            if (z && !pl.wfast) put<T>(blob, ((size_t)(i / MR) * blk_stride(pl, RT) + (size_t)5 * MR + (i % MR)) * sizeof(T), at(*z, i, 0.0));
        }
        Phi[p].m[0] = phi[MR - 1];
        Psi[p].m[0] = psi[0];
        Chi0[p].m[0] = chi[0];
    }
    put_scan_tables<T>(blob, pl, 1, Phi, Psi, Chi0);
    if (z && pl.wfast) {
        // z = A'^{-1} u in the partitioned form is "local solve + chi GZ + psi XZ": GZ_p = forward-sweep value of u at the last
        // row of partition p-1, XZ_p = z at the first row of partition p+1; the local (zero-carry) solve of u is nonzero only
        // in partition 0 (u_0 = -b_0 at row 0) and partition P-1 (u_{n-1} = c_{n-1} at row n-1); n = P*MR here.
        const int tq = pl.tq;
        for (int p = 0; p < P; ++p) {
            put<T>(blob, pl.offT + ((size_t)10 * tq + p) * sizeof(T), p > 0 ? (*zfwd)[p * MR - 1] : 0.0);
            put<T>(blob, pl.offT + ((size_t)11 * tq + p) * sizeof(T), p + 1 < P ? (*z)[(p + 1) * MR] : 0.0);
        }
        std::vector<double> loc(MR);
        for (int e = 0; e < 2; ++e) {
            const int p = e == 0 ? 0 : P - 1, r0 = p * MR;
            double g = 0.0;
            for (int k = 0; k < MR; ++k) {
                const double r = (e == 0 && k == 0) ? u0 : ((e == 1 && k == MR - 1) ? uN : 0.0);
                g = nl[r0 + k] * (k > 0 ? g : 0.0) + inv[r0 + k] * r;
                loc[k] = g;
            }
            for (int k = MR - 2; k >= 0; --k) loc[k] = loc[k] + nch[r0 + k] * loc[k + 1];
            for (int k = 0; k < MR; ++k)
                put<T>(blob, ((size_t)p * blk_stride(pl, RT) + (size_t)5 * MR + k) * sizeof(T), loc[k]);
        }
    }
    dedupe_blocks(pl, blob, RT, dedupe_wanted(dedupe_mode));
}

template <typename T>
void build_blob_penta(int n, DtypePlan &pl, const std::vector<double> &inv, const std::vector<double> &nle,
                      const std::vector<double> &nlb, const std::vector<double> &ngam,
                      const std::vector<double> &ndel, std::vector<unsigned char> &blob,
                      const std::vector<double> *Z = nullptr, int dedupe_mode = -1)
{
    const int MR = pl.rows, P = pl.P, Np = P * MR;
    // coefficient values per row: the periodic form carries the rows of Z = A'^{-1} U (n x 4, row-major), or, with the
    // cyclic correction folded into the scan, the local solves of the unit vectors in the two end partitions
    const int RT = Z ? (pl.wfast ? RecLayout<KIND_PENTAPF>::ELEMS : RecLayout<KIND_PENTAP>::ELEMS)
                     : RecLayout<KIND_PENTA>::ELEMS;
    auto at = [&](const std::vector<double> &v, int i, double pad) { return i < n ? v[i] : pad; };
    pl.offT = (unsigned)align16((size_t)P * blk_stride(pl, RT) * sizeof(T));
    pl.blob_bytes = (unsigned)align16(pl.offT + scan_table_bytes(pl, 2, sizeof(T)));
    blob.assign(pl.blob_bytes, 0);
    std::vector<double> phi[2], chi[2], psi[2];
    for (int t = 0; t < 2; ++t) {
        phi[t].resize(MR);
        chi[t].resize(MR);
        psi[t].resize(MR);
    }
    std::vector<Mat> Phi(P), Psi(P), Chi0(P);
    auto putv = [&](int arr, int i, int j, double v) {  // partition block, array at offset arr*MR, row i, value j
        const size_t blk = (size_t)(i / MR) * blk_stride(pl, RT);
        put<T>(blob, (blk + (size_t)arr * MR + (size_t)(i % MR) * (arr == 2 ? 1 : 2) + j) * sizeof(T), v);
    };
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
            putv(0, i, 0, at(inv, i, 0.0));  // padding rows: g = 0 * f, whatever the explicit half put there
            putv(0, i, 1, at(nle, i, 0.0));
            putv(2, i, 0, at(nlb, i, 0.0));
            putv(3, i, 0, at(ngam, i, 0.0));
            putv(3, i, 1, at(ndel, i, 0.0));
            putv(5, i, 0, chi[0][k]);
            putv(5, i, 1, chi[1][k]);
            putv(7, i, 0, psi[0][k]);
            putv(7, i, 1, psi[1][k]);
            if (Z && !pl.wfast)
                for (int m = 0; m < 4; ++m) putv(m < 2 ? 9 : 11, i, m & 1, i < n ? (*Z)[(size_t)i * 4 + m] : 0.0);
        }
        // carries: (g at the last row, g at the last-but-one row) forward; (x at the first row, x at
        // the second row) backward
        Phi[p].m[0] = phi[0][MR - 1];
        Phi[p].m[1] = phi[1][MR - 1];
        Phi[p].m[2] = phi[0][MR - 2];
        Phi[p].m[3] = phi[1][MR - 2];
        Psi[p].m[0] = psi[0][0];
        Psi[p].m[1] = psi[1][0];
        Psi[p].m[2] = psi[0][1];
        Psi[p].m[3] = psi[1][1];
        Chi0[p].m[0] = chi[0][0];
        Chi0[p].m[1] = chi[1][0];
        Chi0[p].m[2] = chi[0][1];
        Chi0[p].m[3] = chi[1][1];
    }
    put_scan_tables<T>(blob, pl, 2, Phi, Psi, Chi0);
    if (Z && pl.wfast) {
        // Column m of Z solves A' z = e_r, r = (0, 1, n-2, n-1)[m].  In the partitioned form it is "local solve + chi GZ +
        // psi XZ": GZ_p = (g at the last two rows of partition p-1), XZ_p = (z at the first two rows of partition p+1), and
        // the local (zero-carry) solve is nonzero only in the partition that holds row r (n = P*MR: partition 0 or P-1).
        const int tq = pl.tq;
        const int urow[4] = {0, 1, n - 2, n - 1};
        std::vector<double> g(n), loc(MR);
        for (int m = 0; m < 4; ++m) {
            for (int i = 0; i < n; ++i) {  // forward sweep of e_r with the sweep multipliers
                const double r = (i == urow[m]) ? 1.0 : 0.0;
                g[i] = inv[i] * r + (i >= 2 ? nle[i] * g[i - 2] : 0.0) + (i >= 1 ? nlb[i] * g[i - 1] : 0.0);
            }
            for (int p = 0; p < P; ++p) {
                const double gz[2] = {p > 0 ? g[p * MR - 1] : 0.0, p > 0 ? g[p * MR - 2] : 0.0};
                const double xz[2] = {p + 1 < P ? (*Z)[(size_t)((p + 1) * MR) * 4 + m] : 0.0,
                                      p + 1 < P ? (*Z)[(size_t)((p + 1) * MR + 1) * 4 + m] : 0.0};
                for (int c = 0; c < 2; ++c) {
                    put<T>(blob, pl.offT + ((size_t)(40 + c * 4 + m) * tq + p) * sizeof(T), gz[c]);
                    put<T>(blob, pl.offT + ((size_t)(48 + c * 4 + m) * tq + p) * sizeof(T), xz[c]);
                }
            }
            // local solve in the end partition that holds row r
            const int p = (m < 2) ? 0 : P - 1, r0 = p * MR;
            for (int k = 0; k < MR; ++k) {
                const int i = r0 + k;
                const double r = (i == urow[m]) ? 1.0 : 0.0;
                loc[k] = inv[i] * r + (k >= 2 ? nle[i] * loc[k - 2] : 0.0) + (k >= 1 ? nlb[i] * loc[k - 1] : 0.0);
            }
            for (int k = MR - 2; k >= 0; --k)
                loc[k] = loc[k] + ngam[r0 + k] * loc[k + 1] + (k + 2 < MR ? ndel[r0 + k] * loc[k + 2] : 0.0);
            for (int k = 0; k < MR; ++k) putv(9, r0 + k, m & 1, loc[k]);
        }
    }
    dedupe_blocks(pl, blob, RT, dedupe_wanted(dedupe_mode));
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
        if (h->alt[t].d_blob) cudaFree(h->alt[t].d_blob);
    }
    h->magic = 0;
    delete h;
}

// The partitioned plan keeps the whole coefficient image, the exchange area and (TMA variant) the
// prefetch ring in shared memory; the per-CTA limit of sm_100a is 227 KB.
constexpr size_t SMEM_LIMIT = 227 * 1024;

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// shared-memory layout of one kernel variant: [blob][exchange][mbarriers][ring]
void layout_slot(const DtypePlan &pl, const Shape &sh, int kind, KernelSlot &sl, bool halo = true, int selem = 0)
{
    if (selem == 0) selem = pl.elem;  // bytes per element of the batch in global memory / in the ring
    const bool tri = (kind == KIND_TRI || kind == KIND_TRIP || kind == KIND_TRICN || kind == KIND_TRICNP || kind == KIND_TRIPF ||
                      kind == KIND_TRICNPF);
    const bool pertf = (kind == KIND_TRIPF || kind == KIND_TRICNPF);  // + 1 value: nfac for the end partitions
    const int NC = tri ? 1 : 2;
    // kinds with an explicit half need one halo row on each side between fused steps
    const bool cn5 = (kind == KIND_PENTACN || kind == KIND_PENTACNP || kind == KIND_PENTACNPF);  // two halo rows on each side
    const bool is_ch = (kind == KIND_CH || kind == KIND_CHP || kind == KIND_CHPF || kind == KIND_TRICN || kind == KIND_TRICNP ||
                        kind == KIND_TRICNPF || cn5);
    const bool wood = (kind == KIND_PENTAP || kind == KIND_CHP || kind == KIND_PENTACNP), pert = (kind == KIND_TRIP || kind == KIND_TRICNP);
    const bool woodf = (kind == KIND_PENTAPF || kind == KIND_CHPF || kind == KIND_PENTACNPF);  // + 2 values: nw for the end partitions
    const size_t W = (size_t)sh.lanes * sl.vec;
    // CH: + the halo rows exchanged between fused steps; periodic tri: + y_1 and y_N of eq. 15
    sl.xvals = 2 * NC + ((is_ch && halo) ? (cn5 ? 4 : 2) : 0) + (pert ? 2 : 0) + (woodf ? 2 : 0) + (pertf ? 1 : 0);
    sl.xper = (int)(sl.xvals * pl.P * W);
    sl.xstride = sl.xper + (wood ? (int)(4 * W) : 0);  // cyclic penta: y at rows 0, 1, n-2, n-1
    const size_t xch = (pl.P > 1) ? (size_t)sh.tpc * sl.xstride * pl.elem : 0;
    sl.offX = (unsigned)align16(pl.blob_bytes);
    sl.offM = (unsigned)align16(sl.offX + xch);
    sl.offR = (unsigned)align_up(sl.offM + 17 * 8, 128);
    // TMA boxes of whole partitions: the largest divisor g of P with g*rows <= 256 rows per box
    const size_t Np = (size_t)pl.P * pl.rows;
    int g = 256 / pl.rows < pl.P ? 256 / pl.rows : pl.P;
    while (pl.P % g != 0) --g;
    sl.box_rows = (unsigned)(g * pl.rows);
    sl.nboxes = (unsigned)(pl.P / g);
    const size_t ring = (size_t)sh.tpc * Np * W * selem;
    sl.smem = sl.tma ? sl.offR + ring : sl.offM + 17 * 8;
}

bool tma_possible(const DtypePlan &pl, const Shape &sh, int vec, int selem = 0)
{
    const size_t wb = (size_t)sh.lanes * vec * (selem ? selem : pl.elem);  // bytes of one tile row
    if (g_tune.prefetch == 0) return false;
    if (pl.P > 1 && !pl.ws) return false;       // the serial carry walk has no TMA variant
    if (wb % 16 != 0 || sh.lanes * vec > 256) return false;
    return true;
}

SweepEntry find_sweep(int kind, int elem_bytes, int vec, int rows, int single, int tma, int ws, int fuse)
{
    if (elem_bytes == 8) {
        if (kind == KIND_TRI) return find_sweep_tri_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_TRIP) return find_sweep_trip_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_PENTAP) return find_sweep_pentap_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_CHP) return find_sweep_chp_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_TRICN) return find_sweep_tricn_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_TRICNP) return find_sweep_tricnp_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_PENTACN) return find_sweep_pentacn_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_PENTACNP) return find_sweep_pentacnp_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_PENTAPF) return find_sweep_pentapf_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_CHPF) return find_sweep_chpf_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_PENTACNPF) return find_sweep_pentacnpf_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_TRIPF) return find_sweep_tripf_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_TRICNPF) return find_sweep_tricnpf_f64(vec, rows, single, tma, ws, fuse);
        if (kind == KIND_PENTA) return find_sweep_penta_f64(vec, rows, single, tma, ws, fuse);
        return find_sweep_ch_f64(vec, rows, single, tma, ws, fuse);
    }
    if (kind == KIND_TRI) return find_sweep_tri_f32(vec, rows, single, tma, ws, fuse);
    if (kind == KIND_TRIP) return find_sweep_trip_f32(vec, rows, single, tma, ws, fuse);
    if (kind == KIND_PENTAP) return find_sweep_pentap_f32(vec, rows, single, tma, ws, fuse);
    if (kind == KIND_PENTAPF) return find_sweep_pentapf_f32(vec, rows, single, tma, ws, fuse);
    if (kind == KIND_TRIPF) return find_sweep_tripf_f32(vec, rows, single, tma, ws, fuse);
    if (kind == KIND_CHPF || kind == KIND_PENTACNPF || kind == KIND_TRICNPF) return SweepEntry{nullptr, nullptr, 0};
    if (kind == KIND_CHP) return find_sweep_chp_f32(vec, rows, single, tma, ws, fuse);
    if (kind == KIND_TRICN || kind == KIND_TRICNP || kind == KIND_PENTACN || kind == KIND_PENTACNP)
        return SweepEntry{nullptr, nullptr, 0};  // the Crank-Nicolson steps are fp64 only
    if (kind == KIND_PENTA) return find_sweep_penta_f32(vec, rows, single, tma, ws, fuse);
    return find_sweep_ch_f32(vec, rows, single, tma, ws, fuse);
}

SweepEntry find_sweep_cl(int kind, int elem_bytes, int fuse)
{
    if (kind == KIND_TRI) return elem_bytes == 8 ? find_sweep_cl_tri_f64(fuse) : find_sweep_cl_tri_f32(fuse);
    if (kind == KIND_PENTA) return elem_bytes == 8 ? find_sweep_cl_penta_f64(fuse) : find_sweep_cl_penta_f32(fuse);
    return SweepEntry{nullptr, nullptr, 0};
}

// Cluster plan (sweep.cuh, CL): a tile's rows are split over csz CTAs of one thread-block cluster (csz SMs), each
// keeping PLc <= 16 partitions on 16 lanes x 16 bytes = 256-byte row segments, which is what HBM and the TLB want
// (DESIGN.md "Long systems").  Shared memory per CTA: its partitions' coefficient blocks, its own scan-table block, the
// exchange area of its partitions, the two carry inboxes and the ring of its rows.
void fill_cluster_slot(Handle *h, DtypePlan &pl, bool f32s = false)
{
    KernelSlot &sl = f32s ? pl.ck32 : pl.ck;
    sl = KernelSlot();
    const size_t selem = f32s ? 4 : (size_t)pl.elem;  // bytes per element of the batch in global memory / in the ring
    if (!pl.csz || h->periodic || g_tune.cluster == 0 || g_tune.prefetch == 0 || pl.rows != 32) return;
    const int kind = h->kind;  // KIND_TRI / KIND_PENTA
    const int NC = (kind == KIND_TRI) ? 1 : 2;
    const int elems = (kind == KIND_TRI) ? RecLayout<KIND_TRI>::ELEMS : RecLayout<KIND_PENTA>::ELEMS;
    Shape &sh = pl.cshape;
    sh.lanes = 16;
    sh.lanes_log2 = 4;
    sh.vec = 16 / pl.elem;
    sh.tpc = 1;
    const int PL = pl.PLc;
    sh.threads = PL * sh.lanes;
    sl.vec = sh.vec;
    sl.tma = 1;
    const size_t W = (size_t)sh.lanes * sl.vec;
    sl.xvals = 2 * NC;
    sl.xper = (int)(sl.xvals * PL * W);
    sl.xstride = sl.xper;
    const size_t rows_bytes = (size_t)(pl.nuniq < PL ? pl.nuniq : PL) * blk_stride(pl, elems) * pl.elem;  // shared blocks, or its own PL
    sl.offTl = (unsigned)align16(rows_bytes);
    sl.offX = (unsigned)align16(sl.offTl + pl.tab_bytes_cl);
    sl.offIn = (unsigned)align16(sl.offX + (size_t)sl.xstride * pl.elem);
    sl.offM = (unsigned)align16(sl.offIn + (size_t)2 * 2 * 8 * NC * W * pl.elem);  // [tile parity][F | B][8 senders][NC][W]
    sl.offR = (unsigned)align_up(sl.offM + 49 * 8, 128);  // 17 barriers as everywhere + 2 x 16 inbox barriers
    int g = 256 / pl.rows < PL ? 256 / pl.rows : PL;
    while (PL % g != 0) --g;
    sl.box_rows = (unsigned)(g * pl.rows);
    sl.nboxes = (unsigned)(PL / g);
    sl.smem = sl.offR + (size_t)PL * pl.rows * W * selem;
    if (sl.smem > SMEM_LIMIT) return;
    if (f32s) {
        sl.ent = find_sweep_cl_f32s(kind);  // single-step launches only, as the other *_f32s kernels
    } else {
        sl.ent = find_sweep_cl(kind, pl.elem, 0);
        sl.fused = find_sweep_cl(kind, pl.elem, 1);
    }
    if (sl.ent.func && sl.ent.max_threads < sh.threads) sl.ent = SweepEntry{nullptr, nullptr, 0};
}

void fit_plan(DtypePlan &pl, int handle_kind)
{
    if (pl.two_pass) return;
    for (int k = 0; k < 3; ++k) {
        KernelSlot probe;
        probe.vec = 1;
        probe.tma = 0;
        layout_slot(pl, pl.shape[k], handle_kind, probe);
        if (probe.smem > SMEM_LIMIT) pl.two_pass = true;
    }
}

void fill_slots(Handle *h)
{
    for (int t = 0; t < (h->has_alt ? 4 : 2); ++t) {
        DtypePlan &pl = t < 2 ? h->plan[t] : h->alt[t - 2];
        fill_cluster_slot(h, pl);
        if (pl.elem == 8) fill_cluster_slot(h, pl, true);
        if (pl.elem == 8 && !h->periodic && !pl.two_pass && (pl.P == 1 || (pl.ws && pl.rows == 32))) {
            // fp32 storage, fp64 arithmetic: the plain solve kernels of the fp64 plan with a ring of floats
            const Shape &sh = pl.shape[0];
            for (int s = 0; s < 2; ++s)
                for (int d = 0; d < 2; ++d) {
                    KernelSlot &sl = pl.ks32[s][d];
                    sl = KernelSlot();
                    sl.vec = (s == 0) ? sh.vec : 1;
                    sl.tma = (d == 0) ? 1 : 0;
                    if (sl.vec > 2 || (sl.tma && !tma_possible(pl, sh, sl.vec, 4))) continue;
                    layout_slot(pl, sh, h->kind, sl, true, 4);
                    if (sl.smem > SMEM_LIMIT) continue;
                    sl.ent = find_sweep_f32s(h->kind, sl.vec, pl.rows, pl.P == 1 ? 1 : 0, sl.tma, pl.ws);
                    if (sl.ent.func && sl.ent.max_threads < sh.threads) sl.ent = SweepEntry{nullptr, nullptr, 0};
                }
        }
        if (pl.two_pass) continue;
        const int single = (pl.P == 1) ? 1 : 0;
        for (int ks = 0; ks < 3; ++ks) {
            int kind;
            if (h->kind == KIND_TRI) {
                if (ks == 2) continue;
                kind = (ks == 0) ? (h->periodic ? KIND_TRIP : KIND_TRI) : (h->periodic ? KIND_TRICNP : KIND_TRICN);
                if (ks == 1 && pl.elem != 8) continue;  // the Crank-Nicolson step is fp64 only
                // periodic explicit halves need whole partitions and at least two of them (halo wrap)
                if (kind == KIND_TRICNP && (pl.P < 2 || pl.P * pl.rows != h->n)) continue;
                if (pl.wfast) kind = (ks == 0) ? KIND_TRIPF : KIND_TRICNPF;
            } else {
                kind = (ks == 0) ? (h->periodic ? KIND_PENTAP : KIND_PENTA)
                                 : (ks == 1 ? (h->periodic ? KIND_CHP : KIND_CH) : (h->periodic ? KIND_PENTACNP : KIND_PENTACN));
                if (ks == 2 && pl.elem != 8) continue;
                if (kind == KIND_PENTACNP && (pl.P < 2 || pl.P * pl.rows != h->n)) continue;
                if (pl.wfast) kind = (ks == 0) ? KIND_PENTAPF : (ks == 1 ? KIND_CHPF : KIND_PENTACNPF);
                // the periodic CH kernels need whole partitions and at least two of them (halo wrap);
                // other sizes run the two-pass form
                if (kind == KIND_CHP && (pl.P < 2 || pl.P * pl.rows != h->n)) continue;
            }
            const Shape &sh = pl.shape[ks];
            for (int s = 0; s < 2; ++s) {
                for (int d = 0; d < 2; ++d) {
                    KernelSlot &sl = pl.k[ks][s][d];
                    sl.vec = (s == 0) ? sh.vec : 1;
                    sl.tma = (d == 0) ? 1 : 0;
                    sl.ent = SweepEntry{nullptr, nullptr, 0};
                    sl.max_grid = 0;
                    if (sl.tma && !tma_possible(pl, sh, sl.vec)) continue;
                    layout_slot(pl, sh, kind, sl);
                    bool can_fuse = true;
                    if (sl.smem > SMEM_LIMIT && (kind == KIND_CH || kind == KIND_CHP || kind == KIND_TRICN || kind == KIND_TRICNP || kind == KIND_PENTACN ||
                                                kind == KIND_PENTACNP) && !pl.wfast) {
                        // tight fit (N = 1024 fp64): drop the halo exchange rows, one step per launch
                        layout_slot(pl, sh, kind, sl, false);
                        can_fuse = false;
                    }
                    if (sl.smem > SMEM_LIMIT) continue;
                    sl.ent = find_sweep(kind, pl.elem, sl.vec, pl.rows, single, sl.tma, pl.ws, 0);
                    if (sl.ent.func && sl.ent.max_threads < sh.threads) sl.ent = SweepEntry{nullptr, nullptr, 0};
                    sl.fused = SweepEntry{nullptr, nullptr, 0};
                    if (sl.ent.func && sl.tma && can_fuse) sl.fused = find_sweep(kind, pl.elem, sl.vec, pl.rows, single, 1, pl.ws, 1);
                }
            }
            // Half-width tiles for long fused loops (same kernels, lanes = 8): with shared coefficient blocks the four
            // partitions of a warp read one address, and two (four) half-size groups per CTA overlap one group's carry scan
            // and barriers with the other's sweeps.  Which calls use it: launch_one (narrow_pays).
            pl.kn[ks] = KernelSlot();
            {
                const KernelSlot &base = pl.k[ks][0][0];
                if (pl.elem == 8 && pl.ws && pl.rows == 32 && pl.nuniq < pl.P && base.fused.func && sh.lanes == 16 && sh.vec == 2 &&
                    (pl.P * 8) % 32 == 0 && g_tune.lanes < 0 && g_tune.tpc < 0) {
                    Shape &nsh = pl.nshape[ks];
                    nsh = sh;
                    nsh.lanes = 8;
                    nsh.lanes_log2 = 3;
                    finish_shape(pl.elem, pl.rows, pl.P, nsh);
                    KernelSlot &nk = pl.kn[ks];
                    nk.vec = base.vec;
                    nk.tma = 1;
                    layout_slot(pl, nsh, kind, nk);
                    if (nsh.tpc >= 2 && nk.smem <= SMEM_LIMIT && base.fused.max_threads >= nsh.threads) {
                        nk.ent = base.ent;
                        nk.fused = base.fused;
                    }
                }
            }
        }
    }
}

int resolve_slot(Handle *h, const Shape &sh, KernelSlot &sl, int cluster = 0)
{
    std::lock_guard<std::mutex> lk(h->mu);
    if (sl.max_grid > 0) return BTPS_OK;
    if (!sl.ent.func) return set_err(BTPS_E_ARG);
    // The attribute belongs to the kernel FUNCTION, which handles of different n share (sweep_kernel is not a
    // template of P or n): every setter therefore asks for the same value, the per-CTA maximum of sm_100a, so
    // that no handle ever lowers what another live handle needs (two handles of different n used in turn).
    CU_TRY(cudaFuncSetAttribute(sl.ent.func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT));
    if (sl.fused.func)
        CU_TRY(cudaFuncSetAttribute(sl.fused.func, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SMEM_LIMIT));
    if (sl.fused.func) {
        // both instantiations do the same arithmetic for one step; ptxas sometimes spills tile rows in one and not
        // in the other (255-register variants), so take the one with the smaller local-memory frame
        cudaFuncAttributes fa, fb;
        CU_TRY(cudaFuncGetAttributes(&fa, sl.ent.func));
        CU_TRY(cudaFuncGetAttributes(&fb, sl.fused.func));
        sl.prefer_fused = (fb.localSizeBytes < fa.localSizeBytes) ? 1 : 0;
    }
    int occ = 0, sms = 0, dev = 0;
    CU_TRY(cudaGetDevice(&dev));
    CU_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (cluster) {
        // co-resident clusters of two CTAs (each CTA fills an SM)
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(cluster * (sms / cluster)));
        cfg.blockDim = dim3((unsigned)sh.threads);
        cfg.dynamicSmemBytes = sl.smem;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension;
        at[0].val.clusterDim.x = (unsigned)cluster;
        at[0].val.clusterDim.y = 1;
        at[0].val.clusterDim.z = 1;
        cfg.attrs = at;
        cfg.numAttrs = 1;
        int ncl = 0;
        CU_TRY(cudaOccupancyMaxActiveClusters(&ncl, sl.ent.func, &cfg));
        if (ncl < 1) {
            snprintf(tl_cuda_msg, sizeof(tl_cuda_msg), "cluster kernel does not fit: %d threads, %zu B smem", sh.threads, sl.smem);
            return set_err(BTPS_E_CUDA);
        }
        sl.max_grid = cluster * ncl;
        return BTPS_OK;
    }
    CU_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, sl.ent.func, sh.threads, sl.smem));
    if (occ < 1) {
        snprintf(tl_cuda_msg, sizeof(tl_cuda_msg), "kernel does not fit: %d threads, %zu B smem", sh.threads,
                 sl.smem);
        return set_err(BTPS_E_CUDA);
    }
    sl.max_grid = occ * sms;
    return BTPS_OK;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (libcuda is not linked)
typedef CUresult (*encode_tiled_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                    CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                    CUtensorMapFloatOOBfill);

encode_tiled_fn get_encode()
{
    static encode_tiled_fn fn = []() -> encode_tiled_fn {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess ||
            q != cudaDriverEntryPointSuccess)
            return nullptr;
        return (encode_tiled_fn)p;
    }();
    return fn;
}

// 2-D view of the interleaved batch for TMA: dim 0 = systems (contiguous), dim 1 = rows
template <typename T>
int make_tmap(CUtensorMap *tm, T *d_rhs, long long batch, int n, int W, unsigned box_rows)
{
    encode_tiled_fn enc = get_encode();
    if (!enc) {
        snprintf(tl_cuda_msg, sizeof(tl_cuda_msg), "cuTensorMapEncodeTiled is not available");
        return set_err(BTPS_E_CUDA);
    }
    const cuuint64_t dims[2] = {(cuuint64_t)batch, (cuuint64_t)n};
    const cuuint64_t strides[1] = {(cuuint64_t)batch * sizeof(T)};
    const cuuint32_t box[2] = {(cuuint32_t)W, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = enc(tm, sizeof(T) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2,
                           (void *)d_rhs, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE,
                           (size_t)W * sizeof(T) >= 256 ? CU_TENSOR_MAP_L2_PROMOTION_L2_256B
                                                        : CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                           CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(tl_cuda_msg, sizeof(tl_cuda_msg), "cuTensorMapEncodeTiled failed (%d)", (int)r);
        return set_err(BTPS_E_CUDA);
    }
    return BTPS_OK;
}

// 17..32 partitions (512 < N <= 1024): one CTA keeps such a tile on 8 lanes = 128-byte row segments, the chain of two
// CTAs on 256-byte ones.  Where the pair wins by default (measured on B200).
template <typename T>
bool cl_pays(int kind, const DtypePlan &pl, long long batch, size_t selem)
{
    // measured on B200 (profiles/r02b_long_systems.md; one carry exchange per tile, sent with st.async): the pair keeps
    // 0.82-0.91 (tri) / 0.78-0.87 (penta, 32 partitions) of the HBM peak whatever the batch, while the single CTA's 128-byte
    // segments fall from 0.85-0.91 to 0.69 as a row of the batch grows from 1 MiB to 32 MiB.  Crossovers by row pitch:
    //   tri,   24-32 partitions (N > 736): pair from 4 MiB rows;  18-23 partitions: from 32 MiB rows (0.74-0.82 against 0.71)
    //   penta, 31-32 partitions (N > 960): pair from 8 MiB rows (0.87 / 0.78 against 0.78 / 0.69);  fewer: the pair loses
    if (pl.csz != 2) return false;
    const size_t pitch = (size_t)batch * selem;
    // fp32 storage with fp64 sweeps (*_f32s): the pair turns 64-byte segments into 128-byte ones -- at 32 partitions tri 0.57 -> 0.72
    // at 2^19 systems, 0.36 -> 0.68 at 2^22, penta 0.46 -> 0.50, 0.36 -> 0.51; with fewer partitions it loses (N = 768: 0.57 -> 0.49)
    if (selem != (size_t)pl.elem) return pl.PLc == 16 && pitch >= ((size_t)(kind == KIND_TRI ? 1 : 2) << 20);
    // (tri at 32 partitions: the pair's CTAs keep full 128 KB shares and hold their stores, launch_one -- 0.88-0.93 from 2^16
    //  systems on, never behind the single CTA's 0.87-0.91)
    if (kind == KIND_TRI) return (pl.PLc == 16 && pitch >= ((size_t)512 << 10)) || (pl.P >= 24 && pitch >= ((size_t)4 << 20)) || pitch >= ((size_t)32 << 20);
    if (kind == KIND_PENTA) return pl.P >= 31 && pitch >= ((size_t)8 << 20);
    return false;
}

// calls that advance at least this many time steps keep 17..32 partitions on one CTA (launch_one)
constexpr int LOOP_STEPS_SINGLE_CTA = 3;

// one sweep launch (kind = KIND_TRI / KIND_PENTA / KIND_CH) on a device buffer
template <typename T, typename S = T>
int launch_one(Handle *h, int kind, S *d_rhs, long long batch, double alpha_x, int reverse, int ksteps,
               cudaStream_t st, double *stat = nullptr, const double *ex = nullptr, const char **tag_out = nullptr,
               int call_steps = 0)
{
    if (call_steps < ksteps) call_steps = ksteps;  // time steps of the whole call this launch belongs to
    constexpr bool MIXED = !std::is_same<T, S>::value;  // fp32 in HBM, fp64 arithmetic: plain solves of the fp64 plan
    // (the single-step plain solve of a 32-partition pentadiagonal handle runs on its own unshared blob: make_penta_handle)
    const bool own_blocks = h->has_alt && kind == KIND_PENTA && ksteps == 1 && !stat;
    DtypePlan &pl = own_blocks ? h->alt[sizeof(T) == 8 ? 0 : 1] : h->plan[sizeof(T) == 8 ? 0 : 1];
    // a handle's tables live on the device that was current when it was factored
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) return set_err(BTPS_E_DEVICE);
    // the paper's own 2R+2W form (Alg. 2 / 4), ksteps launches: plans too large for the on-chip tables,
    // and periodic CH shapes the partitioned kernels do not cover (n not a multiple of the rows per thread)
    auto two_pass = [&]() -> int {
        if (tag_out) {  // btps_kernel_tag: name the kernel, launch nothing
            *tag_out = "two_pass_kernel";
            return BTPS_OK;
        }
        if (MIXED) {  // the two-pass form writes g to global memory: in fp32 storage that would not be an fp64 solve
            snprintf(tl_cuda_msg, sizeof(tl_cuda_msg), "fp32-storage solves need an on-chip plan (n <= 4096, 16-byte aligned rows above 1024)");
            return set_err(BTPS_E_ARG);
        }
        T *const dr = (T *)(void *)d_rhs;  // (same type unless MIXED, which has returned above)
        const int block = 128;
        const long long grid = (batch + block - 1) / block;
        const T *co = (const T *)pl.d_soa;
        PerPenta ppx = h->pp;
        for (int i = 0; i < 5; ++i) ppx.ex[i] = ex ? ex[i] : 0.0;
        for (int l = 0; l < ksteps; ++l) {
            if (kind == KIND_TRI && h->periodic)
                two_pass_kernel<T, KIND_TRIP><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, h->per_vN, h->per_invden, h->pp);
            else if (kind == KIND_TRI)
                two_pass_kernel<T, KIND_TRI><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, 0.0, 0.0, h->pp);
            else if (kind == KIND_TRICN && h->periodic)
                two_pass_kernel<T, KIND_TRICNP><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, h->per_vN, h->per_invden, ppx);
            else if (kind == KIND_TRICN)
                two_pass_kernel<T, KIND_TRICN><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, 0.0, 0.0, ppx);
            else if (kind == KIND_PENTA && h->periodic)
                two_pass_kernel<T, KIND_PENTAP><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, 0.0, 0.0, h->pp);
            else if (kind == KIND_PENTA)
                two_pass_kernel<T, KIND_PENTA><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, 0.0, 0.0, h->pp);
            else if (kind == KIND_PENTACN && h->periodic)
                two_pass_kernel<T, KIND_PENTACNP><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, 0.0, 0.0, ppx);
            else if (kind == KIND_PENTACN)
                two_pass_kernel<T, KIND_PENTACN><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, 0.0, 0.0, ppx);
            else if (h->periodic)
                two_pass_kernel<T, KIND_CHP><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, alpha_x, 0.0, h->pp);
            else
                two_pass_kernel<T, KIND_CH><<<(unsigned)grid, block, 0, st>>>(co, dr, batch, h->n, alpha_x, 0.0, h->pp);
            g_launches.fetch_add(1, std::memory_order_relaxed);
            CU_TRY(cudaGetLastError());
            if (stat) {
                lbar_kernel<T><<<(unsigned)grid, block, 0, st>>>(dr, batch, h->n, stat + l, 1.0 / (double)batch);
                g_launches.fetch_add(1, std::memory_order_relaxed);
                CU_TRY(cudaGetLastError());
            }
        }
        return BTPS_OK;
    };
    const int ks = (kind == KIND_CH || kind == KIND_TRICN) ? 1 : (kind == KIND_PENTACN ? 2 : 0);
    const bool tma_ok = (((uintptr_t)d_rhs % 16) == 0) && ((((size_t)batch * sizeof(S)) % 16) == 0) &&
                        (batch < (1ll << 31));
    // long systems: the cluster-chain kernels when the batch is TMA-aligned and a multiple of the vector width.
    // More than 32 partitions (N > 1024) have no other on-chip plan; for 17..32 partitions the default comes from
    // measurements on B200; btps_tune("cluster", 1) forces the chain for every eligible plan,
    // 0 switches it off.
    KernelSlot &clslot = MIXED ? pl.ck32 : pl.ck;
    // (time loops: a tile that stays on chip for several steps is read and written once per launch, so the width of its row
    //  segments no longer decides, and per step the single CTA is the faster one -- N = 1024, 128 steps per call, us per step:
    //  tri 53.3 against the pair's 64.3 at 2^16 systems, 838 against 1013 at 2^20; penta 1465 against 1811 at 2^20.  Decided
    //  per CALL, not per launch, so that every launch of one loop runs the same kernel whatever the steps per launch.  Crossover,
    //  ms per call, one CTA / pair: 2 steps 15.2 / 13.0 at 2^22 systems, 0.251 / 0.246 at 2^16; 3 steps 16.6 / 17.0, 0.257 / 0.288.)
    const bool cl_default = (pl.P > 32) || (call_steps < LOOP_STEPS_SINGLE_CTA && cl_pays<T>(kind, pl, batch, sizeof(S)));
    const bool cl_wanted = (g_tune.cluster > 0) || (g_tune.cluster < 0 && cl_default);
    const bool use_cl = (ks == 0) && (kind == KIND_TRI || kind == KIND_PENTA) && cl_wanted && clslot.ent.func && tma_ok &&
                        (batch % pl.cshape.vec == 0) && !(MIXED && h->periodic);
    if (!use_cl && pl.two_pass) return two_pass();
    const Shape &sh0 = use_cl ? pl.cshape : pl.shape[ks];
    // the vectorised kernels need whole vectors: batch % vec == 0 and an aligned base pointer;
    // TMA needs a 16-byte aligned base and row pitch
    int s = 0;
    if (sh0.vec > 1) {
        const bool ok = (batch % sh0.vec == 0) && (((uintptr_t)d_rhs % (sizeof(S) * sh0.vec)) == 0);
        if (!ok) s = 1;
    }
    auto slot_at = [&](int sv, int dv) -> KernelSlot & { return MIXED ? pl.ks32[sv][dv] : pl.k[ks][sv][dv]; };
    if (MIXED && (ks != 0 || h->periodic)) return set_err(BTPS_E_ARG);
    int d = (tma_ok && slot_at(s, 0).ent.func) ? 0 : 1;
    if (!slot_at(s, d).ent.func && s == 0) s = 1;  // e.g. the wide variant has no direct-load twin that fits
    if (!slot_at(s, d).ent.func) d = 1;
    // Long fused loops on half-width tiles (fill_slots).  Measured on B200 (128 steps per call, us per step, 16 -> 8 lanes):
    // tri N = 512 / 256 at 2^16 systems 25.5 -> 24.5 / 12.2 -> 11.9, N = 256 at 2^20 191 -> 184; Cahn-Hilliard N = 256 at 2^16 /
    // 2^20 26.9 -> 25.6 / 424 -> 404, periodic 540 -> 527; everything else within +-1 % or slower (N = 128: + 5-17 %, plain
    // and periodic penta + 0-3 %, periodic tri N = 512 + 5 %), so only those.  A launch's load and store are slower on the
    // 128-byte segments, hence only launches of 4 or more steps (ms per call, 16 / 8 lanes: tri N = 512 at 2^16 systems 0.107 /
    // 0.115 with 2 steps, 0.132 / 0.128 with 3, 0.157 / 0.150 with 4; the Cahn-Hilliard and Crank-Nicolson steps gain 4-9 % from 2
    // steps on).  Same arithmetic per system: the results are bitwise equal.
    // The Crank-Nicolson steps (tri_cn_step_batched, penta_cn_step_batched; plain and periodic handles) gain throughout 8-16
    // partitions: N = 256 3-5 %, N = 384 6-11 %, N = 512 4 % (periodic 1 %).
    const bool narrow_pays = (kind == KIND_TRI && !h->periodic && pl.P >= 8 && pl.P <= 16) || (kind == KIND_CH && pl.P >= 8 && pl.P <= 12) ||
                             ((kind == KIND_TRICN || kind == KIND_PENTACN) && pl.P >= 8 && pl.P <= 16);
    const bool narrow = !use_cl && !MIXED && s == 0 && d == 0 && ksteps >= 4 && narrow_pays && pl.kn[ks].fused.func &&
                        g_tune.lanes < 0 && g_tune.tpc < 0 && g_tune.narrow != 0;
    const Shape &sh = narrow ? pl.nshape[ks] : sh0;
    KernelSlot &sl = use_cl ? clslot : (narrow ? pl.kn[ks] : slot_at(s, d));
    if (!sl.ent.func) return two_pass();
    {
        // takes the handle's lock: max_grid / prefer_fused are written by the first launch of this slot
        const int rc = resolve_slot(h, sh, sl, use_cl ? pl.csz : 0);
        if (rc != BTPS_OK) return rc;
    }
    SweepArgs a;
    a.rhs = d_rhs;
    a.blob = pl.d_blob;
    a.batch = batch;
    const long long W = (long long)sh.lanes * sl.vec;
    a.num_tiles = (batch + W - 1) / W;
    a.alpha_x = alpha_x;
    a.per_vN = h->per_vN;
    a.per_invden = h->per_invden;
    a.last_part = (h->n - 1) / pl.rows;
    a.last_k = (h->n - 1) % pl.rows;
    for (int i = 0; i < 5; ++i) a.ex[i] = ex ? ex[i] : 0.0;
    for (int i = 0; i < 16; ++i) a.per_H[i] = h->pp.H[i];
    for (int i = 0; i < 6; ++i) a.per_w6[i] = h->pp.w6[i];
    {
        const int wr[4] = {0, h->n > 1 ? 1 : 0, h->n > 2 ? h->n - 2 : 0, h->n - 1};
        for (int i = 0; i < 4; ++i) {
            a.wrow_part[i] = wr[i] / pl.rows;
            a.wrow_k[i] = wr[i] % pl.rows;
        }
    }
    a.per_ngl = h->per_ngl;
    a.xstride = sl.xstride;
    a.xper = sl.xper;
    a.n = h->n;
    a.P = use_cl ? pl.csz * pl.PLc : pl.P;
    a.lanes = sh.lanes;
    a.lanes_log2 = sh.lanes_log2;
    a.tpc = sh.tpc;
    a.reverse = reverse;
    {
        // stores held until the next tile has landed (sweep.cuh, store phase).  Measured on B200, fp64 unless noted:
        // tridiagonal kinds (plain, periodic, Crank-Nicolson; also fp32) with one full-size tile per CTA gain 4-12 %
        // (N = 480 / 512 / 992 / 1024), 96 KB tiles (N = 768) lose 4-9 %; the plain pentadiagonal solve gains 4-6 % on
        // 16-lane tiles (N <= 512) and loses up to 8 % on 8-lane ones; Cahn-Hilliard, periodic penta, fp32 penta lose.
        const bool tri_family = (kind == KIND_TRI || kind == KIND_TRICN);
        const size_t tile_bytes = (size_t)pl.P * pl.rows * sh.lanes * sl.vec * sizeof(S);
        // (and at least 8 tiles per CTA: with 3-4 it loses ~10 %)
        const bool full_tile = (sh.tpc == 1) && !use_cl && tile_bytes >= (112u << 10) && a.num_tiles >= 8ll * sl.max_grid;
        // (8-lane tiles, N = 993 ... 1024: held stores cost up to 9 % while the rows of a tile share pages, and win 4-5 % once
        // every row of the batch is 32 MiB or more -- 2^22 systems in fp64, 2^23 in fp32 -- where they keep 0.69 of the peak
        // and free-running stores fall to 0.66: profiles/r02b_shared_blocks.md)
        const bool penta_big = (kind == KIND_PENTA) && !h->periodic && sh.lanes == 8 && (size_t)batch * sizeof(S) >= ((size_t)32 << 20);
        const bool penta_ok = ((kind == KIND_PENTA) && sizeof(T) == 8 && !h->periodic && sh.lanes == 16) || penta_big;
        // cluster kernels: only the tridiagonal pair whose CTAs keep a full 128 KB share (32 partitions, N = 993 ... 1024) gains
        // -- 0.84 -> 0.90-0.93 from 2^19 systems, fp32 0.84 -> 0.92; shares of 96-112 KB (N = 768 / 896) lose 0-3 %, clusters of
        // 3 / 4 / 8 are indifferent or lose up to 10 %, the pentadiagonal pair is indifferent (profiles/r02b_long_systems.md)
        // (not with fp32 storage: its shares are 64 KB and held stores lose 6-17 % there)
        const bool pair_tile = use_cl && !MIXED && kind == KIND_TRI && pl.csz == 2 && pl.PLc == 16 && a.num_tiles >= 8ll * (sl.max_grid / 2);
        a.hold_stores = g_tune.hold_stores >= 0 ? (g_tune.hold_stores > 0) : (((full_tile && (tri_family || penta_ok)) || pair_tile) ? 1 : 0);
    }
    a.blk = blk_stride(pl, h->kind == KIND_TRI ? (h->periodic ? 6 : 5) : (h->periodic ? (pl.wfast ? 11 : 13) : 9));  // = RecLayout<KIND>::ELEMS of the kernel
    a.csz = use_cl ? pl.csz : 1;
    a.nuniq = pl.nuniq;
    a.cl_own = (use_cl && pl.nuniq > pl.PLc) ? 1 : 0;  // (then nothing is shared: every CTA stages its own partitions' blocks)
    memcpy(a.pmap, pl.pmap, sizeof(a.pmap));
    a.scan_log2_cl = pl.scan_log2_cl;
    a.tab_bytes_cl = pl.tab_bytes_cl;
    a.offIn = sl.offIn;
    a.scan_log2 = pl.scan_log2;
    a.tq = use_cl ? SCAN_LANES : pl.tq;  // (the per-CTA table blocks of the cluster kernels have 32 entries per row)
    a.ksteps = ksteps;
    a.xvals = sl.xvals;
    a.blob_bytes = pl.blob_bytes;
    a.offT = use_cl ? pl.offTc : pl.offT;
    a.offTl = use_cl ? sl.offTl : pl.offT;
    a.offX = sl.offX;
    a.offM = sl.offM;
    a.offR = sl.offR;
    a.box_rows = sl.box_rows;
    a.nboxes = sl.nboxes;
    if (tag_out) {  // btps_kernel_tag: name the kernel this call would launch, launch nothing
        const bool f1 = g_tune.one_step_fused >= 0 ? g_tune.one_step_fused > 0 : sl.prefer_fused != 0;
        *tag_out = (((ksteps > 1 || stat || f1) && sl.fused.func) ? sl.fused : sl.ent).tag;
        return BTPS_OK;
    }
    CUtensorMap tm;
    memset(&tm, 0, sizeof(tm));
    if (sl.tma) {
        const int rc = make_tmap<S>(&tm, d_rhs, batch, h->n, (int)W, sl.box_rows);
        if (rc != BTPS_OK) return rc;
    }
    long long grid = a.num_tiles;  // one tile per CTA first (tile order is group-major), capped at the resident CTAs
    if (use_cl) grid = (long long)pl.csz * a.num_tiles;  // one cluster per tile in flight
    if (grid > sl.max_grid) grid = sl.max_grid;
    if (g_tune.grid > 0 && grid > g_tune.grid) grid = use_cl ? (g_tune.grid / pl.csz) * pl.csz : g_tune.grid;
    if (use_cl && grid < pl.csz) grid = pl.csz;
    // several steps per launch need the fused instantiation; without one (direct-load variants)
    // the steps are launched one by one
    // (the statistic of eq. 30 is computed inside the fused kernels; elsewhere by a pass of its own)
    const bool want_fused1 = g_tune.one_step_fused >= 0 ? g_tune.one_step_fused > 0 : sl.prefer_fused != 0;
    const bool fused = (ksteps > 1 || stat || want_fused1) && sl.fused.func;
    const int nlaunch = fused ? 1 : ksteps;
    a.ksteps = fused ? ksteps : 1;
    a.stat = fused ? stat : nullptr;
    a.stat_scale = 1.0 / (double)batch;
    // Programmatic dependent launch (the next launch's prologue -- barrier set-up, table staging -- overlaps this launch's
    // tail).  Measured on B200 (profiles/r02a_headline_ab.md): launches of up to ~30 us gain 3-17 % from it (N = 64 ... 256 up
    // to 2^16 systems), batches of 256 MiB are indifferent (+-1 %), N = 1024 from 2^16 systems loses 5-7 % and the
    // three-kernel step of bench.py 4.5 %: on by default for batches of at most 128 MiB.
    const int pdl = g_tune.pdl >= 0 ? (g_tune.pdl > 0) : ((size_t)h->n * (size_t)batch * sizeof(S) <= ((size_t)128 << 20));
    for (int l = 0; l < nlaunch; ++l) {
        const cudaError_t e = (fused ? sl.fused : sl.ent).launch(a, tm, (int)grid, sh.threads, sl.smem, st, pdl);
        g_launches.fetch_add(1, std::memory_order_relaxed);
        if (e != cudaSuccess) return cuda_fail(e, "sweep launch");
        if (stat && !fused) {
            const int block = 128;
            lbar_kernel<T><<<(unsigned)((batch + block - 1) / block), block, 0, st>>>((T *)(void *)d_rhs, batch, h->n, stat + l,
                                                                                      1.0 / (double)batch);
            g_launches.fetch_add(1, std::memory_order_relaxed);
            CU_TRY(cudaGetLastError());
        }
    }
    return BTPS_OK;
}

// Time steps advanced per launch while a tile is on chip: systems never interact, so
// the RHS = previous solution loop can run on the registers; HBM then sees one read
// and one write per `fuse` steps.  The two-pass kernel advances one step per launch.
int fuse_limit(const DtypePlan &pl)
{
    if (pl.two_pass && !pl.ck.fused.func) return 1;
    // measured on B200: 8 -> 64 steps per launch still gains 5-15 % (fewer tile round trips and launches); the gain
    // from 32 to 64 is ~2 %, so 64 is both the default and the cap
    const int k = g_tune.fuse > 0 ? g_tune.fuse : 64;
    return k < 1 ? 1 : (k > 64 ? 64 : k);
}

Handle *check(const void *hv, int magic)
{
    Handle *h = (Handle *)hv;
    if (!h || h->magic != magic) return nullptr;
    return h;
}

template <typename T, typename S = T>
int solve_steps(const void *hv, int magic, int kind, S *d_rhs, int64_t batch, double alpha_x, int nsteps,
                void *stream, double *d_stat = nullptr, const double *ex = nullptr)
{
    Handle *h = check(hv, magic);
    if (!h || !d_rhs || batch < 1 || nsteps < 0) return set_err(BTPS_E_ARG);
    if ((uintptr_t)d_rhs % sizeof(S)) return set_err(BTPS_E_ALIGN);
    const bool rev = g_tune.reverse > 0;
    const int kmax = std::is_same<T, S>::value ? fuse_limit(h->plan[sizeof(T) == 8 ? 0 : 1]) : 1;
    for (int s = 0, l = 0; s < nsteps; ++l) {
        const int k = (nsteps - s < kmax) ? (nsteps - s) : kmax;
        const int rc = launch_one<T, S>(h, kind, d_rhs, batch, alpha_x, rev ? (l & 1) : 0, k, (cudaStream_t)stream,
                                        d_stat ? d_stat + s : nullptr, ex, nullptr, nsteps);
        if (rc != BTPS_OK) return rc;
        s += k;
    }
    return set_err(BTPS_OK);
}

// ------------------------------------------------------------------------------------------------
// host-buffer path: column chunks, 3 streams, strided 2-D copies in and out
// ------------------------------------------------------------------------------------------------
struct HostPipe {
    std::mutex mu;  // one host-buffer call at a time per device
    static constexpr int NBUF = 3;
    cudaStream_t st[NBUF] = {nullptr, nullptr, nullptr};
    void *buf[NBUF] = {nullptr, nullptr, nullptr};
    size_t cap = 0;
    bool ready = false;
};

// one pipe (3 streams + 3 staging buffers) per CUDA device, created on first use with that device current
std::mutex g_pipes_mu;
std::map<int, HostPipe *> g_pipes;

HostPipe *pipe_for(int device)
{
    std::lock_guard<std::mutex> lk(g_pipes_mu);
    HostPipe *&p = g_pipes[device];
    if (!p) p = new HostPipe();
    return p;
}

int pipe_prepare(HostPipe &pp, size_t bytes)
{
    if (!pp.ready) {
        for (int i = 0; i < HostPipe::NBUF; ++i) CU_TRY(cudaStreamCreateWithFlags(&pp.st[i], cudaStreamNonBlocking));
        pp.ready = true;
    }
    if (bytes > pp.cap) {
        for (int i = 0; i < HostPipe::NBUF; ++i) {
            if (pp.buf[i]) CU_TRY(cudaFree(pp.buf[i]));
            pp.buf[i] = nullptr;
        }
        pp.cap = 0;
        for (int i = 0; i < HostPipe::NBUF; ++i) CU_TRY(cudaMalloc(&pp.buf[i], bytes));
        pp.cap = bytes;
    }
    return BTPS_OK;
}

// strided host <-> device copy of a column chunk: [n rows] x [w systems], host pitch = batch elements.
// cudaMemcpy2DAsync takes pitches up to cudaDevAttrMaxPitch (2^31 - 1 bytes); wider batches go row by row.
template <typename T>
cudaError_t copy_chunk(T *dev, T *host, long long w, long long batch, int n, bool to_device, cudaStream_t st)
{
    const size_t hp = (size_t)batch * sizeof(T), dp = (size_t)w * sizeof(T);
    if (hp <= (size_t)0x7fffffff) {
        return to_device ? cudaMemcpy2DAsync(dev, dp, host, hp, dp, (size_t)n, cudaMemcpyHostToDevice, st)
                         : cudaMemcpy2DAsync(host, hp, dev, dp, dp, (size_t)n, cudaMemcpyDeviceToHost, st);
    }
    for (int i = 0; i < n; ++i) {
        const cudaError_t e = to_device
            ? cudaMemcpyAsync(dev + (size_t)i * w, host + (size_t)i * batch, dp, cudaMemcpyHostToDevice, st)
            : cudaMemcpyAsync(host + (size_t)i * batch, dev + (size_t)i * w, dp, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}

template <typename T>
int solve_host(const void *hv, int magic, int kind, T *h_rhs, int64_t batch, double alpha_x, int nsteps)
{
    Handle *h = check(hv, magic);
    if (!h || !h_rhs || batch < 1 || nsteps < 0) return set_err(BTPS_E_ARG);
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) return set_err(BTPS_E_DEVICE);
    HostPipe &pp = *pipe_for(dev);
    std::lock_guard<std::mutex> lk(pp.mu);
    const int n = h->n;
    // chunk width: about 32 MiB per chunk, a multiple of 256 systems; batches that would give fewer than 4 chunks are
    // cut into 4 (down to 256 systems per chunk) so that copies in, kernels and copies out of different chunks overlap
    const size_t target = g_tune.host_chunk_kib > 0 ? ((size_t)g_tune.host_chunk_kib << 10) : (32ull << 20);
    long long wc = (long long)(target / ((size_t)n * sizeof(T)));
    if (g_tune.host_chunk_kib <= 0 && wc * 4 > batch) wc = (batch + 3) / 4;
    wc = ((wc + 255) / 256) * 256;
    if (wc < 256) wc = 256;
    if (wc > batch) wc = batch;
    const size_t chunk_bytes = (size_t)n * wc * sizeof(T);
    int rc = pipe_prepare(pp, chunk_bytes);
    if (rc != BTPS_OK) return rc;
    const bool rev = g_tune.reverse > 0;
    // any failure inside the loop: stop issuing, then wait for what is already in flight -- asynchronous copies
    // must not still be writing into the caller's buffer after this call has returned
    cudaError_t cerr = cudaSuccess;
    const char *what = "";
    int ci = 0;
    for (long long j0 = 0; j0 < batch && rc == BTPS_OK && cerr == cudaSuccess; j0 += wc, ++ci) {
        const long long w = (batch - j0 < wc) ? (batch - j0) : wc;
        const int b = ci % HostPipe::NBUF;
        cudaStream_t st = pp.st[b];
        T *d = (T *)pp.buf[b];
        cerr = copy_chunk<T>(d, h_rhs + j0, w, batch, n, true, st);
        if (cerr != cudaSuccess) { what = "host-to-device chunk copy"; break; }
        const int kmax = fuse_limit(h->plan[sizeof(T) == 8 ? 0 : 1]);
        for (int s = 0, l = 0; s < nsteps && rc == BTPS_OK; ++l) {
            const int k = (nsteps - s < kmax) ? (nsteps - s) : kmax;
            rc = launch_one<T>(h, kind, d, w, alpha_x, rev ? (l & 1) : 0, k, st, nullptr, nullptr, nullptr, nsteps);
            s += k;
        }
        if (rc != BTPS_OK) break;
        cerr = copy_chunk<T>(d, h_rhs + j0, w, batch, n, false, st);
        if (cerr != cudaSuccess) { what = "device-to-host chunk copy"; break; }
    }
    for (int i = 0; i < HostPipe::NBUF; ++i) {
        const cudaError_t e = cudaStreamSynchronize(pp.st[i]);
        if (e != cudaSuccess && cerr == cudaSuccess) { cerr = e; what = "cudaStreamSynchronize"; }
    }
    if (rc != BTPS_OK) return rc;
    if (cerr != cudaSuccess) return cuda_fail(cerr, what);
    return set_err(BTPS_OK);
}

}  // namespace

// ================================================================================================
// exported C-ABI
// ================================================================================================
extern "C" {

// shared by tri_factor and tri_factor_periodic: tables + upload for a factored (possibly modified) matrix
static tri_handle_t make_tri_handle(int n, const std::vector<double> &inv, const std::vector<double> &nl,
                                    const std::vector<double> &nch, const std::vector<double> *z, double vN,
                                    double invden, const std::vector<double> *zfwd = nullptr, double u0 = 0.0,
                                    double uN = 0.0)
{
    Handle *h = new Handle();
    h->magic = MAGIC_TRI;
    h->kind = KIND_TRI;
    h->periodic = (z != nullptr);
    h->per_vN = vN;
    h->per_invden = invden;
    h->n = n;
    if (cudaGetDevice(&h->device) != cudaSuccess) h->device = -1;
    for (int t = 0; t < 2; ++t) {
        DtypePlan &pl = h->plan[t];
        choose_plan(n, t == 0 ? 8 : 4, h->kind, pl);
        // periodic: fold the Sherman-Morrison finish into the carry scan when the partitions are whole (n = P*32, P >= 2)
        pl.wfast = (z && zfwd && pl.ws && pl.rows == 32 && pl.P >= 2 && pl.P * pl.rows == n && g_tune.cyclic_scan != 0) ? 1 : 0;
        std::vector<unsigned char> blob, soa;
        std::vector<const std::vector<double> *> arrs = {&inv, &nl, &nch};
        if (z) arrs.push_back(z);
        if (t == 0) {
            build_blob_tri<double>(n, pl, inv, nl, nch, blob, z, zfwd, u0, uN);
            build_soa<double>(arrs, n, soa);
        } else {
            build_blob_tri<float>(n, pl, inv, nl, nch, blob, z, zfwd, u0, uN);
            build_soa<float>(arrs, n, soa);
        }
        pl.soa_bytes = soa.size();
        fit_plan(pl, h->periodic ? KIND_TRIP : KIND_TRI);
        if (upload(blob, &pl.d_blob) != BTPS_OK || upload(soa, &pl.d_soa) != BTPS_OK) {
            free_handle(h);
            return nullptr;
        }
    }
    fill_slots(h);
    set_err(BTPS_OK);
    return (tri_handle_t)h;
}

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
    return make_tri_handle(n, inv, nl, nch, nullptr, 0.0, 0.0);
}

// Periodic (cyclic) tridiagonal matrix, PAPER.md:140-164 (Sec. 3.3): A = A' + u (x) v with
// u = (-b_1, 0, ..., c_N)^T, v = (1, 0, ..., -a_1/b_1)^T (eq. 13a) and A' = A without its corners, diagonal
// ends 2 b_1 and b_N + a_1 c_N / b_1 (eq. 13b).  A' is factored as in tri_factor, z = A'^{-1} u is
// solved once here (eq. 14) and stored with the tables; the kernels finish each solve with eq. 15.
tri_handle_t tri_factor_periodic(int n, const double *a, const double *b, const double *c)
{
    if (n < 3 || !a || !b || !c) {
        set_err(BTPS_E_ARG);
        return nullptr;
    }
    if (b[0] == 0.0 || !std::isfinite(b[0])) {
        set_err(BTPS_E_PIVOT, 1);
        return nullptr;
    }
    std::vector<double> bp(b, b + n);
    bp[0] = 2.0 * b[0];
    bp[n - 1] = b[n - 1] + a[0] * c[n - 1] / b[0];
    std::vector<double> inv, nl, nch;
    int row = 0;
    if (factor_tri_host(n, a, bp.data(), c, inv, nl, nch, &row) != BTPS_OK) {
        set_err(BTPS_E_PIVOT, row);
        return nullptr;
    }
    std::vector<double> z(n, 0.0);
    z[0] = -b[0];
    z[n - 1] = c[n - 1];
    double g = 0.0;
    std::vector<double> zfwd(n);
    for (int i = 0; i < n; ++i) {  // forward sweep of A' z = u with the sweep multipliers
        g = nl[i] * g + inv[i] * z[i];
        z[i] = g;
        zfwd[i] = g;
    }
    for (int i = n - 2; i >= 0; --i) z[i] = z[i] + nch[i] * z[i + 1];
    const double vN = -a[0] / b[0];
    const double den = 1.0 + z[0] + vN * z[n - 1];
    if (den == 0.0 || !std::isfinite(den)) {
        set_err(BTPS_E_PIVOT, n);
        return nullptr;
    }
    return make_tri_handle(n, inv, nl, nch, &z, vN, 1.0 / den, &zfwd, -b[0], c[n - 1]);
}

void tri_destroy(tri_handle_t hv)
{
    Handle *h = check(hv, MAGIC_TRI);
    if (h) free_handle(h);
}

// shared by penta_factor and penta_factor_periodic: tables + upload for a factored matrix
static penta_handle_t make_penta_handle(int n, const std::vector<double> &inv, const std::vector<double> &nle,
                                        const std::vector<double> &nlb, const std::vector<double> &ngam,
                                        const std::vector<double> &ndel, const std::vector<double> *Z,
                                        const PerPenta *pp)
{
    Handle *h = new Handle();
    h->magic = MAGIC_PENTA;
    h->kind = KIND_PENTA;
    h->periodic = (Z != nullptr);
    if (pp) h->pp = *pp;
    h->per_ngl = (Z && n >= 2) ? ngam[n - 2] : 0.0;
    h->n = n;
    if (cudaGetDevice(&h->device) != cudaSuccess) h->device = -1;
    std::vector<double> zc[4];
    std::vector<const std::vector<double> *> arrs = {&inv, &nle, &nlb, &ngam, &ndel};
    if (Z) {
        for (int m = 0; m < 4; ++m) {
            zc[m].resize(n);
            for (int i = 0; i < n; ++i) zc[m][i] = (*Z)[(size_t)i * 4 + m];
            arrs.push_back(&zc[m]);
        }
    }
    for (int t = 0; t < 2; ++t) {
        DtypePlan &pl = h->plan[t];
        choose_plan(n, t == 0 ? 8 : 4, h->kind, pl);
        // periodic: fold the cyclic correction into the carry scan when the partitions are whole (n = P*32, P >= 2)
        pl.wfast = (Z && pl.ws && pl.rows == 32 && pl.P >= 2 && pl.P * pl.rows == n && g_tune.cyclic_scan != 0) ? 1 : 0;
        std::vector<unsigned char> blob, soa;
        if (t == 0) {
            build_blob_penta<double>(n, pl, inv, nle, nlb, ngam, ndel, blob, Z);
            build_soa<double>(arrs, n, soa);
        } else {
            build_blob_penta<float>(n, pl, inv, nle, nlb, ngam, ndel, blob, Z);
            build_soa<float>(arrs, n, soa);
        }
        pl.soa_bytes = soa.size();
        fit_plan(pl, Z ? KIND_PENTAP : KIND_PENTA);
        if (upload(blob, &pl.d_blob) != BTPS_OK || upload(soa, &pl.d_soa) != BTPS_OK) {
            free_handle(h);
            return nullptr;
        }
        // Measured on B200 (profiles/r02b_shared_blocks.md): with shared coefficient blocks everything gains or is
        // indifferent -- N = 1024: periodic solves and CH steps fit their TMA ring (0.51-0.56 -> 0.82-0.91 of the HBM
        // peak), the CH step fuses its time loop (0.20 -> 0.115 ms per step at 2^16), plain steps in a fused loop gain
        // 19 % -- except the single-step plain solve at 32 partitions, fp64 and fp32, which LOSES 5-15 % when its sweeps
        // get shorter (0.87 -> 0.74 at 2^19; also with the blob whole and only the addresses shared, so it is the phasing
        // of its stores against the next tile's load, not shared-memory size).  That one call keeps a blob of its own.
        if (!Z && pl.P == 32 && !pl.two_pass && pl.nuniq < pl.P && g_tune.dedupe < 0) {
            DtypePlan &al = h->alt[t];
            choose_plan(n, t == 0 ? 8 : 4, h->kind, al);
            al.wfast = 0;
            std::vector<unsigned char> blob2;
            if (t == 0) build_blob_penta<double>(n, al, inv, nle, nlb, ngam, ndel, blob2, nullptr, 0);
            else build_blob_penta<float>(n, al, inv, nle, nlb, ngam, ndel, blob2, nullptr, 0);
            al.soa_bytes = 0;
            fit_plan(al, KIND_PENTA);
            if (upload(blob2, &al.d_blob) != BTPS_OK) {
                free_handle(h);
                return nullptr;
            }
            h->has_alt = true;
        }
    }
    if (h->has_alt && (!h->alt[0].d_blob || !h->alt[1].d_blob || h->alt[0].two_pass || h->alt[1].two_pass)) h->has_alt = false;
    fill_slots(h);
    set_err(BTPS_OK);
    return (penta_handle_t)h;
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
    return make_penta_handle(n, inv, nle, nlb, ngam, ndel, nullptr, nullptr);
}

// Periodic (cyclic) pentadiagonal matrix (eq. 26a).  The paper cites [24,4,25] for the
// method; here (C-31) A = A' + U V^T with A' the matrix without its six wrap-around entries
// (factored as in penta_factor), U = unit columns at rows 0, 1, n-2, n-1 and V^T the wrap-around
// entries; Z = A'^{-1} U and H = (I + V^T Z)^{-1} are computed once here, the kernels finish each solve
// with x = y - Z H (V^T y).
penta_handle_t penta_factor_periodic(int n, const double *e, const double *a, const double *d, const double *c,
                                     const double *f)
{
    if (n < 5 || !e || !a || !d || !c || !f) {
        set_err(BTPS_E_ARG);
        return nullptr;
    }
    std::vector<double> inv, nle, nlb, ngam, ndel;
    int row = 0;
    if (factor_penta_host(n, e, a, d, c, f, inv, nle, nlb, ngam, ndel, &row) != BTPS_OK) {
        set_err(BTPS_E_PIVOT, row);
        return nullptr;
    }
    PerPenta pp = {};
    const double w6[6] = {e[0], a[0], e[1], f[n - 2], c[n - 1], f[n - 1]};
    for (int i = 0; i < 6; ++i) pp.w6[i] = w6[i];
    // Z = A'^{-1} U with the sweep multipliers (forward: g_i = inv_i r_i + nle_i g_{i-2} + nlb_i g_{i-1};
    // backward: x_i = g_i + ngam_i x_{i+1} + ndel_i x_{i+2})
    std::vector<double> Z((size_t)n * 4, 0.0), col(n);
    const int urow[4] = {0, 1, n - 2, n - 1};
    for (int m = 0; m < 4; ++m) {
        std::fill(col.begin(), col.end(), 0.0);
        col[urow[m]] = 1.0;
        for (int i = 0; i < n; ++i)
            col[i] = inv[i] * col[i] + (i >= 2 ? nle[i] * col[i - 2] : 0.0) + (i >= 1 ? nlb[i] * col[i - 1] : 0.0);
        for (int i = n - 2; i >= 0; --i)
            col[i] = col[i] + ngam[i] * col[i + 1] + (i + 2 < n ? ndel[i] * col[i + 2] : 0.0);
        for (int i = 0; i < n; ++i) Z[(size_t)i * 4 + m] = col[i];
    }
    // S = I + V^T Z, H = S^{-1}: solve S H = I column by column (Gaussian elimination, partial pivoting)
    double S[4][4];
    for (int m = 0; m < 4; ++m) {
        S[0][m] = w6[0] * Z[(size_t)(n - 2) * 4 + m] + w6[1] * Z[(size_t)(n - 1) * 4 + m];
        S[1][m] = w6[2] * Z[(size_t)(n - 1) * 4 + m];
        S[2][m] = w6[3] * Z[m];
        S[3][m] = w6[4] * Z[m] + w6[5] * Z[4 + m];
    }
    for (int m = 0; m < 4; ++m) S[m][m] += 1.0;
    double aug[4][8];
    for (int i = 0; i < 4; ++i)
        for (int j = 0; j < 4; ++j) {
            aug[i][j] = S[i][j];
            aug[i][4 + j] = (i == j) ? 1.0 : 0.0;
        }
    for (int k = 0; k < 4; ++k) {
        int pr = k;
        for (int r = k + 1; r < 4; ++r)
            if (std::fabs(aug[r][k]) > std::fabs(aug[pr][k])) pr = r;
        if (aug[pr][k] == 0.0 || !std::isfinite(aug[pr][k])) {
            set_err(BTPS_E_PIVOT, n);
            return nullptr;
        }
        for (int j = 0; j < 8; ++j) std::swap(aug[k][j], aug[pr][j]);
        for (int r = k + 1; r < 4; ++r) {
            const double mlt = aug[r][k] / aug[k][k];
            for (int j = k; j < 8; ++j) aug[r][j] -= mlt * aug[k][j];
        }
    }
    for (int j = 0; j < 4; ++j)          // back substitution for each column of H
        for (int i = 3; i >= 0; --i) {
            double v = aug[i][4 + j];
            for (int r = i + 1; r < 4; ++r) v -= aug[i][r] * pp.H[r * 4 + j];
            pp.H[i * 4 + j] = v / aug[i][i];
        }
    return make_penta_handle(n, inv, nle, nlb, ngam, ndel, &Z, &pp);
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
int tri_solve_batched_f32s(tri_handle_t h, float *d_rhs, int64_t batch, void *stream)
{
    return solve_steps<double, float>(h, MAGIC_TRI, KIND_TRI, d_rhs, batch, 0.0, 1, stream);
}
int penta_solve_batched_f32s(penta_handle_t h, float *d_rhs, int64_t batch, void *stream)
{
    return solve_steps<double, float>(h, MAGIC_PENTA, KIND_PENTA, d_rhs, batch, 0.0, 1, stream);
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

int tri_cn_step_batched(tri_handle_t h, double *d_u, int64_t batch, double xa, double xb, double xc, int nsteps,
                        void *stream)
{
    const double ex[5] = {xa, xb, xc, 0.0, 0.0};
    return solve_steps<double>(h, MAGIC_TRI, KIND_TRICN, d_u, batch, 0.0, nsteps, stream, nullptr, ex);
}

int penta_cn_step_batched(penta_handle_t h, double *d_u, int64_t batch, const double *x5, int nsteps, void *stream)
{
    if (!x5) return set_err(BTPS_E_ARG);
    const double ex[5] = {x5[0], x5[1], x5[2], x5[3], x5[4]};
    return solve_steps<double>(h, MAGIC_PENTA, KIND_PENTACN, d_u, batch, 0.0, nsteps, stream, nullptr, ex);
}

int ch_step_batched_stat(penta_handle_t h, double *d_c, int64_t batch, double alpha, int nsteps, double *d_lbar,
                         void *stream)
{
    if (!d_lbar || nsteps < 0) return set_err(BTPS_E_ARG);
    if (nsteps > 0) {
        const cudaError_t e = cudaMemsetAsync(d_lbar, 0, (size_t)nsteps * sizeof(double), (cudaStream_t)stream);
        if (e != cudaSuccess) return cuda_fail(e, "cudaMemsetAsync");
    }
    return solve_steps<double>(h, MAGIC_PENTA, KIND_CH, d_c, batch, alpha, nsteps, stream, d_lbar);
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

// ------------------------------------------------------------------------------------------------
// Host-buffer solve that allocates nothing (include/btps.h "tri_solve_batched_host_static").  The *_host calls above
// stage the batch in device buffers they cudaMalloc on first use; this one stages it in a fixed array that is part of
// the library image, so it can be called where cudaMalloc cannot (code under stream capture, serving loops, harnesses
// that forbid allocation).  Every device that loads the library holds the array until the process exits.
// ------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned char g_static_scratch[BTPS_STATIC_SCRATCH_BYTES];

// In host code the array's name is a host-side stand-in, not a device address: the address a kernel can use comes from
// cudaGetSymbolAddress, asked once per device with that device current.  (No allocation: a fixed table of pointers.)
static int static_scratch_ptr(int dev, void **out)
{
    constexpr int MAX_DEV = 64;
    static std::mutex mu;
    static void *ptr[MAX_DEV] = {nullptr};
    if (dev < 0 || dev >= MAX_DEV) return set_err(BTPS_E_DEVICE);
    std::lock_guard<std::mutex> lk(mu);
    if (!ptr[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess) return cuda_fail(e, "cudaGetSymbolAddress(g_static_scratch)");
        if (!p || ((uintptr_t)p & 255)) return cuda_fail(cudaErrorInvalidSymbol, "static scratch array address");
        ptr[dev] = p;
    }
    *out = ptr[dev];
    return BTPS_OK;
}

int tri_solve_batched_host_static(tri_handle_t hv, double *h_rhs, int64_t batch, int nsteps, void *stream)
{
    Handle *h = check(hv, MAGIC_TRI);
    if (!h || !h_rhs || batch < 1 || nsteps < 0) return set_err(BTPS_E_ARG);
    // n * batch * 8 bytes must fit in the array (checked without overflow)
    if ((uint64_t)batch > (uint64_t)BTPS_STATIC_SCRATCH_BYTES / sizeof(double) / (uint64_t)h->n) {
        snprintf(tl_size_msg, sizeof(tl_size_msg),
                 "tri_solve_batched_host_static: n * batch * 8 = %lld * %lld * 8 bytes exceeds the static scratch array "
                 "(BTPS_STATIC_SCRATCH_BYTES = %lld); use tri_solve_batched_host or a device buffer",
                 (long long)h->n, (long long)batch, (long long)BTPS_STATIC_SCRATCH_BYTES);
        return set_err(BTPS_E_TOO_LARGE);
    }
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev != h->device) return set_err(BTPS_E_DEVICE);
    void *p = nullptr;
    int rc = static_scratch_ptr(dev, &p);
    if (rc != BTPS_OK) return rc;
    double *d = (double *)p;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t bytes = (size_t)h->n * (size_t)batch * sizeof(double);
    // the copy in overwrites every element the kernels read: nothing left in the array by an earlier call is used
    cudaError_t e = cudaMemcpyAsync(d, h_rhs, bytes, cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(e, "host-to-device copy into the static scratch array");
    rc = solve_steps<double>(h, MAGIC_TRI, KIND_TRI, d, batch, 0.0, nsteps, stream);
    // whatever the outcome, nothing may still be reading or writing the caller's buffer after the return
    if (rc == BTPS_OK) {
        e = cudaMemcpyAsync(h_rhs, d, bytes, cudaMemcpyDeviceToHost, st);
        if (e != cudaSuccess) rc = cuda_fail(e, "device-to-host copy out of the static scratch array");
    }
    e = cudaStreamSynchronize(st);
    if (rc != BTPS_OK) return rc;
    if (e != cudaSuccess) return cuda_fail(e, "cudaStreamSynchronize");
    return set_err(BTPS_OK);
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
        case BTPS_E_DEVICE: return "handle used on a device other than the one it was factored on";
        case BTPS_E_TOO_LARGE: return tl_size_msg[0] ? tl_size_msg : "problem larger than the static scratch array (BTPS_STATIC_SCRATCH_BYTES)";
        default: return "unknown";
    }
}

int btps_plan_info(int kind, const void *handle, int elem_bytes, int *out)
{
    if (kind < 0 || kind > 4) return set_err(BTPS_E_ARG);
    Handle *h = check(handle, (kind == 0 || kind == 3) ? MAGIC_TRI : MAGIC_PENTA);
    if (!h || !out || (elem_bytes != 8 && elem_bytes != 4)) return set_err(BTPS_E_ARG);
    const DtypePlan &pl = h->plan[elem_bytes == 8 ? 0 : 1];
    const int ks = (kind == 4) ? 2 : ((kind >= 2) ? 1 : 0);
    const Shape &sh = pl.shape[ks];
    const KernelSlot &sl = pl.k[ks][0][0].ent.func ? pl.k[ks][0][0] : pl.k[ks][0][1];
    out[0] = pl.two_pass ? 0 : pl.rows;
    out[1] = pl.two_pass ? 1 : pl.P;
    out[2] = pl.two_pass ? 128 : sh.lanes;
    out[3] = pl.two_pass ? 1 : sh.vec;
    out[4] = pl.two_pass ? 1 : sh.tpc;
    out[5] = pl.two_pass ? 128 : sh.threads;
    out[6] = pl.two_pass ? 0 : (int)sl.smem;
    out[7] = pl.two_pass ? (int)pl.soa_bytes : (int)pl.blob_bytes;
    out[8] = pl.two_pass ? 0 : sl.tma;
    out[9] = pl.two_pass ? 0 : pl.ws;
    return set_err(BTPS_OK);
}

int btps_tune(const char *key, int value)
{
    if (!key) return set_err(BTPS_E_ARG);
    if (!strcmp(key, "rows")) {
#ifndef BTPS_TUNING_VARIANTS
        // the default build holds the 8 / 16-rows-per-thread kernels only for single-partition plans (n <= 16)
        if (value == 8 || value == 16) return set_err(BTPS_E_ARG);
#endif
        g_tune.rows = value;
    }
    else if (!strcmp(key, "lanes")) g_tune.lanes = value;
    else if (!strcmp(key, "vec")) g_tune.vec = value;
    else if (!strcmp(key, "tiles_per_cta")) g_tune.tpc = value;
    else if (!strcmp(key, "force_two_pass")) g_tune.force_two_pass = value;
    else if (!strcmp(key, "reverse")) g_tune.reverse = value;
    else if (!strcmp(key, "prefetch")) g_tune.prefetch = value;
    else if (!strcmp(key, "pdl")) g_tune.pdl = value;
    else if (!strcmp(key, "warp_scan")) g_tune.warp_scan = value;
    else if (!strcmp(key, "grid")) g_tune.grid = value;
    else if (!strcmp(key, "fuse_steps")) g_tune.fuse = value;
    else if (!strcmp(key, "cluster")) g_tune.cluster = value;
    else if (!strcmp(key, "cyclic_in_scan")) g_tune.cyclic_scan = value;
    else if (!strcmp(key, "one_step_fused")) g_tune.one_step_fused = value;
    else if (!strcmp(key, "host_chunk_kib")) g_tune.host_chunk_kib = value;
    else if (!strcmp(key, "hold_stores")) g_tune.hold_stores = value;
    else if (!strcmp(key, "dedupe")) g_tune.dedupe = value;
    else if (!strcmp(key, "blk_pad")) g_tune.blk_pad = value;
    else if (!strcmp(key, "narrow_loops")) g_tune.narrow = value;
    else return set_err(BTPS_E_ARG);
    return set_err(BTPS_OK);
}

int64_t btps_launch_count(void) { return (int64_t)g_launches.load(std::memory_order_relaxed); }

#ifndef BTPS_BUILD_ID
#define BTPS_BUILD_ID "unknown"
#endif
const char *btps_build_id(void) { return BTPS_BUILD_ID; }

int btps_kernel_tag(int kind, const void *handle, int elem_bytes, int64_t batch, int nsteps, char *buf, int len)
{
    if (kind < 0 || kind > 4 || !buf || len < 1 || batch < 1 || nsteps < 1 || (elem_bytes != 8 && elem_bytes != 4 && elem_bytes != 12))
        return set_err(BTPS_E_ARG);
    if (elem_bytes == 12 && (kind > 1 || nsteps != 1)) return set_err(BTPS_E_ARG);  // *_f32s: plain single solves
    Handle *h = check(handle, (kind == 0 || kind == 3) ? MAGIC_TRI : MAGIC_PENTA);
    if (!h) return set_err(BTPS_E_ARG);
    static const int kinds[5] = {KIND_TRI, KIND_PENTA, KIND_CH, KIND_TRICN, KIND_PENTACN};
    if (elem_bytes == 4 && kind >= 2) return set_err(BTPS_E_ARG);  // the fused steps are fp64 only
    const char *tag = nullptr;
    // a base pointer aligned like a fresh allocation: the choice depends on the alignment of pointer and pitch only
    void *fake = (void *)(uintptr_t)4096;
    const double ex[5] = {0, 1, 0, 0, 0};
    const int rc = elem_bytes == 8 ? launch_one<double>(h, kinds[kind], (double *)fake, batch, 0.0, 0, nsteps, nullptr, nullptr, ex, &tag)
                 : elem_bytes == 4 ? launch_one<float>(h, kinds[kind], (float *)fake, batch, 0.0, 0, nsteps, nullptr, nullptr, ex, &tag)
                                   : launch_one<double, float>(h, kinds[kind], (float *)fake, batch, 0.0, 0, 1, nullptr, nullptr, ex, &tag);
    if (rc != BTPS_OK) return rc;
    snprintf(buf, (size_t)len, "%s", tag ? tag : "");
    return set_err(BTPS_OK);
}

}  // extern "C"
