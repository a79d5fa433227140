// api.cu -- the C ABI of include/lsms_tau.h and include/lsms_tau_diag.h: argument checks, the per-handle context,
// workspace layout and the batch scheduler that walks the blocked right-looking elimination.
#include <math.h>
#include <stdint.h>
#include <string.h>
#include <algorithm>
#include <new>
#include <vector>
#include "../../include/lsms_tau.h"
#include "../../include/lsms_tau_diag.h"
#include "common.cuh"
#include "internal.h"

namespace lsms {
thread_local LaunchCounter g_launches = {0};
thread_local Ctx* t_ctx = nullptr;

// ---- optional per-kernel-class timing (lsms_profile_begin / lsms_profile_end): CUDA events recorded on
// the launch stream around each launch, so bench.py can report the Schur update's duration and share
// measured inside the step.  Classes: lsms_tau_diag.h.
ProfScope::ProfScope(int cls, cudaStream_t s, double flops) : st(s), live(t_ctx && t_ctx->prof.on) {
    if (!live) return;
    Prof& p = t_ctx->prof;
    if (p.ev.size() < 2 * (p.used + 1)) {
        cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
        p.ev.push_back(a); p.ev.push_back(b); p.cls.push_back(cls);
    }
    p.cls[p.used] = cls;
    p.flops[cls] += flops;
    cudaEventRecord(p.ev[2 * p.used], st);
}
ProfScope::~ProfScope() { if (live) { Prof& p = t_ctx->prof; cudaEventRecord(p.ev[2 * p.used + 1], st); ++p.used; } }

static inline size_t align256(size_t x) { return (x + 255) / 256 * 256; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static int isqrt_exact(int v) { int r = (int)lround(sqrt((double)v)); return (r * r == v) ? r : -1; }

static inline int eff_nb(const Ctx* c) { return c->opt[LSMS_OPT_NB_OUTER] > 0 ? c->opt[LSMS_OPT_NB_OUTER] : 64; }
static inline int eff_ib(const Ctx* c) { return c->opt[LSMS_OPT_IB_INNER] > 0 ? c->opt[LSMS_OPT_IB_INNER] : 16; }

// First enqueueing call through a handle: bind it to the current device -- opt the kernels into their shared-memory
// sizes there and create the scheduler's streams and events.
static int bind_device(Ctx* c, int dev) {
    LSMS_CUDA_OK(cudaDeviceGetAttribute(&c->sms, cudaDevAttrMultiProcessorCount, dev));
    int rc;
    if ((rc = init_attrs_gemm()) || (rc = init_attrs_lu()) || (rc = init_attrs_assemble()) || (rc = init_attrs_fused()) ||
        (rc = init_attrs_resident()) || (rc = init_attrs_panel()) ||
        (rc = init_attrs_panel_cluster())) return rc;
    // How many clusters of 1 / 2 / 4 / 8 CTAs of each cluster kernel this device -- or the SM partition this process has been
    // given of it (MPS / MIG: the paper's ranks share a GPU) -- can hold at once; 0 = such a cluster cannot
    // be launched here at all, and the scheduler then keeps to the schedules that need none.
    for (int i = 0; i < 4; ++i) {
        c->res_clusters[i] = resident_max_active_clusters(1 << i);
        c->fused_clusters[i] = fused_max_active_clusters(1 << i);
        c->pclu_clusters[i] = i ? panel_cluster_max_active_clusters(1 << i) : 0;
    }
    int lo = 0, hi = 0;
    LSMS_CUDA_OK(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    LSMS_CUDA_OK(cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming));
    for (int g = 0; g < MAX_GROUPS; ++g) {
        GroupStreams& s = c->gs[g];
        if (g > 0) LSMS_CUDA_OK(cudaStreamCreateWithFlags(&s.main, cudaStreamNonBlocking));
        LSMS_CUDA_OK(cudaStreamCreateWithPriority(&s.aux, cudaStreamNonBlocking, hi));
        LSMS_CUDA_OK(cudaEventCreateWithFlags(&s.fork, cudaEventDisableTiming));
        LSMS_CUDA_OK(cudaEventCreateWithFlags(&s.join, cudaEventDisableTiming));
        LSMS_CUDA_OK(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
    }
    c->device = dev;
    return 0;
}

// Entry of every extern "C" call that enqueues work (after its argument checks): the handle is bound to the current
// device on first use and must be used on that device afterwards.
struct CallScope {
    int rc = 0;
    explicit CallScope(Ctx* c) {
        int dev = -1;
        cudaError_t e = cudaGetDevice(&dev);
        if (e != cudaSuccess) { rc = (int)e; return; }
        if (c->device < 0) { rc = bind_device(c, dev); if (rc) return; }
        if (dev != c->device) { rc = (int)cudaErrorInvalidDevice; return; }
        t_ctx = c; g_launches.n = 0;
    }
    ~CallScope() { if (!rc && t_ctx) t_ctx->last_launches = g_launches.n; }
};

// Workspace layout for lsms_tau00_batched:
//   [pivots int32 batch*n][perm int32 batch*(4+3NB)][Ninv c128 batch*NB*NB][Tperm c128 batch*NB*n][K5 scratch]
struct TauWs { int* piv; int* perm; c128* ninv; c128* tperm; void* k5; size_t total; };
static TauWs tau_ws_layout(void* base, int NB, int n, int k, int batch) {
    TauWs w; char* p = (char*)base;
    w.piv = (int*)p; p += align256((size_t)batch * n * sizeof(int));
    w.perm = (int*)p; p += align256((size_t)batch * (4 + 3 * NB) * sizeof(int));
    w.ninv = (c128*)p; p += align256((size_t)batch * NB * NB * sizeof(c128));
    w.tperm = (c128*)p; p += align256((size_t)batch * NB * n * sizeof(c128));
    w.k5 = p; p += align256(final_inverse_ws_bytes(k, batch));
    w.total = (size_t)(p - (char*)base);
    return w;
}
// the same layout seen from item b0 on
static TauWs tau_ws_offset(const TauWs& ws, int NB, int n, int k, int b0) {
    TauWs w = ws;
    w.piv = ws.piv + (size_t)b0 * n;
    w.perm = ws.perm + (size_t)b0 * (4 + 3 * NB);
    w.ninv = ws.ninv + (size_t)b0 * NB * NB;
    w.tperm = ws.tperm + (size_t)b0 * NB * n;
    w.k5 = (char*)ws.k5 + (final_inverse_ws_bytes(k, 1) ? (size_t)b0 * k * k * sizeof(c128) : 0);
    return w;
}
static size_t tau_ws_bytes(const Ctx* c, int n, int k, int batch) { return tau_ws_layout(nullptr, eff_nb(c), n, k, batch).total; }

// Blocked right-looking elimination of the first ne = n-k columns of every item, in lock-step over
// the batch: each launch covers all items, so the latency-bound panel kernels (one CTA per item)
// fill the chip through the batch dimension while the update kernels tile every trailing matrix.
//   outer panel [J, J+W), W <= NB:
//     for each inner panel [c0, c0+w), w <= IB:                       (inside the outer panel only)
//        K2  factor the (n-c0) x w panel, pivots restricted to rows < ne; interchanges and triangular solves
//            inside the outer panel
//        K4  rank-w update of the outer panel's remaining columns
//     K3a fold the W interchanges into one row permutation; Ninv = -(L11^{-1})
//     K3b permute the trailing columns [J+W, n): new top block -> Tperm, displaced rows scattered
//     K4  U12 = -(Ninv * Tperm)        (the triangular solve as a DMMA GEMM, written into the matrix)
//     K4  Schur update A22 -= L21 U12 with inner dimension W          (>95% of the flops)
//
// Look-ahead (the batch scheduler's overlap): after the triangular solve of panel J the
// Schur update is split in two.  The columns of the NEXT panel are updated first; then the next panel is
// factored on a high-priority auxiliary stream while the main stream updates the remaining columns.  The
// latency/L2-bound panel kernels thus run underneath the DMMA-bound update instead of in front of it.
// The two streams touch disjoint columns (the panel's interchanges reach the trailing columns only in K3b,
// after the join).  The streams and events belong to the handle.

// CTAs per matrix for the panel kernel.  A cluster shortens the panel factorisation of a tall panel several times
// (rank 12450, 12 matrices: 303 -> 117 ms per step when timed alone), but its CTAs must be co-scheduled on free SMs, so
// under look-ahead it waits for the Schur update to drain instead of running beneath it and whole steps of batches
// >= 4 got SLOWER (NC 1897 -> 1928 ms, H 629 -> 654, C 440 -> 465, P 121 -> 129).  It pays when there is next to
// nothing to overlap with: one or two tall matrices (rank 12450, batch 1: 369 -> 223 ms; rank 4320: 36.9 -> 32.5 ms).
static inline int ilog2(int cl) { return cl >= 8 ? 3 : cl >= 4 ? 2 : cl >= 2 ? 1 : 0; }
static int panel_cluster_size(const Ctx* c, int m, int batch) {
    const int pc = c->opt[LSMS_OPT_PANEL_CLUSTER];
    if (c->opt[LSMS_OPT_PANEL_THREADS] < 1) return 1;
    if (pc == 1) return 1;
    int cl = 1;
    if (pc > 1) cl = pc;
    else if (batch <= 2 && m >= 4096) cl = 8;
    else if (batch <= 2 && m >= 2048) cl = 4;
    // three or four tall matrices: the panel phase is still most of what look-ahead cannot hide (rank 6750 x 4: ~80 of
    // 130 ms) and the few cluster CTAs find free SMs quickly.  Measured whole eliminations, one-CTA -> this rule:
    // rank 6750 x 3 116.0 -> 95.0 ms, x 4 129.7 -> 116.9; rank 6225 x 3 95.2 -> 80.0, x 4 105.5 -> 96.2; rank 5400 x 3
    // 60.2 -> 56.7, x 4 69.0 -> 66.4; rank 12450 x 3 542.4 -> 485.2, x 4 654.3 -> 635.2 (4 CTAs while the panel is taller
    // than 2 x 5120 rows); rank 4320 unchanged (36.2, 39.8).  A cluster below 4096 rows loses (rank 4320 x 3 with 2 CTAs
    // throughout: 38.8 vs 36.2), and so does one from six matrices on (rank 6750 x 6: 167.8 vs 165.5 ms).
    else if (batch <= 4 && m > 10240) cl = 4;
    else if (batch <= 4 && m >= 4096) cl = 2;
    if (cl > 1 && (m + cl - 1) / cl > 5120) cl = 1;         // taller than the cluster instances cover: one-CTA kernel
    if (cl > 1 && c->pclu_clusters[ilog2(cl)] < 1) cl = 1;  // such a cluster cannot be co-scheduled on this device / partition
    return cl;
}

// Tallest panel the lock-step schedule can factor: the first one, n rows.  The one-CTA panel kernels cover 16384 rows,
// the cluster kernel 5120 per CTA (8 CTAs for one or two matrices, 4 for three or four, see above); later panels are
// shorter and covered whenever the first is.  Checked by every entry point before anything is enqueued (LSMS_ERR_PANEL_TOO_TALL).
static bool rows_supported(const Ctx* c, int n, int batch) {
    return n <= 16384 || panel_cluster_size(c, n, batch) > 1;
}

// factor the outer panel [J, J+W) on stream st: inner panels of width <= IB
static int factor_panel(const Ctx* c, c128* M, int n, int batch, int J, int W, int ne, int IB, int* piv, int* info, cudaStream_t st) {
    const size_t stride = (size_t)n * n;
    const int Jend = J + W;
    GemmShape g; g.strideA = g.strideB = g.strideC = stride; g.ldA = g.ldB = g.ldC = n; g.batch = batch; g.beta0 = 0;
    for (int jj = 0; jj < W; jj += IB) {
        const int c0 = J + jj, w = (W - jj < IB) ? W - jj : IB;
        int rc;
        // register-blocked K2: factors the inner panel, applies its interchanges to the whole outer panel and
        // solves the w x w triangle for the outer panel's columns to the right;
        // small batches of tall panels: a cluster of CTAs per matrix, so that the panel phase spans the chip too
        const int cl = panel_cluster_size(c, n - c0, batch);
        if (cl > 1) { ProfScope ps(1, st); rc = launch_panel_cluster(M, stride, n, J, W, c0, w, ne, batch, piv, info, cl, st); }
        else { ProfScope ps(1, st); rc = launch_panel_reg(M, stride, n, J, W, c0, w, ne, batch, piv, info, c->opt[LSMS_OPT_PANEL_THREADS], st); }
        if (rc) return rc;
        const int rem = Jend - (c0 + w);
        if (rem > 0) {
            g.Mr = n - (c0 + w); g.Nc = rem; g.K = w;
            g.A = M + (size_t)(c0 + w) + (size_t)c0 * n;
            g.B = M + (size_t)c0 + (size_t)(c0 + w) * n;
            g.C = M + (size_t)(c0 + w) + (size_t)(c0 + w) * n;
            { ProfScope ps(3, st, 8.0 * g.Mr * g.Nc * g.K * batch); rc = launch_schur_gemm(g, st); } if (rc) return rc;
        }
    }
    return 0;
}

// A22[:, c_lo:c_hi) -= L21 * U12[:, c_lo:c_hi) for the outer panel [J, J+W)
static int schur_update(c128* M, int n, int batch, int J, int W, int c_lo, int c_hi, cudaStream_t st) {
    if (c_hi <= c_lo) return 0;
    const int Jend = J + W;
    GemmShape g; g.strideA = g.strideB = g.strideC = (size_t)n * n; g.ldA = g.ldB = g.ldC = n; g.batch = batch; g.beta0 = 0;
    g.Mr = n - Jend; g.Nc = c_hi - c_lo; g.K = W;
    g.A = M + (size_t)Jend + (size_t)J * n;
    g.B = M + (size_t)J + (size_t)c_lo * n;
    g.C = M + (size_t)Jend + (size_t)c_lo * n;
    ProfScope ps(4, st, 8.0 * g.Mr * g.Nc * g.K * batch);
    return launch_schur_gemm(g, st);
}

// one batch group [0, batch) of items (pointers already offset to the group's first item)
static int eliminate(const Ctx* c, c128* M, int n, int k, int batch, const TauWs& ws, int* info, cudaStream_t st, const GroupStreams& gs) {
    const int ne = n - k;
    const int NB = eff_nb(c), IB = eff_ib(c);
    const size_t stride = (size_t)n * n;
    int* piv = ws.piv;
    const bool la = c->opt[LSMS_OPT_LOOKAHEAD] != 0;
    if (ne <= 0) return 0;
    // Tile alignment: the first panel is n mod 64 wide (when that is non-zero), so that every trailing matrix
    // the Schur update sees has a multiple of the 64-row DMMA tile in both dimensions; only the last,
    // smallest updates carry a ragged tile (n = 2160, 64-row tiles: 34 tile rows of which one 3/4 full -> 33 full).
    int W0 = ne < NB ? ne : NB;
    if (c->opt[LSMS_OPT_ALIGN_FIRST] && NB % 64 == 0 && n % 64 != 0 && n % 64 < W0) W0 = n % 64;
    int rc = factor_panel(c, M, n, batch, 0, W0, ne, IB, piv, info, st); if (rc) return rc;
    { ProfScope ps(6, st); rc = launch_panel_post(M, stride, n, 0, W0, batch, piv, ws.perm, ws.ninv, NB, st); } if (rc) return rc;
    for (int J = 0, W = W0; J < ne; J += W, W = (ne - J < NB) ? ne - J : NB) {
        const int Jend = J + W;                               // Jend <= ne < n
        { ProfScope ps(6, st); rc = launch_row_permute(M, stride, n, J, W, Jend, n, batch, ws.perm, ws.tperm, (size_t)NB * n, NB, st); } if (rc) return rc;
        GemmShape t; t.batch = batch; t.beta0 = 1; t.triA = 1;
        t.A = ws.ninv; t.strideA = (size_t)NB * NB; t.ldA = NB;
        t.B = ws.tperm + (size_t)Jend * NB; t.strideB = (size_t)NB * n; t.ldB = NB;
        t.C = M + (size_t)J + (size_t)Jend * n; t.strideC = stride; t.ldC = n;
        t.Mr = W; t.Nc = n - Jend; t.K = W;
        { ProfScope ps(7, st, 8.0 * t.Mr * t.Nc * t.K * batch); rc = launch_schur_gemm(t, st); } if (rc) return rc;
        const int W2 = (Jend < ne) ? ((ne - Jend < NB) ? ne - Jend : NB) : 0;     // width of the next panel
        if (W2 > 0 && la) {
            rc = schur_update(M, n, batch, J, W, Jend, Jend + W2, st); if (rc) return rc;
            LSMS_CUDA_OK(cudaEventRecord(gs.fork, st));
            LSMS_CUDA_OK(cudaStreamWaitEvent(gs.aux, gs.fork, 0));
            rc = factor_panel(c, M, n, batch, Jend, W2, ne, IB, piv, info, gs.aux);
            // the next panel's net permutation and -(L11^-1) are also built under the update: perm/Ninv of
            // panel J were last read by the permutation / triangular solve above, before the fork
            if (!rc) { ProfScope ps(6, gs.aux); rc = launch_panel_post(M, stride, n, Jend, W2, batch, piv, ws.perm, ws.ninv, NB, gs.aux); }
            // the auxiliary stream is joined back even when a launch failed, so that the caller's stream stays ordered
            cudaError_t e1 = cudaEventRecord(gs.join, gs.aux);
            int rc2 = rc ? 0 : schur_update(M, n, batch, J, W, Jend + W2, n, st);
            cudaError_t e2 = cudaStreamWaitEvent(st, gs.join, 0);
            if (rc) return rc;
            if (rc2) return rc2;
            LSMS_CUDA_OK(e1); LSMS_CUDA_OK(e2);
        } else {
            rc = schur_update(M, n, batch, J, W, Jend, n, st); if (rc) return rc;
            if (W2 > 0) {
                rc = factor_panel(c, M, n, batch, Jend, W2, ne, IB, piv, info, st); if (rc) return rc;
                { ProfScope ps(6, st); rc = launch_panel_post(M, stride, n, Jend, W2, batch, piv, ws.perm, ws.ninv, NB, st); } if (rc) return rc;
            }
        }
    }
    return 0;
}

// Batch groups (the batch scheduler's second level).  In lock-step over the whole batch
// the poorly parallel phases of every item (net permutation, triangular solve, the narrow look-ahead slice,
// the last small panels) coincide and leave the chip idle.  The batch is therefore cut into `groups`
// contiguous groups that run the same elimination on separate streams: while one group is in such a phase
// the hardware scheduler fills the SMs with another group's Schur-update tiles.  The groups touch disjoint
// items; the caller's stream is forked into the group streams and joined again before the call returns.
static int pick_groups(const Ctx* c, int n, int batch) {
    int g = c->opt[LSMS_OPT_GROUPS];
    // two groups from 16 matrices on, if there is enough work to split (measured, two groups / one: 2160^2 x 16
    // 19.4 / 19.6 ms, 4320^2 x 16 114.7 / 115.5, 2160^2 x 128 115.4 / 116.2 -- but 880^2 x 16 4.13 / 3.87)
    if (g <= 0) g = (batch >= 16 && (long long)batch * n >= 32768) ? 2 : 1;
    if (g > MAX_GROUPS) g = MAX_GROUPS;
    if (g > batch) g = batch;
    return g;
}

static int eliminate_groups(Ctx* c, c128* M, int n, int k, int batch, const TauWs& ws, c128* tau, int* info, cudaStream_t st) {
    const int NB = eff_nb(c);
    const int groups = pick_groups(c, n, batch);
    const size_t stride = (size_t)n * n;
    if (groups > 1) LSMS_CUDA_OK(cudaEventRecord(c->ev_start, st));
    int rc = 0, forked = 0;
    for (int g = 0; g < groups && !rc; ++g) {
        const int b0 = (int)((long long)batch * g / groups), b1 = (int)((long long)batch * (g + 1) / groups);
        if (b1 <= b0) continue;
        cudaStream_t gst = (g == 0) ? st : c->gs[g].main;
        if (g > 0) { rc = (int)cudaStreamWaitEvent(gst, c->ev_start, 0); if (rc) break; }
        const TauWs w = tau_ws_offset(ws, NB, n, k, b0);
        rc = eliminate(c, M + (size_t)b0 * stride, n, k, b1 - b0, w, info + b0, gst, c->gs[g]);
        if (!rc) {
            ProfScope ps(5, gst);
            rc = launch_final_inverse(M + (size_t)b0 * stride, stride, n, k, b1 - b0, tau + (size_t)b0 * k * k, info + b0, w.k5, gst);
        }
        // a group stream that was forked is always joined back, also after a failed launch
        if (g > 0) { cudaEventRecord(c->gs[g].done, gst); forked = g; }
    }
    for (int g = 1; g <= forked; ++g) {
        cudaError_t e = cudaStreamWaitEvent(st, c->gs[g].done, 0);
        if (!rc && e != cudaSuccess) rc = (int)e;
    }
    return rc;
}

// ---- the batch scheduler's first decision (north_star: "packs small LIZ matrices several per SM and lets large
// ones span the whole chip").  Small-matrix mode eliminates a matrix start to finish inside one launch, `cl` CTAs per
// matrix; 0 = lock-step launches over the batch.  See fused.cu for the measurements behind the thresholds.
// Return value: 0 lock-step; cl > 0: one-launch mode through global memory / L2 (fused.cu), cl CTAs per matrix;
// -cl < 0: on-chip mode (resident.cu), the matrix in the distributed shared memory of a cluster of cl CTAs.
static int pick_small_mode(const Ctx* c, int n, int k, int batch) {
    const int sm = c->opt[LSMS_OPT_SMALL_MODE];
    if (sm == 1) return 0;
    int rcl = resident_cluster_size(n, k);
    // clusters of rcl CTAs that can be resident at once (0: the cluster cannot be launched on this device / partition)
    const int ract = rcl > 0 ? std::min(c->res_clusters[ilog2(rcl)], c->sms / rcl) : 0;
    if (ract < 1) rcl = 0;
    if (sm == 7) return rcl > 0 ? -rcl : 0;
    // Default for matrices that fit on chip (n <= ~216 with 4 SMs each), while the batch needs at most ~3.5 waves of
    // clusters: the on-chip kernel is built for latency (208^2 x 32: 0.20 ms against 0.56 ms through L2 and 0.85 ms in
    // lock-step), but it holds 4 SMs per matrix for the whole elimination, and from ~150 matrices of 208^2 on the
    // lock-step schedule has the higher throughput (128 matrices: 0.71 ms on chip, 0.78 lock-step; 192: 1.05 / 0.90;
    // 512: 2.72 / 1.64).
    if (sm == 0 && rcl > 0 && 2LL * batch <= 7LL * ract) return -rcl;
    if (sm == 0) return 0;
    if (!fused_supported(n, k, eff_nb(c), eff_ib(c))) return 0;
    if (sm >= 3) return c->fused_clusters[sm - 3] > 0 ? 1 << (sm - 3) : 0;
    if (c->fused_clusters[0] < 1) return 0;
    // sm == 2: the one-launch mode through L2 (fused.cu).  CTAs per matrix: a CTA is a quarter of an SM, so few matrices
    // get a cluster each until the chip is covered.  Tiny matrices: at most 4 -- their panel chain is serial, rank 0
    // factors under the other ranks' updates, and a third to seventh helper only adds barrier traffic (208^2 x 32:
    // 0.56 ms with 4 CTAs per matrix, 0.61 with 8).  Measured against the other schedules it never wins by default:
    // 208^2 x 32: 0.56 ms (on chip 0.25); 208^2 x 1024: 4.1 ms (lock-step 3.5); 880^2 x 512: 55 ms (lock-step 39: its
    // per-matrix latency phases run with 128 threads and do not overlap the other matrices' updates as hoped).
    const long long slots = 4LL * c->sms;
    const int cl_max = fused_is_tiny(n) ? 4 : 8;
    int cl = 1;
    while (cl < cl_max && (long long)batch * cl * 2 <= slots && c->fused_clusters[ilog2(cl * 2)] > 0) cl *= 2;
    return cl;
}

static int tau00_impl(Ctx* c, c128* M, int n, int k, int batch, c128* tau, int* info, void* workspace, cudaStream_t st) {
    const TauWs ws = tau_ws_layout(workspace, eff_nb(c), n, k, batch);
    const int cl = pick_small_mode(c, n, k, batch);
    c->last_schedule = cl < 0 ? 100 - cl : cl;
    if (cl < 0) {
        int done = 0, rc;
        { ProfScope ps(2, st, 8.0 / 3.0 * (double)n * n * n * batch);
          rc = launch_lu_resident(M, (size_t)n * n, n, k, batch, -cl, ws.piv, tau, info, st, &done); }
        if (rc <= 0) return rc;
        // The cluster launch was refused although bind_device found it feasible (the SMs available to this process can
        // change under it).  A refused launch enqueues nothing and its error code has been taken off the thread: the
        // items not yet enqueued go through the lock-step schedule, which needs no cluster.
        c->last_schedule = 0;
        return eliminate_groups(c, M + (size_t)done * n * n, n, k, batch - done, tau_ws_offset(ws, eff_nb(c), n, k, done),
                                tau + (size_t)done * k * k, info + done, st);
    }
    if (cl > 0) {
        ProfScope ps(2, st, 8.0 / 3.0 * (double)n * n * n * batch);
        return launch_lu_fused(M, (size_t)n * n, n, k, batch, eff_nb(c), eff_ib(c), c->opt[LSMS_OPT_ALIGN_FIRST], cl, ws.piv, tau, info, st);
    }
    return eliminate_groups(c, M, n, k, batch, ws, tau, info, st);
}

static size_t workspace_bytes_impl(const Ctx* c, int n_sites, int lmax, int spin_canted, int batch) {
    if (n_sites < 1 || lmax < 0 || lmax > 8 || batch < 1) return 0;
    int kmax = (lmax + 1) * (lmax + 1), k = kmax * (spin_canted ? 2 : 1);
    size_t n = (size_t)n_sites * k;
    if (n > 46340 || !rows_supported(c, (int)n, batch)) return 0;
    size_t a = align256(gaunt_table_bytes(lmax));
    size_t t = tau_ws_bytes(c, (int)n, k, batch);
    return a > t ? a : t;
}

}  // namespace lsms

using namespace lsms;

#define LSMS_ENTER(h) if (!(h)) return -1
#define LSMS_BIND(h) CallScope scope__(h); if (scope__.rc) return scope__.rc

extern "C" {

const char* lsms_version(void) { return "lsms_tau 0.3 (sm_100a; DMMA.8x8x4 Schur update, TMA-staged; on-chip cluster mode for small matrices)"; }

int lsms_create(lsms_handle_t* handle_out) {
    if (!handle_out) return -1;
    lsms_context* c = new (std::nothrow) lsms_context();
    *handle_out = c;
    if (!c) return (int)cudaErrorMemoryAllocation;
    for (int i = 0; i < LSMS_OPT_COUNT; ++i) c->opt[i] = 0;
    c->opt[LSMS_OPT_LOOKAHEAD] = 1; c->opt[LSMS_OPT_PANEL_THREADS] = 1; c->opt[LSMS_OPT_ALIGN_FIRST] = 1;
    c->device = -1;                      // bound by the first call that enqueues work
    return 0;
}

int lsms_destroy(lsms_handle_t c) {
    if (!c) return -1;
    if (t_ctx == c) t_ctx = nullptr;
    for (int g = 0; g < MAX_GROUPS; ++g) {
        GroupStreams& s = c->gs[g];
        if (s.main) cudaStreamDestroy(s.main);
        if (s.aux) cudaStreamDestroy(s.aux);
        if (s.fork) cudaEventDestroy(s.fork);
        if (s.join) cudaEventDestroy(s.join);
        if (s.done) cudaEventDestroy(s.done);
    }
    if (c->ev_start) cudaEventDestroy(c->ev_start);
    for (cudaEvent_t ev : c->prof.ev) cudaEventDestroy(ev);
    delete c;
    return 0;
}

int lsms_set_option(lsms_handle_t c, int option, int value) {
    if (!c) return -1;
    bool ok = false;
    switch (option) {
        case LSMS_OPT_NB_OUTER: ok = value >= 0 && value <= 96 && value % 4 == 0; break;
        case LSMS_OPT_IB_INNER: ok = value >= 0 && value <= 16; break;
        case LSMS_OPT_LOOKAHEAD: ok = value == 0 || value == 1; break;
        case LSMS_OPT_PANEL_THREADS: ok = value >= 0 && value <= 2; break;
        case LSMS_OPT_ALIGN_FIRST: ok = value == 0 || value == 1; break;
        case LSMS_OPT_GROUPS: ok = value >= 0 && value <= MAX_GROUPS; break;
        case LSMS_OPT_PANEL_CLUSTER: ok = value == 0 || value == 1 || value == 2 || value == 4 || value == 8; break;
        case LSMS_OPT_SMALL_MODE: ok = value >= 0 && value <= 7; break;
        default: return -2;
    }
    if (!ok) return -3;
    c->opt[option] = value;
    return 0;
}

int lsms_get_option(lsms_handle_t c, int option, int* value_host) {
    if (!c) return -1;
    if (option < 0 || option >= LSMS_OPT_COUNT) return -2;
    if (!value_host) return -3;
    *value_host = c->opt[option];
    return 0;
}

size_t lsms_workspace_bytes(lsms_handle_t c, int n_sites, int lmax, int spin_canted, int batch) {
    if (!c) return 0;
    return workspace_bytes_impl(c, n_sites, lmax, spin_canted, batch);
}

size_t lsms_solve_workspace_bytes(lsms_handle_t c, int n_sites, int kmax, int spin_canted, int batch) {
    if (!c || n_sites < 1 || kmax < 1 || batch < 1) return 0;
    int k = kmax * (spin_canted ? 2 : 1);
    size_t n = (size_t)n_sites * k;
    if (n > 46340 || !rows_supported(c, (int)n, batch)) return 0;
    return align256((size_t)batch * n * n * sizeof(c128)) + align256((size_t)batch * k * k * sizeof(c128)) + tau_ws_bytes(c, (int)n, k, batch);
}

int lsms_tinv_from_phase_shifts(lsms_handle_t h, const lsms_c128* delta, const int* species, const lsms_c128* z,
                                int lmax, int n_sites, int spin_canted, int n_species, int batch,
                                lsms_c128* tinv_diag, lsms_c128* kappa, int* info, void* cuda_stream) {
    LSMS_ENTER(h);
    if (!delta || !aligned16(delta)) return -2;
    if (!species) return -3;
    if (!z || !aligned16(z)) return -4;
    if (lmax < 0 || lmax > 8) return -5;
    if (n_sites < 1) return -6;
    if (n_species < 1) return -8;
    if (batch < 1) return -9;
    if (!tinv_diag || !aligned16(tinv_diag)) return -10;
    if (!kappa || !aligned16(kappa)) return -11;
    if (!info) return -12;
    LSMS_BIND(h);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LSMS_CUDA_OK(cudaMemsetAsync(info, 0, (size_t)batch * sizeof(int), st));
    return launch_tinv((const c128*)delta, species, (const c128*)z, lmax, n_sites, spin_canted ? 2 : 1, n_species, batch,
                       (c128*)tinv_diag, (c128*)kappa, info, st);
}

int lsms_build_M_batched(lsms_handle_t h, const lsms_c128* tinv_diag, const double* site_pos, const double* moment_dir,
                         const lsms_c128* kappa, int lmax, int n_sites, int spin_canted, int batch,
                         lsms_c128* M_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    LSMS_ENTER(h);
    if (!tinv_diag || !aligned16(tinv_diag)) return -2;
    if (!site_pos) return -3;
    if (spin_canted && !moment_dir) return -4;
    if (!kappa || !aligned16(kappa)) return -5;
    if (lmax < 0 || lmax > 8) return -6;
    if (n_sites < 1) return -7;
    if (batch < 1) return -9;
    if (!M_out || !aligned16(M_out)) return -10;
    if (!info) return -11;
    if (!workspace || !aligned16(workspace)) return -12;
    if (workspace_bytes < align256(gaunt_table_bytes(lmax))) return -13;
    LSMS_BIND(h);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LSMS_CUDA_OK(cudaMemsetAsync(info, 0, (size_t)batch * sizeof(int), st));
    ProfScope ps(0, st);
    return launch_assemble((const c128*)tinv_diag, site_pos, moment_dir, (const c128*)kappa, lmax, n_sites,
                           spin_canted ? 1 : 0, batch, 1, (c128*)M_out, info, workspace, st);
}

int lsms_build_M_shared_g0_batched(lsms_handle_t h, const lsms_c128* tinv_diag, const double* site_pos, const double* moment_dir,
                                   const lsms_c128* kappa, int lmax, int n_sites, int spin_canted, int n_atoms, int n_energies,
                                   lsms_c128* M_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    LSMS_ENTER(h);
    if (!tinv_diag || !aligned16(tinv_diag)) return -2;
    if (!site_pos) return -3;
    if (spin_canted && !moment_dir) return -4;
    if (!kappa || !aligned16(kappa)) return -5;
    if (lmax < 0 || lmax > 8) return -6;
    if (n_sites < 1) return -7;
    if (n_atoms < 1) return -9;
    if (n_energies < 1) return -10;
    if (!M_out || !aligned16(M_out)) return -11;
    if (!info) return -12;
    if (!workspace || !aligned16(workspace)) return -13;
    if (workspace_bytes < align256(gaunt_table_bytes(lmax))) return -14;
    LSMS_BIND(h);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LSMS_CUDA_OK(cudaMemsetAsync(info, 0, (size_t)n_atoms * n_energies * sizeof(int), st));
    ProfScope ps(0, st);
    return launch_assemble((const c128*)tinv_diag, site_pos, moment_dir, (const c128*)kappa, lmax, n_sites,
                           spin_canted ? 1 : 0, n_energies, n_atoms, (c128*)M_out, info, workspace, st);
}

int lsms_tau00_batched(lsms_handle_t h, lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                       lsms_c128* tau00_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    LSMS_ENTER(h);
    if (!M || !aligned16(M)) return -2;
    if (n_sites < 1) return -3;
    if (kmax < 1 || isqrt_exact(kmax) < 0 || kmax > 81) return -4;
    if (batch < 1) return -6;
    if (!tau00_out || !aligned16(tau00_out)) return -7;
    if (!info) return -8;
    const int k = kmax * (spin_canted ? 2 : 1);
    const long long nll = (long long)n_sites * k;
    if (nll > 46340) return -3;
    const int n = (int)nll;
    if (!rows_supported(h, n, batch)) return LSMS_ERR_PANEL_TOO_TALL;
    if (!workspace || !aligned16(workspace)) return -9;
    if (workspace_bytes < tau_ws_bytes(h, n, k, batch)) return -10;
    LSMS_BIND(h);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LSMS_CUDA_OK(cudaMemsetAsync(info, 0, (size_t)batch * sizeof(int), st));
    return tau00_impl(h, (c128*)M, n, k, batch, (c128*)tau00_out, info, workspace, st);
}

int lsms_solve_central_column_batched(lsms_handle_t h, const lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                                      lsms_c128* X_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    LSMS_ENTER(h);
    if (!M || !aligned16(M)) return -2;
    if (n_sites < 1) return -3;
    if (kmax < 1 || isqrt_exact(kmax) < 0 || kmax > 81) return -4;
    if (batch < 1) return -6;
    if (!X_out || !aligned16(X_out)) return -7;
    if (!info) return -8;
    if (!workspace || !aligned16(workspace)) return -9;
    const size_t need = lsms_solve_workspace_bytes(h, n_sites, kmax, spin_canted, batch);
    if (need == 0) return (long long)n_sites * kmax * (spin_canted ? 2 : 1) > 46340 ? -3 : LSMS_ERR_PANEL_TOO_TALL;
    if (workspace_bytes < need) return -10;
    LSMS_BIND(h);
    const int k = kmax * (spin_canted ? 2 : 1);
    const int n = n_sites * k;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* p = (char*)workspace;
    c128* copy = (c128*)p; p += align256((size_t)batch * n * n * sizeof(c128));
    c128* tau = (c128*)p; p += align256((size_t)batch * k * k * sizeof(c128));
    LSMS_CUDA_OK(cudaMemcpyAsync(copy, M, (size_t)batch * n * n * sizeof(c128), cudaMemcpyDeviceToDevice, st));
    LSMS_CUDA_OK(cudaMemsetAsync(info, 0, (size_t)batch * sizeof(int), st));
    int rc = tau00_impl(h, copy, n, k, batch, tau, info, p, st);
    if (rc) return rc;
    return launch_backsolve_central(copy, (size_t)n * n, n, k, batch, tau, (c128*)X_out, st);
}

size_t lsms_host_call_scratch_bytes(lsms_handle_t c, int n_sites, int lmax, int spin_canted, int n_species, int batch) {
    if (!c || n_sites < 1 || lmax < 0 || lmax > 8 || batch < 1 || n_species < 1) return 0;
    int nspin = spin_canted ? 2 : 1, nl = lmax + 1, kmax = nl * nl, k = kmax * nspin;
    size_t n = (size_t)n_sites * k;
    const size_t wsb = workspace_bytes_impl(c, n_sites, lmax, spin_canted, batch);
    if (wsb == 0) return 0;
    size_t s = 0;
    s += align256((size_t)n_species * nspin * nl * sizeof(c128));          // delta
    s += align256((size_t)batch * n_sites * sizeof(int));                 // species
    s += align256((size_t)batch * sizeof(c128));                          // z
    s += align256((size_t)batch * n_sites * 3 * sizeof(double)) * 2;      // site_pos, moment_dir
    s += align256((size_t)batch * n_sites * nspin * nl * sizeof(c128));   // tinv
    s += align256((size_t)batch * sizeof(c128));                          // kappa
    s += align256((size_t)batch * n * n * sizeof(c128));                  // M
    s += align256((size_t)batch * k * k * sizeof(c128));                  // tau00
    s += align256((size_t)batch * sizeof(int));                           // info
    s += wsb;
    return s;
}

int lsms_tau00_from_host(lsms_handle_t h, const lsms_c128* delta_host, const int* species_host, const lsms_c128* z_host,
                         const double* site_pos_host, const double* moment_dir_host,
                         int lmax, int n_sites, int spin_canted, int n_species, int batch, int n_energies,
                         lsms_c128* tau00_out_host, int* info_host,
                         void* device_scratch, size_t scratch_bytes, void* cuda_stream,
                         size_t* h2d_bytes, size_t* d2h_bytes) {
    LSMS_ENTER(h);
    if (!delta_host) return -2;
    if (!species_host) return -3;
    if (!z_host) return -4;
    if (!site_pos_host) return -5;
    if (spin_canted && !moment_dir_host) return -6;
    if (lmax < 0 || lmax > 8) return -7;
    if (n_sites < 1) return -8;
    if (n_species < 1) return -10;
    if (batch < 1) return -11;
    if (n_energies < 0 || n_energies > batch) return -12;
    if (!tau00_out_host) return -13;
    if (!info_host) return -14;
    if (!device_scratch || !aligned16(device_scratch)) return -15;
    const size_t need = lsms_host_call_scratch_bytes(h, n_sites, lmax, spin_canted, n_species, batch);
    if (need == 0) return (long long)n_sites * (lmax + 1) * (lmax + 1) * (spin_canted ? 2 : 1) > 46340 ? -8 : LSMS_ERR_PANEL_TOO_TALL;
    if (scratch_bytes < need) return -16;
    LSMS_BIND(h);
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nspin = spin_canted ? 2 : 1, nl = lmax + 1, kmax = nl * nl, k = kmax * nspin;
    const size_t n = (size_t)n_sites * k;
    char* p = (char*)device_scratch;
    auto take = [&](size_t bytes) { char* q = p; p += align256(bytes); return (void*)q; };
    const size_t b_delta = (size_t)n_species * nspin * nl * sizeof(c128), b_spec = (size_t)batch * n_sites * sizeof(int),
                 b_z = (size_t)batch * sizeof(c128), b_pos = (size_t)batch * n_sites * 3 * sizeof(double),
                 b_tau = (size_t)batch * k * k * sizeof(c128), b_info = (size_t)batch * sizeof(int);
    c128* d_delta = (c128*)take(b_delta); int* d_spec = (int*)take(b_spec); c128* d_z = (c128*)take(b_z);
    double* d_pos = (double*)take(b_pos); double* d_mom = (double*)take(b_pos);
    c128* d_tinv = (c128*)take((size_t)batch * n_sites * nspin * nl * sizeof(c128)); c128* d_kappa = (c128*)take(b_z);
    c128* d_M = (c128*)take((size_t)batch * n * n * sizeof(c128));
    c128* d_tau = (c128*)take(b_tau); int* d_info = (int*)take(b_info);
    void* ws = p;
    // f3: one g0 per energy when the host inputs show that all atoms share geometry and energies
    int n_atoms = 1, n_e = batch;
    if (n_energies > 0 && n_energies < batch && batch % n_energies == 0) {
        const size_t pos_e = (size_t)n_energies * n_sites * 3 * sizeof(double), z_e = (size_t)n_energies * sizeof(c128);
        bool same = true;
        for (int a = 1; a < batch / n_energies && same; ++a)
            same = memcmp((const char*)site_pos_host + a * pos_e, site_pos_host, pos_e) == 0 &&
                   memcmp((const char*)z_host + a * z_e, z_host, z_e) == 0;
        if (same) { n_atoms = batch / n_energies; n_e = n_energies; }
    }
    size_t h2d = 0;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_delta, delta_host, b_delta, cudaMemcpyHostToDevice, st)); h2d += b_delta;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_spec, species_host, b_spec, cudaMemcpyHostToDevice, st)); h2d += b_spec;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_z, z_host, b_z, cudaMemcpyHostToDevice, st)); h2d += b_z;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_pos, site_pos_host, b_pos, cudaMemcpyHostToDevice, st)); h2d += b_pos;
    if (spin_canted) { LSMS_CUDA_OK(cudaMemcpyAsync(d_mom, moment_dir_host, b_pos, cudaMemcpyHostToDevice, st)); h2d += b_pos; }
    // info is cleared once; every stage records only the FIRST non-zero code of an item
    LSMS_CUDA_OK(cudaMemsetAsync(d_info, 0, b_info, st));
    int rc = launch_tinv(d_delta, d_spec, d_z, lmax, n_sites, nspin, n_species, batch, d_tinv, d_kappa, d_info, st);
    if (rc) return rc;
    { ProfScope ps(0, st);
      rc = launch_assemble(d_tinv, d_pos, spin_canted ? d_mom : nullptr, d_kappa, lmax, n_sites, spin_canted ? 1 : 0, n_e, n_atoms,
                           d_M, d_info, ws, st); }
    if (rc) return rc;
    rc = tau00_impl(h, d_M, (int)n, k, batch, d_tau, d_info, ws, st);
    if (rc) return rc;
    LSMS_CUDA_OK(cudaMemcpyAsync(tau00_out_host, d_tau, b_tau, cudaMemcpyDeviceToHost, st));
    LSMS_CUDA_OK(cudaMemcpyAsync(info_host, d_info, b_info, cudaMemcpyDeviceToHost, st));
    LSMS_CUDA_OK(cudaStreamSynchronize(st));
    if (h2d_bytes) *h2d_bytes = h2d;
    if (d2h_bytes) *d2h_bytes = b_tau + b_info;
    return 0;
}

int lsms_contour_sum_batched(lsms_handle_t h, const lsms_c128* tau00, const lsms_c128* weights, int n_atoms, int n_energies, int k,
                             lsms_c128* out, void* cuda_stream) {
    LSMS_ENTER(h);
    if (!tau00 || !aligned16(tau00)) return -2;
    if (!weights || !aligned16(weights)) return -3;
    if (n_atoms < 1) return -4;
    if (n_energies < 1 || n_energies > 2048) return -5;
    if (k < 1 || k > 4096) return -6;
    if (!out || !aligned16(out)) return -7;
    LSMS_BIND(h);
    return launch_contour_sum((const c128*)tau00, (const c128*)weights, n_atoms, n_energies, k * k, (c128*)out, (cudaStream_t)cuda_stream);
}

// ---------------------------------------------------------------- include/lsms_tau_diag.h

int lsms_last_launch_count(lsms_handle_t h) { return h ? h->last_launches : -1; }
int lsms_last_schedule(lsms_handle_t h) { return h ? h->last_schedule : -1; }

int lsms_max_active_clusters(lsms_handle_t h, int kernel, int cluster_size, int* count_host) {
    LSMS_ENTER(h);
    if (kernel < 0 || kernel > 2) return -2;
    if (cluster_size != 1 && cluster_size != 2 && cluster_size != 4 && cluster_size != 8) return -3;
    if (!count_host) return -4;
    LSMS_BIND(h);
    const int i = ilog2(cluster_size);
    *count_host = kernel == 0 ? h->res_clusters[i] : kernel == 1 ? h->fused_clusters[i] : h->pclu_clusters[i];
    return 0;
}

int lsms_profile_begin(lsms_handle_t h) {
    if (!h) return -1;
    h->prof.on = true; h->prof.used = 0;
    for (int i = 0; i < 8; ++i) h->prof.flops[i] = 0.0;
    return 0;
}

int lsms_profile_end(lsms_handle_t h, double* ms_by_class_host, int* launches_by_class_host, double* flops_by_class_host) {
    if (!h) return -1;
    if (!ms_by_class_host) return -2;
    if (!launches_by_class_host) return -3;
    if (!flops_by_class_host) return -4;
    Prof& p = h->prof;
    p.on = false;
    for (int i = 0; i < 8; ++i) { ms_by_class_host[i] = 0.0; launches_by_class_host[i] = 0; flops_by_class_host[i] = p.flops[i]; }
    for (size_t i = 0; i < p.used; ++i) {
        LSMS_CUDA_OK(cudaEventSynchronize(p.ev[2 * i + 1]));
        float ms = 0.f;
        LSMS_CUDA_OK(cudaEventElapsedTime(&ms, p.ev[2 * i], p.ev[2 * i + 1]));
        ms_by_class_host[p.cls[i]] += ms; launches_by_class_host[p.cls[i]] += 1;
    }
    p.used = 0;
    return 0;
}

int lsms_fp64_peak_probe(lsms_handle_t h, int which, int iters, double* sink, double* tflops_host, void* cuda_stream) {
    LSMS_ENTER(h);
    if (which < 0 || which > 1) return -2;
    if (iters < 1) return -3;
    if (!sink) return -4;
    if (!tflops_host) return -5;
    LSMS_BIND(h);
    return run_peak_probe(which, iters, sink, tflops_host, (cudaStream_t)cuda_stream);
}

int lsms_schur_update_batched(lsms_handle_t h, lsms_c128* M, int n, int c0, int kk, int batch, void* cuda_stream) {
    LSMS_ENTER(h);
    if (!M || !aligned16(M)) return -2;
    if (n < 2) return -3;
    if (c0 < 0 || kk < 1 || c0 + kk >= n) return -4;
    if (batch < 1) return -6;
    LSMS_BIND(h);
    GemmShape g; g.strideA = g.strideB = g.strideC = (size_t)n * n; g.ldA = g.ldB = g.ldC = n; g.batch = batch; g.beta0 = 0;
    const int r0 = c0 + kk;
    c128* base = (c128*)M;
    g.Mr = n - r0; g.Nc = n - r0; g.K = kk;
    g.A = base + (size_t)r0 + (size_t)c0 * n; g.B = base + (size_t)c0 + (size_t)r0 * n; g.C = base + (size_t)r0 + (size_t)r0 * n;
    return launch_schur_gemm(g, (cudaStream_t)cuda_stream);
}

/* host-only debug export for the CPU test-suite: the closed-form Gaunt number used by K1 */
double lsms_debug_gaunt_closed_form(int l, int m, int lp, int mp, int lpp) { return gaunt_closed_form_host(l, m, lp, mp, lpp); }

}  // extern "C"
