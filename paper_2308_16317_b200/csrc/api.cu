// api.cu -- the C ABI of include/lsms_tau.h: argument checks, workspace layout and the batch
// scheduler that walks the blocked right-looking elimination.
#include <math.h>
#include <stdint.h>
#include <vector>
#include "../../include/lsms_tau.h"
#include "common.cuh"
#include "internal.h"

namespace lsms {
thread_local LaunchCounter g_launches = {0};
static int g_nb_outer = 0, g_ib_inner = 0;

// ---- optional per-kernel-class timing (lsms_profile_begin / lsms_profile_end): CUDA events recorded on
// the caller's stream around each launch, so bench.py can report the Schur update's duration and share
// measured inside the step.  Classes: 0 K1 assembly, 1 K2 panel, 2 K3 swap/trsm, 3 K4 inner (K <= IB),
// 4 K4 Schur update (K = NB), 5 K5 final inverse, 6 K3a/K3b net permutation + Ninv, 7 K4 as TRSM (U12 = -Ninv*A12).
struct Prof {
    bool on = false;
    std::vector<cudaEvent_t> ev;     // pairs
    std::vector<int> cls;
    size_t used = 0;
    double flops[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};
static Prof g_prof;
struct ProfScope {
    cudaStream_t st; bool live;
    ProfScope(int cls, cudaStream_t s, double flops = 0.0) : st(s), live(g_prof.on) {
        if (!live) return;
        if (g_prof.ev.size() < 2 * (g_prof.used + 1)) {
            cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
            g_prof.ev.push_back(a); g_prof.ev.push_back(b); g_prof.cls.push_back(cls);
        }
        g_prof.cls[g_prof.used] = cls;
        g_prof.flops[cls] += flops;
        cudaEventRecord(g_prof.ev[2 * g_prof.used], st);
    }
    ~ProfScope() { if (live) { cudaEventRecord(g_prof.ev[2 * g_prof.used + 1], st); ++g_prof.used; } }
};

static inline size_t align256(size_t x) { return (x + 255) / 256 * 256; }
static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; }

static int isqrt_exact(int v) { int r = (int)lround(sqrt((double)v)); return (r * r == v) ? r : -1; }

static inline int eff_nb() { return g_nb_outer > 0 ? g_nb_outer : 64; }
static inline int eff_ib() { return g_ib_inner > 0 ? g_ib_inner : 16; }

// Workspace layout for lsms_tau00_batched:
//   [pivots int32 batch*n][perm int32 batch*(4+3NB)][Ninv c128 batch*NB*NB][Tperm c128 batch*NB*n][K5 scratch]
struct TauWs { int* piv; int* perm; c128* ninv; c128* tperm; void* k5; size_t total; };
static TauWs tau_ws_layout(void* base, int n, int k, int batch) {
    const int NB = eff_nb();
    TauWs w; char* p = (char*)base;
    w.piv = (int*)p; p += align256((size_t)batch * n * sizeof(int));
    w.perm = (int*)p; p += align256((size_t)batch * (4 + 3 * NB) * sizeof(int));
    w.ninv = (c128*)p; p += align256((size_t)batch * NB * NB * sizeof(c128));
    w.tperm = (c128*)p; p += align256((size_t)batch * NB * n * sizeof(c128));
    w.k5 = p; p += align256(final_inverse_ws_bytes(k, batch));
    w.total = (size_t)(p - (char*)base);
    return w;
}
static size_t tau_ws_bytes(int n, int k, int batch) { return tau_ws_layout(nullptr, n, k, batch).total; }

// Blocked right-looking elimination of the first ne = n-k columns of every item, in lock-step over
// the batch: each launch covers all items, so the latency-bound panel kernels (one CTA per item)
// fill the chip through the batch dimension while the update kernels tile every trailing matrix.
//   outer panel [J, J+W), W <= NB:
//     for each inner panel [c0, c0+w), w <= IB:                       (inside the outer panel only)
//        K2  factor the (n-c0) x w panel, pivots restricted to rows < ne
//        K3  interchanges on the outer panel's other columns; TRSM on those to the right
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
// after the join).  The auxiliary stream and two events are the library's only persistent objects.
static int g_lookahead = 1;
static int g_groups = 0;                  // 0 = chosen per shape
static int g_align_first = 1;              // first panel n mod 64 wide (tile-aligned trailing matrices)
static int g_panel_variant = 1;           // -1 L2-resident k_panel, 0 register-blocked 256 threads, 1 register-blocked 512 threads for tall panels
constexpr int MAX_GROUPS = 8;
// Stream set of one batch group (see eliminate_groups): group 0 runs on the caller's stream, the others on
// library-owned streams; every group has a high-priority auxiliary stream for the look-ahead panel.
struct GroupStreams { cudaStream_t main = nullptr, aux = nullptr; cudaEvent_t fork = nullptr, join = nullptr, done = nullptr; };
static GroupStreams g_gs[MAX_GROUPS];
static cudaEvent_t g_ev_start = nullptr;

static int ensure_streams(int groups) {
    int lo = 0, hi = 0;
    LSMS_CUDA_OK(cudaDeviceGetStreamPriorityRange(&lo, &hi));
    if (!g_ev_start) LSMS_CUDA_OK(cudaEventCreateWithFlags(&g_ev_start, cudaEventDisableTiming));
    for (int g = 0; g < groups; ++g) {
        GroupStreams& s = g_gs[g];
        if (s.aux) continue;
        if (g > 0) LSMS_CUDA_OK(cudaStreamCreateWithFlags(&s.main, cudaStreamNonBlocking));
        LSMS_CUDA_OK(cudaStreamCreateWithPriority(&s.aux, cudaStreamNonBlocking, hi));
        LSMS_CUDA_OK(cudaEventCreateWithFlags(&s.fork, cudaEventDisableTiming));
        LSMS_CUDA_OK(cudaEventCreateWithFlags(&s.join, cudaEventDisableTiming));
        LSMS_CUDA_OK(cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
    }
    return 0;
}

static int g_panel_cluster = 0;            // 0 = chosen per shape, 1 = never, 2/4/8 = forced
// CTAs per matrix for the panel kernel.  A cluster shortens the panel factorisation of a tall panel several times
// (rank 12450, 12 matrices: 303 -> 117 ms per step when timed alone), but its CTAs must be co-scheduled on free SMs, so
// under look-ahead it waits for the Schur update to drain instead of running beneath it and whole steps of batches
// >= 4 got SLOWER (NC 1897 -> 1928 ms, H 629 -> 654, C 440 -> 465, P 121 -> 129).  It pays when there is next to
// nothing to overlap with: one or two tall matrices (rank 12450, batch 1: 369 -> 223 ms; rank 4320: 36.9 -> 32.5 ms).
static int panel_cluster_size(int m, int batch) {
    if (g_panel_variant < 1) return 1;
    if (g_panel_cluster == 1) return 1;
    int cl = 1;
    if (g_panel_cluster > 1) cl = g_panel_cluster;
    else if (batch <= 2 && m >= 4096) cl = 8;
    else if (batch <= 2 && m >= 2048) cl = 4;
    if (cl > 1 && (m + cl - 1) / cl > 5120) cl = 1;         // taller than the cluster instances cover: one-CTA kernel
    return cl;
}

// factor the outer panel [J, J+W) on stream st: inner panels of width <= IB
static int factor_panel(c128* M, int n, int batch, int J, int W, int ne, int IB, int* piv, int* info, cudaStream_t st) {
    const size_t stride = (size_t)n * n;
    const int Jend = J + W;
    GemmShape g; g.strideA = g.strideB = g.strideC = stride; g.ldA = g.ldB = g.ldC = n; g.batch = batch; g.beta0 = 0;
    for (int jj = 0; jj < W; jj += IB) {
        const int c0 = J + jj, w = (W - jj < IB) ? W - jj : IB;
        int rc;
        if (g_panel_variant >= 0 && n - c0 <= 16384) {
            // register-blocked K2: factors the inner panel, applies its interchanges to the whole outer panel and
            // solves the w x w triangle for the outer panel's columns to the right
            // small batches of tall panels: a cluster of CTAs per matrix, so that the panel phase spans the chip too
            const int cl = panel_cluster_size(n - c0, batch);
            if (cl > 1) { ProfScope ps(1, st); rc = launch_panel_cluster(M, stride, n, J, W, c0, w, ne, batch, piv, info, cl, st); }
            else { ProfScope ps(1, st); rc = launch_panel_reg(M, stride, n, J, W, c0, w, ne, batch, piv, info, g_panel_variant, st); }
            if (rc) return rc;
        } else {
            { ProfScope ps(1, st); rc = launch_panel(M, stride, n, c0, w, ne, batch, piv, info, st); } if (rc) return rc;
            { ProfScope ps(2, st); rc = launch_swap_trsm(M, stride, n, c0, w, J, c0, 1, batch, piv, st); } if (rc) return rc;
            { ProfScope ps(2, st); rc = launch_swap_trsm(M, stride, n, c0, w, c0 + w, Jend, 3, batch, piv, st); } if (rc) return rc;
        }
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
static int eliminate(c128* M, int n, int k, int batch, const TauWs& ws, int* info, cudaStream_t st, const GroupStreams& gs) {
    const int ne = n - k;
    const int NB = eff_nb(), IB = eff_ib();
    const size_t stride = (size_t)n * n;
    int* piv = ws.piv;
    const bool la = g_lookahead != 0;
    if (ne <= 0) return 0;
    // Tile alignment: the first panel is n mod 64 wide (when that is non-zero), so that every trailing matrix
    // the Schur update sees has a multiple of the 64 x 64 DMMA tile in both dimensions; only the last,
    // smallest updates carry a ragged tile (n = 2160, 64-row tiles: 34 tile rows of which one 3/4 full -> 33 full).
    int W0 = ne < NB ? ne : NB;
    if (g_align_first && NB % 64 == 0 && n % 64 != 0 && n % 64 < W0) W0 = n % 64;
    int rc = factor_panel(M, n, batch, 0, W0, ne, IB, piv, info, st); if (rc) return rc;
    { ProfScope ps(6, st); rc = launch_panel_post(M, stride, n, 0, W0, batch, piv, ws.perm, ws.ninv, NB, st); } if (rc) return rc;
    for (int J = 0, W = W0; J < ne; J += W, W = (ne - J < NB) ? ne - J : NB) {
        const int Jend = J + W;                               // Jend <= ne < n
        { ProfScope ps(6, st); rc = launch_row_permute(M, stride, n, J, W, Jend, n, batch, ws.perm, ws.tperm, (size_t)NB * n, NB, st); } if (rc) return rc;
        GemmShape t; t.batch = batch; t.beta0 = 1;
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
            rc = factor_panel(M, n, batch, Jend, W2, ne, IB, piv, info, gs.aux); if (rc) return rc;
            // the next panel's net permutation and -(L11^-1) are also built under the update: perm/Ninv of
            // panel J were last read by the permutation / triangular solve above, before the fork
            { ProfScope ps(6, gs.aux); rc = launch_panel_post(M, stride, n, Jend, W2, batch, piv, ws.perm, ws.ninv, NB, gs.aux); } if (rc) return rc;
            LSMS_CUDA_OK(cudaEventRecord(gs.join, gs.aux));
            rc = schur_update(M, n, batch, J, W, Jend + W2, n, st); if (rc) return rc;
            LSMS_CUDA_OK(cudaStreamWaitEvent(st, gs.join, 0));
        } else {
            rc = schur_update(M, n, batch, J, W, Jend, n, st); if (rc) return rc;
            if (W2 > 0) {
                rc = factor_panel(M, n, batch, Jend, W2, ne, IB, piv, info, st); if (rc) return rc;
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
static int pick_groups(int n, int batch) {
    int g = g_groups;
    if (g <= 0) g = (batch >= 16) ? 2 : 1;
    if (g > MAX_GROUPS) g = MAX_GROUPS;
    if (g > batch) g = batch;
    (void)n;
    return g;
}

static int eliminate_groups(c128* M, int n, int k, int batch, const TauWs& ws, c128* tau, int* info, cudaStream_t st) {
    const int NB = eff_nb();
    const int groups = pick_groups(n, batch);
    int rc = ensure_streams(groups); if (rc) return rc;
    const size_t stride = (size_t)n * n;
    if (groups > 1) LSMS_CUDA_OK(cudaEventRecord(g_ev_start, st));
    for (int g = 0; g < groups; ++g) {
        const int b0 = (int)((long long)batch * g / groups), b1 = (int)((long long)batch * (g + 1) / groups);
        if (b1 <= b0) continue;
        cudaStream_t gst = (g == 0) ? st : g_gs[g].main;
        if (g > 0) LSMS_CUDA_OK(cudaStreamWaitEvent(gst, g_ev_start, 0));
        TauWs w = ws;
        w.piv = ws.piv + (size_t)b0 * n;
        w.perm = ws.perm + (size_t)b0 * (4 + 3 * NB);
        w.ninv = ws.ninv + (size_t)b0 * NB * NB;
        w.tperm = ws.tperm + (size_t)b0 * NB * n;
        w.k5 = (char*)ws.k5 + (final_inverse_ws_bytes(k, 1) ? (size_t)b0 * k * k * sizeof(c128) : 0);
        rc = eliminate(M + (size_t)b0 * stride, n, k, b1 - b0, w, info + b0, gst, g_gs[g]); if (rc) return rc;
        { ProfScope ps(5, gst);
          rc = launch_final_inverse(M + (size_t)b0 * stride, stride, n, k, b1 - b0, tau + (size_t)b0 * k * k, info + b0, w.k5, gst); }
        if (rc) return rc;
        if (g > 0) LSMS_CUDA_OK(cudaEventRecord(g_gs[g].done, gst));
    }
    for (int g = 1; g < groups; ++g) {
        const int b0 = (int)((long long)batch * g / groups), b1 = (int)((long long)batch * (g + 1) / groups);
        if (b1 > b0) LSMS_CUDA_OK(cudaStreamWaitEvent(st, g_gs[g].done, 0));
    }
    return 0;
}

}  // namespace lsms

using namespace lsms;

extern "C" {

const char* lsms_version(void) { return "lsms_tau 0.1 (sm_100a; DMMA.8x8x4 Schur update, TMA-staged)"; }

size_t lsms_workspace_bytes(int n_sites, int lmax, int spin_canted, int batch) {
    if (n_sites < 1 || lmax < 0 || lmax > 8 || batch < 1) return 0;
    int kmax = (lmax + 1) * (lmax + 1), k = kmax * (spin_canted ? 2 : 1);
    size_t n = (size_t)n_sites * k;
    size_t a = align256(gaunt_table_bytes(lmax));
    size_t t = tau_ws_bytes((int)n, k, batch);
    return a > t ? a : t;
}

size_t lsms_solve_workspace_bytes(int n_sites, int kmax, int spin_canted, int batch) {
    if (n_sites < 1 || kmax < 1 || batch < 1) return 0;
    int k = kmax * (spin_canted ? 2 : 1);
    size_t n = (size_t)n_sites * k;
    return align256((size_t)batch * n * n * sizeof(c128)) + align256((size_t)batch * k * k * sizeof(c128)) + tau_ws_bytes((int)n, k, batch);
}

int lsms_tinv_from_phase_shifts(const lsms_c128* delta, const int* species, const lsms_c128* z,
                                int lmax, int n_sites, int spin_canted, int n_species, int batch,
                                lsms_c128* tinv_diag, lsms_c128* kappa, void* cuda_stream) {
    if (!delta || !aligned16(delta)) return -1;
    if (!species) return -2;
    if (!z || !aligned16(z)) return -3;
    if (lmax < 0 || lmax > 8) return -4;
    if (n_sites < 1) return -5;
    if (n_species < 1) return -7;
    if (batch < 1) return -8;
    if (!tinv_diag || !aligned16(tinv_diag)) return -9;
    if (!kappa || !aligned16(kappa)) return -10;
    g_launches.n = 0;
    return launch_tinv((const c128*)delta, species, (const c128*)z, lmax, n_sites, spin_canted ? 2 : 1, batch,
                       (c128*)tinv_diag, (c128*)kappa, (cudaStream_t)cuda_stream);
}

int lsms_build_M_batched(const lsms_c128* tinv_diag, const double* site_pos, const double* moment_dir,
                         const lsms_c128* kappa, int lmax, int n_sites, int spin_canted, int batch,
                         lsms_c128* M_out, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!tinv_diag || !aligned16(tinv_diag)) return -1;
    if (!site_pos) return -2;
    if (spin_canted && !moment_dir) return -3;
    if (!kappa || !aligned16(kappa)) return -4;
    if (lmax < 0 || lmax > 8) return -5;
    if (n_sites < 1) return -6;
    if (batch < 1) return -8;
    if (!M_out || !aligned16(M_out)) return -9;
    if (!workspace || !aligned16(workspace)) return -10;
    if (workspace_bytes < align256(gaunt_table_bytes(lmax))) return -11;
    g_launches.n = 0;
    ProfScope ps(0, (cudaStream_t)cuda_stream);
    return launch_assemble((const c128*)tinv_diag, site_pos, moment_dir, (const c128*)kappa, lmax, n_sites,
                           spin_canted ? 1 : 0, batch, 1, (c128*)M_out, workspace, (cudaStream_t)cuda_stream);
}

int lsms_build_M_shared_g0_batched(const lsms_c128* tinv_diag, const double* site_pos, const double* moment_dir,
                                   const lsms_c128* kappa, int lmax, int n_sites, int spin_canted, int n_atoms, int n_energies,
                                   lsms_c128* M_out, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!tinv_diag || !aligned16(tinv_diag)) return -1;
    if (!site_pos) return -2;
    if (spin_canted && !moment_dir) return -3;
    if (!kappa || !aligned16(kappa)) return -4;
    if (lmax < 0 || lmax > 8) return -5;
    if (n_sites < 1) return -6;
    if (n_atoms < 1) return -8;
    if (n_energies < 1) return -9;
    if (!M_out || !aligned16(M_out)) return -10;
    if (!workspace || !aligned16(workspace)) return -11;
    if (workspace_bytes < align256(gaunt_table_bytes(lmax))) return -12;
    g_launches.n = 0;
    ProfScope ps(0, (cudaStream_t)cuda_stream);
    return launch_assemble((const c128*)tinv_diag, site_pos, moment_dir, (const c128*)kappa, lmax, n_sites,
                           spin_canted ? 1 : 0, n_energies, n_atoms, (c128*)M_out, workspace, (cudaStream_t)cuda_stream);
}

int lsms_tau00_batched(lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                       lsms_c128* tau00_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!M || !aligned16(M)) return -1;
    if (n_sites < 1) return -2;
    if (kmax < 1 || isqrt_exact(kmax) < 0 || kmax > 81) return -3;
    if (batch < 1) return -5;
    if (!tau00_out || !aligned16(tau00_out)) return -6;
    if (!info) return -7;
    const int k = kmax * (spin_canted ? 2 : 1);
    const long long nll = (long long)n_sites * k;
    if (nll > 46340) return -2;
    const int n = (int)nll;
    if (!workspace || !aligned16(workspace)) return -8;
    if (workspace_bytes < tau_ws_bytes(n, k, batch)) return -9;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    g_launches.n = 0;
    const TauWs ws = tau_ws_layout(workspace, n, k, batch);
    LSMS_CUDA_OK(cudaMemsetAsync(info, 0, (size_t)batch * sizeof(int), st));
    return eliminate_groups((c128*)M, n, k, batch, ws, (c128*)tau00_out, info, st);
}

int lsms_solve_central_column_batched(const lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                                      lsms_c128* X_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream) {
    if (!M || !aligned16(M)) return -1;
    if (n_sites < 1) return -2;
    if (kmax < 1 || isqrt_exact(kmax) < 0 || kmax > 81) return -3;
    if (batch < 1) return -5;
    if (!X_out || !aligned16(X_out)) return -6;
    if (!info) return -7;
    if (!workspace || !aligned16(workspace)) return -8;
    if (workspace_bytes < lsms_solve_workspace_bytes(n_sites, kmax, spin_canted, batch)) return -9;
    const int k = kmax * (spin_canted ? 2 : 1);
    const int n = n_sites * k;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    char* p = (char*)workspace;
    c128* copy = (c128*)p; p += align256((size_t)batch * n * n * sizeof(c128));
    c128* tau = (c128*)p; p += align256((size_t)batch * k * k * sizeof(c128));
    LSMS_CUDA_OK(cudaMemcpyAsync(copy, M, (size_t)batch * n * n * sizeof(c128), cudaMemcpyDeviceToDevice, st));
    int rc = lsms_tau00_batched((lsms_c128*)copy, n_sites, kmax, spin_canted, batch, (lsms_c128*)tau, info, p,
                                tau_ws_bytes(n, k, batch), cuda_stream);
    if (rc) return rc;
    return launch_backsolve_central(copy, (size_t)n * n, n, k, batch, tau, (c128*)X_out, st);
}

size_t lsms_host_call_scratch_bytes(int n_sites, int lmax, int spin_canted, int n_species, int batch) {
    if (n_sites < 1 || lmax < 0 || lmax > 8 || batch < 1 || n_species < 1) return 0;
    int nspin = spin_canted ? 2 : 1, nl = lmax + 1, kmax = nl * nl, k = kmax * nspin;
    size_t n = (size_t)n_sites * k;
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
    s += lsms_workspace_bytes(n_sites, lmax, spin_canted, batch);
    return s;
}

int lsms_tau00_from_host(const lsms_c128* delta_host, const int* species_host, const lsms_c128* z_host,
                         const double* site_pos_host, const double* moment_dir_host,
                         int lmax, int n_sites, int spin_canted, int n_species, int batch,
                         lsms_c128* tau00_out_host, int* info_host,
                         void* device_scratch, size_t scratch_bytes, void* cuda_stream,
                         size_t* h2d_bytes, size_t* d2h_bytes) {
    if (!delta_host) return -1;
    if (!species_host) return -2;
    if (!z_host) return -3;
    if (!site_pos_host) return -4;
    if (spin_canted && !moment_dir_host) return -5;
    if (lmax < 0 || lmax > 8) return -6;
    if (n_sites < 1) return -7;
    if (n_species < 1) return -9;
    if (batch < 1) return -10;
    if (!tau00_out_host) return -11;
    if (!info_host) return -12;
    if (!device_scratch || !aligned16(device_scratch)) return -13;
    if (scratch_bytes < lsms_host_call_scratch_bytes(n_sites, lmax, spin_canted, n_species, batch)) return -14;
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
    void* ws = p; const size_t ws_bytes = lsms_workspace_bytes(n_sites, lmax, spin_canted, batch);
    size_t h2d = 0;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_delta, delta_host, b_delta, cudaMemcpyHostToDevice, st)); h2d += b_delta;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_spec, species_host, b_spec, cudaMemcpyHostToDevice, st)); h2d += b_spec;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_z, z_host, b_z, cudaMemcpyHostToDevice, st)); h2d += b_z;
    LSMS_CUDA_OK(cudaMemcpyAsync(d_pos, site_pos_host, b_pos, cudaMemcpyHostToDevice, st)); h2d += b_pos;
    if (spin_canted) { LSMS_CUDA_OK(cudaMemcpyAsync(d_mom, moment_dir_host, b_pos, cudaMemcpyHostToDevice, st)); h2d += b_pos; }
    int rc = lsms_tinv_from_phase_shifts((lsms_c128*)d_delta, d_spec, (lsms_c128*)d_z, lmax, n_sites, spin_canted, n_species, batch,
                                         (lsms_c128*)d_tinv, (lsms_c128*)d_kappa, cuda_stream);
    if (rc) return rc;
    int launches = g_launches.n;
    rc = lsms_build_M_batched((lsms_c128*)d_tinv, d_pos, spin_canted ? d_mom : nullptr, (lsms_c128*)d_kappa, lmax, n_sites, spin_canted,
                              batch, (lsms_c128*)d_M, ws, ws_bytes, cuda_stream);
    if (rc) return rc;
    launches += g_launches.n;
    rc = lsms_tau00_batched((lsms_c128*)d_M, n_sites, kmax, spin_canted, batch, (lsms_c128*)d_tau, d_info, ws, ws_bytes, cuda_stream);
    if (rc) return rc;
    launches += g_launches.n;
    g_launches.n = launches;
    LSMS_CUDA_OK(cudaMemcpyAsync(tau00_out_host, d_tau, b_tau, cudaMemcpyDeviceToHost, st));
    LSMS_CUDA_OK(cudaMemcpyAsync(info_host, d_info, b_info, cudaMemcpyDeviceToHost, st));
    LSMS_CUDA_OK(cudaStreamSynchronize(st));
    if (h2d_bytes) *h2d_bytes = h2d;
    if (d2h_bytes) *d2h_bytes = b_tau + b_info;
    return 0;
}

int lsms_contour_sum_batched(const lsms_c128* tau00, const lsms_c128* weights, int n_atoms, int n_energies, int k,
                             lsms_c128* out, void* cuda_stream) {
    if (!tau00 || !aligned16(tau00)) return -1;
    if (!weights || !aligned16(weights)) return -2;
    if (n_atoms < 1) return -3;
    if (n_energies < 1 || n_energies > 2048) return -4;
    if (k < 1 || k > 4096) return -5;
    if (!out || !aligned16(out)) return -6;
    g_launches.n = 0;
    return launch_contour_sum((const c128*)tau00, (const c128*)weights, n_atoms, n_energies, k * k, (c128*)out, (cudaStream_t)cuda_stream);
}

int lsms_set_blocking(int nb_outer, int ib_inner) {
    if (nb_outer < 0 || nb_outer > 96 || (nb_outer % 4) != 0) return -1;
    if (ib_inner < 0 || ib_inner > 16) return -2;
    g_nb_outer = nb_outer; g_ib_inner = ib_inner;
    return 0;
}

int lsms_set_lookahead(int on) { g_lookahead = on ? 1 : 0; return 0; }

int lsms_set_align_first(int on) { g_align_first = on ? 1 : 0; return 0; }

int lsms_set_panel_cluster(int cl) {
    if (cl != 0 && cl != 1 && cl != 2 && cl != 4 && cl != 8) return -1;
    g_panel_cluster = cl;
    return 0;
}

int lsms_set_panel_variant(int variant) {
    if (variant < -1 || variant > 1) return -1;
    g_panel_variant = variant;
    return 0;
}

int lsms_set_groups(int groups) {
    if (groups < 0 || groups > MAX_GROUPS) return -1;
    g_groups = groups;
    return 0;
}

int lsms_last_launch_count(void) { return g_launches.n; }

int lsms_profile_begin(void) {
    g_prof.on = true; g_prof.used = 0;
    for (int i = 0; i < 8; ++i) g_prof.flops[i] = 0.0;
    return 0;
}

int lsms_profile_end(double* ms_by_class_host, int* launches_by_class_host, double* flops_by_class_host) {
    if (!ms_by_class_host) return -1;
    if (!launches_by_class_host) return -2;
    if (!flops_by_class_host) return -3;
    g_prof.on = false;
    for (int i = 0; i < 8; ++i) { ms_by_class_host[i] = 0.0; launches_by_class_host[i] = 0; flops_by_class_host[i] = g_prof.flops[i]; }
    for (size_t i = 0; i < g_prof.used; ++i) {
        LSMS_CUDA_OK(cudaEventSynchronize(g_prof.ev[2 * i + 1]));
        float ms = 0.f;
        LSMS_CUDA_OK(cudaEventElapsedTime(&ms, g_prof.ev[2 * i], g_prof.ev[2 * i + 1]));
        ms_by_class_host[g_prof.cls[i]] += ms; launches_by_class_host[g_prof.cls[i]] += 1;
    }
    g_prof.used = 0;
    return 0;
}

int lsms_fp64_peak_probe(int which, int iters, double* tflops_host, void* cuda_stream) {
    if (which < 0 || which > 1) return -1;
    if (iters < 1) return -2;
    if (!tflops_host) return -3;
    return run_peak_probe(which, iters, tflops_host, (cudaStream_t)cuda_stream);
}

int lsms_schur_update_batched(lsms_c128* M, int n, int c0, int kk, int batch, void* cuda_stream) {
    if (!M || !aligned16(M)) return -1;
    if (n < 2) return -2;
    if (c0 < 0 || kk < 1 || c0 + kk >= n) return -3;
    if (batch < 1) return -5;
    GemmShape g; g.strideA = g.strideB = g.strideC = (size_t)n * n; g.ldA = g.ldB = g.ldC = n; g.batch = batch; g.beta0 = 0;
    const int r0 = c0 + kk;
    c128* base = (c128*)M;
    g.Mr = n - r0; g.Nc = n - r0; g.K = kk;
    g.A = base + (size_t)r0 + (size_t)c0 * n; g.B = base + (size_t)c0 + (size_t)r0 * n; g.C = base + (size_t)r0 + (size_t)r0 * n;
    g_launches.n = 0;
    return launch_schur_gemm(g, (cudaStream_t)cuda_stream);
}

/* host-only debug export for the CPU test-suite: the closed-form Gaunt number used by K1 */
double lsms_debug_gaunt_closed_form(int l, int m, int lp, int mp, int lpp) { return gaunt_closed_form_host(l, m, lp, mp, lpp); }

}  // extern "C"
