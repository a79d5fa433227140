// internal.h -- host-side launchers and the per-handle context shared between the translation units of liblsms_tau.so.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <vector>
#include "../../include/lsms_tau.h"
#include "common.cuh"

namespace lsms {

// ---- per-handle state (include/lsms_tau.h "State and threads"): options, scheduler streams/events, profiling events.
constexpr int MAX_GROUPS = 8;
// Stream set of one batch group: group 0 runs on the caller's stream, the others on handle-owned streams; every group
// has a high-priority auxiliary stream for the look-ahead panel.
struct GroupStreams { cudaStream_t main = nullptr, aux = nullptr; cudaEvent_t fork = nullptr, join = nullptr, done = nullptr; };
struct Prof {
    bool on = false;
    std::vector<cudaEvent_t> ev;     // pairs
    std::vector<int> cls;
    size_t used = 0;
    double flops[8] = {0, 0, 0, 0, 0, 0, 0, 0};
};
struct Ctx {
    int device = 0;
    int sms = 148;
    int opt[LSMS_OPT_COUNT];
    // clusters of 1 / 2 / 4 / 8 CTAs that fit the device (or this process's SM partition) at once, per cluster kernel:
    // on-chip elimination, one-launch elimination through L2, cluster panel kernel.  Filled by bind_device; an unbound
    // handle (host-side size queries) assumes they all fit.
    int res_clusters[4] = {1 << 20, 1 << 20, 1 << 20, 1 << 20};
    int fused_clusters[4] = {1 << 20, 1 << 20, 1 << 20, 1 << 20};
    int pclu_clusters[4] = {0, 1 << 20, 1 << 20, 1 << 20};
    GroupStreams gs[MAX_GROUPS];
    cudaEvent_t ev_start = nullptr;
    Prof prof;
    int last_launches = 0;
    int last_schedule = -1;
};
}  // namespace lsms
struct lsms_context : lsms::Ctx {};
namespace lsms {

// the handle whose call is running on this host thread (set on entry of every extern "C" call)
extern thread_local Ctx* t_ctx;

// Brackets a launch with CUDA events of the handle's profiler when profiling is on (lsms_tau_diag.h classes).
struct ProfScope {
    cudaStream_t st; bool live;
    ProfScope(int cls, cudaStream_t s, double flops = 0.0);
    ~ProfScope();
};

// one-time per-device opt-in to dynamic shared-memory sizes (called from bind_device, at a handle's first enqueueing call)
int init_attrs_gemm();
int init_attrs_lu();
int init_attrs_assemble();
int init_attrs_fused();
int init_attrs_resident();
int init_attrs_panel();
int init_attrs_panel_cluster();

// assemble.cu
size_t gaunt_table_bytes(int lmax);
double gaunt_closed_form_host(int l, int m, int lp, int mp, int lpp);
int launch_tinv(const c128* delta, const int* species, const c128* z, int lmax, int n_sites, int nspin, int n_species, int batch,
                c128* tinv, c128* kappa, int* info, cudaStream_t st);
int launch_assemble(const c128* tinv, const double* site_pos, const double* moment, const c128* kappa, int lmax,
                    int n_sites, int canted, int batch, int n_rep, c128* M, int* info, void* ws, cudaStream_t st);

// gemm.cu -- K4: C[Mr x Nc] -= A[Mr x K] * B[K x Nc] inside the same column-major matrices (ld = n)
struct GemmShape {
    const c128* A; const c128* B; c128* C;   // item 0 of each operand: A is Mr x K, B is K x Nc, C is Mr x Nc (column-major)
    size_t strideA, strideB, strideC;        // elements between batch items
    int ldA, ldB, ldC;
    int Mr, Nc, K;
    int beta0;                               // 0: C -= A*B ;  1: C = -(A*B)  (C is not read)
    int triA = 0;                            // 1: A is lower triangular, Mr <= 64 (one tile row): zero blocks are skipped
    int batch;
};
int launch_schur_gemm(const GemmShape& g, cudaStream_t st);

// panel.cu -- K2 with the sub-panel in registers; also applies the interchanges to the whole outer panel [J, J+Wout)
int launch_panel_reg(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                     int variant, cudaStream_t st);
// panel_cluster.cu -- the same with a cluster of cl CTAs per matrix (small batches of tall panels)
int launch_panel_cluster(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                         int cl, cudaStream_t st);
// lu.cu -- K3a, K3b, K5 and the verification back-substitution
int launch_panel_post(const c128* base, size_t stride, int n, int J, int W, int batch, const int* piv, int* perm, c128* ninv,
                      int nbmax, cudaStream_t st);
int launch_row_permute(c128* base, size_t stride, int n, int J, int W, int col_lo, int col_hi, int batch, const int* perm,
                       c128* tperm, size_t tperm_stride, int nbmax, cudaStream_t st);
int launch_final_inverse(c128* base, size_t stride, int n, int k, int batch, c128* tau, int* info, void* ws, cudaStream_t st);
int launch_backsolve_central(const c128* LU, size_t stride, int n, int k, int batch, const c128* tau, c128* X, cudaStream_t st);
size_t final_inverse_ws_bytes(int k, int batch);

// fused.cu -- small-matrix mode: the whole elimination of a matrix in one launch, cl CTAs per matrix
bool fused_supported(int n, int k, int NB, int IB);
bool fused_is_tiny(int n);
int launch_lu_fused(c128* base, size_t stride, int n, int k, int batch, int NB, int IB, int align_first, int cl,
                    int* piv, c128* tau, int* info, cudaStream_t st);

// resident.cu -- small-matrix mode, on-chip variant: the matrix lives in the distributed shared memory of a cluster
int resident_cluster_size(int n, int k);             // smallest cluster that holds an n x n matrix on chip (0: none)
// *enqueued (optional) receives the number of leading items whose launch was accepted, also when a launch is refused
int launch_lu_resident(c128* base, size_t stride, int n, int k, int batch, int cl, int* piv, c128* tau, int* info, cudaStream_t st,
                       int* enqueued = nullptr);
// cudaOccupancyMaxActiveClusters of the cluster kernels for clusters of cl CTAs at their largest shared-memory size
// (the minimum over a kernel family's instances); 0 when such a cluster cannot be launched on the current device
int resident_max_active_clusters(int cl);
int fused_max_active_clusters(int cl);
int panel_cluster_max_active_clusters(int cl);

// reduce.cu
int launch_contour_sum(const c128* tau, const c128* w, int n_atoms, int n_e, int kk, c128* out, cudaStream_t st);

// probe.cu
int run_peak_probe(int which, int iters, double* sink, double* tflops, cudaStream_t st);

}  // namespace lsms
