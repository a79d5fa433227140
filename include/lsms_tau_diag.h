/* lsms_tau_diag.h -- measurement and debugging entry points of liblsms_tau.so.
 *
 * NOT part of the method's boundary (include/lsms_tau.h): nothing here is needed to compute
 * tau^{00}.  These calls exist so that bench.py and the tests can time kernel classes inside a step, measure the
 * FP64 roofline denominator on the box, run the Schur update alone for ncu
 * (BASELINE.json north_star: "evidenced by ncu") and check the closed-form Gaunt table without a device.
 * Same conventions as lsms_tau.h: device pointers unless named *_host, per-handle state only.
 */
#ifndef LSMS_TAU_DIAG_H
#define LSMS_TAU_DIAG_H

#include "lsms_tau.h"

#ifdef __cplusplus
extern "C" {
#endif

/* How many kernels the last call made through this handle enqueued (counted on the host at launch time). */
int lsms_last_launch_count(lsms_handle_t handle);

/* Which schedule the last lsms_tau00_batched call through this handle used: 0 lock-step launches over the batch,
 * 1 <= c <= 8: small-matrix mode through L2 with c CTAs per matrix; 100 + c: on-chip small-matrix mode, the matrix held
 * in the distributed shared memory of a cluster of c CTAs.  -1 before the first call. */
int lsms_last_schedule(lsms_handle_t handle);

/* How many thread-block clusters of `cluster_size` (1, 2, 4, 8) CTAs of a cluster kernel fit on the handle's device at
 * once -- as this process sees it, so under MPS / MIG the answer is for its SM partition (cudaOccupancyMaxActiveClusters at the
 * kernel's largest shared-memory size, asked once when the handle is bound).  kernel: 0 on-chip elimination
 * (k_lu_resident), 1 one-launch elimination through L2 (k_lu_fused / k_lu_tiny), 2 cluster panel kernel (k_panel_clu;
 * cluster_size 1 gives 0).  0 means the scheduler never picks that kernel with that cluster size on this device and
 * uses the lock-step / one-CTA schedule instead.  Binds the handle.  Errors: -1 handle, -2 kernel, -3 cluster_size, -4 count_host. */
int lsms_max_active_clusters(lsms_handle_t handle, int kernel, int cluster_size, int* count_host);

/* Per-kernel-class timing.  Between lsms_profile_begin and lsms_profile_end every kernel enqueued through the
 * handle is bracketed by CUDA events on the stream it is launched on (the events belong to the handle and are
 * created on demand).  lsms_profile_end synchronises those events and returns, per class, the summed device time
 * in ms, the number of launches and the algorithmic flops (K4 classes only):
 *   0 K1 assembly, 1 K2 panel LU, 2 small-matrix mode (whole elimination in one launch), 3 K4 inner rank-IB updates,
 *   4 K4 Schur update (inner dimension NB), 5 K5 final inverse, 6 K3a/K3b net row permutation + -(L11^-1),
 *   7 K4 used as the triangular solve U12 = -(Ninv * A12).
 * All three arrays are HOST arrays of 8 entries.  Meaningful with one batch group and no look-ahead, when every
 * event pair brackets one kernel running alone. */
int lsms_profile_begin(lsms_handle_t handle);
int lsms_profile_end(lsms_handle_t handle, double* ms_by_class_host, int* launches_by_class_host, double* flops_by_class_host);

/* FP64 peak probe (the roofline denominator): runs a register-resident DMMA.8x8x4
 * (which = 0) or DFMA (which = 1) chain on every SM for `iters` iterations and returns the achieved TFLOP/s in
 * *tflops_host; synchronises.  `sink` is 8 bytes of device memory the kernel may write (never does). */
int lsms_fp64_peak_probe(lsms_handle_t handle, int which, int iters, double* sink, double* tflops_host, void* cuda_stream);

/* Schur update alone (the K4 kernel): for each item C -= A B with A = M[r0:, c0:c0+kk],
 * B = M[c0:c0+kk, r0:], C = M[r0:, r0:], r0 = c0 + kk, on the n x n column-major matrices. */
int lsms_schur_update_batched(lsms_handle_t handle, lsms_c128* M, int n, int c0, int kk, int batch, void* cuda_stream);

/* Host only, no handle: the closed-form Gaunt number C(L,L',L'') = Int Y_L^* Y_L' Y_L''^* dOmega, m'' = m' - m,
 * that K1 tabulates (two Wigner 3j symbols, Racah's sum). */
double lsms_debug_gaunt_closed_form(int l, int m, int lp, int mp, int lpp);

#ifdef __cplusplus
}
#endif
#endif /* LSMS_TAU_DIAG_H */
