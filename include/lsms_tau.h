/* lsms_tau.h -- C ABI of the B200-native LSMS tau^{00} library (liblsms_tau.so).
 *
 * The hot path of arxiv 2308.16317 ("High Performance GPU Accelerated MuST Software"):
 *     tau(e) = [ t^{-1}(e) - g0(e) ]^{-1}                       PAPER.md:54, eq. (4)
 * of which "only the first block of the inverted matrix is needed"  PAPER.md:62,
 * i.e. tau^{00}, the central-site block of the inverse of the LIZ KKR matrix
 * M = t^{-1} - g0, for many (atom, energy) items at once.
 * The paper's boundary is "Fortran subroutine -> C interface -> CUDA";
 * this header is that boundary with the matrix built on the device (the paper's stated
 * future work) and without cuSOLVER.
 *
 * Conventions:
 *   - every floating-point number is IEEE binary64; complex = interleaved (re,im), 16 B
 *   - matrices are column-major, ld = n, batch stride n*n
 *   - n_sites sites per LIZ, API site 0 is the central site; it is STORED in the LAST
 *     diagonal block so that it is eliminated last (sites 1..N-1 -> blocks 0..N-2)
 *   - kmax = (lmax+1)^2, L = l(l+1)+m; k = kmax*(1+spin_canted); n = n_sites*k;
 *     spin-canted within-site index = s*kmax + L, s = 0 (up), 1 (down)
 *   - Rydberg atomic units: kappa = sqrt(z), Im kappa >= 0, lengths in Bohr
 *
 * Pointers are DEVICE pointers unless the name ends in _host.  The caller owns every
 * buffer, including the workspace; the library allocates no device memory.  Its only
 * persistent objects are the internal streams and events of lsms_tau00_batched's scheduler
 * (look-ahead and batch-group streams, created on first use) and the process-wide tuning
 * knobs below.  All device work is ordered after what is already enqueued on `cuda_stream`
 * (a cudaStream_t passed as void*), later work on `cuda_stream` is ordered after it, and the
 * calls return without synchronising (the *_host entry point synchronises the stream
 * before returning because it hands results back in host memory).  Because the internal
 * streams are shared, calls from several host threads must be serialised by the caller;
 * successive calls on different caller streams are correct and run one after the other.
 *
 * Return value (LAPACK-like): 0 = enqueued; -i = i-th argument invalid (null pointer,
 * out-of-range size, workspace too small, pointer not 16-byte aligned); >0 = CUDA runtime
 * error code.  Numerical failure is per item in info[], never a return code.
 */
#ifndef LSMS_TAU_H
#define LSMS_TAU_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double re, im; } lsms_c128;   /* == double _Complex == cuDoubleComplex */

/* Library version string (static storage). */
const char* lsms_version(void);

/* Bytes of device workspace that lsms_build_M_batched / lsms_tau00_batched need for these
 * shapes (host function, no GPU work).  0 if an argument is out of range. */
size_t lsms_workspace_bytes(int n_sites, int lmax, int spin_canted, int batch);

/* Bytes of device workspace for lsms_solve_central_column_batched (holds a copy of M). */
size_t lsms_solve_workspace_bytes(int n_sites, int kmax, int spin_canted, int batch);

/* Bytes of device scratch for lsms_tau00_from_host (inputs, M, outputs and workspace). */
size_t lsms_host_call_scratch_bytes(int n_sites, int lmax, int spin_canted, int n_species, int batch);

/* Single-site inverse t-matrices from phase shifts (BASELINE.json configs[0]):
 *   kappa_b = sqrt(z_b) (principal root, Im >= 0),
 *   t_l = -(1/kappa) sin(delta_l) e^{i delta_l},   tinv = 1/t_l = -kappa / (sin(delta_l) e^{i delta_l}).
 *   delta     [n_species][n_spin][lmax+1]   phase shifts, n_spin = 1 + spin_canted
 *   species   [batch][n_sites]              int32 in [0, n_species)
 *   z         [batch]                       complex energies (Ry), Im z >= 0
 *   tinv_diag [batch][n_sites][n_spin][lmax+1]  (out)
 *   kappa     [batch]                       (out)                                              */
int lsms_tinv_from_phase_shifts(const lsms_c128* delta, const int* species, const lsms_c128* z,
                                int lmax, int n_sites, int spin_canted, int n_species, int batch,
                                lsms_c128* tinv_diag, lsms_c128* kappa, void* cuda_stream);

/* Assemble the KKR matrices M = t^{-1} - g0 on the device.
 *   off-site blocks (i != j): -g0_{LL'}(R_i - R_j; kappa), with
 *     g0_{LL'}(R) = -4 pi i kappa sum_{l''} i^{l-l'+l''} h_{l''}(kappa R) Y_{l'',m'-m}(R^) C(L,L',L''),
 *     C = Int Y_L^* Y_L' Y_L''^* dOmega (Gaunt), h = spherical Hankel of the first kind,
 *     Y complex with Condon-Shortley phase; (x) 1_2 in spin space when spin_canted;
 *   site-diagonal blocks: diag_L(tinv_l); spin-canted: 1/2(a+b) (x) 1 + 1/2(a-b) (x) (sigma . e_i),
 *     a/b = up/down tinv (App. A (A3)).
 *   tinv_diag  [batch][n_sites][n_spin][lmax+1]
 *   site_pos   [batch][n_sites][3]  Bohr, site 0 = central
 *   moment_dir [batch][n_sites][3]  unit vectors; may be NULL iff !spin_canted
 *   kappa      [batch]  Im >= 0
 *   M_out      [batch][n*n] column-major (out)
 * lmax in [0,8].  Errors: -1..-4 null inputs, -5 lmax, -6 n_sites, -8 batch, -9 M_out,
 * -10/-11 workspace.                                                                           */
int lsms_build_M_batched(const lsms_c128* tinv_diag, const double* site_pos, const double* moment_dir,
                         const lsms_c128* kappa, int lmax, int n_sites, int spin_canted, int batch,
                         lsms_c128* M_out, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* de-duplicated assembly.  g0 depends on the LIZ geometry and on kappa only, so when the batch
 * is (central atoms) x (energies) on one lattice (reading A19: item = atom * n_energies + energy) and every atom's
 * LIZ has the same site positions, each g0 block is evaluated once per energy and stored into the matrices of all
 * n_atoms atoms; only the site-diagonal t^{-1} blocks (and moments) are per item.  Arguments as for
 * lsms_build_M_batched with batch = n_atoms * n_energies, except that site_pos and kappa are READ FOR ATOM 0 ONLY
 * (items 0 .. n_energies-1): the caller guarantees site_pos[a][e] == site_pos[0][e] and kappa[a][e] == kappa[0][e].
 * The result is bit-identical to lsms_build_M_batched on such input.
 * Errors: -1..-4 null inputs, -5 lmax, -6 n_sites, -8 n_atoms, -9 n_energies, -10 M_out, -11/-12 workspace.        */
int lsms_build_M_shared_g0_batched(const lsms_c128* tinv_diag, const double* site_pos, const double* moment_dir,
                                   const lsms_c128* kappa, int lmax, int n_sites, int spin_canted,
                                   int n_atoms, int n_energies,
                                   lsms_c128* M_out, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* tau^{00}_b = central-site k x k block of M_b^{-1} by a blocked right-looking
 * LU with panel partial pivoting restricted to the non-central rows; the trailing k x k block after
 * n-k columns is the Schur complement of the central site and tau^{00} is its inverse (no
 * back-substitution).  Any nonsingular M of this shape is legal input (it need not come from
 * lsms_build_M_batched: the paper's own use is a CPU-built M).
 *   M         [batch][n*n]  OVERWRITTEN (factorised in place), n = n_sites*k, k = kmax*(1+spin_canted)
 *   tau00_out [batch][k*k]  column-major (out)
 *   info      [batch]       0 ok; j>0 = zero or non-finite pivot met at elimination step j (1-based)
 * Errors: -1 M, -2 n_sites, -3 kmax, -5 batch, -6 tau00_out, -7 info, -8/-9 workspace.         */
int lsms_tau00_batched(lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                       lsms_c128* tau00_out, int* info,
                       void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Verification only (not on the timed path): the whole central block column X = M^{-1} E,
 * E = last k columns of I_n, for the residual test ||M X - E|| ("solving X'X = I").
 *   M     [batch][n*n]  NOT modified (a copy is factorised in the workspace)
 *   X_out [batch][n*k]  column-major, ld = n (out);  info [batch] as above.                     */
int lsms_solve_central_column_batched(const lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                                      lsms_c128* X_out, int* info,
                                      void* workspace, size_t workspace_bytes, void* cuda_stream);

/* End-to-end call with HOST inputs and outputs: copies the (small) inputs to the device,
 * runs lsms_tinv_from_phase_shifts + lsms_build_M_batched + lsms_tau00_batched on `cuda_stream`,
 * copies tau00 and info back and synchronises the stream.  Host buffers should be pinned.
 *   delta_host [n_species][n_spin][lmax+1], species_host [batch][n_sites], z_host [batch],
 *   site_pos_host [batch][n_sites][3], moment_dir_host [batch][n_sites][3] or NULL,
 *   tau00_out_host [batch][k*k], info_host [batch];
 *   device_scratch: >= lsms_host_call_scratch_bytes(...) bytes of DEVICE memory.
 * h2d_bytes / d2h_bytes (may be NULL) receive the bytes copied in each direction.               */
int lsms_tau00_from_host(const lsms_c128* delta_host, const int* species_host, const lsms_c128* z_host,
                         const double* site_pos_host, const double* moment_dir_host,
                         int lmax, int n_sites, int spin_canted, int n_species, int batch,
                         lsms_c128* tau00_out_host, int* info_host,
                         void* device_scratch, size_t scratch_bytes, void* cuda_stream,
                         size_t* h2d_bytes, size_t* d2h_bytes);

/* the tau part of the energy-contour integral of eq. (2)/(3): for every
 * central atom a,  out_a = sum_q weights_q * tau00_{a,q},  with the batch index = a * n_energies + q of
 * lsms_tau00_batched (reading A19).  The caller supplies the complex quadrature weights (rule weight x dz/dq).
 *   tau00   [n_atoms][n_energies][k*k]  device (the tau00_out of lsms_tau00_batched)
 *   weights [n_energies]                device
 *   out     [n_atoms][k*k]              device (out), column-major k x k like tau00
 * Errors: -1 tau00, -2 weights, -3 n_atoms, -4 n_energies (1..2048), -5 k, -6 out.               */
int lsms_contour_sum_batched(const lsms_c128* tau00, const lsms_c128* weights, int n_atoms, int n_energies, int k,
                             lsms_c128* out, void* cuda_stream);

/* Tuning knobs (process-wide, not thread-safe; defaults chosen per shape when 0):
 *   outer panel width NB (multiple of 4, <= 96; the workspace size depends on it: query
 *   lsms_workspace_bytes after setting it) and inner panel width IB (<= 16).             */
int lsms_set_blocking(int nb_outer, int ib_inner);

/* Look-ahead (default on): the next panel is factored on a library-owned high-priority stream while the
 * caller's stream runs the Schur update of the remaining columns; the two are joined with events before
 * the call returns to the next panel, so the caller still sees one ordered stream.  The auxiliary streams
 * and their events are created on first use and are the library's only persistent objects. */
int lsms_set_lookahead(int on);

/* Batch groups (default 0 = chosen per shape: two groups for batches of 16 or more, else one): the batch is cut into `groups` (<= 8) contiguous groups that
 * run the elimination on separate library-owned streams, forked from and joined back into the caller's
 * stream inside lsms_tau00_batched, so that the poorly parallel phases of one group (net permutation,
 * triangular solve, look-ahead slice, last panels) run under another group's Schur updates.  Results do
 * not depend on the setting (every item is eliminated independently).  Errors: -1 groups out of range. */
int lsms_set_groups(int groups);

/* Panel kernel (K2) variant: 1 (default) register-blocked sub-panels, 512 threads for panels taller than 1280
 * rows and 256 below; 0 register-blocked, 256 threads throughout (half an SM, narrower sub-panels for tall
 * panels); -1 the L2-resident column-at-a-time kernel.  All variants pick the same pivots (|re|+|im|, ties to
 * the lowest row) and perform the same arithmetic per element.  Errors: -1 out of range. */
int lsms_set_panel_variant(int variant);

/* CTAs per matrix in the panel kernel (thread-block cluster, rows dealt round-robin, exchange through distributed
 * shared memory): 0 (default) chosen per shape -- 8 (4) CTAs for batches of one or two matrices while the panel is
 * taller than 4096 (2048) rows, else one: under look-ahead a cluster has to wait for co-scheduled SMs and larger
 * batches lose --, 1 never, 2 / 4 / 8 forced.  Same pivots and arithmetic as the one-CTA kernel.  Errors: -1. */
int lsms_set_panel_cluster(int cl);

/* Tile alignment (default on): the first outer panel is n mod 64 columns wide, so that all later trailing
 * matrices are whole multiples of 64 rows and columns (the Schur-update tile is 64 x 32).  Off: every panel is NB wide. */
int lsms_set_align_first(int on);

/* How many kernels the last lsms_tau00_batched / lsms_build_M_batched call on this thread enqueued. */
int lsms_last_launch_count(void);

/* Optional per-kernel-class timing (measurement aid; process-wide, not thread-safe).  Between
 * lsms_profile_begin() and lsms_profile_end() every kernel the library enqueues is bracketed by CUDA
 * events on the caller's stream.  lsms_profile_end synchronises those events and returns, per class,
 * the summed device time in ms, the number of launches and the algorithmic flops (K4 classes only):
 *   0 K1 assembly, 1 K2 panel LU, 2 K3 interchanges+TRSM, 3 K4 inner rank-IB updates,
 *   4 K4 Schur update (inner dimension NB), 5 K5 final inverse, 6 K3a/K3b net row permutation + -(L11^-1),
 *   7 K4 used as the triangular solve U12 = -(Ninv * A12).
 * All three arrays are HOST arrays of 8 entries. */
int lsms_profile_begin(void);
int lsms_profile_end(double* ms_by_class_host, int* launches_by_class_host, double* flops_by_class_host);

/* FP64 peak probe (measurement aid for the roofline denominator):
 * runs a register-resident DMMA.8x8x4 (which = 0) or DFMA (which = 1) chain on every SM for
 * `iters` iterations and returns the achieved TFLOP/s in *tflops (host pointer); synchronises. */
int lsms_fp64_peak_probe(int which, int iters, double* tflops_host, void* cuda_stream);

/* Schur update alone (the K4 kernel): for each item C -= A B with A = M[r0:, c0:c0+kk],
 * B = M[c0:c0+kk, r0:], C = M[r0:, r0:], r0 = c0 + kk, on the n x n column-major matrices.
 * Exposed so the update can be timed and profiled in isolation (BASELINE.json north_star). */
int lsms_schur_update_batched(lsms_c128* M, int n, int c0, int kk, int batch, void* cuda_stream);

/* Host-only debug export (no GPU work): the closed-form Gaunt number
 * C(L,L',L'') = Int Y_L^* Y_L' Y_L''^* dOmega, m'' = m' - m, that K1 tabulates (two Wigner 3j
 * symbols, Racah's sum).  Lets the CPU test-suite check the table without a device. */
double lsms_debug_gaunt_closed_form(int l, int m, int lp, int mp, int lpp);

#ifdef __cplusplus
}
#endif
#endif /* LSMS_TAU_H */
