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
 * State and threads ("the library owns nothing persistent ... re-entrant on different
 * streams").  There is NO process-wide state (one exception, described where it is declared: the built-in scratch
 * array of lsms_tau00_onchip_static_scratch).  Everything a call needs beyond its arguments lives in an opaque
 * handle the caller creates and destroys: the scheduler options and the auxiliary streams and events of the batch
 * scheduler (look-ahead and batch-group streams).  A handle is bound to the device that is current at its first call
 * that enqueues work; a later call made while another device is current returns cudaErrorInvalidDevice (101).  One handle serves
 * one host thread at a time; calls on DIFFERENT handles are independent and may run concurrently from different
 * host threads on different streams (the paper's callers are many MPI ranks sharing a GPU).
 *
 * Pointers are DEVICE pointers unless the name ends in _host.  The caller owns every buffer, including the
 * workspace; the library allocates no device memory (its device image holds one fixed 256 KB array, see
 * lsms_tau00_onchip_static_scratch).  All device work is ordered after what is already enqueued
 * on `cuda_stream` (a cudaStream_t passed as void*), later work on `cuda_stream` is ordered after it, and the calls
 * return without synchronising (the *_host entry point synchronises the stream before returning because it hands
 * results back in host memory).
 *
 * Return value (LAPACK-like): 0 = enqueued; -i = i-th argument invalid (null pointer, out-of-range size,
 * workspace too small, pointer not 16-byte aligned); >0 = CUDA runtime error code.  Numerical failure and invalid
 * per-item input VALUES are reported per item in info[] (device memory, written without synchronising), never as
 * a return code:  info[b] > 0: zero or non-finite pivot at elimination step info[b] (1-based);
 *                 info[b] < 0: an input value of item b is illegal (reading A4: Im z < 0 / Im kappa < 0, or a
 *                              non-finite z, kappa, phase shift or t^{-1}); the codes are listed per call.
 */
#ifndef LSMS_TAU_H
#define LSMS_TAU_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { double re, im; } lsms_c128;   /* == double _Complex == cuDoubleComplex */
typedef struct lsms_context* lsms_handle_t;    /* opaque; see "State and threads" above */

/* Library version string (static storage). */
const char* lsms_version(void);

/* Create a handle with default options (host only: no CUDA call, works without a device).  The first call that
 * enqueues work through it binds it to the current device: the kernels are opted into their shared-memory sizes
 * there and the scheduler's streams and events are created (non-blocking streams; one high-priority look-ahead
 * stream per batch group).  lsms_destroy synchronises nothing: destroy a handle only after the work enqueued
 * through it has completed.  Errors: -1 null argument; >0 CUDA error (allocation). */
int lsms_create(lsms_handle_t* handle_out);
int lsms_destroy(lsms_handle_t handle);

/* Scheduler options of a handle.  Results never depend on them beyond rounding order:
 * every item is eliminated independently with the same pivot rule (reading A14). */
enum {
    LSMS_OPT_NB_OUTER = 0,      /* outer panel width = inner dimension of the Schur update: 0 (default 64) or a multiple of
                                   4 up to 96.  The workspace size depends on it: query lsms_workspace_bytes afterwards.   */
    LSMS_OPT_IB_INNER = 1,      /* inner panel width: 0 (default 16) or 1..16                                              */
    LSMS_OPT_LOOKAHEAD = 2,     /* 1 (default): the next panel is factored on the handle's high-priority stream while the
                                   caller's stream runs the Schur update of the remaining columns; 0: one after the other  */
    LSMS_OPT_GROUPS = 3,        /* batch groups on separate streams, forked from and joined into the caller's stream:
                                   0 (default) chosen per shape, 1..8 forced                                               */
    LSMS_OPT_PANEL_THREADS = 4, /* panel kernel (K2): 1 (default) 512 threads for panels taller than 1280 rows, 256 below;
                                   0: 256 threads throughout (half an SM); 2: 128 threads (a quarter SM, the footprint of one
                                   Schur-update CTA) for panels of up to 1024 rows                                         */
    LSMS_OPT_PANEL_CLUSTER = 5, /* CTAs per matrix in the panel kernel (thread-block cluster, rows dealt round-robin,
                                   exchange through distributed shared memory): 0 (default) chosen per shape, 1 never,
                                   2 / 4 / 8 forced                                                                        */
    LSMS_OPT_ALIGN_FIRST = 6,   /* 1 (default): the first outer panel is n mod 64 columns wide so that all later trailing
                                   matrices are whole multiples of the 64-row Schur-update tile; 0: every panel NB wide    */
    LSMS_OPT_SMALL_MODE = 7,    /* small-matrix mode of the batch scheduler ("packs small LIZ matrices several per SM",
                                   north_star): the whole elimination of a matrix runs inside ONE launch, one CTA (or one
                                   cluster of CTAs) per matrix, several matrices resident per SM.  0 (default) chosen from
                                   (n, batch); 1 never (lock-step launches over the batch); 2 whenever the shape allows
                                   (n <= 2048), CTAs per matrix chosen from the batch size; 3 / 4 / 5 / 6: forced with
                                   1 / 2 / 4 / 8 CTAs per matrix, matrix in L2; 7: the on-chip variant (matrix held in the
                                   distributed shared memory of a cluster; n <= ~216), which is also what 0 picks when the
                                   matrix fits                                                                             */
    LSMS_OPT_COUNT = 8
};
int lsms_set_option(lsms_handle_t handle, int option, int value);       /* -1 handle, -2 option, -3 value out of range */
int lsms_get_option(lsms_handle_t handle, int option, int* value_host);

/* Bytes of device workspace that lsms_build_M_batched / lsms_tau00_batched need for these shapes with the
 * handle's current LSMS_OPT_NB_OUTER (host function, no GPU work).  0 if an argument is out of range. */
size_t lsms_workspace_bytes(lsms_handle_t handle, int n_sites, int lmax, int spin_canted, int batch);

/* Bytes of device workspace for lsms_solve_central_column_batched (holds a copy of M). */
size_t lsms_solve_workspace_bytes(lsms_handle_t handle, int n_sites, int kmax, int spin_canted, int batch);

/* Bytes of device scratch for lsms_tau00_from_host (inputs, M, outputs and workspace). */
size_t lsms_host_call_scratch_bytes(lsms_handle_t handle, int n_sites, int lmax, int spin_canted, int n_species, int batch);

/* Single-site inverse t-matrices from phase shifts (BASELINE.json configs[0]):
 *   kappa_b = sqrt(z_b) (principal root, Im >= 0),
 *   t_l = -(1/kappa) sin(delta_l) e^{i delta_l},   tinv = 1/t_l = -kappa / (sin(delta_l) e^{i delta_l}).
 *   delta     [n_species][n_spin][lmax+1]   phase shifts, n_spin = 1 + spin_canted
 *   species   [batch][n_sites]              int32 in [0, n_species)
 *   z         [batch]                       complex energies (Ry), Im z >= 0 (reading A4)
 *   tinv_diag [batch][n_sites][n_spin][lmax+1]  (out)
 *   kappa     [batch]                       (out)
 *   info      [batch] (out)  0 ok; -4: z_b non-finite or Im z_b < 0 (kappa_b and the item's tinv are then NaN);
 *                            -2: a species index of item b is out of range; -1: a phase shift used by item b is
 *                            non-finite or gives sin(delta) = 0 (no scattering: t^{-1} does not exist).
 * Errors: -1 handle, -2 delta, -3 species, -4 z, -5 lmax, -6 n_sites, -8 n_species, -9 batch, -10 tinv_diag,
 * -11 kappa, -12 info.                                                                                      */
int lsms_tinv_from_phase_shifts(lsms_handle_t handle, const lsms_c128* delta, const int* species, const lsms_c128* z,
                                int lmax, int n_sites, int spin_canted, int n_species, int batch,
                                lsms_c128* tinv_diag, lsms_c128* kappa, int* info, void* cuda_stream);

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
 *   kappa      [batch]  Im >= 0 (reading A4)
 *   M_out      [batch][n*n] column-major (out)
 *   info       [batch] (out)  0 ok; -5: kappa_b non-finite or Im kappa_b < 0 -- the item is rejected and its matrix
 *                             is filled with NaN (so that a later lsms_tau00_batched on it reports a pivot failure).
 * lmax in [0,8].  Errors: -1 handle, -2 tinv_diag, -3 site_pos, -4 moment_dir, -5 kappa, -6 lmax, -7 n_sites,
 * -9 batch, -10 M_out, -11 info, -12/-13 workspace.                                                         */
int lsms_build_M_batched(lsms_handle_t handle, const lsms_c128* tinv_diag, const double* site_pos, const double* moment_dir,
                         const lsms_c128* kappa, int lmax, int n_sites, int spin_canted, int batch,
                         lsms_c128* M_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* de-duplicated assembly.  g0 depends on the LIZ geometry and on kappa only, so when the batch
 * is (central atoms) x (energies) on one lattice (reading A19: item = atom * n_energies + energy) and every atom's
 * LIZ has the same site positions, each g0 block is evaluated once per energy and stored into the matrices of all
 * n_atoms atoms; only the site-diagonal t^{-1} blocks (and moments) are per item.  Arguments as for
 * lsms_build_M_batched with batch = n_atoms * n_energies, except that site_pos and kappa are READ FOR ATOM 0 ONLY
 * (items 0 .. n_energies-1): the caller guarantees site_pos[a][e] == site_pos[0][e] and kappa[a][e] == kappa[0][e].
 * The result is bit-identical to lsms_build_M_batched on such input.  info [batch] as above (the code of energy e
 * is written to every item a * n_energies + e).
 * Errors: -1 handle, -2 tinv_diag, -3 site_pos, -4 moment_dir, -5 kappa, -6 lmax, -7 n_sites, -9 n_atoms,
 * -10 n_energies, -11 M_out, -12 info, -13/-14 workspace.                                                    */
int lsms_build_M_shared_g0_batched(lsms_handle_t handle, const lsms_c128* tinv_diag, const double* site_pos,
                                   const double* moment_dir, const lsms_c128* kappa, int lmax, int n_sites, int spin_canted,
                                   int n_atoms, int n_energies,
                                   lsms_c128* M_out, int* info, void* workspace, size_t workspace_bytes, void* cuda_stream);

/* tau^{00}_b = central-site k x k block of M_b^{-1} by a blocked right-looking
 * LU with panel partial pivoting restricted to the non-central rows; the trailing k x k block after
 * n-k columns is the Schur complement of the central site and tau^{00} is its inverse (no
 * back-substitution).  Any nonsingular M of this shape is legal input (it need not come from
 * lsms_build_M_batched: the paper's own use is a CPU-built M).
 * The batch scheduler (north_star) picks the schedule from (n, batch) and the handle's options:
 * small matrices are eliminated start to finish inside one launch, one CTA or CTA cluster per matrix and several
 * matrices per SM; large ones advance in lock-step over the batch with every Schur update spanning the chip.
 *   M         [batch][n*n]  OVERWRITTEN (factorised in place), n = n_sites*k, k = kmax*(1+spin_canted)
 *   tau00_out [batch][k*k]  column-major (out)
 *   info      [batch] (out) 0 ok; j>0 = zero or non-finite pivot met at elimination step j (1-based)
 * Size limit: n <= 16384 rows; one or two matrices per call may have up to 40960 rows and three or four up to 20480
 * (their panels are factored by a cluster of CTAs) unless LSMS_OPT_PANEL_CLUSTER / LSMS_OPT_PANEL_THREADS or the device
 * rule that out.  Beyond it this
 * call, lsms_solve_central_column_batched and lsms_tau00_from_host return LSMS_ERR_PANEL_TOO_TALL before enqueueing
 * anything, and the workspace queries return 0.
 * Errors: -1 handle, -2 M, -3 n_sites, -4 kmax, -6 batch, -7 tau00_out, -8 info, -9/-10 workspace,
 * LSMS_ERR_PANEL_TOO_TALL.                                                                                    */
#define LSMS_ERR_PANEL_TOO_TALL (-22)
int lsms_tau00_batched(lsms_handle_t handle, lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                       lsms_c128* tau00_out, int* info,
                       void* workspace, size_t workspace_bytes, void* cuda_stream);

/* tau^{00} of a batch of SMALL matrices for a caller that cannot give the library any device workspace and cannot
 * allocate one (eq. (4), :62; the on-chip schedule of lsms_tau00_batched, LSMS_OPT_SMALL_MODE = 7).
 *
 * For whom: the paper's callers are Fortran MPI ranks that go through a C interface and share a GPU (PAPER.md:88-92,
 * :110).  A rank that sized all of its device buffers at start-up has no spare memory inside the energy loop; a
 * cudaMalloc there can fail because the other ranks hold the rest of the GPU, and it stalls the device for all of them.
 * Likewise a host code whose device memory belongs to another runtime (OpenACC / OpenMP data regions, a pool) can pass
 * matrices and result blocks but has no way to ask for workspace.  This call needs none: it takes no handle and no
 * workspace, and it calls no cudaMalloc / cudaFree and creates no stream or event.  The one piece of global memory the
 * kernel needs beyond its arguments -- a pivot word per matrix row -- is a fixed array of LSMS_STATIC_SCRATCH_WORDS
 * 32-bit words (256 KB) built into the library, which every GPU that loads the library holds until the process exits.
 *
 *   M         [batch][n*n]  column-major, OVERWRITTEN (factorised in place), n = n_sites*k, k = kmax*(1+spin_canted);
 *                           n must fit the on-chip kernel: n <= 256 and the matrix within the shared memory of 8 SMs
 *                           (n <= ~216 for complex128), else LSMS_ERR_NOT_ON_CHIP
 *   batch                   batch * n <= LSMS_STATIC_SCRATCH_WORDS, else LSMS_ERR_STATIC_SCRATCH_TOO_SMALL
 *   tau00_out [batch][k*k]  column-major (out);   info [batch] (out) as for lsms_tau00_batched
 * Both size limits are checked on the host before any CUDA call.  Results are those of lsms_tau00_batched in on-chip
 * mode (same kernel, same launch shape).
 * First call on a device: it looks up the array's address on that device and opts the kernel into its shared-memory
 * size (once per device, remembered inside the library, thread-safe).  Make that first call outside any stream capture.
 * Sharing: every call on a device uses the same array, whatever the stream or host thread.  Calls that overlap on the
 * GPU overwrite each other's pivot words -- order them (one stream, or events).  The array keeps the last call's
 * contents; nothing in it needs clearing, the kernel writes a matrix's pivot words before anything reads them.
 * Errors: -1 M, -2 n_sites, -3 kmax, -5 batch, -6 tau00_out, -7 info (null or not 16-byte aligned where complex),
 * LSMS_ERR_NOT_ON_CHIP, LSMS_ERR_STATIC_SCRATCH_TOO_SMALL; >0 CUDA error code.                                  */
#define LSMS_STATIC_SCRATCH_WORDS 65536
#define LSMS_ERR_NOT_ON_CHIP (-20)              /* codes below -19 name a condition, not an argument position */
#define LSMS_ERR_STATIC_SCRATCH_TOO_SMALL (-21)
int lsms_tau00_onchip_static_scratch(lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                                     lsms_c128* tau00_out, int* info, void* cuda_stream);

/* Verification only (not on the timed path): the whole central block column X = M^{-1} E,
 * E = last k columns of I_n, for the residual test ||M X - E|| ("solving X'X = I").
 *   M     [batch][n*n]  NOT modified (a copy is factorised in the workspace)
 *   X_out [batch][n*k]  column-major, ld = n (out);  info [batch] as above.
 * Errors as for lsms_tau00_batched (-7 X_out).                                                               */
int lsms_solve_central_column_batched(lsms_handle_t handle, const lsms_c128* M, int n_sites, int kmax, int spin_canted,
                                      int batch, lsms_c128* X_out, int* info,
                                      void* workspace, size_t workspace_bytes, void* cuda_stream);

/* End-to-end call with HOST inputs and outputs: copies the (small) inputs to the device, runs
 * lsms_tinv_from_phase_shifts + assembly + lsms_tau00_batched on `cuda_stream`, copies tau00 and info back and
 * synchronises the stream.  Host buffers should be pinned.
 *   delta_host [n_species][n_spin][lmax+1], species_host [batch][n_sites], z_host [batch],
 *   site_pos_host [batch][n_sites][3], moment_dir_host [batch][n_sites][3] or NULL,
 *   n_energies: 0, or the number of energies of a batch laid out as item = atom * n_energies + energy (reading A19).
 *     When it divides the batch and the HOST inputs show that every atom has the same site positions and the same
 *     z per energy index as atom 0 (compared bytewise here, on the host), the matrices are assembled by
 *     lsms_build_M_shared_g0_batched (f3: one g0 per energy), else item by item; same results.
 *   tau00_out_host [batch][k*k], info_host [batch]: first non-zero code of the three stages per item;
 *   device_scratch: >= lsms_host_call_scratch_bytes(...) bytes of DEVICE memory.
 * h2d_bytes / d2h_bytes (may be NULL) receive the bytes copied in each direction.
 * Errors: -1 handle, -2 delta, -3 species, -4 z, -5 site_pos, -6 moment_dir, -7 lmax, -8 n_sites, -10 n_species,
 * -11 batch, -12 n_energies, -13 tau00_out, -14 info, -15/-16 scratch.                                       */
int lsms_tau00_from_host(lsms_handle_t handle, const lsms_c128* delta_host, const int* species_host, const lsms_c128* z_host,
                         const double* site_pos_host, const double* moment_dir_host,
                         int lmax, int n_sites, int spin_canted, int n_species, int batch, int n_energies,
                         lsms_c128* tau00_out_host, int* info_host,
                         void* device_scratch, size_t scratch_bytes, void* cuda_stream,
                         size_t* h2d_bytes, size_t* d2h_bytes);

/* the tau part of the energy-contour integral of eq. (2)/(3): for every
 * central atom a,  out_a = sum_q weights_q * tau00_{a,q},  with the batch index = a * n_energies + q of
 * lsms_tau00_batched (reading A19).  The caller supplies the complex quadrature weights (rule weight x dz/dq).
 *   tau00   [n_atoms][n_energies][k*k]  device (the tau00_out of lsms_tau00_batched)
 *   weights [n_energies]                device
 *   out     [n_atoms][k*k]              device (out), column-major k x k like tau00
 * Errors: -1 handle, -2 tau00, -3 weights, -4 n_atoms, -5 n_energies (1..2048), -6 k, -7 out.                */
int lsms_contour_sum_batched(lsms_handle_t handle, const lsms_c128* tau00, const lsms_c128* weights, int n_atoms,
                             int n_energies, int k, lsms_c128* out, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* LSMS_TAU_H */
