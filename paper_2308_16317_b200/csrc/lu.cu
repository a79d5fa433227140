// lu.cu -- K3a/K3b (net row permutation of an outer panel, -(L11^-1), row gather/scatter of the trailing
// columns), K5 (inverse of the final k x k Schur complement) and the verification-only back-substitution.
// SURVEY.md 8(a) a4, a6; "LU factorization of the matrix" PAPER.md:92; "only the first block of the inverted
// matrix is needed" PAPER.md:62.  (K2, the panel factorisation itself, is in panel.cu / panel_cluster.cu.)
#include "common.cuh"
#include "internal.h"
#include "lu_body.cuh"

namespace lsms {

// ---------------------------------------------------------------- K3a: after an outer panel
// One CTA per matrix, once the outer panel [J, J+W) is fully factored:
//  * warp 0 folds the W interchanges (applied in order) into one row permutation:
//      perm[0] = nd, top_src[i] = row whose content ends in top position J+i,
//      (down_dst[j], down_top[j]) = row below the top block that receives original top row J+down_top[j];
//    (a row that enters the top block at step i stays there, so every displaced row is an original top row)
//  * the other warps stage L11 (unit lower W x W) in shared memory; then the whole CTA inverts it by 16 x 16
//    blocks (diagonal blocks by forward substitution, block rows X_{ij} = -D_i^{-1} sum_k L_{ik} X_{kj} in place)
//    and stores Ninv = -(L11)^{-1}, so that U12 = L11^{-1} A12 becomes a GEMM on the DMMA path: U12 = -(Ninv * A12).
constexpr int POST_THREADS = 256;

__global__ void __launch_bounds__(POST_THREADS)
k_panel_post(const c128* __restrict__ base, size_t stride, int n, int J, int W, const int* __restrict__ piv,
             int* __restrict__ perm_all, c128* __restrict__ ninv_all, int nbmax) {
    extern __shared__ __align__(16) unsigned char post_smem[];
    const int nb16 = (W + 15) / 16, Wp = nb16 * 16;
    c128* X = reinterpret_cast<c128*>(post_smem);                 // [Wp][Wp] column-major: L11 (padded with I), then L11^{-1} in place
    c128* T = X + (size_t)Wp * Wp;                                // [16][Wp]   scratch block row
    int* cur_top = reinterpret_cast<int*>(T + (size_t)16 * Wp);
    int* bpos = cur_top + W;
    int* bcon = bpos + W;
    const c128* A = base + (size_t)blockIdx.x * stride;
    const int* pv = piv + (size_t)blockIdx.x * n + J;
    int* perm = perm_all + (size_t)blockIdx.x * (4 + 3 * nbmax);
    c128* ninv = ninv_all + (size_t)blockIdx.x * nbmax * nbmax;
    const int tid = threadIdx.x;

    if (tid < 32) {
        // ---- net permutation (warp 0)
        net_permutation(pv, J, W, cur_top, bpos, bcon, perm, perm + 1, perm + 1 + nbmax, perm + 1 + 2 * nbmax);
    } else {
        // ---- L11 -> shared memory (strictly lower part; unit diagonal; identity padding up to Wp)
        for (int e = tid - 32; e < Wp * Wp; e += POST_THREADS - 32) {
            const int i = e % Wp, j = e / Wp;
            c128 v = cmake(i == j ? 1.0 : 0.0, 0.0);
            if (i > j && i < W) v = A[(size_t)(J + i) + (size_t)(J + j) * n];
            X[i + j * Wp] = v;
        }
    }
    __syncthreads();
    // ---- diagonal 16 x 16 blocks: D^{-1} in place, one thread per column (unit lower: x_jj = 1)
    {
        const int b0 = (tid / 16) * 16, j = tid % 16;
        c128 x[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = cmake(i == j ? 1.0 : 0.0, 0.0);
        if (tid < Wp) {
#pragma unroll
            for (int i = 1; i < 16; ++i) {
                if (i > j) {
                    c128 acc = cmake(0.0, 0.0);
#pragma unroll
                    for (int k = 0; k < i; ++k) if (k >= j) cfms(acc, X[(b0 + i) + (b0 + k) * Wp], x[k]);
                    x[i] = acc;
                }
            }
        }
        __syncthreads();       // every read of a diagonal block precedes the writes below
        if (tid < Wp) {
#pragma unroll
            for (int i = 0; i < 16; ++i) if (i > j) X[(b0 + i) + (b0 + j) * Wp] = x[i];
        }
    }
    __syncthreads();
    // ---- block rows: X_{bi,bj} = -D_bi^{-1} * sum_{bk = bj}^{bi-1} L_{bi,bk} X_{bk,bj}, written over L_{bi,bj}
    for (int bi = 1; bi < nb16; ++bi) {
        const int ncol = bi * 16;
        for (int e = tid; e < 16 * ncol; e += POST_THREADS) {
            const int i = e % 16, j = e / 16, bj = j / 16;
            c128 acc = cmake(0.0, 0.0);
            for (int k = bj * 16; k < ncol; ++k) cfma(acc, X[(bi * 16 + i) + k * Wp], X[k + j * Wp]);
            T[i + j * 16] = acc;
        }
        __syncthreads();
        for (int e = tid; e < 16 * ncol; e += POST_THREADS) {
            const int i = e % 16, j = e / 16;
            c128 acc = cmake(0.0, 0.0);
            for (int k = 0; k <= i; ++k) cfms(acc, X[(bi * 16 + i) + (bi * 16 + k) * Wp], T[k + j * 16]);
            X[(bi * 16 + i) + j * Wp] = acc;       // block row bi of L is dead: only T and D_bi^{-1} are read in this phase
        }
        __syncthreads();
    }
    for (int e = tid; e < W * W; e += POST_THREADS) {
        const int i = e % W, j = e / W;
        ninv[i + (size_t)j * nbmax] = (i >= j) ? cneg(X[i + j * Wp]) : cmake(0.0, 0.0);
    }
}

// ---------------------------------------------------------------- K3b: apply the net row permutation
// to the trailing columns [col_lo, col_hi): the new top block (rows J..J+W) goes, packed with ld = nbmax,
// to tperm (the B operand of the TRSM-GEMM that writes U12 back into the matrix); displaced original top
// rows are scattered to their final rows below.  One CTA per strip of PERM_TN columns: 16 for matrices of up to ~4000
// rows, 8 for taller ones, whose scattered row accesses of a strip span more DRAM pages (measured, K3a + K3b per step:
// H (6750 rows) 26.5 -> 24.0 ms with 8 columns; M (880) 2.9 -> 3.2 and P (2160) 5.8 -> 5.8, so those keep 16).
constexpr int PERM_THREADS = 256;

template <int PERM_TN>
__global__ void __launch_bounds__(PERM_THREADS)
k_row_permute(c128* __restrict__ base, size_t stride, int n, int J, int W, int col_lo, int col_hi,
              const int* __restrict__ perm_all, c128* __restrict__ tperm_all, size_t tperm_stride, int nbmax) {
    extern __shared__ __align__(16) unsigned char perm_smem[];
    c128* Told = reinterpret_cast<c128*>(perm_smem);               // [PERM_TN][W]
    int* s_perm = reinterpret_cast<int*>(perm_smem + (size_t)PERM_TN * W * sizeof(c128));   // [1 + 3W]
    c128* A = base + (size_t)blockIdx.y * stride;
    const int* perm = perm_all + (size_t)blockIdx.y * (4 + 3 * nbmax);
    c128* T = tperm_all + (size_t)blockIdx.y * tperm_stride;
    const int tid = threadIdx.x;
    const int c_first = col_lo + blockIdx.x * PERM_TN;
    const int ncol = min(PERM_TN, col_hi - c_first);
    const int nd = perm[0];
    if (tid == 0) s_perm[0] = nd;
    for (int i = tid; i < W; i += PERM_THREADS) {
        s_perm[1 + i] = perm[1 + i];
        if (i < nd) { s_perm[1 + W + i] = perm[1 + nbmax + i]; s_perm[1 + 2 * W + i] = perm[1 + 2 * nbmax + i]; }
    }
    for (int e = tid; e < ncol * W; e += PERM_THREADS) {
        const int i = e % W, c = e / W;
        Told[c * W + i] = A[(size_t)(J + i) + (size_t)(c_first + c) * n];
    }
    __syncthreads();
    // gather the new top block (rows from below are read before any scatter of this CTA's columns)
    for (int e = tid; e < ncol * W; e += PERM_THREADS) {
        const int i = e % W, c = e / W;
        const int src = s_perm[1 + i];
        c128 v = (src < J + W) ? Told[c * W + (src - J)] : A[(size_t)src + (size_t)(c_first + c) * n];
        T[(size_t)i + (size_t)(c_first + c) * nbmax] = v;
    }
    __syncthreads();
    for (int e = tid; e < ncol * nd; e += PERM_THREADS) {
        const int j = e % nd, c = e / nd;
        A[(size_t)s_perm[1 + W + j] + (size_t)(c_first + c) * n] = Told[c * W + s_perm[1 + 2 * W + j]];
    }
}

// ---------------------------------------------------------------- K5: tau00 = S^{-1}
// One CTA per matrix: in-place Gauss-Jordan inversion with partial pivoting of the trailing k x k
// block, in shared memory when it fits (k <= 96), else in a global scratch buffer.
constexpr int K5_THREADS = 256;

__global__ void __launch_bounds__(K5_THREADS)
k_final_inverse(const c128* __restrict__ base, size_t stride, int n, int k, c128* __restrict__ tau, int* __restrict__ info,
                c128* __restrict__ gscratch, int use_smem) {
    extern __shared__ __align__(16) unsigned char k5_smem[];
    __shared__ K5Shared sh;
    c128* S = use_smem ? reinterpret_cast<c128*>(k5_smem) : gscratch + (size_t)blockIdx.x * k * k;
    final_inverse_body<K5_THREADS>(base + (size_t)blockIdx.x * stride, n, k, tau + (size_t)blockIdx.x * k * k, info + blockIdx.x, S, sh);
}

size_t final_inverse_ws_bytes(int k, int batch) { return k > 96 ? (size_t)batch * k * k * sizeof(c128) : 0; }

// ---------------------------------------------------------------- verification: X = M^{-1} E
// After the restricted-pivot elimination the system reads [U11 U12; 0 S] X = [0; I] (the
// interchanges never touch the central rows, where E is non-zero), so X2 = S^{-1} = tau00 and
// X1 = -U11^{-1} (U12 X2).  One CTA per (item, column of X).  Slow by design; not timed.
__global__ void __launch_bounds__(256)
k_backsolve_central(const c128* __restrict__ LU, size_t stride, int n, int k, const c128* __restrict__ tau, c128* __restrict__ X) {
    const c128* A = LU + (size_t)blockIdx.y * stride;
    const c128* T = tau + (size_t)blockIdx.y * k * k + (size_t)blockIdx.x * k;     // column of tau00
    c128* x = X + ((size_t)blockIdx.y * k + blockIdx.x) * n;
    const int ne = n - k, tid = threadIdx.x;
    __shared__ c128 s_x;
    for (int i = tid; i < k; i += 256) x[ne + i] = T[i];
    // rhs = -U12 * X2
    for (int i = tid; i < ne; i += 256) {
        c128 s = cmake(0.0, 0.0);
        for (int c = 0; c < k; ++c) cfms(s, A[i + (size_t)(ne + c) * n], T[c]);
        x[i] = s;
    }
    __syncthreads();
    for (int j = ne - 1; j >= 0; --j) {
        if (tid == 0) { c128 v = cdiv(x[j], A[j + (size_t)j * n]); x[j] = v; s_x = v; }
        __syncthreads();
        const c128 xj = s_x;
        for (int i = tid; i < j; i += 256) { c128 v = x[i]; cfms(v, A[i + (size_t)j * n], xj); x[i] = v; }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- host launchers

int init_attrs_lu() {
    // largest outer panel the ABI accepts: W = 96 (LSMS_OPT_NB_OUTER)
    const size_t Wp = 96;
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_panel_post, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                      (int)((Wp * Wp + 16 * Wp) * sizeof(c128) + 3 * Wp * sizeof(int))));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_final_inverse, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 96 * 16));
    return 0;
}

int launch_panel_post(const c128* base, size_t stride, int n, int J, int W, int batch, const int* piv, int* perm, c128* ninv,
                      int nbmax, cudaStream_t st) {
    const size_t Wp = (size_t)(W + 15) / 16 * 16;
    size_t smem = (Wp * Wp + 16 * Wp) * sizeof(c128) + 3 * (size_t)W * sizeof(int);
    k_panel_post<<<batch, POST_THREADS, smem, st>>>(base, stride, n, J, W, piv, perm, ninv, nbmax);
    LSMS_LAUNCH_CHECK();
    return 0;
}

int launch_row_permute(c128* base, size_t stride, int n, int J, int W, int col_lo, int col_hi, int batch, const int* perm,
                       c128* tperm, size_t tperm_stride, int nbmax, cudaStream_t st) {
    if (col_hi <= col_lo) return 0;
    const int tn = n > 4000 ? 8 : 16;
    size_t smem = (size_t)tn * W * sizeof(c128) + (1 + 3 * (size_t)W) * sizeof(int);
    for (int b0 = 0; b0 < batch; b0 += 65535) {
        int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        dim3 grid((col_hi - col_lo + tn - 1) / tn, nb);
        if (tn == 8)
            k_row_permute<8><<<grid, PERM_THREADS, smem, st>>>(base + (size_t)b0 * stride, stride, n, J, W, col_lo, col_hi,
                                                              perm + (size_t)b0 * (4 + 3 * nbmax), tperm + (size_t)b0 * tperm_stride, tperm_stride, nbmax);
        else
            k_row_permute<16><<<grid, PERM_THREADS, smem, st>>>(base + (size_t)b0 * stride, stride, n, J, W, col_lo, col_hi,
                                                               perm + (size_t)b0 * (4 + 3 * nbmax), tperm + (size_t)b0 * tperm_stride, tperm_stride, nbmax);
        LSMS_LAUNCH_CHECK();
    }
    return 0;
}

int launch_final_inverse(c128* base, size_t stride, int n, int k, int batch, c128* tau, int* info, void* ws, cudaStream_t st) {
    const int use_smem = k <= 96;
    size_t smem = use_smem ? (size_t)k * k * sizeof(c128) : 0;
    k_final_inverse<<<batch, K5_THREADS, smem, st>>>(base, stride, n, k, tau, info, (c128*)ws, use_smem);
    LSMS_LAUNCH_CHECK();
    return 0;
}

int launch_backsolve_central(const c128* LU, size_t stride, int n, int k, int batch, const c128* tau, c128* X, cudaStream_t st) {
    dim3 grid(k, batch);
    k_backsolve_central<<<grid, 256, 0, st>>>(LU, stride, n, k, tau, X);
    LSMS_LAUNCH_CHECK();
    return 0;
}

}  // namespace lsms
