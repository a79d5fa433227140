// lu.cu -- K2 (panel LU with restricted partial pivoting), K3 (row interchanges + unit-lower
// triangular solve), K5 (inverse of the final k x k Schur complement) and the verification-only
// back-substitution.  SURVEY.md 8(a) a3, a4, a6; "LU factorization of the matrix" PAPER.md:92;
// "only the first block of the inverted matrix is needed" PAPER.md:62.
//
// Pivot rule (reading A14): for the first ne = n-k columns the pivot search covers rows
// [j, ne) only, so the central-site rows are updated but never selected; the trailing k x k block
// is then exactly the Schur complement D - C A^{-1} B of the central site.
#include "common.cuh"
#include "internal.h"

namespace lsms {

constexpr int PANEL_THREADS = 256;     // 256 x 128 regs: fits beside one Schur-update CTA (look-ahead)
constexpr int MAX_IB = 16;

// ---------------------------------------------------------------- K2: panel factorisation
// One CTA per matrix.  Columns [c0, c0+w) of rows [c0, n); w <= MAX_IB.  Unblocked right-looking
// elimination inside the panel; the max search of column j+1 is fused into the update of step j.
__global__ void __launch_bounds__(PANEL_THREADS)
k_panel(c128* __restrict__ base, size_t stride, int n, int c0, int w, int ne, int* __restrict__ piv, int* __restrict__ info) {
    c128* A = base + (size_t)blockIdx.x * stride;
    int* pv = piv + (size_t)blockIdx.x * n;
    __shared__ c128 urow[MAX_IB];
    __shared__ double red_v[PANEL_THREADS / 32];
    __shared__ int red_i[PANEL_THREADS / 32];
    __shared__ int s_piv;
    __shared__ int s_bad;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    // candidate of this thread for the current column: (value, row); rows j..ne-1
    double bv = -1.0; int bi = 0x7fffffff;
    for (int i = c0 + tid; i < ne; i += PANEL_THREADS) {
        double v = cabs1(A[i + (size_t)c0 * n]);
        if (v > bv) { bv = v; bi = i; }
    }
    for (int jj = 0; jj < w; ++jj) {
        const int j = c0 + jj;
        // ---- block arg-max (ties -> smallest row)
        double v = bv; int ix = bi;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            double ov = __shfl_xor_sync(0xffffffffu, v, o); int oi = __shfl_xor_sync(0xffffffffu, ix, o);
            if (ov > v || (ov == v && oi < ix)) { v = ov; ix = oi; }
        }
        if (lane == 0) { red_v[warp] = v; red_i[warp] = ix; }
        __syncthreads();
        if (warp == 0) {
            v = (lane < PANEL_THREADS / 32) ? red_v[lane] : -1.0; ix = (lane < PANEL_THREADS / 32) ? red_i[lane] : 0x7fffffff;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                double ov = __shfl_xor_sync(0xffffffffu, v, o); int oi = __shfl_xor_sync(0xffffffffu, ix, o);
                if (ov > v || (ov == v && oi < ix)) { v = ov; ix = oi; }
            }
            if (lane == 0) {
                const bool bad = !(v > 0.0) || !(v < 1.0e300 * 1.0e300);     // zero, NaN or Inf pivot
                s_bad = bad ? 1 : 0;
                s_piv = bad ? j : ix;
                pv[j] = bad ? j : ix;
                if (bad) atomicCAS(&info[blockIdx.x], 0, j + 1);
            }
        }
        __syncthreads();
        const int p = s_piv;
        const bool bad = s_bad != 0;
        // ---- swap rows j and p inside the panel, publish the pivot row
        if (tid < w) {
            c128 a = A[j + (size_t)(c0 + tid) * n];
            if (p != j) { c128 bq = A[p + (size_t)(c0 + tid) * n]; A[p + (size_t)(c0 + tid) * n] = a; A[j + (size_t)(c0 + tid) * n] = bq; a = bq; }
            urow[tid] = a;
        }
        __syncthreads();
        // ---- scale column j, rank-1 update of the remaining panel columns, next column's max
        bv = -1.0; bi = 0x7fffffff;
        if (!bad) {
            const c128 rp = crecip(urow[jj]);
            // all loads of a row are issued before any of its stores (independent L2 round trips in
            // flight instead of one dependent load->fma->store chain per column)
            for (int i = j + 1 + tid; i < n; i += PANEL_THREADS) {
                c128 a[MAX_IB];
                const c128 l0 = A[i + (size_t)j * n];
#pragma unroll
                for (int t = 1; t < MAX_IB; ++t)
                    if (jj + t < w) a[t] = A[i + (size_t)(j + t) * n];
                const c128 l = cmul(l0, rp);
                A[i + (size_t)j * n] = l;
#pragma unroll
                for (int t = 1; t < MAX_IB; ++t)
                    if (jj + t < w) {
                        cfms(a[t], l, urow[jj + t]);
                        A[i + (size_t)(j + t) * n] = a[t];
                    }
                if (jj + 1 < w && i < ne) { double vv = cabs1(a[1]); if (vv > bv) { bv = vv; bi = i; } }
            }
        } else if (jj + 1 < w) {
            for (int i = j + 1 + tid; i < ne; i += PANEL_THREADS) {
                double vv = cabs1(A[i + (size_t)(j + 1) * n]);
                if (vv > bv) { bv = vv; bi = i; }
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- K3: interchanges + U12 = L11^{-1} A12
// One thread per target column c in [col_lo, col_hi) (columns of the panel itself are skipped by the
// caller's ranges).  mode bit 0: apply the w interchanges of panel [c0, c0+w) in order; mode bit 1:
// solve the w x w unit-lower triangle L11 against rows [c0, c0+w) of the column.
constexpr int K3_THREADS = 128;

__global__ void __launch_bounds__(K3_THREADS)
k_swap_trsm(c128* __restrict__ base, size_t stride, int n, int c0, int w, int col_lo, int col_hi, int mode,
            const int* __restrict__ piv) {
    const bool do_swap = mode & 1, do_trsm = mode & 2;
    c128* A = base + (size_t)blockIdx.y * stride;
    const int* pv = piv + (size_t)blockIdx.y * n + c0;
    __shared__ c128 L[MAX_IB * MAX_IB];
    __shared__ int sp[MAX_IB];
    if (threadIdx.x < w) sp[threadIdx.x] = pv[threadIdx.x];
    if (do_trsm)
        for (int e = threadIdx.x; e < w * w; e += K3_THREADS) { int r = e % w, c = e / w; L[r + MAX_IB * c] = A[(c0 + r) + (size_t)(c0 + c) * n]; }
    __syncthreads();
    const int c = col_lo + blockIdx.x * K3_THREADS + threadIdx.x;
    if (c >= col_hi) return;
    c128* col = A + (size_t)c * n;
    c128 x[MAX_IB];
#pragma unroll
    for (int i = 0; i < MAX_IB; ++i) x[i] = (i < w) ? col[c0 + i] : cmake(0.0, 0.0);
    // interchanges, in order (a row index may appear more than once)
#pragma unroll
    for (int i = 0; i < MAX_IB; ++i) {
        if (do_swap && i < w) {
            const int p = sp[i];
            if (p != c0 + i) {
                if (p < c0 + w) {
                    // both rows are in registers: static indexing through a select chain
                    c128 xi = x[i], xp = xi;
#pragma unroll
                    for (int t = 0; t < MAX_IB; ++t) if (t == p - c0) xp = x[t];
#pragma unroll
                    for (int t = 0; t < MAX_IB; ++t) if (t == p - c0) x[t] = xi;
                    x[i] = xp;
                } else {
                    c128 t = col[p]; col[p] = x[i]; x[i] = t;
                }
            }
        }
    }
    if (do_trsm) {
#pragma unroll
        for (int j = 0; j < MAX_IB; ++j)
#pragma unroll
            for (int i = j + 1; i < MAX_IB; ++i)
                if (i < w) cfms(x[i], L[i + MAX_IB * j], x[j]);
    }
#pragma unroll
    for (int i = 0; i < MAX_IB; ++i) if (i < w) col[c0 + i] = x[i];
}

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
        // ---- net permutation (warp 0; the below-list is searched lane-parallel)
        const int lane = tid;
        for (int i = lane; i < W; i += 32) cur_top[i] = J + i;
        __syncwarp();
        int nb = 0;
        for (int i = 0; i < W; ++i) {
            const int p = pv[i];
            if (p == J + i) continue;
            if (p < J + W) {
                if (lane == 0) { int t = cur_top[i]; cur_top[i] = cur_top[p - J]; cur_top[p - J] = t; }
            } else {
                int found = -1;
                for (int b0 = 0; b0 < nb; b0 += 32) {
                    const int idx = b0 + lane;
                    const unsigned m = __ballot_sync(0xffffffffu, idx < nb && bpos[idx] == p);
                    if (m) { found = b0 + __ffs(m) - 1; break; }
                }
                if (found < 0) { found = nb; if (lane == 0) { bpos[nb] = p; bcon[nb] = p; } ++nb; }
                __syncwarp();
                if (lane == 0) { int t = cur_top[i]; cur_top[i] = bcon[found]; bcon[found] = t; }
            }
            __syncwarp();
        }
        __syncwarp();
        // compact the displaced rows (content differs from position); serial over <= W entries
        if (lane == 0) {
            int nd = 0;
            for (int j = 0; j < nb; ++j)
                if (bcon[j] != bpos[j]) { perm[1 + nbmax + nd] = bpos[j]; perm[1 + 2 * nbmax + nd] = bcon[j] - J; ++nd; }
            perm[0] = nd;
        }
        for (int i = lane; i < W; i += 32) perm[1 + i] = cur_top[i];
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
// rows are scattered to their final rows below.  One CTA per strip of PERM_TN columns.
constexpr int PERM_TN = 16, PERM_THREADS = 256;

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
    const c128* A = base + (size_t)blockIdx.x * stride;
    const int ne = n - k;
    c128* S = use_smem ? reinterpret_cast<c128*>(k5_smem) : gscratch + (size_t)blockIdx.x * k * k;
    __shared__ int cpiv[256];
    __shared__ int s_p;
    __shared__ c128 s_rp;
    __shared__ double wv[K5_THREADS / 32];
    __shared__ int wi[K5_THREADS / 32];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int e = tid; e < k * k; e += K5_THREADS) { int r = e % k, c = e / k; S[e] = A[(ne + r) + (size_t)(ne + c) * n]; }
    __syncthreads();
    bool failed = false;
    for (int j = 0; j < k; ++j) {
        double bv = -1.0; int bi = 0x7fffffff;
        for (int i = j + tid; i < k; i += K5_THREADS) { double v = cabs1(S[i + (size_t)j * k]); if (v > bv) { bv = v; bi = i; } }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            double ov = __shfl_xor_sync(0xffffffffu, bv, o); int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) { wv[warp] = bv; wi[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            for (int t = 1; t < K5_THREADS / 32; ++t) if (wv[t] > bv || (wv[t] == bv && wi[t] < bi)) { bv = wv[t]; bi = wi[t]; }
            const bool bad = !(bv > 0.0) || !(bv < 1.0e300 * 1.0e300);
            s_p = bad ? -1 : bi;
            if (bad) atomicCAS(&info[blockIdx.x], 0, ne + j + 1);
            else { cpiv[j] = bi; s_rp = crecip(S[bi + (size_t)j * k]); }
        }
        __syncthreads();
        const int p = s_p;
        if (p < 0) { failed = true; break; }
        // swap rows j <-> p
        if (p != j) for (int c = tid; c < k; c += K5_THREADS) { c128 t = S[j + (size_t)c * k]; S[j + (size_t)c * k] = S[p + (size_t)c * k]; S[p + (size_t)c * k] = t; }
        __syncthreads();
        // row j <- row j / pivot, with a_jj := 1 first
        const c128 rp = s_rp;
        for (int c = tid; c < k; c += K5_THREADS) {
            c128 v = (c == j) ? cmake(1.0, 0.0) : S[j + (size_t)c * k];
            S[j + (size_t)c * k] = cmul(v, rp);
        }
        __syncthreads();
        // eliminate column j from every other row: f = a_ij, a_ij := 0, row_i -= f * row_j
        for (int e = tid; e < k * k; e += K5_THREADS) {
            int i = e % k, c = e / k;
            if (i == j) continue;
            c128 f = S[i + (size_t)j * k];
            if (c == j) continue;                  // column j itself is handled after the sweep
            c128 v = S[i + (size_t)c * k];
            cfms(v, f, S[j + (size_t)c * k]);
            S[i + (size_t)c * k] = v;
        }
        __syncthreads();
        for (int i = tid; i < k; i += K5_THREADS) {
            if (i == j) continue;
            c128 f = S[i + (size_t)j * k];
            S[i + (size_t)j * k] = cneg(cmul(f, S[j + (size_t)j * k]));
        }
        __syncthreads();
    }
    if (!failed) {
        // undo the row interchanges as column interchanges, in reverse order
        for (int j = k - 1; j >= 0; --j) {
            const int p = cpiv[j];
            if (p != j) for (int r = tid; r < k; r += K5_THREADS) { c128 t = S[r + (size_t)j * k]; S[r + (size_t)j * k] = S[r + (size_t)p * k]; S[r + (size_t)p * k] = t; }
            __syncthreads();
        }
    }
    c128* out = tau + (size_t)blockIdx.x * k * k;
    for (int e = tid; e < k * k; e += K5_THREADS) out[e] = S[e];
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

int launch_panel(c128* base, size_t stride, int n, int c0, int w, int ne, int batch, int* piv, int* info, cudaStream_t st) {
    k_panel<<<batch, PANEL_THREADS, 0, st>>>(base, stride, n, c0, w, ne, piv, info);
    LSMS_LAUNCH_CHECK();
    return 0;
}

int launch_swap_trsm(c128* base, size_t stride, int n, int c0, int w, int col_lo, int col_hi, int mode, int batch,
                     const int* piv, cudaStream_t st) {
    if (col_hi <= col_lo) return 0;
    for (int b0 = 0; b0 < batch; b0 += 65535) {
        int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        dim3 grid((col_hi - col_lo + K3_THREADS - 1) / K3_THREADS, nb);
        k_swap_trsm<<<grid, K3_THREADS, 0, st>>>(base + (size_t)b0 * stride, stride, n, c0, w, col_lo, col_hi, mode, piv + (size_t)b0 * n);
        LSMS_LAUNCH_CHECK();
    }
    return 0;
}

int launch_panel_post(const c128* base, size_t stride, int n, int J, int W, int batch, const int* piv, int* perm, c128* ninv,
                      int nbmax, cudaStream_t st) {
    const size_t Wp = (size_t)(W + 15) / 16 * 16;
    size_t smem = (Wp * Wp + 16 * Wp) * sizeof(c128) + 3 * (size_t)W * sizeof(int);
    static size_t attr = 0;
    if (smem > attr && smem > 48 * 1024) { LSMS_CUDA_OK(cudaFuncSetAttribute(k_panel_post, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); attr = smem; }
    k_panel_post<<<batch, POST_THREADS, smem, st>>>(base, stride, n, J, W, piv, perm, ninv, nbmax);
    LSMS_LAUNCH_CHECK();
    return 0;
}

int launch_row_permute(c128* base, size_t stride, int n, int J, int W, int col_lo, int col_hi, int batch, const int* perm,
                       c128* tperm, size_t tperm_stride, int nbmax, cudaStream_t st) {
    if (col_hi <= col_lo) return 0;
    size_t smem = (size_t)PERM_TN * W * sizeof(c128) + (1 + 3 * (size_t)W) * sizeof(int);
    static size_t attr = 0;
    if (smem > attr && smem > 48 * 1024) { LSMS_CUDA_OK(cudaFuncSetAttribute(k_row_permute, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); attr = smem; }
    for (int b0 = 0; b0 < batch; b0 += 65535) {
        int nb = batch - b0 < 65535 ? batch - b0 : 65535;
        dim3 grid((col_hi - col_lo + PERM_TN - 1) / PERM_TN, nb);
        k_row_permute<<<grid, PERM_THREADS, smem, st>>>(base + (size_t)b0 * stride, stride, n, J, W, col_lo, col_hi,
                                                       perm + (size_t)b0 * (4 + 3 * nbmax), tperm + (size_t)b0 * tperm_stride, tperm_stride, nbmax);
        LSMS_LAUNCH_CHECK();
    }
    return 0;
}

int launch_final_inverse(c128* base, size_t stride, int n, int k, int batch, c128* tau, int* info, void* ws, cudaStream_t st) {
    const int use_smem = k <= 96;
    size_t smem = use_smem ? (size_t)k * k * sizeof(c128) : 0;
    static bool attr_set = false;
    if (!attr_set) { LSMS_CUDA_OK(cudaFuncSetAttribute(k_final_inverse, cudaFuncAttributeMaxDynamicSharedMemorySize, 96 * 96 * 16)); attr_set = true; }
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
