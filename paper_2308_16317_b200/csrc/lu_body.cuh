// lu_body.cuh -- device-side pieces of K3a and K5 shared by the lock-step kernels (lu.cu) and the small-matrix
// kernel (fused.cu): the net row permutation of an outer panel and the inverse of the final k x k Schur complement.
#pragma once
#include "common.cuh"

namespace lsms {

// Fold the W row interchanges of the outer panel [J, J+W) (pv[i] = pivot row of step J+i, applied in order) into one
// row permutation.  ONE WARP (all 32 lanes) calls this; cur_top / bpos / bcon are scratch arrays of W ints.
//   top_src[i]            row whose content ends in top position J+i
//   *nd_out, ddst, dsrc   displaced rows: row ddst[j] (below the top block) receives the ORIGINAL top row J+dsrc[j]
// (a row that enters the top block at step i stays there, so every displaced row is an original top row).
__device__ __forceinline__ void net_permutation(const int* __restrict__ pv, int J, int W, int* cur_top, int* bpos, int* bcon,
                                                int* nd_out, int* top_src, int* ddst, int* dsrc) {
    const int lane = threadIdx.x & 31;
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
            if (bcon[j] != bpos[j]) { ddst[nd] = bpos[j]; dsrc[nd] = bcon[j] - J; ++nd; }
        *nd_out = nd;
    }
    for (int i = lane; i < W; i += 32) top_src[i] = cur_top[i];
}

// ---------------------------------------------------------------- K5: tau00 = S^{-1}
// The whole CTA (THREADS threads): in-place Gauss-Jordan inversion with partial pivoting of the trailing k x k block of
// A (column-major, ld = n), done in the scratch array S (k*k elements, shared or global), result to `out` (k x k).
// A zero / non-finite pivot at step j sets *info = n-k+j+1 (if still 0).  k <= 256.
struct K5Shared { int cpiv[256]; int s_p; c128 s_rp; double wv[32]; int wi[32]; };

template <int THREADS>
__device__ __forceinline__ void final_inverse_body(const c128* __restrict__ A, int n, int k, c128* __restrict__ out,
                                                   int* __restrict__ info, c128* S, K5Shared& sh) {
    const int ne = n - k;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    for (int e = tid; e < k * k; e += THREADS) { int r = e % k, c = e / k; S[e] = A[(ne + r) + (size_t)(ne + c) * n]; }
    __syncthreads();
    bool failed = false;
    for (int j = 0; j < k; ++j) {
        double bv = -1.0; int bi = 0x7fffffff;
        for (int i = j + tid; i < k; i += THREADS) { double v = cabs1(S[i + (size_t)j * k]); if (v > bv) { bv = v; bi = i; } }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            double ov = __shfl_xor_sync(0xffffffffu, bv, o); int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) { sh.wv[warp] = bv; sh.wi[warp] = bi; }
        __syncthreads();
        if (tid == 0) {
            for (int t = 1; t < THREADS / 32; ++t) if (sh.wv[t] > bv || (sh.wv[t] == bv && sh.wi[t] < bi)) { bv = sh.wv[t]; bi = sh.wi[t]; }
            const bool bad = !(bv > 0.0) || !(bv < 1.0e300 * 1.0e300);
            sh.s_p = bad ? -1 : bi;
            if (bad) atomicCAS(info, 0, ne + j + 1);
            else { sh.cpiv[j] = bi; sh.s_rp = crecip(S[bi + (size_t)j * k]); }
        }
        __syncthreads();
        const int p = sh.s_p;
        if (p < 0) { failed = true; break; }
        // swap rows j <-> p
        if (p != j) for (int c = tid; c < k; c += THREADS) { c128 t = S[j + (size_t)c * k]; S[j + (size_t)c * k] = S[p + (size_t)c * k]; S[p + (size_t)c * k] = t; }
        __syncthreads();
        // row j <- row j / pivot, with a_jj := 1 first
        const c128 rp = sh.s_rp;
        for (int c = tid; c < k; c += THREADS) {
            c128 v = (c == j) ? cmake(1.0, 0.0) : S[j + (size_t)c * k];
            S[j + (size_t)c * k] = cmul(v, rp);
        }
        __syncthreads();
        // eliminate column j from every other row: f = a_ij, a_ij := 0, row_i -= f * row_j
        for (int e = tid; e < k * k; e += THREADS) {
            int i = e % k, c = e / k;
            if (i == j) continue;
            c128 f = S[i + (size_t)j * k];
            if (c == j) continue;                  // column j itself is handled after the sweep
            c128 v = S[i + (size_t)c * k];
            cfms(v, f, S[j + (size_t)c * k]);
            S[i + (size_t)c * k] = v;
        }
        __syncthreads();
        for (int i = tid; i < k; i += THREADS) {
            if (i == j) continue;
            c128 f = S[i + (size_t)j * k];
            S[i + (size_t)j * k] = cneg(cmul(f, S[j + (size_t)j * k]));
        }
        __syncthreads();
    }
    if (!failed) {
        // undo the row interchanges as column interchanges, in reverse order
        for (int j = k - 1; j >= 0; --j) {
            const int p = sh.cpiv[j];
            if (p != j) for (int r = tid; r < k; r += THREADS) { c128 t = S[r + (size_t)j * k]; S[r + (size_t)j * k] = S[r + (size_t)p * k]; S[r + (size_t)p * k] = t; }
            __syncthreads();
        }
    }
    for (int e = tid; e < k * k; e += THREADS) out[e] = S[e];
}

// K5 for a SMALL block (k <= 32, k*k <= 4*THREADS), trimmed for latency: one thread per element (up to four); every WARP
// finds the pivot of column j for itself (lane i takes row i: two redux.sync on a 64-bit key, the reciprocal of every
// candidate computed under the reduction and fetched from the winner by shuffles), the new value of each element is
// computed from the OLD matrix, then written: two CTA barriers per elimination step instead of six plus a serial
// section.  Same in-place Gauss-Jordan arithmetic as final_inverse_body; pivot = largest |re|+|im| (ties, up to 2^-47,
// to the lowest row).
template <int THREADS>
__device__ __forceinline__ void final_inverse_small(const c128* __restrict__ A, int n, int k, c128* __restrict__ out,
                                                    int* __restrict__ info, c128* S, int* cpiv) {
    const int ne = n - k, tid = threadIdx.x, lane = tid & 31, kk = k * k;
    for (int e = tid; e < kk; e += THREADS) { const int r = e % k, c = e / k; S[e] = A[(ne + r) + (size_t)(ne + c) * n]; }
    __syncthreads();
    bool failed = false;
    for (int j = 0; j < k; ++j) {
        const bool elig = lane >= j && lane < k;
        const c128 cand = elig ? S[lane + j * k] : cmake(0.0, 0.0);
        const c128 rinv = crecip_fast(cand);
        const unsigned long long kb = elig ? ((((unsigned long long)__double_as_longlong(cabs1(cand))) & ~31ull) | (unsigned long long)(31 - lane)) : 0ull;
        const uint32_t khi = (uint32_t)(kb >> 32), klo = (uint32_t)kb;
        const uint32_t mhi = __reduce_max_sync(0xffffffffu, khi);
        const uint32_t mlo = __reduce_max_sync(0xffffffffu, (khi == mhi) ? klo : 0u);
        const unsigned long long wkey = ((unsigned long long)mhi << 32) | mlo;
        if ((wkey >> 5) == 0ull || (uint32_t)(wkey >> 52) >= 0x7FFu) {       // zero, NaN or Inf pivot; the same in every thread
            if (tid == 0) atomicCAS(info, 0, ne + j + 1);
            failed = true;
            break;
        }
        const int p = 31 - (int)(wkey & 31ull);
        c128 rp;
        rp.x = __shfl_sync(0xffffffffu, rinv.x, p); rp.y = __shfl_sync(0xffffffffu, rinv.y, p);
        if (tid == 0) cpiv[j] = p;
        c128 nv[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int e = tid + u * THREADS;
            if (e < kk) {
                const int i = e % k, c = e / k;
                const c128 rowj = cmul((c == j) ? cmake(1.0, 0.0) : S[p + c * k], rp);      // new row j, column c
                if (i == j) nv[u] = rowj;
                else {
                    const int src = (i == p) ? j : i;                                        // rows j and p change places
                    const c128 f = S[src + j * k];
                    if (c == j) nv[u] = cneg(cmul(f, rp));
                    else { c128 x = S[src + c * k]; cfms(x, f, rowj); nv[u] = x; }
                }
            }
        }
        __syncthreads();
#pragma unroll
        for (int u = 0; u < 4; ++u) { const int e = tid + u * THREADS; if (e < kk) S[e] = nv[u]; }
        __syncthreads();
    }
    if (!failed && tid < k) {
        // undo the row interchanges as column interchanges, in reverse order; thread r owns row r
        for (int j = k - 1; j >= 0; --j) {
            const int p = cpiv[j];
            if (p != j) { const c128 t = S[tid + j * k]; S[tid + j * k] = S[tid + p * k]; S[tid + p * k] = t; }
        }
    }
    __syncthreads();
    for (int e = tid; e < kk; e += THREADS) out[e] = S[e];
}

}  // namespace lsms
