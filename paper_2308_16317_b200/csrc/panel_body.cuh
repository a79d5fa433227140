// panel_body.cuh -- K2: register-blocked panel LU with restricted partial pivoting (
// "LU factorization of the matrix" PAPER.md:92; pivot rule: DESIGN.md reading A14).
//
// One CTA per matrix factors the inner panel: columns [c0, c0+w), w <= 16, rows [c0, n).  The panel is
// too tall for shared memory (2160 x 16 x 16 B = 553 KB), so it lives in L2/HBM and the kernel is bound
// by the latency of its sequential column steps, not by bandwidth or flops.  The steps are therefore
// taken on a SUB-PANEL of S columns held in registers (thread t owns rows c0 + t + r*THREADS, r < R):
//
//   for each sub-panel [cs, cs+S):
//     1  load the sub-panel (R*S independent loads per thread, one L2 round trip)
//     2  S column steps entirely on chip: block arg-max (shuffles + one shared-memory exchange), the
//        pivot row and row j swap through shared memory, scale + rank-1 update in registers
//     3  store the sub-panel; publish L11 (S x S), the S pivots and their duplicate map
//     4  one thread per OTHER column of the outer panel [J, J+W): the S interchanges applied with all
//        loads issued together; for the inner panel's columns to the right also the S x S unit-lower
//        solve, whose result (rows of U) is published in shared memory
//     5  rank-S update of the inner panel's remaining columns, L from registers, U from shared memory
//
//   after the last sub-panel:
//     6  the w x w unit-lower solve for the outer panel's columns to the right of the inner panel
//
// The row interchanges and triangular solves inside an outer panel are thus all done here (K3's launches
// inside the outer panel are gone); what remains per inner panel is the rank-w update of those columns (K4).
#pragma once
#include "common.cuh"

namespace lsms {

constexpr int P2_MAXW = 16;       // inner panel width limit
constexpr int P2_MAXOUT = 128;    // outer panel width limit (column threads of step 4)

// Shared-memory state of one panel factorisation (sized for the widest sub-panel, S = 4, and 16 warps).
struct PanelShared {
    c128 prow[4], jrow[4];
    c128 L11[4 * 4];                 // L11[i*S + q] = multiplier of row cs+i, column cs+q (q < i)
    c128 Us[4 * P2_MAXW];            // Us[q*P2_MAXW + c] = U(cs+q, cs+sw+c)
    c128 Lw[P2_MAXW * P2_MAXW];      // step 6: the w x w unit-lower triangle
    double red_v[16];
    int red_i[16];
    int spiv[4], canon[4];
};

// The whole CTA (THREADS threads) factors the inner panel [c0, c0+w) of the matrix A (column-major, ld = n) and
// applies its interchanges / triangular solves to the outer panel [J, J+Wout).  pv = the matrix's pivot vector,
// info = the matrix's status word.  Callers: k_panel_reg (one CTA per matrix, lock-step schedule) and the
// small-matrix kernel of fused.cu.  Ends with the CTA's threads NOT synchronised (global stores may be pending).
template <int THREADS, int R, int S>
__device__ __forceinline__ void panel_body(c128* __restrict__ A, int n, int J, int Wout, int c0, int w, int ne,
                                           int* __restrict__ pv, int* __restrict__ info, PanelShared& sh) {
    constexpr int NW = THREADS / 32;
    static_assert(S <= 4 && NW <= 16, "PanelShared is sized for S <= 4 and <= 16 warps");
    double* red_v = sh.red_v; int* red_i = sh.red_i;
    c128* prow = sh.prow; c128* jrow = sh.jrow; c128* L11 = sh.L11; c128* Us = sh.Us;
    int* spiv = sh.spiv; int* canon = sh.canon;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const c128 zero = cmake(0.0, 0.0);

    for (int s0 = 0; s0 < w; s0 += S) {
        const int cs = c0 + s0, sw = min(S, w - s0);
        // ---- 1: sub-panel -> registers
        c128 v[R][S];
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int row = c0 + tid + r * THREADS;
#pragma unroll
            for (int q = 0; q < S; ++q) v[r][q] = (row < n && q < sw) ? A[row + (size_t)(cs + q) * n] : zero;
        }
        // ---- 2: column steps
#pragma unroll
        for (int q = 0; q < S; ++q) {
            if (q < sw) {
                const int j = cs + q;
                double bv = -1.0; int bi = 0x7fffffff;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int row = c0 + tid + r * THREADS;
                    const double a = cabs1(v[r][q]);
                    if (row >= j && row < ne && a > bv) { bv = a; bi = row; }
                }
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) {
                    const double ov = __shfl_xor_sync(0xffffffffu, bv, o); const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
                }
                if (lane == 0) { red_v[warp] = bv; red_i[warp] = bi; }
                __syncthreads();
                bv = red_v[lane % NW]; bi = red_i[lane % NW];
#pragma unroll
                for (int o = NW / 2; o > 0; o >>= 1) {
                    const double ov = __shfl_xor_sync(0xffffffffu, bv, o); const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
                    if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
                }
                const bool bad = !(bv > 0.0) || !(bv < 1.0e300 * 1.0e300);     // zero, NaN or Inf pivot
                const int p = bad ? j : bi;
                if (tid == 0) { spiv[q] = p; pv[j] = p; if (bad) atomicCAS(info, 0, j + 1); }
                // ---- pivot row and row j through shared memory
                const int tj = (j - c0) % THREADS, rj = (j - c0) / THREADS;
                const int tp = (p - c0) % THREADS, rp_ = (p - c0) / THREADS;
                if (tid == tp) {
#pragma unroll
                    for (int r = 0; r < R; ++r) if (r == rp_) {
#pragma unroll
                        for (int t = 0; t < S; ++t) prow[t] = v[r][t];
                    }
                }
                if (p != j && tid == tj) {
#pragma unroll
                    for (int r = 0; r < R; ++r) if (r == rj) {
#pragma unroll
                        for (int t = 0; t < S; ++t) jrow[t] = v[r][t];
                    }
                }
                __syncthreads();
                if (p != j) {
                    if (tid == tj) {
#pragma unroll
                        for (int r = 0; r < R; ++r) if (r == rj) {
#pragma unroll
                            for (int t = 0; t < S; ++t) v[r][t] = prow[t];
                        }
                    }
                    if (tid == tp) {
#pragma unroll
                        for (int r = 0; r < R; ++r) if (r == rp_) {
#pragma unroll
                            for (int t = 0; t < S; ++t) v[r][t] = jrow[t];
                        }
                    }
                }
                // ---- scale column j and rank-1 update of the sub-panel's remaining columns
                if (!bad) {
                    const c128 rp = crecip(prow[q]);
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const int row = c0 + tid + r * THREADS;
                        if (row > j && row < n) {
                            const c128 l = cmul(v[r][q], rp);
                            v[r][q] = l;
#pragma unroll
                            for (int t = q + 1; t < S; ++t) if (t < sw) cfms(v[r][t], l, prow[t]);
                        }
                    }
                }
            }
        }
        // ---- 3: store the sub-panel (rows above cs hold finished U entries and are unchanged), publish L11
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const int row = c0 + tid + r * THREADS;
            if (row >= cs && row < n) {
#pragma unroll
                for (int q = 0; q < S; ++q) if (q < sw) A[row + (size_t)(cs + q) * n] = v[r][q];
                if (row < cs + sw) {
#pragma unroll
                    for (int q = 0; q < S; ++q) L11[(row - cs) * S + q] = v[r][q];
                }
            }
        }
        if (tid == 0) {
            // canon[i] = first step whose pivot row equals that of step i (rows below the sub-panel only)
            for (int i = 0; i < sw; ++i) {
                int c = -1;
                if (spiv[i] >= cs + sw) { c = i; for (int t = 0; t < i; ++t) if (spiv[t] == spiv[i]) { c = t; break; } }
                canon[i] = c;
            }
        }
        __syncthreads();
        // ---- 4: the other columns of the outer panel: interchanges (+ S x S solve for the inner panel's right part)
        const int nright = (c0 + w) - (cs + sw);          // inner-panel columns still to be updated
        if (tid < Wout) {
            const int cu = J + tid;
            if (cu < cs || cu >= cs + sw) {
                c128* col = A + (size_t)cu * n;
                c128 x[S], y[S];
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    x[i] = (i < sw) ? col[cs + i] : zero;
                    y[i] = (i < sw && canon[i] == i) ? col[spiv[i]] : zero;
                }
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    if (i < sw) {
                        const int p = spiv[i];
                        if (p != cs + i) {
                            const int k = (p < cs + sw) ? (p - cs) : canon[i];
                            const bool top = p < cs + sw;
                            const c128 xi = x[i];
                            c128 other = xi;
#pragma unroll
                            for (int t = 0; t < S; ++t) if (t == k) other = top ? x[t] : y[t];
#pragma unroll
                            for (int t = 0; t < S; ++t) if (t == k) { if (top) x[t] = xi; else y[t] = xi; }
                            x[i] = other;
                        }
                    }
                }
                const bool right = cu >= cs + sw && cu < c0 + w;
                if (right) {
#pragma unroll
                    for (int jq = 0; jq < S; ++jq)
#pragma unroll
                        for (int i = jq + 1; i < S; ++i)
                            if (i < sw) cfms(x[i], L11[i * S + jq], x[jq]);
#pragma unroll
                    for (int i = 0; i < S; ++i) if (i < sw) Us[i * P2_MAXW + (cu - cs - sw)] = x[i];
                }
#pragma unroll
                for (int i = 0; i < S; ++i) {
                    if (i < sw) {
                        col[cs + i] = x[i];
                        if (canon[i] == i) col[spiv[i]] = y[i];
                    }
                }
            }
        }
        __syncthreads();
        // ---- 5: rank-sw update of the inner panel's remaining columns (rows below the sub-panel).
        // Software-pipelined over (column, row chunk): the loads of the next chunk are issued before the
        // current chunk is updated and stored, so that one L2 round trip is always in flight.
        if (nright > 0) {
            constexpr int RC = (R % 5 == 0) ? 5 : ((R % 4 == 0) ? 4 : R);      // rows per chunk (R in {1,2,5,10,20,32})
            constexpr int NCH = R / RC;
            c128 cur[RC], nxt[RC];
#pragma unroll
            for (int i = 0; i < RC; ++i) {
                const int row = c0 + tid + i * THREADS;
                cur[i] = (row >= cs + sw && row < n) ? A[row + (size_t)(cs + sw) * n] : zero;
            }
            for (int c = 0; c < nright; ++c) {
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) {
                    const int nch = (ch + 1 == NCH) ? 0 : ch + 1;
                    const int nc = c + ((ch + 1 == NCH) ? 1 : 0);
#pragma unroll
                    for (int i = 0; i < RC; ++i) {
                        const int row = c0 + tid + (nch * RC + i) * THREADS;
                        nxt[i] = (nc < nright && row >= cs + sw && row < n) ? A[row + (size_t)(cs + sw + nc) * n] : zero;
                    }
#pragma unroll
                    for (int i = 0; i < RC; ++i) {
                        const int r = ch * RC + i;
                        const int row = c0 + tid + r * THREADS;
                        if (row >= cs + sw && row < n) {
#pragma unroll
                            for (int q = 0; q < S; ++q) if (q < sw) cfms(cur[i], v[r][q], Us[q * P2_MAXW + c]);
                            A[row + (size_t)(cs + sw + c) * n] = cur[i];
                        }
                    }
#pragma unroll
                    for (int i = 0; i < RC; ++i) cur[i] = nxt[i];
                }
            }
        }
        __syncthreads();
    }
    // ---- 6: U12 of the outer panel's columns to the RIGHT of this inner panel: solve the w x w unit-lower L11
    // against rows [c0, c0+w) of each such column (their interchanges were applied in step 4).  One thread per
    // column; L11 is read back from the panel this CTA has just stored.
    const int nr = (J + Wout) - (c0 + w);
    if (nr > 0) {
        c128* Lw = sh.Lw;
        for (int e = tid; e < w * w; e += THREADS) { const int r = e % w, c = e / w; Lw[r + P2_MAXW * c] = A[(c0 + r) + (size_t)(c0 + c) * n]; }
        __syncthreads();
        if (tid < nr) {
            c128* col = A + (size_t)(c0 + w + tid) * n + c0;
            c128 x[P2_MAXW];
#pragma unroll
            for (int i = 0; i < P2_MAXW; ++i) x[i] = (i < w) ? col[i] : zero;
#pragma unroll
            for (int jq = 0; jq < P2_MAXW; ++jq)
#pragma unroll
                for (int i = jq + 1; i < P2_MAXW; ++i)
                    if (i < w) cfms(x[i], Lw[i + P2_MAXW * jq], x[jq]);
#pragma unroll
            for (int i = 0; i < P2_MAXW; ++i) if (i < w) col[i] = x[i];
        }
    }
}

}  // namespace lsms
