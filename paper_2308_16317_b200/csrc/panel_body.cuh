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
    // column-step exchange, double-buffered by the parity of the column: per warp the arg-max candidate's row (S
    // entries), the reciprocal of its would-be pivot and the arg-max key; the row that stands at the pivot position
    c128 cand[2][16][4 + 2];
    c128 jrow[2][4];
    c128 L11[4 * 4];                 // L11[i*S + q] = multiplier of row cs+i, column cs+q (q < i)
    c128 Us[4 * P2_MAXW];            // Us[q*P2_MAXW + c] = U(cs+q, cs+sw+c)
    c128 Lw[P2_MAXW * P2_MAXW];      // step 6: the w x w unit-lower triangle
    int spiv[4], canon[4];
};

// The whole CTA (THREADS threads) factors the inner panel [c0, c0+w) of the matrix A (column-major, ld = n) and
// applies its interchanges / triangular solves to the outer panel [J, J+Wout).  pv = the matrix's pivot vector,
// info = the matrix's status word.  Callers: k_panel_reg (one CTA per matrix, lock-step schedule) and the
// small-matrix kernel of fused.cu.  Ends with the CTA's threads NOT synchronised (global stores may be pending).
__device__ __forceinline__ void cp_async16(void* dst_smem, const void* src_gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"((uint32_t)__cvta_generic_to_shared(dst_smem)), "l"(src_gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// DEPTH > 0: step 5 streams the columns it updates through `stage` (DEPTH slots of R*THREADS complex numbers of shared
// memory) with per-thread asynchronous copies, DEPTH columns ahead -- the step is bound by the bytes a CTA keeps in
// flight towards L2/HBM, and registers hold one column only.  DEPTH = 0: the register-pipelined loop (one column ahead).
template <int THREADS, int R, int S, int DEPTH = 0>
__device__ __forceinline__ void panel_body(c128* __restrict__ A, int n, int J, int Wout, int c0, int w, int ne,
                                           int* __restrict__ pv, int* __restrict__ info, PanelShared& sh, c128* stage = nullptr) {
    constexpr int NW = THREADS / 32;
    static_assert(S <= 4 && NW <= 16, "PanelShared is sized for S <= 4 and <= 16 warps");
    static_assert(R * THREADS <= 16384, "arg-max key: 14 bits for the row offset within the panel (16383 - offset), 4 for the warp");
    c128* L11 = sh.L11; c128* Us = sh.Us;
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
        // ---- 2: column steps, ONE CTA barrier each.  Arg-max key of a row: the bits of |re|+|im| with the low 18
        // mantissa bits replaced by (16383 - (row - c0), warp), so that one unsigned 64-bit maximum picks the largest
        // magnitude and, among (nearly) equal ones, the lowest row (LAPACK's izamax up to 2^-34); 0 = not eligible.  Every warp
        // finds its candidate with two redux.sync and publishes the candidate's row TOGETHER with the key (and with
        // the reciprocal of the would-be pivot, computed under the reduction), the owner of row j publishes that row:
        // when the barrier opens every thread has what it needs for the interchange and the rank-1 update.
        int piv_reg[S];
#pragma unroll
        for (int q = 0; q < S; ++q) {
            piv_reg[q] = cs + q;
            if (q < sw) {
                const int j = cs + q, par = q & 1;
                // local best row by magnitude (ascending rows, strict >: the lowest row among equal ones), then ONE key
                double ba = -1.0; int rb = 0;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int row = c0 + tid + r * THREADS;
                    const double a = cabs1(v[r][q]);
                    if (row >= j && row < ne && (a > ba || a != a)) { ba = a; rb = r; }   // a NaN entry is taken, kept and flagged
                }
                unsigned long long key = 0ull;
                if (ba >= 0.0 || ba != ba)
                    key = ((unsigned long long)__double_as_longlong(ba) & ~0x3FFFFull) |
                          ((unsigned long long)(16383 - (tid + rb * THREADS)) << 4) | (unsigned long long)warp;
                c128 vq = v[0][q];
#pragma unroll
                for (int r = 1; r < R; ++r) if (r == rb) vq = v[r][q];
                const c128 rinv = crecip_fast(vq);
                const uint32_t khi = (uint32_t)(key >> 32), klo = (uint32_t)key;
                const uint32_t mhi = __reduce_max_sync(0xffffffffu, khi);
                const uint32_t mlo = __reduce_max_sync(0xffffffffu, (khi == mhi) ? klo : 0u);
                c128* slot = sh.cand[par][warp];
                if (key != 0ull && khi == mhi && klo == mlo) {
#pragma unroll
                    for (int r = 0; r < R; ++r) if (r == rb) {
#pragma unroll
                        for (int t = 0; t < S; ++t) slot[t] = v[r][t];
                    }
                    slot[4] = rinv;
                }
                if (lane == 0) reinterpret_cast<unsigned long long*>(slot + 5)[0] = ((unsigned long long)mhi << 32) | mlo;
                const int tj = j - c0;                      // row j belongs to thread j - c0 (< w <= 16 <= THREADS), its first row
                if (tid == tj) {
#pragma unroll
                    for (int t = 0; t < S; ++t) sh.jrow[par][t] = v[0][t];
                }
                __syncthreads();
                // winner among the NW warp candidates: lane l takes candidate l mod NW, two more redux.sync
                const unsigned long long ck = reinterpret_cast<const unsigned long long*>(&sh.cand[par][lane % NW][5])[0];
                const uint32_t chi = (uint32_t)(ck >> 32), clo = (uint32_t)ck;
                const uint32_t whi = __reduce_max_sync(0xffffffffu, chi);
                const uint32_t wlo = __reduce_max_sync(0xffffffffu, (chi == whi) ? clo : 0u);
                const unsigned long long wkey = ((unsigned long long)whi << 32) | wlo;
                const int wsel = (int)(wkey & 15ull);
                const bool bad = (wkey >> 18) == 0ull || (uint32_t)(wkey >> 52) >= 0x7FFu;     // zero, NaN or Inf pivot
                const int p = bad ? j : c0 + 16383 - (int)((wkey >> 4) & 0x3FFFull);
                piv_reg[q] = bad ? -1 - j : p;
                if (!bad) {
                    c128 prow[S];
#pragma unroll
                    for (int t = 0; t < S; ++t) prow[t] = sh.cand[par][wsel][t];
                    const c128 rp = sh.cand[par][wsel][4];
                    const int tp = (p - c0) % THREADS, rp_ = (p - c0) / THREADS;
                    if (p != j) {
                        if (tid == tp) {
#pragma unroll
                            for (int r = 0; r < R; ++r) if (r == rp_) {
#pragma unroll
                                for (int t = 0; t < S; ++t) v[r][t] = sh.jrow[par][t];
                            }
                        }
                        if (tid == tj) {
#pragma unroll
                            for (int t = 0; t < S; ++t) v[0][t] = prow[t];
                        }
                    }
                    // ---- scale column j and rank-1 update of the sub-panel's remaining columns
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
#pragma unroll
            for (int q = 0; q < S; ++q) {
                if (q < sw) {
                    const int pq = piv_reg[q] < 0 ? -1 - piv_reg[q] : piv_reg[q];
                    spiv[q] = pq; pv[cs + q] = pq;
                    if (piv_reg[q] < 0) atomicCAS(info, 0, cs + q + 1);
                }
            }
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
        if (nright > 0 && DEPTH > 0) {
            // every thread copies, updates and stores its own rows only: no barrier inside the loop; a slot is refilled
            // after the stores that consumed it have been issued
            auto issue = [&](int c) {
                if (c < nright) {
                    c128* dst = stage + (size_t)(c % (DEPTH > 0 ? DEPTH : 1)) * (R * THREADS) + tid;
                    const c128* src = A + (size_t)(cs + sw + c) * n + c0 + tid;
#pragma unroll
                    for (int r = 0; r < R; ++r) {
                        const int row = c0 + tid + r * THREADS;
                        if (row >= cs + sw && row < n) cp_async16(dst + r * THREADS, src + r * THREADS);
                    }
                }
                cp_async_commit();
            };
            for (int d = 0; d < DEPTH; ++d) issue(d);
            for (int c = 0; c < nright; ++c) {
                cp_async_wait<(DEPTH > 0 ? DEPTH - 1 : 0)>();
                const c128* src = stage + (size_t)(c % (DEPTH > 0 ? DEPTH : 1)) * (R * THREADS) + tid;
                c128 u[S];
#pragma unroll
                for (int q = 0; q < S; ++q) u[q] = (q < sw) ? Us[q * P2_MAXW + c] : zero;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    const int row = c0 + tid + r * THREADS;
                    if (row >= cs + sw && row < n) {
                        c128 x = src[r * THREADS];
#pragma unroll
                        for (int q = 0; q < S; ++q) if (q < sw) cfms(x, v[r][q], u[q]);
                        A[row + (size_t)(cs + sw + c) * n] = x;
                    }
                }
                issue(c + DEPTH);
            }
            cp_async_wait<0>();
        } else if (nright > 0) {
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
