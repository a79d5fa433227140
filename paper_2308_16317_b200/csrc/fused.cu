// fused.cu -- the SMALL-MATRIX MODE of the batch scheduler (BASELINE.json north_star: "a batch
// scheduler that packs small LIZ matrices several per SM and lets large ones span the whole chip").
//
// The lock-step schedule (api.cu: eliminate) needs ~10 launches per 16 columns; on a 208 x 208 matrix that is 40
// launches for 0.8 GFLOP, and on 880 x 880 the latency-bound phases of all items coincide between launches.  Here the
// WHOLE elimination of a matrix -- every panel, interchange, triangular solve, Schur update and the final k x k
// inverse -- runs inside ONE launch:
//
//   * one CTA of 128 threads per matrix (or a thread-block cluster of 2 / 4 / 8 CTAs per matrix when the batch is too
//     small to fill the chip that way), FOUR such CTAs resident per SM: while one matrix is in a latency-bound phase
//     (pivot search, interchanges) the other three keep the SM's FP64 tensor pipe busy -- the overlap that the
//     lock-step schedule cannot get from the block scheduler;
//   * the phases are the device-side bodies of the lock-step kernels: panel_body (K2, panel_body.cuh), gemm_tile (K4:
//     DMMA.8x8x4, operands staged by TMA bulk copies, gemm_body.cuh), final_inverse_body (K5, lu_body.cuh), glued by
//     __syncthreads() (cluster barriers when a cluster shares a matrix) instead of kernel boundaries;
//   * the matrix stays where the caller put it (L2 / HBM); CTAs of a cluster exchange nothing but global memory
//     ordered by barrier.cluster (release / acquire), so every CTA count runs the same code.
//
// Two-level right-looking blocking, the same arithmetic per element as the lock-step schedule:
//   outer panel [J, J+W), W <= NB:
//     for each inner panel [c0, c0+w), w <= IB:
//        P1  panel_body: factor, interchanges + triangular solves inside the outer panel         (rank 0 of the cluster)
//        P2  rank-w DMMA update of the outer panel's remaining columns                            (tiles dealt to all CTAs)
//     P3  net row permutation of the W interchanges (every CTA computes it from the pivot vector)
//     P4  permute the trailing columns in place, strips of columns staged in shared memory         (strips dealt to all CTAs)
//     P5  U12 = L11^{-1} A12 by 16-row blocks: thread-per-column forward substitution, then a rank-16 DMMA update of
//         the block rows below (inside the outer panel's rows)
//     P6  Schur update A22 -= L21 U12 on DMMA, inner dimension W                                   (>95 % of the flops)
//   K5  tau00 = inverse of the trailing k x k block                                                (rank 0)
// The tile order of P6 is row-major over the tile grid: the CTA's 64 x W tile of L21 then stays in L2 for a whole tile
// row and only U12 streams (HBM traffic 1.5x the C traffic instead of 2.5x when hundreds of matrices are in flight).
#include "common.cuh"
#include "internal.h"
#include "gemm_body.cuh"
#include "lu_body.cuh"
#include "panel_body.cuh"

namespace lsms {

constexpr int FT = 128;                       // threads per CTA (4 warps = one 64 x 32 DMMA tile)
constexpr int F_STAGES = 2, F_BN = 32;
constexpr int F_MAXNB = 96, F_MAXIB = 16;
constexpr size_t F_RING_BYTES = (size_t)F_STAGES * stage_elems<F_BN>() * sizeof(c128);      // 54272
// dynamic shared memory: [ring | phase scratch (aliased)] [mbarriers] [perm ints]
constexpr size_t F_BAR_OFF = F_RING_BYTES;
constexpr size_t F_PERM_OFF = F_BAR_OFF + 16;
constexpr size_t F_SMEM = F_PERM_OFF + (6 * F_MAXNB + 4) * sizeof(int);                        // 56608 <= 57344 (4 CTAs / SM)
static_assert(sizeof(PanelShared) <= F_RING_BYTES, "panel state is aliased onto the operand ring");
static_assert(sizeof(K5Shared) + 16 <= 8192, "K5 state");
static_assert((2 * 96 * F_MAXIB + F_MAXIB * F_MAXIB) * sizeof(c128) <= F_RING_BYTES, "tiny-mode strip staging");

__device__ __forceinline__ uint32_t f_cluster_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t f_cluster_size() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }

// Phase boundary.  Orders generic-proxy stores (global and shared) before the TMA (async-proxy) reads and writes of the
// next phase, and synchronises the CTA -- or, when a cluster shares the matrix, all its CTAs, with release / acquire
// semantics at cluster scope for the global-memory traffic between them.
__device__ __forceinline__ void phase_sync(uint32_t ncl) {
    asm volatile("fence.proxy.async;" ::: "memory");
    if (ncl == 1) __syncthreads();
    else asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

// C[Mr x Nc] -= A[Mr x K] B[K x Nc] of ONE matrix: the tiles are dealt round-robin to the CTAs of the cluster,
// row-major over the tile grid.  Ends with the CTA synchronised.
__device__ __forceinline__ void gemm_phase(const c128* A, const c128* B, c128* C, int ld, int Mr, int Nc, int K,
                                           int rank, int ncl, c128* ring, uint64_t* full, uint32_t& cc) {
    if (Mr <= 0 || Nc <= 0 || K <= 0) return;
    GemmShape g;
    g.A = A; g.B = B; g.C = C; g.strideA = g.strideB = g.strideC = 0; g.ldA = g.ldB = g.ldC = ld;
    g.Mr = Mr; g.Nc = Nc; g.K = K; g.beta0 = 0; g.batch = 1;
    const int tiles_m = (Mr + BM - 1) / BM, tiles_n = (Nc + F_BN - 1) / F_BN;
    for (int t = rank; t < tiles_m * tiles_n; t += ncl) {
        const int tm = t / tiles_n, tn = t % tiles_n;
        const int m0 = tm * BM, n0 = tn * F_BN;
        gemm_tile<F_STAGES, F_BN>(g, A + m0, B + (size_t)n0 * ld, C + m0 + (size_t)n0 * ld, min(BM, Mr - m0), min(F_BN, Nc - n0),
                                  ring, full, cc);
        __syncthreads();                      // every warp is done with the ring before the next tile refills it
    }
}

// P1 for one inner panel: pick the register blocking from the panel height (128 threads: R rows per thread).
__device__ __forceinline__ void panel_phase(c128* A, int n, int J, int W, int c0, int w, int ne, int* pv, int* info, PanelShared& sh) {
    const int m = n - c0;
    if (m <= 128) panel_body<FT, 1, 4>(A, n, J, W, c0, w, ne, pv, info, sh);
    else if (m <= 256) panel_body<FT, 2, 4>(A, n, J, W, c0, w, ne, pv, info, sh);
    else if (m <= 512) panel_body<FT, 4, 4>(A, n, J, W, c0, w, ne, pv, info, sh);
    else if (m <= 1024) panel_body<FT, 8, 2>(A, n, J, W, c0, w, ne, pv, info, sh);
    else panel_body<FT, 16, 1>(A, n, J, W, c0, w, ne, pv, info, sh);
}

// P1 for TINY matrices (the whole inner panel, (n-c0) x w complex numbers, fits the shared-memory scratch): the panel is
// loaded once, all w column steps run on chip (two CTA barriers per column: arg-max exchange, row swap), and it is
// stored once -- two global round trips per inner panel instead of ~20 for the register-blocked sub-panels of
// panel_body.  Same pivot rule and per-element arithmetic as panel_body (|re|+|im|, ties to the lowest row, rows >= ne
// never eligible).  Requires W == w (single-level blocking): there are no other outer-panel columns to interchange.
// Tried and dropped: a WARP-LEVEL variant (warp 0 holds 4-column sub-panels in registers, 7 rows per lane, column steps
// by shuffles only, no CTA barrier): 36 us per 16-column panel against 26 us here -- one warp issuing the ~1000
// dependent instructions of a column step is slower than four warps sharing them with two barriers.
__device__ __forceinline__ void panel_smem(c128* __restrict__ A, int n, int c0, int w, int ne, int* __restrict__ pv,
                                           int* __restrict__ info, c128* P, double* red_v, int* red_i) {
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int m = n - c0;
    for (int e = tid; e < m * w; e += FT) { const int r = e % m, c = e / m; P[e] = A[(size_t)(c0 + r) + (size_t)(c0 + c) * n]; }
    __syncthreads();
    for (int q = 0; q < w; ++q) {
        const int j = c0 + q;
        double bv = -1.0; int bi = 0x7fffffff;
        for (int r = q + tid; r < ne - c0; r += FT) {
            const double a = cabs1(P[q * m + r]);
            if (a > bv) { bv = a; bi = c0 + r; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bv, o); const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if (lane == 0) { red_v[warp] = bv; red_i[warp] = bi; }
        __syncthreads();
        bv = red_v[lane & (FT / 32 - 1)]; bi = red_i[lane & (FT / 32 - 1)];
#pragma unroll
        for (int o = FT / 64; o > 0; o >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bv, o); const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        const bool bad = !(bv > 0.0) || !(bv < 1.0e300 * 1.0e300);     // zero, NaN or Inf pivot
        const int p = bad ? j : bi;
        if (tid == 0) { pv[j] = p; if (bad) atomicCAS(info, 0, j + 1); }
        if (p != j && tid < w) { const c128 t = P[tid * m + q]; P[tid * m + q] = P[tid * m + (p - c0)]; P[tid * m + (p - c0)] = t; }
        __syncthreads();
        if (!bad) {
            // every thread updates its rows; the columns are taken four at a time so that four independent
            // load -> fma -> store chains are in flight (a one-column-at-a-time loop is bound by shared-memory latency)
            const c128 rp = crecip_fast(P[q * m + q]);
            for (int r = q + 1 + tid; r < m; r += FT) {
                const c128 l = cmul(P[q * m + r], rp);
                P[q * m + r] = l;
                for (int t0 = q + 1; t0 < w; t0 += 4) {
                    c128 x[4], u[4];
#pragma unroll
                    for (int i = 0; i < 4; ++i) if (t0 + i < w) { x[i] = P[(t0 + i) * m + r]; u[i] = P[(t0 + i) * m + q]; }
#pragma unroll
                    for (int i = 0; i < 4; ++i) if (t0 + i < w) { cfms(x[i], l, u[i]); P[(t0 + i) * m + r] = x[i]; }
                }
            }
        }
    }
    __syncthreads();
    for (int e = tid; e < m * w; e += FT) { const int r = e % m, c = e / m; A[(size_t)(c0 + r) + (size_t)(c0 + c) * n] = P[e]; }
}

__global__ void __launch_bounds__(FT, 4)
k_lu_fused(c128* __restrict__ base, size_t stride, int n, int k, int NB, int IB, int W0, int* __restrict__ piv,
           c128* __restrict__ tau, int* __restrict__ info) {
    extern __shared__ __align__(128) unsigned char fsm[];
    c128* ring = reinterpret_cast<c128*>(fsm);
    uint64_t* full = reinterpret_cast<uint64_t*>(fsm + F_BAR_OFF);
    int* perm = reinterpret_cast<int*>(fsm + F_PERM_OFF);          // [nd][top_src W][ddst W][dsrc W][cur_top W][bpos W][bcon W]
    PanelShared& psh = *reinterpret_cast<PanelShared*>(fsm);       // aliases the ring (P1 only)
    c128* scratch = ring;                                          // aliases the ring (P4: Told, P5: Lw, K5: S)

    const uint32_t ncl = f_cluster_size(), rank = f_cluster_rank();
    const int item = blockIdx.x / ncl;
    c128* A = base + (size_t)item * stride;
    int* pv = piv + (size_t)item * n;
    int* inf = info + item;
    const int tid = threadIdx.x;
    const int ne = n - k;
    const int TT = FT * (int)ncl, g0 = (int)rank * FT + tid;       // the cluster's threads, for column-parallel phases

    if (tid == 0) {
        for (int s = 0; s < F_STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    phase_sync(ncl);
    uint32_t cc = 0;

    for (int J = 0, W = W0; J < ne; J += W, W = min(NB, ne - J)) {
        const int Jend = J + W;
        // ---------------- inner panels
        for (int c0 = J; c0 < Jend; c0 += IB) {
            const int w = min(IB, Jend - c0);
            if (rank == 0) panel_phase(A, n, J, W, c0, w, ne, pv, inf, psh);                                  // P1
            phase_sync(ncl);
            const int rem = Jend - (c0 + w);
            if (rem > 0) {                                                                                     // P2
                gemm_phase(A + (size_t)(c0 + w) + (size_t)c0 * n, A + (size_t)c0 + (size_t)(c0 + w) * n,
                           A + (size_t)(c0 + w) + (size_t)(c0 + w) * n, n, n - (c0 + w), rem, w, (int)rank, (int)ncl, ring, full, cc);
                phase_sync(ncl);
            }
        }
        const int ntrail = n - Jend;                               // > 0: Jend <= ne < n
        // ---------------- P3: net permutation of the outer panel's W interchanges (pv was written by rank 0 before the
        // last phase_sync; every CTA folds it for itself)
        int* top_src = perm + 1; int* ddst = top_src + W; int* dsrc = ddst + W;
        if (tid < 32) net_permutation(pv + J, J, W, dsrc + W, dsrc + 2 * W, dsrc + 3 * W, perm, top_src, ddst, dsrc);
        __syncthreads();
        const int nd = perm[0];
        // ---------------- P4: trailing columns [Jend, n): new top block gathered in place, displaced rows scattered
        {
            c128* Told = scratch;                                  // [strip][W]: as many columns as the scratch holds, split evenly
            const int strip = max(1, min((int)(F_RING_BYTES / sizeof(c128)) / W, (ntrail + (int)ncl - 1) / (int)ncl));
            const int nstrips = (ntrail + strip - 1) / strip;
            for (int sidx = (int)rank; sidx < nstrips; sidx += (int)ncl) {
                const int c_first = Jend + sidx * strip, ncol = min(strip, n - c_first);
                for (int e = tid; e < ncol * W; e += FT) {
                    const int i = e % W, c = e / W;
                    Told[c * W + i] = A[(size_t)(J + i) + (size_t)(c_first + c) * n];
                }
                __syncthreads();
                for (int e = tid; e < ncol * W; e += FT) {
                    const int i = e % W, c = e / W;
                    const int src = top_src[i];
                    if (src != J + i)
                        A[(size_t)(J + i) + (size_t)(c_first + c) * n] =
                            (src < Jend) ? Told[c * W + (src - J)] : A[(size_t)src + (size_t)(c_first + c) * n];
                }
                __syncthreads();              // rows below are read (gather) before they are overwritten (scatter)
                for (int e = tid; e < ncol * nd; e += FT) {
                    const int j = e % nd, c = e / nd;
                    A[(size_t)ddst[j] + (size_t)(c_first + c) * n] = Told[c * W + dsrc[j]];
                }
                __syncthreads();
            }
        }
        phase_sync(ncl);
        // ---------------- P5: U12 = L11^{-1} A12 by IB-row blocks
        for (int c0 = J; c0 < Jend; c0 += IB) {
            const int w = min(IB, Jend - c0);
            c128* Lw = scratch;                                    // [F_MAXIB][F_MAXIB], unit lower
            for (int e = tid; e < w * w; e += FT) { const int r = e % w, c = e / w; Lw[r + F_MAXIB * c] = A[(size_t)(c0 + r) + (size_t)(c0 + c) * n]; }
            __syncthreads();
            for (int cj = g0; cj < ntrail; cj += TT) {
                c128* col = A + (size_t)(Jend + cj) * n + c0;
                c128 x[F_MAXIB];
#pragma unroll
                for (int i = 0; i < F_MAXIB; ++i) x[i] = (i < w) ? col[i] : cmake(0.0, 0.0);
#pragma unroll
                for (int jq = 0; jq < F_MAXIB; ++jq)
#pragma unroll
                    for (int i = jq + 1; i < F_MAXIB; ++i)
                        if (i < w) cfms(x[i], Lw[i + F_MAXIB * jq], x[jq]);
#pragma unroll
                for (int i = 0; i < F_MAXIB; ++i) if (i < w) col[i] = x[i];
            }
            phase_sync(ncl);
            const int below = Jend - (c0 + w);
            if (below > 0) {
                gemm_phase(A + (size_t)(c0 + w) + (size_t)c0 * n, A + (size_t)c0 + (size_t)Jend * n,
                           A + (size_t)(c0 + w) + (size_t)Jend * n, n, below, ntrail, w, (int)rank, (int)ncl, ring, full, cc);
                phase_sync(ncl);
            }
        }
        // ---------------- P6: Schur update
        gemm_phase(A + (size_t)Jend + (size_t)J * n, A + (size_t)J + (size_t)Jend * n, A + (size_t)Jend + (size_t)Jend * n,
                   n, ntrail, ntrail, W, (int)rank, (int)ncl, ring, full, cc);
        phase_sync(ncl);
    }
    // ---------------- K5: tau00 = inverse of the trailing k x k block
    if (rank == 0) {
        K5Shared& ksh = *reinterpret_cast<K5Shared*>(fsm);
        c128* S = reinterpret_cast<c128*>(fsm + 8192);
        final_inverse_body<FT>(A, n, k, tau + (size_t)item * k * k, inf, S, ksh);
    }
    if (ncl > 1) phase_sync(ncl);             // no CTA of a cluster exits while another may still be at a barrier
}

// ---------------------------------------------------------------- TINY matrices (n <= 212: BASELINE.json configs[0])
// A whole 16-column panel fits the shared-memory scratch, so the blocking is single-level (W = w <= 16) and every
// phase is trimmed for latency -- at this size nothing but the chain of dependent steps costs time:
//   T1  panel_smem: panel loaded once, w column steps on chip, stored once                          (rank 0)
//   T2  net permutation of the w interchanges                                                       (every CTA, warp 0)
//   T3  trailing columns, strips staged in shared memory: interchanges in place, then the w x w unit-lower solve
//       straight from the staged rows (no second pass over the matrix)
//   T4  rank-w DMMA update of the trailing matrix
// LOOK-AHEAD inside the cluster: the panel factorisation is the critical path (16 dependent column steps, ~26 us) and
// only one CTA can work on it.  So rank 0 takes the NEXT panel's columns through T3 and T4 by itself and factors that
// panel at once, while ranks 1.. do T3 and T4 on all other trailing columns.  The cluster barrier is split
// (barrier.cluster.arrive / .wait): rank 0 arrives before it starts the panel and waits after it, so the other ranks
// never wait for the panel unless they run out of work.  Two cluster barriers per panel.
constexpr int TINY_MAXCOLS = 96;              // trailing columns per strip: 2 x 96 x 16 staged values + L11 = 52 KB

__device__ __forceinline__ void cluster_arrive() {
    asm volatile("fence.proxy.async;" ::: "memory");
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
}
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

// T3 for the columns [col_lo, col_hi) by this CTA: permutation of the panel's w interchanges (top_src / ddst / dsrc, nd
// in perm[0]) applied in place and U rows = L11^{-1} (permuted top block).  Ends with the CTA synchronised.
__device__ __forceinline__ void tiny_t3(c128* __restrict__ A, int n, int c0, int w, int col_lo, int col_hi, c128* ring, const int* perm) {
    const int tid = threadIdx.x, cend = c0 + w;
    const int* top_src = perm + 1; const int* ddst = top_src + w; const int* dsrc = ddst + w;
    c128* Told = ring;                                      // [cols][w]   old top block
    c128* Tnew = ring + TINY_MAXCOLS * F_MAXIB;             // [cols][w]   permuted top block
    c128* L11 = ring + 2 * TINY_MAXCOLS * F_MAXIB;          // [16][16]    unit lower triangle of the panel
    __syncthreads();                                        // T2's result (warp 0) before its use; scratch free
    for (int c_first = col_lo; c_first < col_hi; c_first += TINY_MAXCOLS) {
        const int ncol = min(TINY_MAXCOLS, col_hi - c_first);
        for (int e = tid; e < ncol * w; e += FT) {
            const int i = e % w, c = e / w;
            Told[c * w + i] = A[(size_t)(c0 + i) + (size_t)(c_first + c) * n];
        }
        for (int e = tid; e < w * w; e += FT) { const int r = e % w, c = e / w; L11[r + F_MAXIB * c] = A[(size_t)(c0 + r) + (size_t)(c0 + c) * n]; }
        __syncthreads();
        const int nd = perm[0];
        for (int e = tid; e < ncol * w; e += FT) {
            const int i = e % w, c = e / w;
            const int src = top_src[i];
            Tnew[c * w + i] = (src < cend) ? Told[c * w + (src - c0)] : A[(size_t)src + (size_t)(c_first + c) * n];
        }
        __syncthreads();              // rows below are read (gather) before they are overwritten (scatter)
        for (int e = tid; e < ncol * nd; e += FT) {
            const int j = e % nd, c = e / nd;
            A[(size_t)ddst[j] + (size_t)(c_first + c) * n] = Told[c * w + dsrc[j]];
        }
        for (int c = tid; c < ncol; c += FT) {             // U rows of this column: forward substitution from the staged values
            c128 x[F_MAXIB];
#pragma unroll
            for (int i = 0; i < F_MAXIB; ++i) x[i] = (i < w) ? Tnew[c * w + i] : cmake(0.0, 0.0);
#pragma unroll
            for (int jq = 0; jq < F_MAXIB; ++jq)
#pragma unroll
                for (int i = jq + 1; i < F_MAXIB; ++i)
                    if (i < w) cfms(x[i], L11[i + F_MAXIB * jq], x[jq]);
            c128* col = A + (size_t)(c_first + c) * n + c0;
#pragma unroll
            for (int i = 0; i < F_MAXIB; ++i) if (i < w) col[i] = x[i];
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(FT, 3)
k_lu_tiny(c128* __restrict__ base, size_t stride, int n, int k, int IB, int* __restrict__ piv,
          c128* __restrict__ tau, int* __restrict__ info) {
    extern __shared__ __align__(128) unsigned char fsm[];
    c128* ring = reinterpret_cast<c128*>(fsm);
    uint64_t* full = reinterpret_cast<uint64_t*>(fsm + F_BAR_OFF);
    int* perm = reinterpret_cast<int*>(fsm + F_PERM_OFF);
    double* red_v = reinterpret_cast<double*>(perm + 6 * F_MAXNB - 32);   // arg-max exchange of panel_smem (spare room of the perm region)
    int* red_i = perm + 6 * F_MAXNB - 16;
    const uint32_t ncl = f_cluster_size(), rank = f_cluster_rank();
    const int item = blockIdx.x / ncl;
    c128* A = base + (size_t)item * stride;
    int* pv = piv + (size_t)item * n;
    int* inf = info + item;
    const int tid = threadIdx.x;
    const int ne = n - k;

    if (tid == 0) {
        for (int s = 0; s < F_STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    phase_sync(ncl);
    uint32_t cc = 0;
    bool factored = false;                  // is the current panel already factored (by the previous iteration's look-ahead)?
    for (int c0 = 0; c0 < ne; c0 += IB) {
        const int w = min(IB, ne - c0), cend = c0 + w, ntrail = n - cend;
        if (!factored) {
            if (rank == 0) panel_smem(A, n, c0, w, ne, pv, inf, ring, red_v, red_i);                         // T1
            phase_sync(ncl);
        }
        int* top_src = perm + 1; int* ddst = top_src + w; int* dsrc = ddst + w;
        if (tid < 32) net_permutation(pv + c0, c0, w, dsrc + w, dsrc + 2 * w, dsrc + 3 * w, perm, top_src, ddst, dsrc);   // T2
        const int w2 = (cend < ne) ? min(IB, ne - cend) : 0;           // width of the next panel
        const c128* L21 = A + (size_t)cend + (size_t)c0 * n;           // rows below the panel, its columns
        if (ncl > 1 && w2 > 0) {
            // ---- look-ahead: rank 0 alone brings the next panel's columns up to date and factors them
            if (rank == 0) {
                tiny_t3(A, n, c0, w, cend, cend + w2, ring, perm);
                phase_sync(1);
                gemm_phase(L21, A + (size_t)c0 + (size_t)cend * n, A + (size_t)cend + (size_t)cend * n, n, ntrail, w2, w, 0, 1, ring, full, cc);
                cluster_arrive();
                panel_smem(A, n, cend, w2, ne, pv, inf, ring, red_v, red_i);
                cluster_wait();
                cluster_arrive(); cluster_wait();
            } else {
                const int lo = cend + w2, rest = n - lo, nr = (int)ncl - 1, r1 = (int)rank - 1;
                const int per = (rest + nr - 1) / nr;
                tiny_t3(A, n, c0, w, min(n, lo + r1 * per), min(n, lo + (r1 + 1) * per), ring, perm);
                cluster_arrive(); cluster_wait();
                gemm_phase(L21, A + (size_t)c0 + (size_t)lo * n, A + (size_t)cend + (size_t)lo * n, n, ntrail, rest, w, r1, nr, ring, full, cc);
                cluster_arrive(); cluster_wait();
            }
            factored = true;
        } else {
            const int per = (ntrail + (int)ncl - 1) / (int)ncl;
            tiny_t3(A, n, c0, w, min(n, cend + (int)rank * per), min(n, cend + ((int)rank + 1) * per), ring, perm);
            phase_sync(ncl);
            gemm_phase(L21, A + (size_t)c0 + (size_t)cend * n, A + (size_t)cend + (size_t)cend * n, n, ntrail, ntrail, w, (int)rank, (int)ncl, ring, full, cc);
            phase_sync(ncl);
            factored = false;
        }
    }
    if (rank == 0) {
        K5Shared& ksh = *reinterpret_cast<K5Shared*>(fsm);
        c128* S = reinterpret_cast<c128*>(fsm + 8192);
        final_inverse_body<FT>(A, n, k, tau + (size_t)item * k * k, inf, S, ksh);
    }
    if (ncl > 1) phase_sync(ncl);
}

// k x k Gauss-Jordan scratch (after 8 KB of K5 state) has to fit the ring region
bool fused_supported(int n, int k, int NB, int IB) {
    if (n > 2048 || n - k < 0) return false;
    if (NB < 4 || NB > F_MAXNB || IB < 1 || IB > F_MAXIB) return false;
    if (8192 + (size_t)k * k * sizeof(c128) > F_RING_BYTES) return false;
    return true;
}

// n for which the tiny kernel (panel on chip, single-level blocking) applies
bool fused_is_tiny(int n) { return (size_t)n * F_MAXIB * sizeof(c128) <= F_RING_BYTES; }

int init_attrs_fused() {
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_lu_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_lu_tiny, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)F_SMEM));
    return 0;
}

int fused_max_active_clusters(int cl) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)cl); cfg.blockDim = dim3(FT); cfg.dynamicSmemBytes = F_SMEM;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = (unsigned)cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    int a = 0, b = 0;
    if (cudaOccupancyMaxActiveClusters(&a, k_lu_fused, &cfg) != cudaSuccess ||
        cudaOccupancyMaxActiveClusters(&b, k_lu_tiny, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return a < b ? a : b;
}

int launch_lu_fused(c128* base, size_t stride, int n, int k, int batch, int NB, int IB, int align_first, int cl,
                    int* piv, c128* tau, int* info, cudaStream_t st) {
    if (!fused_supported(n, k, NB, IB) || (cl != 1 && cl != 2 && cl != 4 && cl != 8)) return -1;
    const int ne = n - k;
    // TINY matrices: a whole 16-column panel fits the shared-memory scratch (n <= 212).  Single-level blocking with the
    // panel factored on chip (panel_smem); the rank-16 Schur updates are latency-bound either way at this size.
    const bool tiny = fused_is_tiny(n);
    int W0 = ne < NB ? ne : NB;
    if (align_first && NB % 64 == 0 && n % 64 != 0 && n % 64 < W0) W0 = n % 64;
    for (int b0 = 0; b0 < batch; b0 += 32768) {
        const int nb = batch - b0 < 32768 ? batch - b0 : 32768;
        cudaLaunchConfig_t cfg = {};
        cfg.gridDim = dim3((unsigned)(nb * cl)); cfg.blockDim = dim3(FT); cfg.dynamicSmemBytes = F_SMEM; cfg.stream = st;
        cudaLaunchAttribute at[1];
        at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = (unsigned)cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
        cfg.attrs = at; cfg.numAttrs = 1;
        if (tiny)
            LSMS_CUDA_OK(cudaLaunchKernelEx(&cfg, k_lu_tiny, base + (size_t)b0 * stride, stride, n, k, IB < F_MAXIB ? IB : F_MAXIB,
                                            piv + (size_t)b0 * n, tau + (size_t)b0 * k * k, info + b0));
        else
            LSMS_CUDA_OK(cudaLaunchKernelEx(&cfg, k_lu_fused, base + (size_t)b0 * stride, stride, n, k, NB, IB, W0, piv + (size_t)b0 * n,
                                            tau + (size_t)b0 * k * k, info + b0));
        LSMS_LAUNCH_CHECK();
    }
    return 0;
}

}  // namespace lsms
