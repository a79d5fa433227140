// resident.cu -- small-matrix mode, ON-CHIP variant (SURVEY.md 8(a) a7 / 7.3 hard part 5; BASELINE.json north_star:
// "a batch scheduler that packs small LIZ matrices several per SM and lets large ones span the whole chip").
//
// For matrices of a few hundred rows (BASELINE.json configs[0]: 208 x 208, 692 KB) nothing but the chain of n-k
// dependent pivot steps costs time, and every trip to L2 lengthens it.  Here a matrix never leaves the chip between its
// first and its last elimination step: a thread-block CLUSTER of 1 / 2 / 4 / 8 CTAs (one CTA per SM) holds it in
// distributed shared memory, column blocks of RW = 8 dealt round-robin over the CTAs, and the whole elimination
// ("LU factorization"; restricted pivoting, reading A14; only the central block of
// the inverse is wanted) runs in one launch:
//
//   for each panel p (columns [8p, 8p+8), owner = CTA p mod ncl; R1 of panel p+1 runs DURING step p, see below):
//     R1  owner, one matrix row per thread, the row's 8 panel entries in registers: 8 pivot steps with ONE barrier
//         each (every warp publishes its arg-max candidate -- found by two redux.sync on a 64-bit key -- TOGETHER
//         with that row's entries and the reciprocal of the would-be pivot, so the winner's row is already in shared
//         memory when the barrier opens); rows never move between threads, each thread tracks the position of its
//         row in the pivoted arrangement; result -> staged in the panel's own (now dead) columns of the matrix
//     R2  the staged panel is sent to the other CTAs' panel buffers by the TMA engine: bulk copies shared -> remote
//         shared (cp.async.bulk.shared::cluster.shared::cta), completion counted on an mbarrier of the RECEIVING CTA.
//         A receiver declares its panel buffer free by a release-store of a flag into the next owner's shared memory;
//         the owner's warp 15 (the "shipper") polls the flags and serves each CTA as soon as it is free, the next
//         owner first -- no cluster-wide barrier inside the loop, and nobody waits for a CTA that is behind
//     R3  every CTA, its own trailing columns: the panel's interchanges as ONE net row permutation (eight threads per
//         column) and the 8 x 8 unit-lower solve (rows of U -> a small operand buffer and, for the verification
//         export, to global memory)
//     R4  rank-8 update of its trailing columns on the FP64 tensor pipe (DMMA.8x8x4 from shared memory; operand
//         strides chosen conflict-free: ld = 1, ldp = 2, ldu = 4 (mod 8) complex units)
//   K5  the trailing k x k block goes to global memory and rank 0 inverts it (final_inverse_small).
// LOOK-AHEAD: the CTA that owns panel p+1 updates that block first (R3, R4 on its 8 columns) and factors panel p+1 (R1)
// at once, with its SM to itself, while the other CTAs finish step p.  It catches up on step p for its other columns
// only after panel p+1 is on its way (its own panel buffer still holds panel p): warps 0-14 do that while warp 15 ships
// -- off the critical path, while the next owner works.  Measured chain per panel (208^2, first -> last): ship 1.0 ->
// 0.65 us, block update 1.7 -> 1.45, R1 3.6 -> 2.8, staging 0.7 -> 0.55: 7.0 -> 5.5 us.
//
// Global traffic: the matrix is read once (TMA bulk loads, one per column); U and the final block are written once.
#include "common.cuh"
#include "internal.h"
#include "gemm_body.cuh"
#include "lu_body.cuh"

namespace lsms {

constexpr int RS_T = 512;            // threads per CTA
constexpr int RS_PT = 256;           // panel threads = largest n
constexpr int RW = 8;                // panel width = column-block width
constexpr int RS_LDU = RW + 4;       // U operand buffer stride (complex), == 4 (mod 8)
constexpr size_t RS_SMEM_MAX = 232448;
static_assert(RS_PT <= 256 && RS_PT / 32 <= 8, "arg-max key of the panel step: 8 bits for the row position (255 - pos), 3 for the warp");

struct ResLayout {
    int ld, ldp, ncols_max;
    size_t off_L, off_piv, off_U, off_red, off_bar, total;
};
// red region: 2 parities x 8 warp slots x (8 row entries + 1/candidate + key)
constexpr size_t RS_SLOT = (RW + 2) * sizeof(c128);               // row entries, reciprocal of the candidate, arg-max key
constexpr size_t RS_RED_PAR = 8 * RS_SLOT;
__host__ __device__ inline ResLayout res_layout(int n, int ncl) {
    ResLayout L;
    const int nblk = (n + RW - 1) / RW, blk_max = (nblk + ncl - 1) / ncl;
    L.ncols_max = blk_max * RW;
    L.ld = (n + 6) / 8 * 8 + 1;                  // >= n, == 1 (mod 8)
    L.ldp = (n + 5) / 8 * 8 + 2;                 // >= n, == 2 (mod 8)
    size_t o = (size_t)L.ncols_max * L.ld * sizeof(c128);
    L.off_L = o; o += (size_t)RW * L.ldp * sizeof(c128);
    L.off_piv = o; o += 32 * sizeof(c128);       // net row permutation of the panel (96 B, bulk-copied) + slack for tile over-reads
    L.off_U = o; o += (size_t)L.ncols_max * RS_LDU * sizeof(c128);
    L.off_red = o; o += 2 * RS_RED_PAR;
    L.off_bar = o; o += 128;                    // two mbarriers + the per-CTA 'panel buffer free' flags
    L.total = o;
    return L;
}

__device__ __forceinline__ uint32_t rs_rank() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t rs_ncl() { uint32_t r; asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r)); return r; }
__device__ __forceinline__ uint32_t rs_mapa(uint32_t addr, uint32_t rank) {
    uint32_t r; asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank)); return r;
}
__device__ __forceinline__ void rs_cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void rs_st_release_remote(uint32_t addr_cluster, int v) {
    asm volatile("st.release.cluster.shared::cluster.s32 [%0], %1;" ::"r"(addr_cluster), "r"(v) : "memory");
}
__device__ __forceinline__ int rs_ld_acquire(const int* p) {
    int v; asm volatile("ld.acquire.cluster.shared::cta.s32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory"); return v;
}
// shared (this CTA) -> shared of another CTA of the cluster, by the TMA engine; completion on the receiver's mbarrier
__device__ __forceinline__ void rs_bulk_s2r(uint32_t dst_cluster, uint32_t src_cta, uint32_t bytes, uint32_t bar_cluster) {
    asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(dst_cluster), "r"(src_cta), "r"(bytes), "r"(bar_cluster) : "memory");
}
__global__ void __launch_bounds__(RS_T, 1)
k_lu_resident(c128* __restrict__ base, size_t stride, int n, int k, int* __restrict__ piv, c128* __restrict__ tau,
              int* __restrict__ info) {
    extern __shared__ __align__(128) unsigned char rsm[];
    const int ncl = (int)rs_ncl(), rank = (int)rs_rank();
    const ResLayout L = res_layout(n, ncl);
    c128* Aloc = reinterpret_cast<c128*>(rsm);
    c128* Lbuf = reinterpret_cast<c128*>(rsm + L.off_L);
    int* spiv = reinterpret_cast<int*>(rsm + L.off_piv);
    int* spiv2 = spiv + 32;                              // staging copy of the next panel's permutation
    c128* Ubuf = reinterpret_cast<c128*>(rsm + L.off_U);
    unsigned char* red = rsm + L.off_red;
    uint64_t* bar_load = reinterpret_cast<uint64_t*>(rsm + L.off_bar);
    uint64_t* bar_full = bar_load + 1;
    int* ready = reinterpret_cast<int*>(bar_load + 2);   // ready[r] (written by CTA r): r's panel buffer may receive panel ready[r]
    const int ld = L.ld, ldp = L.ldp;

    const int item = blockIdx.x / ncl;
    c128* A = base + (size_t)item * stride;
    int* pv = piv + (size_t)item * n;
    int* inf = info + item;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int ne = n - k;
    const int nblk = (n + RW - 1) / RW;
    const int my_blocks = (nblk > rank) ? (nblk - rank + ncl - 1) / ncl : 0;
    const int my_cols = my_blocks * RW;                       // local columns incl. the padding of a ragged last block
    auto gcol = [&](int lc) { return ((lc / RW) * ncl + rank) * RW + lc % RW; };

    if (tid < 8) ready[tid] = 0;
    if (tid == 0) {
        mbar_init(bar_load, 1); mbar_init(bar_full, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    // padding columns of a ragged last block and the U buffer start as zeros
    for (int lc = tid; lc < my_cols; lc += RS_T) if (gcol(lc) >= n) for (int r = 0; r < ld; ++r) Aloc[(size_t)lc * ld + r] = cmake(0.0, 0.0);
    for (int e = tid; e < L.ncols_max * RS_LDU; e += RS_T) Ubuf[e] = cmake(0.0, 0.0);
    for (int e = tid; e < RW * ldp + 32; e += RS_T) Lbuf[e] = cmake(0.0, 0.0);      // incl. the permutation ints and the slack behind them
    asm volatile("fence.proxy.async;" ::: "memory");
    __syncthreads();
    // ---- the CTA's column blocks -> shared memory: one TMA bulk copy per column
    {
        int nvalid = 0;
        for (int lc = 0; lc < my_cols; ++lc) nvalid += gcol(lc) < n;
        if (tid == 0) mbar_expect_tx(bar_load, (uint32_t)((size_t)nvalid * n * sizeof(c128)));
        __syncthreads();
        for (int lc = tid; lc < my_cols; lc += RS_T) {
            const int g = gcol(lc);
            if (g < n) tma_bulk_g2s(Aloc + (size_t)lc * ld, A + (size_t)g * n, (uint32_t)(n * sizeof(c128)), bar_load);
        }
    }
    rs_cluster_sync();                           // every CTA of the cluster is running and its mbarriers are initialised
    mbar_wait(bar_load, 0);
    uint32_t full_parity = 0;
    const int np = (ne + RW - 1) / RW;

    // ---- state of a panel factorisation: lives in the registers of the owner's panel threads from R1 (which may run
    // during the PREVIOUS panel's update, see the look-ahead below) to the publication at the top of the panel's own step
    c128 v[RW];
    int pos = 0, ppos_all[RW];
#pragma unroll
    for (int c = 0; c < RW; ++c) { v[c] = cmake(0.0, 0.0); ppos_all[c] = c; }

    // ================= R1: panel factorisation, one row per thread (threads < npt of the owner).  Rows are never moved
    // between threads: thread t keeps the row it loaded and tracks the POSITION (row index relative to c0) at which
    // that row stands in the pivoted arrangement; pivot rows are published through shared memory only.
    auto panel_factor = [&](int p) {
        const int c0 = p * RW, wv = min(RW, ne - c0), m = n - c0;
        const int lcp = (p / ncl) * RW;                                // the panel's first local column in its owner
        const int npt = ((m + 31) / 32) * 32;                          // panel threads: whole warps covering the m rows
        if (tid >= npt) return;
        const int t = tid;
        pos = t;
#pragma unroll
        for (int c = 0; c < RW; ++c) v[c] = (t < m) ? Aloc[(size_t)(lcp + c) * ld + c0 + t] : cmake(0.0, 0.0);
        if (t < 2 * (RS_PT / 32)) {                                    // keys of the warps that sit this panel out
            const int w8 = t >> 1;
            if (w8 >= npt / 32) reinterpret_cast<unsigned long long*>(reinterpret_cast<c128*>(red + (size_t)(t & 1) * RS_RED_PAR + (size_t)w8 * RS_SLOT) + RW + 1)[0] = 0ull;
        }
        // reciprocal of every row's own entry of the coming column: only the pivot row's is used, but computed here
        // (and, for the later columns, right after the entry's last update) its latency hides behind the rest of the
        // rank-1 update and the arg-max reduction
        c128 rinv = crecip_fast(v[0]);
#pragma unroll
        for (int j = 0; j < RW; ++j) {
            ppos_all[j] = j;
            if (j < wv) {
                unsigned char* rp_ = red + (size_t)(j & 1) * RS_RED_PAR;
                // Arg-max key: the bits of |re|+|im| with the low 11 mantissa bits replaced by (255 - pos, warp): one
                // unsigned 64-bit maximum picks the largest magnitude and, among (nearly) equal ones, the lowest row of
                // the current arrangement (LAPACK's rule up to 2^-41); 0 = not eligible.  Two redux.sync per warp
                // instead of fifteen shuffles.
                const bool elig = (pos >= j && t < m && c0 + pos < ne);
                uint32_t khi = 0, klo = 0;
                if (elig) {
                    const unsigned long long kb = (unsigned long long)__double_as_longlong(cabs1(v[j]));
                    khi = (uint32_t)(kb >> 32); klo = ((uint32_t)kb & ~0x7FFu) | ((uint32_t)(255 - pos) << 3) | (uint32_t)warp;
                }
                const uint32_t mhi = __reduce_max_sync(0xffffffffu, khi);
                const uint32_t mlo = __reduce_max_sync(0xffffffffu, (khi == mhi) ? klo : 0u);
                c128* slot = reinterpret_cast<c128*>(rp_ + (size_t)warp * RS_SLOT);
                if (elig && khi == mhi && klo == mlo) {
#pragma unroll
                    for (int c = j + 1; c < RW; ++c) slot[c] = v[c];
                    slot[RW] = rinv;
                }
                if (lane == 0) reinterpret_cast<unsigned long long*>(slot + RW + 1)[0] = ((unsigned long long)mhi << 32) | mlo;
                asm volatile("bar.sync 1, %0;" ::"r"(npt) : "memory");
                // every thread picks the winner among the warp candidates
                unsigned long long wk[RS_PT / 32];
#pragma unroll
                for (int w8 = 0; w8 < RS_PT / 32; ++w8)
                    wk[w8] = reinterpret_cast<const unsigned long long*>(reinterpret_cast<const c128*>(rp_ + (size_t)w8 * RS_SLOT) + RW + 1)[0];
#pragma unroll
                for (int o = RS_PT / 64; o > 0; o >>= 1)
#pragma unroll
                    for (int w8 = 0; w8 < o; ++w8) wk[w8] = wk[w8] > wk[w8 + o] ? wk[w8] : wk[w8 + o];
                const unsigned long long wkey = wk[0];
                const bool bad = (wkey >> 11) == 0ull || (uint32_t)(wkey >> 52) >= 0x7FFu;    // zero, NaN or Inf pivot
                const int ppos = bad ? j : 255 - (int)((wkey >> 3) & 0xFFull);                // position of the pivot row
                ppos_all[j] = bad ? -1 - j : ppos;
                if (!bad) {
                    const c128* ps = reinterpret_cast<const c128*>(rp_ + (size_t)(wkey & 7ull) * RS_SLOT);
                    c128 prow[RW];
#pragma unroll
                    for (int c = j + 1; c < RW; ++c) prow[c] = ps[c];
                    const c128 rp = ps[RW];
                    // the pivot row takes position j, the row that stood there takes the pivot row's position
                    if (pos == ppos) pos = j; else if (pos == j) pos = ppos;
                    if (pos > j && t < m) {
                        const c128 l = cmul(v[j], rp);
                        v[j] = l;
                        if (j + 1 < RW) { cfms(v[j + 1], l, prow[j + 1]); rinv = crecip_fast(v[j + 1]); }
#pragma unroll
                        for (int c = j + 2; c < RW; ++c) cfms(v[c], l, prow[c]);
                    }
                }
            }
        }
    };
    // The factored panel -> shared memory: L (and U11) into the panel buffer, rows in their pivoted positions, and the net
    // row permutation of the panel's interchanges (spiv[8..16): top_src, row whose content ends in top position i;
    // spiv[16..24): ddst, row below the top block that receives the ORIGINAL top row i, or -1).  Columns beyond wv
    // (central columns inside the last panel's block) have received all their updates in R1 and go back to the matrix.
    auto panel_publish = [&](int p) {
        const int c0 = p * RW, wv = min(RW, ne - c0), m = n - c0;
        const int lcp = (p / ncl) * RW;
        if (tid < m) {
            // staging area = the panel's own columns of the matrix (dead once they are in registers); columns beyond wv
            // of a ragged last panel hold live central entries: they are not part of L and are stored where they belong
#pragma unroll
            for (int c = 0; c < RW; ++c) Aloc[(size_t)(lcp + c) * ld + c0 + pos] = v[c];
            if (pos < wv) spiv2[RW + pos] = c0 + tid;
            if (tid < RW) {
                spiv2[2 * RW + tid] = (tid < wv && pos >= wv) ? c0 + pos : -1;
                if (tid >= wv) spiv2[RW + tid] = c0 + tid;         // positions of a ragged last panel that are no pivots
            }
        }
    };
    // staged panel -> this CTA's own panel buffer (the other CTAs get it by bulk copy)
    auto panel_to_lbuf = [&](int p) {
        const int c0 = p * RW, wv = min(RW, ne - c0), m = n - c0;
        const int lcp = (p / ncl) * RW;
        for (int e = tid; e < RW * m; e += RS_T) {
            const int c = e / m, r = e % m;
            Lbuf[(size_t)c * ldp + r] = (c < wv) ? Aloc[(size_t)(lcp + c) * ld + c0 + r] : cmake(0.0, 0.0);
        }
        if (tid < 3 * RW) spiv[tid] = spiv2[tid];
    };
    // ... -> global memory (off the critical path: after the panel has been shipped): pivot vector, status, and the rows
    // of U held by this block for the verification export (k_backsolve_central reads U11, U12)
    auto panel_export = [&](int p) {
        const int c0 = p * RW, wv = min(RW, ne - c0), m = n - c0;
        if (tid == 0) {
#pragma unroll
            for (int j = 0; j < RW; ++j) {
                const int pp = ppos_all[j] < 0 ? -1 - ppos_all[j] : ppos_all[j];
                if (j < wv) { pv[c0 + j] = c0 + pp; if (ppos_all[j] < 0) atomicCAS(inf, 0, c0 + j + 1); }
            }
        }
        if (tid < m && pos < wv) {
#pragma unroll
            for (int c = 0; c < RW; ++c) if (c >= pos && c0 + c < n) A[(size_t)(c0 + pos) + (size_t)(c0 + c) * n] = v[c];
        }
    };
    // ================= R3: panel p's interchanges + 8 x 8 unit-lower solve for the local columns [lc_lo, lc_hi) by the
    // threads tbase .. tbase+nthr-1: EIGHT threads per column (same warp) apply the net permutation -- thread i reads
    // the old and the new content of top position i, then the displaced rows are written -- and the first of them
    // solves for the column's rows of U.
    auto swap_solve = [&](int p, int lc_lo, int lc_hi, int tbase, int nthr) {
        const int c0 = p * RW, wv = min(RW, ne - c0);
        const int i = tid & 7;
        const int top_src = spiv[RW + i], ddst = spiv[2 * RW + i];
        const int ncols = lc_hi - lc_lo, rounds = (ncols * 8 + nthr - 1) / nthr;
        for (int r = 0; r < rounds; ++r) {
            const int lc = lc_lo + (r * nthr + (tid - tbase)) / 8;
            const bool live = lc < lc_hi;
            c128* col = Aloc + (size_t)(live ? lc : lc_lo) * ld;
            const c128 a = col[c0 + i], b = col[top_src];
            __syncwarp();
            if (live && ddst >= 0) col[ddst] = a;
            if (live) Ubuf[(size_t)lc * RS_LDU + i] = b;
            __syncwarp();
            if (live && i == 0) {
                c128 x[RW];
#pragma unroll
                for (int q = 0; q < RW; ++q) x[q] = (q < wv) ? Ubuf[(size_t)lc * RS_LDU + q] : cmake(0.0, 0.0);
#pragma unroll
                for (int jq = 0; jq < RW; ++jq)
#pragma unroll
                    for (int q = jq + 1; q < RW; ++q)
                        if (q < wv) cfms(x[q], Lbuf[(size_t)jq * ldp + q], x[jq]);
                const int g = gcol(lc);
#pragma unroll
                for (int q = 0; q < RW; ++q) {
                    Ubuf[(size_t)lc * RS_LDU + q] = x[q];
                    if (q < wv && g < n) A[(size_t)(c0 + q) + (size_t)g * n] = x[q];
                }
            }
        }
    };
    // ================= R4: rank-8 update of rows [c0+wv, n) x local columns [lc_lo, lc_hi) on DMMA, warp tiles of
    // 32 x 8 dealt to the warps wbase .. wbase+nw-1
    auto rank8_update = [&](int p, int lc_lo, int lc_hi, int wbase, int nw) {
        const int c0 = p * RW, wv = min(RW, ne - c0);
        const int r_lo = c0 + wv, mrows = n - r_lo;
        const int tiles_m = (mrows + 31) / 32, tiles_n = (lc_hi - lc_lo) / RW;
        const int gq = lane >> 2, q = lane & 3;
        for (int tt = warp - wbase; tt < tiles_m * tiles_n; tt += nw) {
            const int tm = tt % tiles_m, tn = tt / tiles_m;
            const int r0 = r_lo + tm * 32, lc0 = lc_lo + tn * RW;
            double cr[4][2], ci[4][2];
            c128* Cb = Aloc + (size_t)(lc0 + 2 * q) * ld + r0 + gq;
#pragma unroll
            for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                for (int e = 0; e < 2; ++e) { const c128 cv = Cb[(size_t)e * ld + mt * 8]; cr[mt][e] = cv.x; ci[mt][e] = cv.y; }
#pragma unroll
            for (int ks = 0; ks < RW / 4; ++ks) {
                const c128 b = Ubuf[(size_t)(lc0 + gq) * RS_LDU + ks * 4 + q];
                const double nbr = -b.x, nbi = -b.y;
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    const c128 a = Lbuf[(size_t)(ks * 4 + q) * ldp + (r0 - c0) + mt * 8 + gq];
                    dmma884(cr[mt][0], cr[mt][1], a.x, nbr);
                    dmma884(ci[mt][0], ci[mt][1], a.x, nbi);
                    dmma884(cr[mt][0], cr[mt][1], a.y, b.y);
                    dmma884(ci[mt][0], ci[mt][1], a.y, nbr);
                }
            }
#pragma unroll
            for (int mt = 0; mt < 4; ++mt)
#pragma unroll
                for (int e = 0; e < 2; ++e)
                    if (r0 + mt * 8 + gq < n) Cb[(size_t)e * ld + mt * 8] = cmake(cr[mt][e], ci[mt][e]);
        }
    };

    // ship panel p (staged in its own columns) to the CTAs rank+d_lo .. rank+d_hi-1 (mod ncl), each as soon as IT has
    // declared its panel buffer free -- no cluster-wide barrier: the next owner, which is served first, never waits for
    // a CTA that is still catching up
    auto ship = [&](int p, int d_lo, int d_hi) {
        const int c0 = p * RW, wv = min(RW, ne - c0), m = n - c0, lcp = (p / ncl) * RW;
        if (tid >= RS_T - 32 && tid < RS_T - 32 + RW + 1) {          // the shipper: warp 15
            const int c = tid - (RS_T - 32);
            for (int d = d_lo; d < d_hi; ++d) {
                const uint32_t dst = (uint32_t)((rank + d) % ncl);
                while (rs_ld_acquire(&ready[dst]) < p) {}
                const uint32_t rbar = rs_mapa(smem_u32(bar_full), dst);
                if (c < wv) rs_bulk_s2r(rs_mapa(smem_u32(Lbuf + (size_t)c * ldp), dst), smem_u32(Aloc + (size_t)(lcp + c) * ld + c0), (uint32_t)(m * sizeof(c128)), rbar);
                else if (c == RW) rs_bulk_s2r(rs_mapa(smem_u32(spiv), dst), smem_u32(spiv2), (uint32_t)(3 * RW * sizeof(int)), rbar);
            }
        }
    };
    // this CTA is done with the panel buffer's content: arm the mbarrier for panel q and tell q's owner
    auto declare_free = [&](int q) {
        if (q < np && q % ncl != rank && tid == 0) {
            const int mq = n - q * RW, wq = min(RW, ne - q * RW);
            mbar_expect_tx(bar_full, (uint32_t)((size_t)wq * mq * sizeof(c128) + 3 * RW * sizeof(int)));
            rs_st_release_remote(rs_mapa(smem_u32(&ready[rank]), (uint32_t)(q % ncl)), q);
        }
    };

    if (np > 0 && rank == 0) panel_factor(0);            // the first panel has nothing to hide behind
    if (np > 0 && rank != 0 && tid == 0) {               // (ready[] = 0 everywhere since before the start-up cluster barrier)
        const int wq = min(RW, ne);
        mbar_expect_tx(bar_full, (uint32_t)((size_t)wq * n * sizeof(c128) + 3 * RW * sizeof(int)));
    }
    if (ncl > 1) rs_cluster_sync();                      // every receiver is armed for panel 0
    for (int p = 0; p < np; ++p) {
        const int owner = p % ncl;
        const int lcp = (p / ncl) * RW;
        if (rank == owner) {
            panel_publish(p);
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
            __syncthreads();
            // ================= R2 and, off the critical path, the catch-up: warp 15 ships the panel -- next owner first, each
            // CTA as soon as it has declared its panel buffer free -- while warps 0-14 do the part of the PREVIOUS step that
            // this CTA put off while it factored panel p (panel p-1 through its columns right of block p); then panel p goes
            // into this CTA's own panel buffer
            if (warp == RS_T / 32 - 1) {
                if (ncl > 1) ship(p, 1, ncl);
            } else if (p > 0) {
                swap_solve(p - 1, lcp + RW, my_cols, 0, RS_T - 32);
                asm volatile("bar.sync 5, %0;" ::"r"(RS_T - 32) : "memory");
                rank8_update(p - 1, lcp + RW, my_cols, 0, RS_T / 32 - 1);
            }
            __syncthreads();
            panel_to_lbuf(p);
            panel_export(p);
            __syncthreads();
        } else {
            mbar_wait(bar_full, full_parity); full_parity ^= 1;
        }
        const int tl0 = (p >= rank) ? ((p - rank) / ncl + 1) * RW : 0;          // first local column right of block p
        if (p + 1 < np && (p + 1) % ncl == rank) {
            // ---- LOOK-AHEAD: this CTA owns the next panel, whose factorisation is the critical path (8 dependent pivot
            // steps): it brings that block (local columns [tl0, tl0+8)) up to date and factors it at once, with the SM to
            // itself; panel p's update of its other columns waits until panel p+1 has been shipped (above).
            swap_solve(p, tl0, tl0 + RW, 0, RS_T);
            __syncthreads();
            rank8_update(p, tl0, tl0 + RW, 0, RS_T / 32);
            __syncthreads();
            panel_factor(p + 1);
        } else {
            swap_solve(p, tl0, my_cols, 0, RS_T);
            __syncthreads();
            rank8_update(p, tl0, my_cols, 0, RS_T / 32);
            __syncthreads();
            declare_free(p + 1);
        }
        __syncthreads();
    }
    // ================= K5: the trailing k x k block -> global memory, inverted by rank 0
    for (int e = tid; e < my_cols * k; e += RS_T) {
        const int lc = e / k, r = e % k, g = gcol(lc);
        if (g >= ne && g < n) A[(size_t)(ne + r) + (size_t)g * n] = Aloc[(size_t)lc * ld + ne + r];
    }
    if (ncl > 1) { __threadfence(); rs_cluster_sync(); } else __syncthreads();
    if (rank == 0) {
        c128* S = reinterpret_cast<c128*>(rsm + 8192);
        if (k <= 32 && k * k <= 4 * RS_T) final_inverse_small<RS_T>(A, n, k, tau + (size_t)item * k * k, inf, S, reinterpret_cast<int*>(rsm));
        else final_inverse_body<RS_T>(A, n, k, tau + (size_t)item * k * k, inf, S, *reinterpret_cast<K5Shared*>(rsm));
    }
    if (ncl > 1) rs_cluster_sync();             // no CTA leaves while its shared memory may still be a copy target
}

// smallest cluster whose CTAs can hold the matrix (0: none)
int resident_cluster_size(int n, int k) {
    if (n < 1 || n > RS_PT || k < 1 || k > n || 8192 + (size_t)k * k * sizeof(c128) > 160 * 1024) return 0;
    for (int cl = 1; cl <= 8; cl *= 2)
        if (res_layout(n, cl).total <= RS_SMEM_MAX && 8192 + (size_t)k * k * sizeof(c128) <= res_layout(n, cl).total) return cl;
    return 0;
}

int init_attrs_resident() {
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_lu_resident, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)RS_SMEM_MAX));
    return 0;
}

// cluster launch configuration shared by the launcher and the occupancy query
static void cluster_config(cudaLaunchConfig_t& cfg, cudaLaunchAttribute* at, unsigned grid, unsigned threads, size_t smem, int cl, cudaStream_t st) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(threads); cfg.dynamicSmemBytes = smem; cfg.stream = st;
    at[0].id = cudaLaunchAttributeClusterDimension; at[0].val.clusterDim.x = (unsigned)cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
}

int resident_max_active_clusters(int cl) {
    cudaLaunchConfig_t cfg; cudaLaunchAttribute at[1];
    cluster_config(cfg, at, (unsigned)cl, RS_T, RS_SMEM_MAX, cl, nullptr);
    int nclu = 0;
    if (cudaOccupancyMaxActiveClusters(&nclu, k_lu_resident, &cfg) != cudaSuccess) { cudaGetLastError(); return 0; }
    return nclu;
}

int launch_lu_resident(c128* base, size_t stride, int n, int k, int batch, int cl, int* piv, c128* tau, int* info, cudaStream_t st,
                       int* enqueued) {
    if (enqueued) *enqueued = 0;
    const int cl_min = resident_cluster_size(n, k);
    if (cl_min == 0 || cl < cl_min || (cl != 1 && cl != 2 && cl != 4 && cl != 8)) return -1;
    const size_t smem = res_layout(n, cl).total;
    for (int b0 = 0; b0 < batch; b0 += 16384) {
        const int nb = batch - b0 < 16384 ? batch - b0 : 16384;
        cudaLaunchConfig_t cfg; cudaLaunchAttribute at[1];
        cluster_config(cfg, at, (unsigned)(nb * cl), RS_T, smem, cl, st);
        LSMS_CUDA_OK(cudaLaunchKernelEx(&cfg, k_lu_resident, base + (size_t)b0 * stride, stride, n, k, piv + (size_t)b0 * n,
                                        tau + (size_t)b0 * k * k, info + b0));
        LSMS_LAUNCH_CHECK();
        if (enqueued) *enqueued = b0 + nb;
    }
    return 0;
}

}  // namespace lsms
