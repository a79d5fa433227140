// gemm_body.cuh -- the DMMA tile of K4 (see gemm.cu for the design notes): shared by k_schur_gemm and the
// small-matrix kernel of fused.cu.
#pragma once
#include "common.cuh"
#include "internal.h"

namespace lsms {

constexpr int BM = 64, KS = 16;
constexpr int LDA_S = BM + 2;      // complex units; == 2 (mod 8): conflict-free LDS.128 of A fragments
constexpr int LDB_S = KS + 4;      // complex units; == 4 (mod 8): conflict-free LDS.128 of B fragments
constexpr int A_STAGE = KS * LDA_S;        // complex elements
// tile width BN = 64 with 256 threads (8 warps as 2 x 4) or BN = 32 with 128 threads (4 warps as 2 x 2); warp tile 32 x 16
template <int BN> __host__ __device__ constexpr int stage_elems() { return A_STAGE + BN * LDB_S; }
template <int STAGES, int BN> constexpr size_t gemm_smem() { return (size_t)STAGES * stage_elems<BN>() * sizeof(c128) + STAGES * sizeof(uint64_t); }

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
// TMA bulk copy global -> shared, completion counted in bytes on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void tma_bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b) {
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// Fill ring slot s with K-chunk kc of the A and B tiles: one bulk copy per tile column, issued by
// threads 0..KS+BN-1; thread 0 also posts the expected byte count on the slot's mbarrier.
template <int STAGES, int BN>
__device__ __forceinline__ void issue_chunk(const GemmShape& g, const c128* A, const c128* B, c128* ring, uint64_t* full,
                                            uint32_t cc0, int kc, int mvalid, int nvalid) {
    const int s = (cc0 + kc) % STAGES, t = threadIdx.x;
    const int k0 = kc * KS, kvalid = min(KS, g.K - k0);
    c128* As = ring + (size_t)s * stage_elems<BN>();
    c128* Bs = As + A_STAGE;
    if (t == 0) mbar_expect_tx(&full[s], (uint32_t)((kvalid * mvalid + nvalid * kvalid) * sizeof(c128)));
    if (t < KS) {
        if (t < kvalid)      // column k0+t of A: mvalid contiguous elements
            tma_bulk_g2s(As + t * LDA_S, A + (size_t)(k0 + t) * g.ldA, (uint32_t)(mvalid * sizeof(c128)), &full[s]);
    } else if (t < KS + BN) {
        const int nn = t - KS;
        if (nn < nvalid)     // column n0+nn of B: kvalid contiguous elements
            tma_bulk_g2s(Bs + nn * LDB_S, B + (size_t)nn * g.ldB + k0, (uint32_t)(kvalid * sizeof(c128)), &full[s]);
    }
}

// One C tile (BM x BN at (m0, n0) of the item's C) of C -= A B (or C = -(A B)) by the CTA's BN*4 threads: operands staged
// by TMA bulk copies into the ring, C in the accumulators.  `cc` counts the K-chunks this CTA has pushed through the
// ring since its mbarriers were initialised (slot = cc % STAGES, parity = (cc / STAGES) & 1), so that a persistent
// CTA can call this for tile after tile; the caller separates two calls by a __syncthreads() (ring reuse).
// Used by k_schur_gemm (one tile per CTA, cc = 0) and by the small-matrix kernel of fused.cu.
// TRI: A is LOWER TRIANGULAR with its diagonal at the tile's origin (the triangular solve as a GEMM, U12 = -(Ninv * T) with
// Ninv = -(L11^-1), one tile row): the 8-row fragment blocks of A that lie wholly above the diagonal are exact zeros and
// their DMMAs are skipped (56 % of the dense count at 64 rows); the result is unchanged.
template <int STAGES, int BN, bool TRI = false>
__device__ __forceinline__ void gemm_tile(const GemmShape& g, const c128* __restrict__ A, const c128* __restrict__ B,
                                          c128* __restrict__ C, int mvalid, int nvalid, c128* ring, uint64_t* full, uint32_t& cc) {
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int nchunks = (g.K + KS - 1) / KS;
    const uint32_t cc0 = cc;
    for (int kc = 0; kc < STAGES && kc < nchunks; ++kc) issue_chunk<STAGES, BN>(g, A, B, ring, full, cc0, kc, mvalid, nvalid);

    // C tile -> accumulators (issued before the first wait so that it overlaps the TMA fill)
    const int gq = lane >> 2, q = lane & 3;              // fragment coordinates: A[gq][q], B[q][gq], C[gq][2q..2q+1]
    const int wm = (warp & 1) * 32, wn = (warp >> 1) * 16;
    double cr[4][2][2], ci[4][2][2];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 2; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int r = wm + mt * 8 + gq, c = wn + nt * 8 + 2 * q + e;
                c128 v = cmake(0.0, 0.0);
                if (!g.beta0 && r < mvalid && c < nvalid) v = C[r + (size_t)c * g.ldC];
                cr[mt][nt][e] = v.x; ci[mt][nt][e] = v.y;
            }

    for (int kc = 0; kc < nchunks; ++kc) {
        const int s = (cc0 + kc) % STAGES;
        mbar_wait(&full[s], ((cc0 + kc) / STAGES) & 1);
        const int kvalid = min(KS, g.K - kc * KS);
        const c128* As = ring + (size_t)s * stage_elems<BN>();
        const c128* Bs = As + A_STAGE;
        const int nfull = kvalid >> 2;
#pragma unroll 1
        for (int ks = 0; ks < nfull; ++ks) {
            const int k0 = ks * 4;
            if constexpr (TRI) {
                // rows wm + mt*8 .. +7 of A are zero in columns > row: block mt is live iff its last row >= first column
                const int kglob = kc * KS + k0;
                if (wm + 31 < kglob) continue;                       // the whole 32-row warp tile lies above the diagonal
                c128 b[2];
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) b[nt] = Bs[(wn + nt * 8 + gq) * LDB_S + k0 + q];
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    if (wm + mt * 8 + 7 >= kglob) {
                        const c128 a = As[(k0 + q) * LDA_S + wm + mt * 8 + gq];
#pragma unroll
                        for (int nt = 0; nt < 2; ++nt) {
                            dmma884(cr[mt][nt][0], cr[mt][nt][1], a.x, -b[nt].x);
                            dmma884(ci[mt][nt][0], ci[mt][nt][1], a.x, -b[nt].y);
                            dmma884(cr[mt][nt][0], cr[mt][nt][1], a.y, b[nt].y);
                            dmma884(ci[mt][nt][0], ci[mt][nt][1], a.y, -b[nt].x);
                        }
                    }
                }
            } else {
                c128 a[4], b[2];
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) a[mt] = As[(k0 + q) * LDA_S + wm + mt * 8 + gq];
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) b[nt] = Bs[(wn + nt * 8 + gq) * LDB_S + k0 + q];
#pragma unroll
                for (int nt = 0; nt < 2; ++nt) {
#pragma unroll
                    for (int mt = 0; mt < 4; ++mt) {
                        dmma884(cr[mt][nt][0], cr[mt][nt][1], a[mt].x, -b[nt].x);
                        dmma884(ci[mt][nt][0], ci[mt][nt][1], a[mt].x, -b[nt].y);
                        dmma884(cr[mt][nt][0], cr[mt][nt][1], a[mt].y, b[nt].y);
                        dmma884(ci[mt][nt][0], ci[mt][nt][1], a[mt].y, -b[nt].x);
                    }
                }
            }
        }
        if (kvalid & 3) {                      // ragged K tail: fragments beyond kvalid are zeroed
            const int k0 = nfull * 4;
            const bool live = (k0 + q) < kvalid;
            c128 a[4], b[2];
#pragma unroll
            for (int mt = 0; mt < 4; ++mt) { a[mt] = As[(k0 + q) * LDA_S + wm + mt * 8 + gq]; if (!live) a[mt] = cmake(0.0, 0.0); }
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) { b[nt] = Bs[(wn + nt * 8 + gq) * LDB_S + k0 + q]; if (!live) b[nt] = cmake(0.0, 0.0); }
#pragma unroll
            for (int nt = 0; nt < 2; ++nt) {
                const double nbr = -b[nt].x, nbi = -b[nt].y, bi = b[nt].y;
#pragma unroll
                for (int mt = 0; mt < 4; ++mt) {
                    dmma884(cr[mt][nt][0], cr[mt][nt][1], a[mt].x, nbr);
                    dmma884(ci[mt][nt][0], ci[mt][nt][1], a[mt].x, nbi);
                    dmma884(cr[mt][nt][0], cr[mt][nt][1], a[mt].y, bi);
                    dmma884(ci[mt][nt][0], ci[mt][nt][1], a[mt].y, nbr);
                }
            }
        }
        if (kc + STAGES < nchunks) {          // refill this slot once every warp is done with it
            __syncthreads();
            issue_chunk<STAGES, BN>(g, A, B, ring, full, cc0, kc + STAGES, mvalid, nvalid);
        }
    }

#pragma unroll
    for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 2; ++nt)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int r = wm + mt * 8 + gq, c = wn + nt * 8 + 2 * q + e;
                if (r < mvalid && c < nvalid) C[r + (size_t)c * g.ldC] = cmake(cr[mt][nt][e], ci[mt][nt][e]);
            }
    cc = cc0 + (uint32_t)nchunks;
}

}  // namespace lsms
