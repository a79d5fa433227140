// gemm.cu -- K4: the trailing Schur-complement update A22 <- A22 - L21 * U12,
// the contraction in which "more than 90% of the computing time" goes.
//
// complex128 GEMM on the FP64 tensor path: PTX mma.sync.m8n8k4.f64 -> SASS DMMA.8x8x4 (tcgen05 has
// no f64 kind, so the warp-level DMMA is the FP64 tensor instruction on sm_100a).  One complex MAC =
// 4 real MMAs:  Cr += Ar*(-Br) + Ai*Bi ;  Ci += Ar*(-Bi) + Ai*(-Br)   (so that C -= A*B).
// Operand tiles are staged into shared memory by the TMA engine (cp.async.bulk, one bulk copy per
// tile column, completion on an mbarrier) in a 2- or 1-stage ring (see launch_schur_gemm).
// A and B are read where the LU left them (column-major, interleaved complex), C lives in the
// accumulators: it is loaded once, updated over the whole inner dimension, stored once.
#include "common.cuh"
#include "internal.h"
#include "gemm_body.cuh"

namespace lsms {

template <int STAGES, int BN, bool TRI>
__global__ void __launch_bounds__(BN * 4, (STAGES == 1 ? 6 : 4) * 128 / (BN * 4))
k_schur_gemm(GemmShape g, int tiles_m) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    c128* ring = reinterpret_cast<c128*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(smem_raw + (size_t)STAGES * stage_elems<BN>() * sizeof(c128));
    const int tm = blockIdx.x % tiles_m, tn = blockIdx.x / tiles_m;
    const int m0 = tm * BM, n0 = tn * BN;
    const int mvalid = min(BM, g.Mr - m0), nvalid = min(BN, g.Nc - n0);
    const c128* A = g.A + (size_t)blockIdx.y * g.strideA + m0;                        // A(m0, 0)
    const c128* B = g.B + (size_t)blockIdx.y * g.strideB + (size_t)n0 * g.ldB;        // B(0, n0)
    c128* C = g.C + (size_t)blockIdx.y * g.strideC + m0 + (size_t)n0 * g.ldC;         // C(m0, n0)
    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(&full[s], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    uint32_t cc = 0;
    gemm_tile<STAGES, BN, TRI>(g, A, B, C, mvalid, nvalid, ring, full, cc);
}

template <int STAGES, int BN, bool TRI>
static int launch_classic(const GemmShape& g, cudaStream_t st) {
    const int tiles_m = (g.Mr + BM - 1) / BM, tiles_n = (g.Nc + BN - 1) / BN;
    for (int b0 = 0; b0 < g.batch; b0 += 65535) {
        GemmShape h = g;
        h.A = g.A + (size_t)b0 * g.strideA; h.B = g.B + (size_t)b0 * g.strideB; h.C = g.C + (size_t)b0 * g.strideC;
        h.batch = g.batch - b0 < 65535 ? g.batch - b0 : 65535;
        dim3 grid((unsigned)(tiles_m * tiles_n), (unsigned)h.batch);
        k_schur_gemm<STAGES, BN, TRI><<<grid, BN * 4, gemm_smem<STAGES, BN>(), st>>>(h, tiles_m);
        LSMS_LAUNCH_CHECK();
    }
    return 0;
}

// Tile shapes.  K > 16 (Schur updates, triangular solve as GEMM): 64 x 32 tiles, 4 warps, 2-stage ring (54 KB), FOUR
// CTAs per SM.  Why four small CTAs: ptxas keeps the two products of an accumulator four DMMAs apart whatever the
// source order, and a warp then waits on the DMMA result, so the pipe needs about 3.4 warps per scheduler to stay
// full (measured: 8 warps per SM reach 21.8 of 36.9 TFLOP/s, 16 warps 34.1).  With two 8-warp CTAs per SM the pipe
// therefore starves whenever one of them loads or stores its C tile (92 % DMMA-active); with four 4-warp CTAs three
// are still in their main loop: 34.6 TFLOP/s.  K <= 16 (rank-IB updates inside an outer panel, bound by the C-tile
// traffic): the same 64 x 32 tiles with one ring stage (6.2 -> 4.9 ms per P step against 64 x 64 tiles) and SIX CTAs per
// SM (80 registers, 27 KB): each CTA is one load -> 4 k-steps -> store chain, so more of them in flight hide more of the
// C-tile latency (4.9 -> 4.4 ms per P step, 9.6 -> 8.9 on C).  Tried and dropped: a one-DMMA-per-accumulator loop body with operands picked by 64-bit loads
// (31.7 TFLOP/s, bank-conflicted LDS.64) and a persistent one-CTA-per-SM variant with the next C tile prefetched
// into shared memory (23.3 TFLOP/s).
int init_attrs_gemm() {
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_schur_gemm<1, 32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gemm_smem<1, 32>()));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_schur_gemm<2, 32, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gemm_smem<2, 32>()));
    LSMS_CUDA_OK(cudaFuncSetAttribute(k_schur_gemm<2, 32, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)gemm_smem<2, 32>()));
    return 0;
}

int launch_schur_gemm(const GemmShape& g, cudaStream_t st) {
    if (g.Mr <= 0 || g.Nc <= 0 || g.K <= 0 || g.batch <= 0) return 0;
    if (g.K <= KS) return launch_classic<1, 32, false>(g, st);
    if (g.triA && g.Mr <= BM) return launch_classic<2, 32, true>(g, st);
    return launch_classic<2, 32, false>(g, st);
}

}  // namespace lsms
