// panel.cu -- K2 of the lock-step schedule: one CTA per matrix runs panel_body (panel_body.cuh) on the inner panel
// [c0, c0+w) of every item of the batch.
#include "common.cuh"
#include "internal.h"
#include "panel_body.cuh"

namespace lsms {

template <int THREADS, int R, int S, int DEPTH>
__global__ void __launch_bounds__(THREADS, (THREADS <= 128) ? 4 : (THREADS <= 256) ? 2 : 1)
k_panel_reg(c128* __restrict__ base, size_t stride, int n, int J, int Wout, int c0, int w, int ne,
            int* __restrict__ piv, int* __restrict__ info) {
    extern __shared__ __align__(16) unsigned char panel_stage[];
    __shared__ PanelShared sh;
    panel_body<THREADS, R, S, DEPTH>(base + (size_t)blockIdx.x * stride, n, J, Wout, c0, w, ne, piv + (size_t)blockIdx.x * n,
                                     info + blockIdx.x, sh, reinterpret_cast<c128*>(panel_stage));
}

template <int THREADS, int R, int DEPTH> constexpr size_t stage_bytes() { return (size_t)DEPTH * R * THREADS * sizeof(c128); }

template <int THREADS, int R, int S, int DEPTH>
static int launch_one(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                      cudaStream_t st) {
    k_panel_reg<THREADS, R, S, DEPTH><<<batch, THREADS, stage_bytes<THREADS, R, DEPTH>(), st>>>(base, stride, n, J, Wout, c0, w, ne, piv, info);
    LSMS_LAUNCH_CHECK();
    return 0;
}

// Instantiations (THREADS, R rows per thread, S sub-panel width, DEPTH columns in flight in step 5).  S <= 4: the column
// threads of step 4 hold 2*S more values beside the sub-panel; R*S complex numbers per thread are the sub-panel.
// DEPTH * R * THREADS * 16 B of shared memory per CTA: 160 KB for the 512-thread kernels (one CTA per SM), 80 KB for
// the 256-thread ones (two per SM), <= 32 KB for the 128-thread ones with R <= 4 (four per SM, the slot of one
// Schur-update CTA); X(128, 8, 2, 3) stages 48 KB beside ~8.6 KB of static PanelShared, so THREE of those fit an SM.
// GPU tests that reach each instance (tests/test_gpu_parity.py):
//   128-thread row, 256-thread row, <512,5,4,4>, <512,10,2,2>: test_panel_kernel_variants_match_oracle[threads = 2 / 0 / 1]
//   <512,20,1,0> (5121-10240 rows): test_tau00_full_size_against_stored_oracle_values[H_0, H_23, N_23; panel_cluster = 1],
//                                   test_tau00_high_l_small_batches_through_a_default_handle (default handle, batch 5)
//   <512,32,1,0> (> 10240 rows):    test_tau00_full_size_against_stored_oracle_values[NC_5; panel_cluster = 1]
#define LSMS_P2_LIST(X)                                                                                     \
    X(128, 1, 4, 4) X(128, 2, 4, 4) X(128, 4, 4, 4) X(128, 8, 2, 3)                                         \
    X(256, 1, 4, 4) X(256, 2, 4, 4) X(256, 5, 4, 4) X(256, 10, 2, 2) X(256, 20, 1, 0)                       \
    X(512, 5, 4, 4) X(512, 10, 2, 2) X(512, 20, 1, 0) X(512, 32, 1, 0)

int init_attrs_panel() {
#define LSMS_P2_ATTR(T, R, S, D)                                                                                        \
    if (D > 0)                                                                                                          \
        LSMS_CUDA_OK(cudaFuncSetAttribute(k_panel_reg<T, R, S, D>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)stage_bytes<T, R, D>()));
    LSMS_P2_LIST(LSMS_P2_ATTR)
#undef LSMS_P2_ATTR
    return 0;
}

// variant: 0 = half-SM footprint (256 threads x <= 128 registers), 1 = full-SM footprint (512 threads) for panels taller
// than 1280 rows: wider sub-panels for the same panel height, 2 = quarter-SM footprint (128 threads) for panels of up to
// 1024 rows: all matrices of a large batch resident at once.
int launch_panel_reg(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                     int variant, cudaStream_t st) {
    if (w < 1 || w > P2_MAXW || Wout > P2_MAXOUT) return -1;
    const int m = n - c0;
#define LSMS_P2(T, R, S, D) return launch_one<T, R, S, D>(base, stride, n, J, Wout, c0, w, ne, batch, piv, info, st)
    if (variant == 2) {
        if (m <= 128) LSMS_P2(128, 1, 4, 4);
        if (m <= 256) LSMS_P2(128, 2, 4, 4);
        if (m <= 512) LSMS_P2(128, 4, 4, 4);
        if (m <= 1024) LSMS_P2(128, 8, 2, 3);
    }
    if (m <= 256) LSMS_P2(256, 1, 4, 4);
    if (m <= 512) LSMS_P2(256, 2, 4, 4);
    if (m <= 1280) LSMS_P2(256, 5, 4, 4);
    if (variant == 0) {
        if (m <= 2560) LSMS_P2(256, 10, 2, 2);
        if (m <= 5120) LSMS_P2(256, 20, 1, 0);
    }
    if (m <= 2560) LSMS_P2(512, 5, 4, 4);
    if (m <= 5120) LSMS_P2(512, 10, 2, 2);
    if (m <= 10240) LSMS_P2(512, 20, 1, 0);
    if (m <= 16384) LSMS_P2(512, 32, 1, 0);
#undef LSMS_P2
    return -1;
}

}  // namespace lsms
