// panel.cu -- K2 of the lock-step schedule: one CTA per matrix runs panel_body (panel_body.cuh) on the inner panel
// [c0, c0+w) of every item of the batch.
#include "common.cuh"
#include "internal.h"
#include "panel_body.cuh"

namespace lsms {

template <int THREADS, int R, int S>
__global__ void __launch_bounds__(THREADS, (THREADS <= 256) ? 2 : 1)
k_panel_reg(c128* __restrict__ base, size_t stride, int n, int J, int Wout, int c0, int w, int ne,
            int* __restrict__ piv, int* __restrict__ info) {
    __shared__ PanelShared sh;
    panel_body<THREADS, R, S>(base + (size_t)blockIdx.x * stride, n, J, Wout, c0, w, ne, piv + (size_t)blockIdx.x * n,
                              info + blockIdx.x, sh);
}

template <int THREADS, int R, int S>
static int launch_one(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                      cudaStream_t st) {
    k_panel_reg<THREADS, R, S><<<batch, THREADS, 0, st>>>(base, stride, n, J, Wout, c0, w, ne, piv, info);
    LSMS_LAUNCH_CHECK();
    return 0;
}

// variant: 0 = half-SM footprint (256 threads x <= 128 registers, co-resident with a Schur-update CTA),
//          1 = full-SM footprint (512 threads), wider sub-panels for the same panel height.
int launch_panel_reg(c128* base, size_t stride, int n, int J, int Wout, int c0, int w, int ne, int batch, int* piv, int* info,
                     int variant, cudaStream_t st) {
    if (w < 1 || w > P2_MAXW || Wout > P2_MAXOUT) return -1;
    const int m = n - c0;
#define LSMS_P2(T, R, S) return launch_one<T, R, S>(base, stride, n, J, Wout, c0, w, ne, batch, piv, info, st)
    // sub-panel width S <= 4: the column threads of step 4 hold 2*S more values beside the sub-panel
    if (m <= 256) LSMS_P2(256, 1, 4);
    if (m <= 512) LSMS_P2(256, 2, 4);
    if (m <= 1280) LSMS_P2(256, 5, 4);
    if (variant == 0) {
        if (m <= 2560) LSMS_P2(256, 10, 2);
        if (m <= 5120) LSMS_P2(256, 20, 1);
    }
    if (m <= 2560) LSMS_P2(512, 5, 4);
    if (m <= 5120) LSMS_P2(512, 10, 2);
    if (m <= 10240) LSMS_P2(512, 20, 1);
    if (m <= 16384) LSMS_P2(512, 32, 1);
#undef LSMS_P2
    return -1;
}

#ifdef LSMS_PANEL_TIMING
extern "C" int lsms_work_panel_cycles(unsigned long long* out_host, int reset) {
    if (out_host) cudaMemcpyFromSymbol(out_host, g_panel_cyc, sizeof(unsigned long long) * 8);
    if (reset) { unsigned long long z[8] = {0}; cudaMemcpyToSymbol(g_panel_cyc, z, sizeof(z)); }
    return 0;
}
#endif

}  // namespace lsms
