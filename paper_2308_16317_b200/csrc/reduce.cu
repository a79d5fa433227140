// reduce.cu -- SURVEY.md 8(f) f4: the tau part of the energy-contour integral of eq. (2)/(3),
//   out_a = sum_q w_q tau00_{a,q}   for every central atom a (batch index = a * n_energies + q, reading A19).
// The step right after the hot path: a batched reduction over the energy axis of the k x k outputs.  HBM-bound
// on reading tau00 once (16 * n_atoms * n_energies * k^2 bytes; 1 MB for workload P) -- i.e. launch-bound.
#include "common.cuh"
#include "internal.h"

namespace lsms {

constexpr int RED_THREADS = 128;

__global__ void __launch_bounds__(RED_THREADS)
k_contour_sum(const c128* __restrict__ tau, const c128* __restrict__ w, int n_e, int kk, c128* __restrict__ out) {
    extern __shared__ __align__(16) unsigned char red_smem[];
    c128* ws = reinterpret_cast<c128*>(red_smem);
    for (int q = threadIdx.x; q < n_e; q += RED_THREADS) ws[q] = w[q];
    __syncthreads();
    const int e = blockIdx.x * RED_THREADS + threadIdx.x;
    if (e >= kk) return;
    const c128* t = tau + (size_t)blockIdx.y * n_e * kk + e;       // consecutive threads read consecutive elements
    c128 acc = cmake(0.0, 0.0);
    for (int q = 0; q < n_e; ++q) cfma(acc, ws[q], t[(size_t)q * kk]);
    out[(size_t)blockIdx.y * kk + e] = acc;
}

int launch_contour_sum(const c128* tau, const c128* w, int n_atoms, int n_e, int kk, c128* out, cudaStream_t st) {
    for (int a0 = 0; a0 < n_atoms; a0 += 65535) {
        const int na = n_atoms - a0 < 65535 ? n_atoms - a0 : 65535;
        dim3 grid((kk + RED_THREADS - 1) / RED_THREADS, na);
        k_contour_sum<<<grid, RED_THREADS, (size_t)n_e * sizeof(c128), st>>>(tau + (size_t)a0 * n_e * kk, w, n_e, kk, out + (size_t)a0 * kk);
        LSMS_LAUNCH_CHECK();
    }
    return 0;
}

}  // namespace lsms
