// internal.h -- host-side launchers shared between the translation units of liblsms_tau.so.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include "common.cuh"

namespace lsms {

// assemble.cu
size_t gaunt_table_bytes(int lmax);
double gaunt_closed_form_host(int l, int m, int lp, int mp, int lpp);
int launch_tinv(const c128* delta, const int* species, const c128* z, int lmax, int n_sites, int nspin, int batch,
                c128* tinv, c128* kappa, cudaStream_t st);
int launch_assemble(const c128* tinv, const double* site_pos, const double* moment, const c128* kappa, int lmax,
                    int n_sites, int canted, int batch, c128* M, void* ws, cudaStream_t st);

// gemm.cu -- K4: C[Mr x Nc] -= A[Mr x K] * B[K x Nc] inside the same column-major matrices (ld = n)
struct GemmShape {
    c128* base;            // item 0 of the batch
    size_t batch_stride;   // elements between items
    int ld;                // leading dimension (= n)
    int Mr, Nc, K;         // C is Mr x Nc, inner dimension K
    size_t offA, offB, offC;   // element offsets of A(0,0), B(0,0), C(0,0) inside an item
    int batch;
};
int launch_schur_gemm(const GemmShape& g, cudaStream_t st);

// lu.cu -- K2, K3, K5 and the verification back-substitution
int launch_panel(c128* base, size_t stride, int n, int c0, int w, int ne, int batch, int* piv, int* info, cudaStream_t st);
int launch_swap_trsm(c128* base, size_t stride, int n, int c0, int w, int col_lo, int col_hi, int mode /*1 swap | 2 trsm*/, int batch,
                     const int* piv, cudaStream_t st);
int launch_final_inverse(c128* base, size_t stride, int n, int k, int batch, c128* tau, int* info, void* ws, cudaStream_t st);
int launch_backsolve_central(const c128* LU, size_t stride, int n, int k, int batch, const c128* tau, c128* X, cudaStream_t st);
size_t final_inverse_ws_bytes(int k, int batch);

// probe.cu
int run_peak_probe(int which, int iters, double* tflops, cudaStream_t st);

}  // namespace lsms
