// static_scratch.cu -- lsms_tau00_onchip_static_scratch (include/lsms_tau.h): tau^{00} of a batch of small LIZ matrices
// (eq. (4), :62) for callers that have no device memory to give the library as workspace and no way to get any.
//
// Who that is.  The paper's callers are Fortran MPI ranks that reach CUDA through a thin C interface and share one GPU,
// several ranks per device.  Such a rank typically sizes its device buffers once, at start-up, to
// fill its share of the GPU; inside the energy loop it has nothing left over, a cudaMalloc there may fail because the
// neighbouring ranks hold the rest of the memory, and cudaMalloc / cudaFree stall the device for every rank on it.  The
// same goes for a host code whose device memory is owned by another runtime (an OpenACC / OpenMP data region, a pool
// allocator) that hands out the matrices and the result blocks but has no call for "a little extra".
//
// What this file does about it.  The on-chip elimination kernel (resident.cu, k_lu_resident) needs, besides its input
// matrices and its outputs, one word of global memory per matrix row for the pivot vector.  Every other entry point takes
// that from the caller's workspace.  Here it lives in a fixed array inside the library image, below, so the caller passes
// inputs and outputs only and the call itself allocates nothing: no cudaMalloc, no cudaFree, no stream, event or handle.
//
// The price.  LSMS_STATIC_SCRATCH_WORDS * 4 bytes = 256 KB of device memory are taken on every GPU on which this
// library is loaded, from the moment its device code is loaded until the process exits, used or not.  batch * n must not
// exceed LSMS_STATIC_SCRATCH_WORDS.  All calls on a device -- from any host thread, on any stream -- use the SAME array,
// so two of them that run on the GPU at the same time write over each other's pivot words: keep them on one stream, or
// order them with events.  The array keeps whatever the last call left there; the kernel writes a matrix's pivot words
// before anything reads them, so there is nothing to clear between calls.
#include <mutex>
#include "../../include/lsms_tau.h"
#include "common.cuh"
#include "internal.h"

namespace lsms {

// The scratch itself.  In device code this name is the array.  In HOST code the same name is only a stand-in the runtime
// uses to look the array up: it is not a device address and must never be handed to a kernel -- the kernel would fault,
// or, on a system where the GPU can reach host memory, quietly scribble over host memory instead.  The device address
// is asked for once per device with cudaGetSymbolAddress (device_setup below), and that is what the kernel gets.
static __device__ __align__(256) int g_static_pivots[LSMS_STATIC_SCRATCH_WORDS];

constexpr int SS_MAX_DEVICES = 64;
struct DeviceSetup { int* pivots = nullptr; bool ready = false; };
static DeviceSetup g_setup[SS_MAX_DEVICES];
static std::mutex g_setup_mutex;

// Once per device, with that device current: the array's address ON THAT DEVICE (every device that loads the library has
// its own copy at its own address) and the kernel's opt-in to its shared-memory size.  Neither allocates device memory
// through the runtime's allocator; the first of them makes the runtime load this library's device code on the device if
// no earlier call has, which is why the first call on a device belongs before any stream capture.
static int device_setup(int dev, int** pivots_out) {
    if (dev < 0 || dev >= SS_MAX_DEVICES) return (int)cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    DeviceSetup& s = g_setup[dev];
    if (!s.ready) {
        int* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_static_pivots);
        if (e != cudaSuccess) { cudaGetLastError(); return (int)e; }
        if (!p) return (int)cudaErrorInvalidSymbol;
        int rc = init_attrs_resident();
        if (rc) { cudaGetLastError(); return rc; }
        s.pivots = p; s.ready = true;
    }
    *pivots_out = s.pivots;
    return 0;
}

}  // namespace lsms

using namespace lsms;

extern "C" int lsms_tau00_onchip_static_scratch(lsms_c128* M, int n_sites, int kmax, int spin_canted, int batch,
                                                lsms_c128* tau00_out, int* info, void* cuda_stream) {
    auto aligned16 = [](const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15) == 0; };
    if (!M || !aligned16(M)) return -1;
    if (n_sites < 1) return -2;
    int lp1 = 1; while (lp1 * lp1 < kmax) ++lp1;
    if (kmax < 1 || kmax > 81 || lp1 * lp1 != kmax) return -3;
    if (batch < 1) return -5;
    if (!tau00_out || !aligned16(tau00_out)) return -6;
    if (!info) return -7;
    const int k = kmax * (spin_canted ? 2 : 1);
    const long long n = (long long)n_sites * k;
    // the two size limits, checked on the host before any CUDA call: the matrix must fit on chip, and the batch's pivot
    // vectors must fit in the built-in array
    const int cl = n <= 46340 ? resident_cluster_size((int)n, k) : 0;
    if (cl == 0) return LSMS_ERR_NOT_ON_CHIP;
    if (n * batch > (long long)LSMS_STATIC_SCRATCH_WORDS) return LSMS_ERR_STATIC_SCRATCH_TOO_SMALL;
    int dev = -1;
    LSMS_CUDA_OK(cudaGetDevice(&dev));
    int* pivots = nullptr;
    int rc = device_setup(dev, &pivots);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    LSMS_CUDA_OK(cudaMemsetAsync(info, 0, (size_t)batch * sizeof(int), st));     // info is an output: cleared like everywhere else
    return launch_lu_resident((c128*)M, (size_t)n * n, (int)n, k, batch, cl, pivots, (c128*)tau00_out, info, st);
}
