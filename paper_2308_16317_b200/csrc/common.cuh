// common.cuh -- shared device helpers for the sm_100a kernels of liblsms_tau.so.
// Complex numbers are double2 (x = re, y = im), 16-byte aligned, as in include/lsms_tau.h.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lsms {

typedef double2 c128;

__host__ __device__ __forceinline__ c128 cmake(double re, double im) { c128 r; r.x = re; r.y = im; return r; }
__host__ __device__ __forceinline__ c128 cadd(c128 a, c128 b) { return cmake(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ c128 csub(c128 a, c128 b) { return cmake(a.x - b.x, a.y - b.y); }
__host__ __device__ __forceinline__ c128 cmul(c128 a, c128 b) { return cmake(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__host__ __device__ __forceinline__ c128 cscale(double s, c128 a) { return cmake(s * a.x, s * a.y); }
__host__ __device__ __forceinline__ c128 cneg(c128 a) { return cmake(-a.x, -a.y); }
// a -= b*c
__device__ __forceinline__ void cfms(c128& a, c128 b, c128 c) {
    a.x = fma(-b.x, c.x, a.x); a.x = fma(b.y, c.y, a.x);
    a.y = fma(-b.x, c.y, a.y); a.y = fma(-b.y, c.x, a.y);
}
// a += b*c
__device__ __forceinline__ void cfma(c128& a, c128 b, c128 c) {
    a.x = fma(b.x, c.x, a.x); a.x = fma(-b.y, c.y, a.x);
    a.y = fma(b.x, c.y, a.y); a.y = fma(b.y, c.x, a.y);
}
// 1/a, scaled (Smith) so that it neither overflows nor loses accuracy for ordinary magnitudes
__device__ __forceinline__ c128 crecip(c128 a) {
    if (fabs(a.x) >= fabs(a.y)) { double r = a.y / a.x, d = a.x + a.y * r; return cmake(1.0 / d, -r / d); }
    double r = a.x / a.y, d = a.x * r + a.y; return cmake(r / d, -1.0 / d);
}
// 1/a without a division instruction, for the latency-bound pivot steps of the small-matrix kernels: a is scaled by a
// power of two taken from the exponent of |re|+|im|, so that the squared modulus d lies in [1/2, 4] for any finite
// non-zero a; 1/d = hardware seed (rcp.approx.ftz.f64, ~20 bits) + three Newton steps (6 dependent DFMAs, no special
// cases to branch on).  Within 2 ulp of crecip.  a = 0 / Inf / NaN give garbage (callers flag such pivots themselves).
__device__ __forceinline__ c128 crecip_fast(c128 a) {
    long long e = (__double_as_longlong(fabs(a.x) + fabs(a.y)) >> 52) & 0x7FF;
    e = e < 2 ? 2 : (e > 2044 ? 2044 : e);
    const double sc = __longlong_as_double((2046 - e) << 52);           // 2^(1023 - e): sc * (|re|+|im|) in [1, 2)
    const double xs = a.x * sc, ys = a.y * sc;
    const double d = fma(xs, xs, ys * ys);
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(d));
#pragma unroll
    for (int i = 0; i < 3; ++i) r = fma(r, fma(-d, r, 1.0), r);
    const double inv = r * sc;
    return cmake(xs * inv, -ys * inv);
}
__device__ __forceinline__ c128 cdiv(c128 a, c128 b) { return cmul(a, crecip(b)); }
// LAPACK's cabs1: |re| + |im| (the pivot-search magnitude of izamax)
__device__ __forceinline__ double cabs1(c128 a) { return fabs(a.x) + fabs(a.y); }

struct LaunchCounter { int n; };
extern thread_local LaunchCounter g_launches;

}  // namespace lsms

// A failed runtime call or launch leaves its code pending on the host thread; it is taken off there (cudaGetLastError)
// before it is returned, so that it is reported once, by the call that caused it, and neither a later library call nor
// the caller's own checks (torch's, say) trip over a stale code.
#define LSMS_CUDA_OK(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { cudaGetLastError(); return (int)e__; } } while (0)
#define LSMS_LAUNCH_CHECK() do { ++lsms::g_launches.n; cudaError_t e__ = cudaGetLastError(); if (e__ != cudaSuccess) return (int)e__; } while (0)
