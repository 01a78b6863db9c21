// common.cuh -- shared by the CUDA translation units of libkspw.so (never by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <cstdio>
#include <cstdint>
#include <string>

typedef double2 cplx;   // (re, im), 16-byte aligned

__host__ __device__ __forceinline__ cplx cmake(double a, double b) { return make_double2(a, b); }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return make_double2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return make_double2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {  // a * conj(b)
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
__device__ __forceinline__ cplx cconj(cplx a) { return make_double2(a.x, -a.y); }
__device__ __forceinline__ cplx cscale(double s, cplx a) { return make_double2(s * a.x, s * a.y); }
__device__ __forceinline__ cplx cfma(cplx a, cplx b, cplx c) {  // a*b + c
  return make_double2(fma(a.x, b.x, fma(-a.y, b.y, c.x)), fma(a.x, b.y, fma(a.y, b.x, c.y)));
}

#define KS_OK 0
#define KS_NOTCONV 1
#define KS_EINVAL -1
#define KS_EGRID -2
#define KS_ENOMEM -3
#define KS_ECUDA -4
#define KS_EVLOC -5

// thread-local text of the last failure outside a context
std::string& ks_global_error();

#define KS_CUDA_CHECK(expr, errstr)                                                          \
  do {                                                                                       \
    cudaError_t e__ = (expr);                                                                \
    if (e__ != cudaSuccess) {                                                                \
      char b__[512];                                                                         \
      snprintf(b__, sizeof b__, "%s:%d %s: %s", __FILE__, __LINE__, #expr, cudaGetErrorString(e__)); \
      (errstr) = b__;                                                                        \
      return (e__ == cudaErrorMemoryAllocation) ? KS_ENOMEM : KS_ECUDA;                      \
    }                                                                                        \
  } while (0)

static inline int ceil_div(long a, long b) { return (int)((a + b - 1) / b); }
