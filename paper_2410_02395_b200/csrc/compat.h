// compat.h -- lets the kernel bodies compile both under nvcc (device code, the product) and under a
// plain host C++ compiler (tests/host_emulation_test.cpp: one std::thread per CUDA thread, used only
// to check index arithmetic on a machine without a GPU; it is not a CPU fallback and is not linked
// into the library).
#pragma once

#ifdef __CUDACC__
#include <cuda_runtime.h>
#define MBS_DEV __device__ __forceinline__
#define MBS_HD __host__ __device__ __forceinline__
#define MBS_SYNC() __syncthreads()
#define MBS_RESTRICT __restrict__
#else
#include <cmath>
struct float2 { float x, y; };
struct double2 { double x, y; };
static inline float2 make_float2(float x, float y) { float2 r; r.x = x; r.y = y; return r; }
static inline double2 make_double2(double x, double y) { double2 r; r.x = x; r.y = y; return r; }
#define MBS_DEV inline
#define MBS_HD inline
void mbs_host_barrier();
#define MBS_SYNC() mbs_host_barrier()
#define MBS_RESTRICT __restrict__
static inline float __ldg(const float* p) { return *p; }
static inline float2 __ldg(const float2* p) { return *p; }
#endif

namespace mbs {
typedef float2 cf;

MBS_HD cf cmul(cf a, cf b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// Complex add / subtract: on sm_100 one packed fp32x2 instruction (FADD2 / FFMA2) instead of two scalar
// ones -- the FFT sweeps are issue-limited, and the butterflies are mostly additions.
#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ >= 1000)
MBS_DEV cf cadd(cf a, cf b) { return __fadd2_rn(a, b); }
MBS_DEV cf csub(cf a, cf b) { return __ffma2_rn(b, make_float2(-1.f, -1.f), a); }
#else
MBS_HD cf cadd(cf a, cf b) { return make_float2(a.x + b.x, a.y + b.y); }
MBS_HD cf csub(cf a, cf b) { return make_float2(a.x - b.x, a.y - b.y); }
#endif
MBS_HD cf cswap(cf a) { return make_float2(a.y, a.x); }
MBS_HD cf cscale(cf a, float s) { return make_float2(a.x * s, a.y * s); }
// a * (-i)
MBS_HD cf cmul_mi(cf a) { return make_float2(a.y, -a.x); }
// a * (+i)
MBS_HD cf cmul_pi(cf a) { return make_float2(-a.y, a.x); }
}  // namespace mbs
