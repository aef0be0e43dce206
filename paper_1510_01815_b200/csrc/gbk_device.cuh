// Device helpers shared by the kernels of libgbk (CUDA side only): packed-FP32 arithmetic for
// Blackwell (fma.rn.f32x2 / mul.rn.f32x2 -> FFMA2 / FMUL2: two FP32 lanes per issued instruction),
// the approximate MUFU functions, the arctangent polynomial and the multiply-high division.
#pragma once
#include <cuda_runtime.h>

namespace gbk {
namespace {

typedef unsigned long long u64;  // two packed floats {lo, hi}

// Bounds checks of the shared-memory indexing, compiled in with -DGBK_DEBUG_BOUNDS only (the pool
// this was developed on has compute-sanitizer closed, so the checks a memcheck run would do are
// written out at the sites that index with run-time strides): a violation traps, the launch fails
// and every test that follows reports a CUDA error.
#ifdef GBK_DEBUG_BOUNDS
#define GBK_CHECK(cond) do { if (!(cond)) __trap(); } while (0)
#else
#define GBK_CHECK(cond) do { } while (0)
#endif

__device__ __forceinline__ u64 pk(float lo, float hi) {
  u64 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ u64 pk1(float v) { return pk(v, v); }
__device__ __forceinline__ void upk(u64 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ u64 fma2(u64 a, u64 b, u64 c) {
  u64 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}
__device__ __forceinline__ u64 mul2(u64 a, u64 b) {
  u64 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ u64 add2(u64 a, u64 b) {
  u64 r;
  asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float lg2_approx(float x) {
  float y;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rsqrt_approx(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float sqrt_approx(float x) {
  float y;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
  float y;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
__host__ __device__ __forceinline__ int round_up4(int v) { return (v + 3) & ~3; }

// n / d by multiply-high: exact for n * d < 2^32 (indices inside one tile).  d = 1 has no 32-bit
// magic number (it would be 2^32) and is passed through.
__device__ __forceinline__ unsigned div_magic(int d) { return d > 1 ? 0xFFFFFFFFu / (unsigned)d + 1u : 0u; }
__device__ __forceinline__ int div_fast(int n, unsigned magic) {
  return magic ? (int)__umulhi((unsigned)n, magic) : n;
}

// Order-preserving map float -> int (and back: it is an involution), for redux.sync min / max.
__device__ __forceinline__ int ordered_key(float f) {
  const int i = __float_as_int(f);
  return i ^ ((i >> 31) & 0x7fffffff);
}
__device__ __forceinline__ float ordered_float(int k) { return __int_as_float(k ^ ((k >> 31) & 0x7fffffff)); }

__device__ __forceinline__ float f_inf() { return __int_as_float(0x7f800000); }
__device__ __forceinline__ float f_nan() { return __int_as_float(0x7fc00000); }

// atan(z) for z in [0, 1] as z * P(z^2) (8 terms, max error 1.4e-7 rad evaluated in FP32;
// DESIGN.md "Precision"), packed for a pixel pair.
__device__ __forceinline__ u64 atan01_2(u64 z) {
  const u64 t = mul2(z, z);
  u64 p = pk1(-0.00405439967289567f);
  p = fma2(p, t, pk1(0.02186231128871441f));
  p = fma2(p, t, pk1(-0.05591132491827011f));
  p = fma2(p, t, pk1(0.09642117470502853f));
  p = fma2(p, t, pk1(-0.13908594846725464f));
  p = fma2(p, t, pk1(0.1994655877351761f));
  p = fma2(p, t, pk1(-0.33329859375953674f));
  p = fma2(p, t, pk1(0.9999993443489075f));
  return mul2(p, z);
}

}  // namespace
}  // namespace gbk
