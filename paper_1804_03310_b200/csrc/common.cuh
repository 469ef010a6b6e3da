// common.cuh -- small device helpers shared by the ph-AFQMC kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <math.h>

namespace afq {

template <typename T> struct __align__(2 * sizeof(T)) cplx { T x, y; };
typedef cplx<double> zcplx;

template <typename T> __host__ __device__ __forceinline__ cplx<T> mk(T a, T b) { cplx<T> r; r.x = a; r.y = b; return r; }
template <typename T> __device__ __forceinline__ cplx<T> cmul(cplx<T> a, cplx<T> b) {
  return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
template <typename T> __device__ __forceinline__ cplx<T> cadd(cplx<T> a, cplx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <typename T> __device__ __forceinline__ cplx<T> csub(cplx<T> a, cplx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <typename T> __device__ __forceinline__ void cfma(cplx<T>& acc, cplx<T> a, cplx<T> b) {
  acc.x = fma(a.x, b.x, acc.x); acc.x = fma(-a.y, b.y, acc.x);
  acc.y = fma(a.x, b.y, acc.y); acc.y = fma(a.y, b.x, acc.y);
}
template <typename T> __device__ __forceinline__ cplx<T> cinv(cplx<T> a) {
  // Smith's algorithm: no overflow of |a|^2
  if (fabs(a.x) >= fabs(a.y)) {
    T r = a.y / a.x, d = a.x + a.y * r;
    return mk<T>(T(1) / d, -r / d);
  } else {
    T r = a.x / a.y, d = a.x * r + a.y;
    return mk<T>(r / d, T(-1) / d);
  }
}
template <typename T> __device__ __forceinline__ T cabs2(cplx<T> a) { return a.x * a.x + a.y * a.y; }
template <typename T> __device__ __forceinline__ zcplx to_z(cplx<T> a) { return mk<double>((double)a.x, (double)a.y); }

__device__ __forceinline__ zcplx zdiv(zcplx a, zcplx b) {
  if (fabs(b.x) >= fabs(b.y)) {
    double r = b.y / b.x, d = b.x + b.y * r;
    return mk<double>((a.x + a.y * r) / d, (a.y - a.x * r) / d);
  } else {
    double r = b.x / b.y, d = b.x * r + b.y;
    return mk<double>((a.x * r + a.y) / d, (a.y * r - a.x) / d);
  }
}

// Round an FP32 value to TF32 (10-bit mantissa), round-to-nearest-even on the dropped 13 bits.
// The tensor pipe ignores the low 13 bits of a kind::tf32 operand, so values stored this way are
// consumed exactly.  Used for the 3xTF32 hi/lo operand split.
__device__ __forceinline__ float tf32_rn(float v) {
  uint32_t u = __float_as_uint(v);
  u += 0x00000fffu + ((u >> 13) & 1u);
  u &= 0xffffe000u;
  return __uint_as_float(u);
}
__device__ __forceinline__ void tf32_split(float v, float& hi, float& lo) {
  hi = tf32_rn(v);
  lo = tf32_rn(v - hi);
}

// The tensor pipe ignores the low 13 mantissa bits of a kind::tf32 operand, i.e. it consumes raw FP32 v as trunc13(v).  The
// matching low part d = v - trunc13(v) (exact, <= 13 significant bits) is itself truncated to 11 bits by the pipe; scaling it
// by 1 + 2^-11 first centres that truncation (error within +-2^-11 |d| <= 2^-21 |v|, zero mean).  One LOP3, one FADD, one
// FMUL per element: cvt.rna.tf32.f32 is a quarter-rate conversion and made the splitter warps the Taylor kernel's bottleneck.
__device__ __forceinline__ uint32_t tf32_lo_bits(uint32_t vbits) {
  const float d = __uint_as_float(vbits) - __uint_as_float(vbits & 0xffffe000u);
  return __float_as_uint(d * 1.00048828125f);
}

// The same split for values produced in registers: hi = v itself (consumed as trunc13(v)), lo = centred low part.
__device__ __forceinline__ void tf32_split_raw(float v, float& hi, float& lo) {
  hi = v;
  lo = __uint_as_float(tf32_lo_bits(__float_as_uint(v)));
}

// cp.async 16-byte global -> shared (LDGSTS)
__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
  uint32_t s = (uint32_t)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

template <typename T> __device__ __forceinline__ T warp_sum(T v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

enum { FLAG_SINGULAR = 1, FLAG_NONFINITE = 2, FLAG_KILLED = 4 };

}  // namespace afq
