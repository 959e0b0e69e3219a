// hsg_prim.cuh — the hardware primitives the arithmetic of hsg_math.cuh is written in: individually rounded IEEE-754
// binary32 operations on one value (float) or on two values at once (F2, the packed f32x2 instructions of sm_100), the
// approximate reciprocal / reciprocal-square-root seeds.  Everything in hsg_math.cuh is plain C++ over these and over
// the compiler's __fmaf_rn-style intrinsics, so that tests/test_device_math_on_host.py can compile the very same move
// templates for the host, against a host restatement of THIS file, and compare them with the serial reference bit for bit.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace hsg {

// number types: float and the packed pair F2
struct F2 { unsigned long long v; };     // two binary32 lanes (lo, hi) in an aligned register pair

__device__ __forceinline__ F2 make_f2(float lo, float hi) {
  F2 r;
  asm("mov.b64 %0, {%1,%2};" : "=l"(r.v) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ float f2_lo(F2 a) { float lo, hi; asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); return lo; }
__device__ __forceinline__ float f2_hi(F2 a) { float lo, hi; asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v)); return hi; }

// the rounded operations
__device__ __forceinline__ float fma_rn(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ float mul_rn(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float add_rn(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float sub_rn(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float neg(float a) { return -a; }
__device__ __forceinline__ F2 fma_rn(F2 a, F2 b, F2 c) { F2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d.v) : "l"(a.v), "l"(b.v), "l"(c.v)); return d; }
__device__ __forceinline__ F2 mul_rn(F2 a, F2 b) { F2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ F2 add_rn(F2 a, F2 b) { F2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
__device__ __forceinline__ F2 sub_rn(F2 a, F2 b) { F2 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d.v) : "l"(a.v), "l"(b.v)); return d; }
// (a float negation of both lanes: ptxas folds it into the operand modifier of the consuming packed instruction)
__device__ __forceinline__ F2 neg(F2 a) { return make_f2(-f2_lo(a), -f2_hi(a)); }
// approximate seeds of div_rn / sqrt_rn (any seed within 2^-21 relative gives the same correctly rounded result)
__device__ __forceinline__ float rcp_approx(float b) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(b)); return r; }
__device__ __forceinline__ float rsqrt_approx(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }


// special-function unit approximations of the fast-math heat-bath VARIANT only (HSG_FLAG_FAST_MATH, hb_draw_fast): PTX ISA
// error bounds — ex2: 2^-22 relative; lg2: 2^-22 absolute for arguments in (0.5, 2), 2^-22 relative otherwise;
// sin, cos: 2^-20.5 absolute on [-pi, pi] (hb_draw_fast keeps the argument there); sqrt: 2^-23 relative
__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float lg2_approx(float x) { float y; asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sin_approx(float x) { float y; asm("sin.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float cos_approx(float x) { float y; asm("cos.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float sqrt_approx(float x) { float y; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

}  // namespace hsg
