// mhd_pack.cuh -- f2: two fp32 cells in one aligned register pair, computed with the packed fp32
// instructions of sm_100a (PTX add/mul/fma.rn.f32x2 -> SASS FADD2 / FMUL2 / FFMA2).
//
// Why: the fp32 sweep kernels are bound by instruction issue, not by HBM or by the FMA pipe
// (round-1 ncu capture of the scalar kernels: ~165 of ~280 issued instructions per cell are FADD/FMUL/FFMA).
// A packed instruction occupies the FMA pipe for two cycles but only ONE issue slot
// (measured on B200 with a throw-away issue-rate loop: FFMA 3.83 warp-inst/clk/SM, FFMA2 1.97), so
// a thread that advances two adjacent pencils in f2 arithmetic issues half the floating-point
// instructions for the same flops, and its 64-bit shared-memory loads and global stores halve the
// load/store instructions too.  What has no packed form stays per lane: MUFU (rcp, sqrt), |x|, and
// the two discrete switches of the scheme (FSETP/FSEL).
//
// The arithmetic templates of mhd_device.cuh (right_left, vl_full, FluidPipe, BPipe) are written in
// terms of + - * fma_ fnma_ rcp_ sqrt_ pos_or_zero pick_pos freeze_speed, all of which are defined
// here for f2, so the SAME source is instantiated for float, double and f2.
#pragma once
#include <cuda_runtime.h>

namespace mhd {

struct f2 {
  float2 v;
  __device__ __forceinline__ f2() {}
  __device__ __forceinline__ explicit f2(float s) { v.x = s; v.y = s; }
  __device__ __forceinline__ explicit f2(double s) { v.x = (float)s; v.y = (float)s; }
  __device__ __forceinline__ explicit f2(int s) { v.x = (float)s; v.y = (float)s; }
  __device__ __forceinline__ f2(float a, float b) { v.x = a; v.y = b; }
  __device__ __forceinline__ explicit f2(float2 a) : v(a) {}
};

__device__ __forceinline__ f2 operator-(f2 a) { return f2(-a.v.x, -a.v.y); }           // folds into operand modifiers
__device__ __forceinline__ f2 operator+(f2 a, f2 b) { return f2(__fadd2_rn(a.v, b.v)); }
__device__ __forceinline__ f2 operator-(f2 a, f2 b) { return f2(__fadd2_rn(a.v, (-b).v)); }
__device__ __forceinline__ f2 operator*(f2 a, f2 b) { return f2(__fmul2_rn(a.v, b.v)); }
#ifndef MHD_F32_IEEE
__device__ __forceinline__ f2 fma_(f2 a, f2 b, f2 c) { return f2(__ffma2_rn(a.v, b.v, c.v)); }
__device__ __forceinline__ f2 fnma_(f2 a, f2 b, f2 c) { return f2(__ffma2_rn((-a).v, b.v, c.v)); }
#else
__device__ __forceinline__ f2 fma_(f2 a, f2 b, f2 c) { return f2(__fadd2_rn(__fmul2_rn(a.v, b.v), c.v)); }
__device__ __forceinline__ f2 fnma_(f2 a, f2 b, f2 c) { return f2(__fadd2_rn(__fmul2_rn((-a).v, b.v), c.v)); }
#endif

// per-lane operations (no packed form in the ISA)
__device__ __forceinline__ float rcp_(float x);
__device__ __forceinline__ float sqrt_(float x);
__device__ __forceinline__ f2 rcp_(f2 x) { return f2(rcp_(x.v.x), rcp_(x.v.y)); }
__device__ __forceinline__ f2 sqrt_(f2 x) { return f2(sqrt_(x.v.x), sqrt_(x.v.y)); }
__device__ __forceinline__ f2 abs_(f2 x) { return f2(fabsf(x.v.x), fabsf(x.v.y)); }
__device__ __forceinline__ f2 pos_or_zero(f2 s, f2 r) { return f2(s.v.x > 0.0f ? r.v.x : 0.0f, s.v.y > 0.0f ? r.v.y : 0.0f); }
__device__ __forceinline__ f2 pick_pos(f2 s, f2 a, f2 b) { return f2(s.v.x > 0.0f ? a.v.x : b.v.x, s.v.y > 0.0f ? a.v.y : b.v.y); }
// x + a b / (a + b) where a*b > 0, else x (vl_add of mhd_device.cuh): products and sums packed, the reciprocal, the test and
// the final multiply-add per lane, so that the select folds into a predicated FFMA (one instruction per lane instead of
// half an FFMA2 plus an FSEL)
__device__ __forceinline__ f2 vl_add(f2 x, f2 a, f2 b) {
  const f2 ab = a * b, s = a + b;
  const float rx = rcp_(s.v.x), ry = rcp_(s.v.y);
  f2 y = x;
  if (ab.v.x > 0.0f) y.v.x = fmaf(ab.v.x, rx, x.v.x);
  if (ab.v.y > 0.0f) y.v.y = fmaf(ab.v.y, ry, x.v.y);
  return y;
}
__device__ __forceinline__ f2 freeze_speed(f2 v, f2 t, f2 inv) {
  return f2(fabsf(v.v.x) + sqrt_(fabsf(t.v.x) * inv.v.x), fabsf(v.v.y) + sqrt_(fabsf(t.v.y) * inv.v.y));
}

}  // namespace mhd
