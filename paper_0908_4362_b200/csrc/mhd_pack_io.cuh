// mhd_pack_io.cuh -- loads, stores and lane shuffles of a lane pack T (f2: two fp32 cells; float / double: one).
#pragma once
#include "mhd_device.cuh"

namespace mhd {

// lane-pack plumbing: T = double (1 cell) or f2 (2 cells)
template <class T> struct PackOf;
template <> struct PackOf<double> { typedef double scalar; enum { L = 1 }; };
template <> struct PackOf<float> { typedef float scalar; enum { L = 1 }; };
template <> struct PackOf<f2> { typedef float scalar; enum { L = 2 }; };

__device__ __forceinline__ double ld_pack(const double* p, double*) { return *p; }
__device__ __forceinline__ float ld_pack(const float* p, float*) { return *p; }
__device__ __forceinline__ f2 ld_pack(const float* p, f2*) { return f2(*reinterpret_cast<const float2*>(p)); }
__device__ __forceinline__ void st_pack(double* p, double v) { *p = v; }
__device__ __forceinline__ void st_pack(float* p, float v) { *p = v; }
__device__ __forceinline__ void st_pack(float* p, f2 v) { *reinterpret_cast<float2*>(p) = v.v; }
// (s, a[0..L-2]): the pack one column to the left;  a[L-1]: the last lane
__device__ __forceinline__ double shift_in_left(double, double s) { return s; }
__device__ __forceinline__ float shift_in_left(float, float s) { return s; }
__device__ __forceinline__ f2 shift_in_left(f2 a, float s) { return f2(s, a.v.x); }
__device__ __forceinline__ double shift_in_right(double, double s) { return s; }
__device__ __forceinline__ float shift_in_right(float, float s) { return s; }
__device__ __forceinline__ f2 shift_in_right(f2 a, float s) { return f2(a.v.y, s); }
__device__ __forceinline__ double last_lane(double a) { return a; }
__device__ __forceinline__ float last_lane(float a) { return a; }
__device__ __forceinline__ float last_lane(f2 a) { return a.v.y; }

// Largest c of eq (18) over the lanes of a pack, as an order-preserving integer key.  NaN must win the maximum (it
// poisons dt): compare bit patterns, not floats.  c >= 0 or NaN, and the bit pattern of a non-negative float orders
// like an unsigned integer with every NaN above +Inf (a NaN with the sign bit set is larger still), so fp32 kernels
// keep a 32-bit key per thread and widen it to the accumulator's double pattern once, at the end (key_bits).
__device__ __forceinline__ unsigned long long pack_speed_key(const double u[5], double hb2, double gamma) {
  return speed_bits(cfl_speed_hb2(u, hb2, gamma));
}
__device__ __forceinline__ unsigned int pack_speed_key(const float u[5], float hb2, float gamma) {
  return __float_as_uint(cfl_speed_hb2(u, hb2, gamma));
}
// two cells: everything that has a packed form runs packed; rcp, sqrt, |x| and the maxima per lane
__device__ __forceinline__ unsigned int pack_speed_key(const f2 u[5], f2 hb2, float gamma) {
  const f2 inv = rcp_(u[0]);
  const f2 ke = f2(0.5f) * fma_(u[1], u[1], fma_(u[2], u[2], u[3] * u[3])) * inv;
  const f2 p = f2(gamma - 1.0f) * (u[4] - ke - hb2);
  const f2 t = fma_(f2(gamma), p, f2(2.0f) * hb2);
  const float ca = fmaxf(fmaxf(fabsf(u[1].v.x), fabsf(u[2].v.x)), fabsf(u[3].v.x)) * inv.v.x + sqrt_(fabsf(t.v.x) * inv.v.x);
  const float cb = fmaxf(fmaxf(fabsf(u[1].v.y), fabsf(u[2].v.y)), fabsf(u[3].v.y)) * inv.v.y + sqrt_(fabsf(t.v.y) * inv.v.y);
  const unsigned int ka = __float_as_uint(ca), kb = __float_as_uint(cb);
  return ka > kb ? ka : kb;
}
__device__ __forceinline__ unsigned long long key_bits(unsigned long long k) { return k; }
__device__ __forceinline__ unsigned long long key_bits(unsigned int k) { return speed_bits(__uint_as_float(k)); }

// kept for the x kernels: the same as a 64-bit pattern per call
__device__ __forceinline__ unsigned long long pack_speed_bits(const double u[5], double hb2, double gamma) { return pack_speed_key(u, hb2, gamma); }
__device__ __forceinline__ unsigned long long pack_speed_bits(const float u[5], float hb2, float gamma) { return key_bits(pack_speed_key(u, hb2, gamma)); }
__device__ __forceinline__ unsigned long long pack_speed_bits(const f2 u[5], f2 hb2, float gamma) { return key_bits(pack_speed_key(u, hb2, gamma)); }

}  // namespace mhd
