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

// largest c of eq (18) over the lanes of a pack, as the order-preserving bit pattern of mhd_device.cuh.
// NaN must win the maximum (it poisons dt): compare the bit patterns, not the floats.
__device__ __forceinline__ unsigned long long pack_speed_bits(const double u[5], double hb2, double gamma) {
  return speed_bits(cfl_speed_hb2(u, hb2, gamma));
}
__device__ __forceinline__ unsigned long long pack_speed_bits(const float u[5], float hb2, float gamma) {
  return speed_bits(cfl_speed_hb2(u, hb2, gamma));
}
__device__ __forceinline__ unsigned long long pack_speed_bits(const f2 u[5], f2 hb2, float gamma) {
  const float ua[5] = {u[0].v.x, u[1].v.x, u[2].v.x, u[3].v.x, u[4].v.x};
  const float ub[5] = {u[0].v.y, u[1].v.y, u[2].v.y, u[3].v.y, u[4].v.y};
  const unsigned long long ba = speed_bits(cfl_speed_hb2(ua, hb2.v.x, gamma));
  const unsigned long long bb = speed_bits(cfl_speed_hb2(ub, hb2.v.y, gamma));
  return ba > bb ? ba : bb;
}

}  // namespace mhd
