// mhd_viz.cuh -- headless restatement of the paper's visualisation stage (section 8) as
// CUDA kernels that read the state where the solver keeps it.  The paper maps the
// result buffers into OpenGL objects: a vertex buffer for 1-D runs (one vertex per grid point, x = position,
// y = selected value), a pixel buffer for 2-D runs (one pixel per grid point, colour = transfer function of the
// selected value), and a texture-based volume renderer for 3-D runs.  Graphics APIs are unavailable on this box;
// the buffers here are plain device memory.  The paper gives no formulas for the mappings, so they are fixed in
// include/mhd.h (DESIGN.md "parity unpinned by the paper" applies to this stage).
//
// Every float operation below is a single IEEE fp32 operation spelled with an intrinsic (no FMA contraction), in
// the order include/mhd.h states, so that the NumPy restatement under oracle/ reproduces the bytes exactly.
#pragma once
#include <cuda_runtime.h>
#include "mhd_device.cuh"

namespace mhd {

template <class real>
struct VizArgs {
  const real* f[8];
  int nx, ny, nz, bc;
  int field;            // 0..7 a stored field; 8 gas pressure p = (gamma-1)(E - |m|^2/(2 rho) - |B_c|^2/2)
  float gamma;
  float vmin, inv;      // inv = 1 / (vmax - vmin) rounded to fp32 on the host
};

// selected value of one cell as fp32
template <class real>
__device__ __forceinline__ float viz_value(const VizArgs<real>& A, int i, int j, int k) {
  const long long sy = A.nx, sz = (long long)A.nx * A.ny;
  const long long idx = i + j * sy + k * sz;
  if (A.field < 8) return (float)A.f[A.field][idx];
  // pressure: every term converted to fp32 first, then single fp32 operations (mhd.h)
  const float rho = (float)A.f[0][idx], mx = (float)A.f[1][idx], my = (float)A.f[2][idx], mz = (float)A.f[3][idx];
  const float E = (float)A.f[4][idx];
  const long long ip = map_index1(i + 1, A.nx, A.bc) + j * sy + k * sz;
  const long long jp = i + map_index1(j + 1, A.ny, A.bc) * sy + k * sz;
  const long long kp = i + j * sy + map_index1(k + 1, A.nz, A.bc) * sz;
  const float bx = __fmul_rn(0.5f, __fadd_rn((float)A.f[5][idx], (float)A.f[5][ip]));
  const float by = __fmul_rn(0.5f, __fadd_rn((float)A.f[6][idx], (float)A.f[6][jp]));
  const float bz = __fmul_rn(0.5f, __fadd_rn((float)A.f[7][idx], (float)A.f[7][kp]));
  const float m2 = __fadd_rn(__fadd_rn(__fmul_rn(mx, mx), __fmul_rn(my, my)), __fmul_rn(mz, mz));
  const float b2 = __fadd_rn(__fadd_rn(__fmul_rn(bx, bx), __fmul_rn(by, by)), __fmul_rn(bz, bz));
  const float ke = __fdiv_rn(__fmul_rn(0.5f, m2), rho);
  return __fmul_rn(__fsub_rn(A.gamma, 1.0f), __fsub_rn(__fsub_rn(E, ke), __fmul_rn(0.5f, b2)));
}

// t = clamp((v - vmin) * inv, 0, 1); NaN maps to 0
__device__ __forceinline__ float viz_unit(float v, float vmin, float inv) {
  const float t = __fmul_rn(__fsub_rn(v, vmin), inv);
  return t > 0.0f ? (t < 1.0f ? t : 1.0f) : 0.0f;
}
__device__ __forceinline__ int viz_byte(float t) { return __float2int_rz(__fadd_rn(__fmul_rn(t, 255.0f), 0.5f)); }

// min and max of the selected value over all cells (order-preserving integer keys; NaN cells are skipped)
__device__ __forceinline__ unsigned int viz_key(float v) {
  const unsigned int b = __float_as_uint(v);
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}
__device__ __forceinline__ float viz_unkey(unsigned int k) {
  return __uint_as_float((k & 0x80000000u) ? (k & 0x7fffffffu) : ~k);
}

template <class real>
__global__ void __launch_bounds__(256) viz_range_kernel(const VizArgs<real> A, unsigned int* lohi) {
  const long long N = (long long)A.nx * A.ny * A.nz;
  const long long sz = (long long)A.nx * A.ny;
  unsigned int lo = 0xffffffffu, hi = 0u;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < N; idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx % A.nx), j = (int)((idx / A.nx) % A.ny), k = (int)(idx / sz);
    const float v = viz_value(A, i, j, k);
    if (isfinite(v)) {                 // NaN and +-Inf cells are skipped (mhd.h: smallest and largest FINITE value)
      const unsigned int key = viz_key(v);
      lo = key < lo ? key : lo;
      hi = key > hi ? key : hi;
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned int a = __shfl_xor_sync(0xffffffffu, lo, o), b = __shfl_xor_sync(0xffffffffu, hi, o);
    lo = a < lo ? a : lo;
    hi = b > hi ? b : hi;
  }
  if ((threadIdx.x & 31) == 0) { atomicMin(&lohi[0], lo); atomicMax(&lohi[1], hi); }
}

// 1-D: one vertex per grid point of the row (j, k): x = -1 + (2 i + 1) / nx, y = -1 + 2 t
template <class real>
__global__ void __launch_bounds__(256) viz_curve_kernel(const VizArgs<real> A, int j, int k, float invn, float2* xy) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= A.nx) return;
  const float t = viz_unit(viz_value(A, i, j, k), A.vmin, A.inv);
  xy[i] = make_float2(__fadd_rn(-1.0f, __fmul_rn((float)(2 * i + 1), invn)), __fadd_rn(-1.0f, __fmul_rn(2.0f, t)));
}

// 2-D: one RGBA8 pixel per grid point of the plane k, colour = lut[byte(t)]
template <class real>
__global__ void __launch_bounds__(256) viz_slice_kernel(const VizArgs<real> A, int k, const uchar4* __restrict__ lut,
                                                        uchar4* __restrict__ rgba) {
  __shared__ uchar4 slut[256];
  slut[threadIdx.x] = lut[threadIdx.x];
  __syncthreads();
  const long long n2 = (long long)A.nx * A.ny;
  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n2; p += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(p % A.nx), j = (int)(p / A.nx);
    rgba[p] = slut[viz_byte(viz_unit(viz_value(A, i, j, k), A.vmin, A.inv))];
  }
}

// 3-D: orthographic front-to-back compositing along +z, one ray per (i, j) column (lanes along x: every plane read is
// coalesced).  Sample colour c_s = lut.rgb / 255, opacity a_s = min(lut.a / 255 * opacity, 1);
// C += (1 - A) a_s c_s;  A += (1 - A) a_s;  the ray stops once A >= 0.99.  Output byte(C), byte(A).
template <class real>
__global__ void __launch_bounds__(256) viz_volume_kernel(const VizArgs<real> A, const uchar4* __restrict__ lut, float opacity,
                                                         uchar4* __restrict__ rgba) {
  __shared__ uchar4 slut[256];
  slut[threadIdx.x] = lut[threadIdx.x];
  __syncthreads();
  const long long n2 = (long long)A.nx * A.ny;
  const float inv255 = __fdiv_rn(1.0f, 255.0f);
  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < n2; p += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(p % A.nx), j = (int)(p / A.nx);
    float cr = 0.0f, cg = 0.0f, cb = 0.0f, al = 0.0f;
    for (int k = 0; k < A.nz; ++k) {
      const uchar4 s = slut[viz_byte(viz_unit(viz_value(A, i, j, k), A.vmin, A.inv))];
      float as = __fmul_rn(__fmul_rn((float)s.w, inv255), opacity);
      as = as < 1.0f ? as : 1.0f;
      const float w = __fmul_rn(__fsub_rn(1.0f, al), as);
      cr = __fadd_rn(cr, __fmul_rn(w, __fmul_rn((float)s.x, inv255)));
      cg = __fadd_rn(cg, __fmul_rn(w, __fmul_rn((float)s.y, inv255)));
      cb = __fadd_rn(cb, __fmul_rn(w, __fmul_rn((float)s.z, inv255)));
      al = __fadd_rn(al, w);
      if (al >= 0.99f) break;
    }
    const float one = 1.0f;
    rgba[p] = make_uchar4((unsigned char)viz_byte(cr < one ? cr : one), (unsigned char)viz_byte(cg < one ? cg : one),
                          (unsigned char)viz_byte(cb < one ? cb : one), (unsigned char)viz_byte(al < one ? al : one));
  }
}

}  // namespace mhd
