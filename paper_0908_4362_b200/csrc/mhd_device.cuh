// mhd_device.cuh -- per-cell arithmetic of the relaxing-TVD scheme, shared by all CUDA kernels.
// PRODUCT code (CUDA path); shares nothing with oracle/.
//
// Citations are to /root/reference/PAPER.md (arxiv/paper_0908_4362), section 3.
//
// Arithmetic policy: the step is close to the ALU/issue roofline, so the
// special functions are the cheap ones.  fp32: MUFU.RCP / MUFU.SQRT (rcp.approx.ftz, sqrt.approx.ftz,
// <= 1-2 ulp, no slow path) -- far inside the 1e-5 per-step tolerance.  fp64: MUFU.RCP64H / MUFU.RSQ64H seed plus one
// third-order correction (rcp_, sqrt_ below: an ulp or two, no slow path; the 1e-12 tolerance leaves 10^4).
// No --use_fast_math: the discrete switches (a*b > 0, vh > 0) see IEEE products.
#pragma once
#include <cuda_runtime.h>
#include "mhd_pack.cuh"

namespace mhd {

enum { BC_PERIODIC = 0, BC_OUTFLOW = 1 };

// Boundary rule (reading R9): map an out-of-range index by wrap or clamp.
__device__ __forceinline__ int map_index(int q, int n, int bc) {
  if (bc == BC_PERIODIC) {
    while (q < 0) q += n;
    while (q >= n) q -= n;
    return q;
  }
  return q < 0 ? 0 : (q >= n ? n - 1 : q);
}
// same, valid only for -n <= q < 2n (one wrap); both rules evaluated and one selected, so that the producers of the ring
// kernels (uniform datapath, a dozen calls per stage) get straight-line code instead of a branch on bc with two arms
__device__ __forceinline__ int map_index1(int q, int n, int bc) {
  const int per = q + ((q >> 31) & n) - (q >= n ? n : 0);
  const int cl = min(max(q, 0), n - 1);
  return bc == BC_PERIODIC ? per : cl;
}

// MHD_F32_IEEE (diagnostic builds only, R15): IEEE division and square root and no fused multiply-add in
// fp32, to measure how much of the fp32 distance to the oracle comes from MUFU and contraction (answer: none of it).
#ifndef MHD_F32_IEEE
__device__ __forceinline__ float rcp_(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
#else
__device__ __forceinline__ float rcp_(float x) { return __fdiv_rn(1.0f, x); }
#endif
#ifndef MHD_F64_IEEE_DIV
// fp64: MUFU.RCP64H seed (relative error e <= 2^-23) + ONE third-order step  r (1 + e + e^2),  e = 1 - x r:  error e^3
// = 2^-69, three dependent DFMAs, no slow path and no range check (IEEE division: ~10 DFMAs plus a slow path; two
// Newton steps: four).  The fp64 kernels are bound by the FP64 pipe and by the latency of exactly these chains
// (profiles/r02_c5_step_ncu_full.md).  x = 0 or denormal gives NaN, which only ever reaches a discarded select
// operand (vl_full with a*b <= 0).
__device__ __forceinline__ double rcp_(double x) {
  double r;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double e = fma(-x, r, 1.0);
  const double e2 = fma(e, e, e);
  return fma(r, e2, r);
}
#else
__device__ __forceinline__ double rcp_(double x) { return 1.0 / x; }
#endif
#ifndef MHD_F32_IEEE
__device__ __forceinline__ float sqrt_(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
#else
__device__ __forceinline__ float sqrt_(float x) { return __fsqrt_rn(x); }
#endif
#ifndef MHD_F64_IEEE_DIV
// fp64 square root of x >= 0: MUFU.RSQ64H seed y (relative error <= 2^-23), one third-order step on the reciprocal
// root  y (1 + e/2 + 3 e^2/8),  e = 1 - x y^2  (error ~ e^3), then sqrt = x y: six dependent operations, result within
// an ulp or two (the 1e-12 per-step tolerance leaves 10^4).
__device__ __forceinline__ double sqrt_(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double t = x * y;
  const double e = fma(-t, y, 1.0);
  const double p = fma(0.375, e, 0.5) * e;
  y = fma(y, p, y);
  return x > 0.0 ? x * y : 0.0;
}
#else
__device__ __forceinline__ double sqrt_(double x) { return sqrt(x); }
#endif
__device__ __forceinline__ float abs_(float x) { return fabsf(x); }
__device__ __forceinline__ double abs_(double x) { return fabs(x); }
// a*b + c and c - a*b as one rounding (the scalar forms are what nvcc's contraction produces anyway;
// they are spelled out so that the packed type f2 of mhd_pack.cuh gets FFMA2 in the same places)
#ifndef MHD_F32_IEEE
__device__ __forceinline__ float fma_(float a, float b, float c) { return fmaf(a, b, c); }
#else
__device__ __forceinline__ float fma_(float a, float b, float c) { return __fadd_rn(__fmul_rn(a, b), c); }
#endif
__device__ __forceinline__ double fma_(double a, double b, double c) { return fma(a, b, c); }
#ifndef MHD_F32_IEEE
__device__ __forceinline__ float fnma_(float a, float b, float c) { return fmaf(-a, b, c); }
#else
__device__ __forceinline__ float fnma_(float a, float b, float c) { return __fadd_rn(__fmul_rn(-a, b), c); }
#endif
__device__ __forceinline__ double fnma_(double a, double b, double c) { return fma(-a, b, c); }
// the two discrete switches of the scheme (reading R8: strict > 0)
__device__ __forceinline__ float pos_or_zero(float s, float r) { return s > 0.0f ? r : 0.0f; }
__device__ __forceinline__ double pos_or_zero(double s, double r) { return s > 0.0 ? r : 0.0; }
__device__ __forceinline__ float pick_pos(float s, float a, float b) { return s > 0.0f ? a : b; }
__device__ __forceinline__ double pick_pos(double s, double a, double b) { return s > 0.0 ? a : b; }
// |v| + sqrt(|t| * inv): the freezing speed of PAPER.md:126 from v, t = gamma p + B^2, inv = 1/rho
__device__ __forceinline__ float freeze_speed(float v, float t, float inv) { return fabsf(v) + sqrt_(fabsf(t) * inv); }
__device__ __forceinline__ double freeze_speed(double v, double t, double inv) { return fabs(v) + sqrt_(fabs(t) * inv); }

// van Leer limiter of two HALF differences, eq (14), written for the FULL differences
// a, b:  vanleer(a/2, b/2) = 2 (a/2)(b/2) / (a/2 + b/2) = a b / (a + b).  Zero unless a*b > 0
// strictly (reading R8).
template <class real>
__device__ __forceinline__ real vl_full(real a, real b) {
  const real ab = a * b;
  const real r = ab * rcp_(a + b);
  return pos_or_zero(ab, r);
}
// x + vl_full(a, b) with the correction folded into one multiply-add:  a b / (a + b) + x  where a*b > 0, else x
template <class real>
__device__ __forceinline__ real vl_add(real x, real a, real b) {
  const real ab = a * b;
  const real y = fma_(ab, rcp_(a + b), x);
  return pick_pos(ab, y, x);
}

// Cell-centred field of one cell (held fixed through both stages) and what the two
// flux evaluations need from it.
template <class real>
struct BCell {
  real b0, b1, b2;   // sweep roles: b0 along the sweep
  real hb2;          // |b|^2 / 2
  __device__ __forceinline__ void set(real x, real y, real z) {
    b0 = x; b1 = y; b2 = z;
    hb2 = real(0.5) * fma_(x, x, fma_(y, y, z * z));
  }
};

// Right- and left-going fluxes R = c u + F, G = c u - F (2c u^R and 2c u^L of eqs (9)-(10),
// PAPER.md:85-89) for one cell.  u = (rho, m1, m2, m3, E) in sweep roles.  F is eq (6) PAPER.md:76;
// P* = P + B^2/2, P = (gamma-1)(E - rho v^2/2 - B^2/2); the freezing speed
// c = |v| + sqrt(|gamma p + B^2| / rho) is PAPER.md:126 (|.|: reading R3).
template <class real>
__device__ __forceinline__ void right_left(const real u[5], const BCell<real>& B, real gamma, real R[5], real G[5]) {
  const real m1 = u[1], m2 = u[2], m3 = u[3], E = u[4];
  const real inv = rcp_(u[0]);
  const real v = m1 * inv;
  const real ke2 = fma_(m1, m1, fma_(m2, m2, m3 * m3));
  const real p = (gamma - real(1)) * fnma_(real(0.5) * ke2, inv, E - B.hb2);
  const real ps = p + B.hb2;
  const real bdotv = fma_(B.b0, m1, fma_(B.b1, m2, B.b2 * m3)) * inv;
  real F[5];
  F[0] = m1;
  F[1] = fma_(m1, v, fnma_(B.b0, B.b0, ps));
  F[2] = fnma_(B.b1, B.b0, m2 * v);
  F[3] = fnma_(B.b2, B.b0, m3 * v);
  F[4] = fnma_(B.b0, bdotv, (E + ps) * v);
  const real c = freeze_speed(v, fma_(gamma, p, real(2) * B.hb2), inv);
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    R[k] = fma_(c, u[k], F[k]);
    G[k] = fma_(c, u[k], -F[k]);
  }
}

// c of eq (18): max(|vx|,|vy|,|vz|) + sqrt(|gamma p + B^2| / rho)
template <class real>
__device__ __forceinline__ real cfl_speed(real rho, real mx, real my, real mz, real E, real bx, real by, real bz,
                                          real gamma) {
  const real inv = rcp_(rho);
  const real b2 = bx * bx + by * by + bz * bz;
  const real ke = real(0.5) * (mx * mx + my * my + mz * mz) * inv;
  const real p = (gamma - real(1)) * (E - ke - real(0.5) * b2);
  const real vmax = fmax(fmax(abs_(mx), abs_(my)), abs_(mz)) * inv;
  return vmax + sqrt_(abs_(gamma * p + b2) * inv);
}

// same from sweep-role quantities: u = (rho, m1, m2, m3, E), hb2 = |B_c|^2 / 2
template <class real>
__device__ __forceinline__ real cfl_speed_hb2(const real u[5], real hb2, real gamma) {
  const real inv = rcp_(u[0]);
  const real ke = real(0.5) * (u[1] * u[1] + u[2] * u[2] + u[3] * u[3]) * inv;
  const real p = (gamma - real(1)) * (u[4] - ke - hb2);
  const real vmax = fmax(fmax(abs_(u[1]), abs_(u[2])), abs_(u[3])) * inv;
  return vmax + sqrt_(abs_(gamma * p + real(2) * hb2) * inv);
}

__device__ __forceinline__ unsigned long long speed_bits(float c) { return (unsigned long long)__double_as_longlong((double)c); }
__device__ __forceinline__ unsigned long long speed_bits(double c) { return (unsigned long long)__double_as_longlong(c); }

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const unsigned long long w = __shfl_xor_sync(0xffffffffu, v, o);
    v = w > v ? w : v;
  }
  return v;
}

// Fold a warp's maximum into the global accumulator.  A million warps hitting one address with atomicMax
// serialise in L2 (measured: +1.4 ms on fluid_x at 512^3), so the atomic is issued only when the value
// beats what the accumulator already holds; a stale read merely costs one redundant atomic.  The result
// is still the exact maximum, independent of order.
__device__ __forceinline__ void publish_max(unsigned long long* acc, unsigned long long v) {
  if (v > *reinterpret_cast<volatile unsigned long long*>(acc)) atomicMax(acc, v);
}

// ---------------------------------------------------------------------------------------------
// Register pipeline of fluid_d for one pencil, fed one cell per call in sweep order.
// Algorithm 1: first-order upwind half step eq (16), then the second-order TVD
// full step eqs (11)-(15),(17) from u^{t+dt/2}.  After push() of cell q the updated u of cell q-3
// is returned (valid once 7 cells have been pushed).  Fluxes are carried as twice their value
// (the 1/2 of  Phi = (R - G)/2  is folded into the dt factors).
// ---------------------------------------------------------------------------------------------
template <class real>
struct FluidPipe {
  real u1_[5], u2_[5], u3_[5];   // u(q-1), u(q-2), u(q-3)
  BCell<real> B1_;               // B_c(q-1)
  real hb2_2_, hb2_3_;           // |B_c|^2/2 of cells q-2, q-3 (for the fused c_max reduction)
  real R0_[5];                   // R of u^t at q-1
  real d1_[5];                   // 2 * first-order flux at face (q-2)+1/2
  real Rb_[5], dRa_[5];          // R^{1}(q-2) and R^{1}(q-2) - R^{1}(q-3)          (R^{1}: from u^{t+dt/2})
  real Gb_[5], dGa_[5];          // G^{1}(q-2) and G^{1}(q-3) - G^{1}(q-2)
  real Rp_[5];                   // limited right-going value at face (q-3)+1/2
  real phi2_[5];                 // 2 * second-order flux at face (q-4)+1/2

  __device__ __forceinline__ void init() {
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      u1_[k] = u2_[k] = u3_[k] = real(1);
      R0_[k] = d1_[k] = Rb_[k] = dRa_[k] = Gb_[k] = dGa_[k] = Rp_[k] = phi2_[k] = real(0);
    }
    B1_.set(real(0), real(0), real(0));
    hb2_2_ = hb2_3_ = real(0);
  }
  // |B_c|^2/2 of the cell whose update the last push() returned
  __device__ __forceinline__ real hb2_out() const { return hb2_out_; }
  real hb2_out_;

  // u, B: cell q.  out: updated u of cell q-3.  hdt = dt/2, qdt = dt/4.
  __device__ __forceinline__ void push(const real u[5], const BCell<real>& B, real gamma, real hdt, real qdt, real out[5]) {
    advance(u, u1_, u3_, B, gamma, hdt, qdt, out);
#pragma unroll
    for (int k = 0; k < 5; ++k) { u3_[k] = u2_[k]; u2_[k] = u1_[k]; u1_[k] = u[k]; }
  }

  // The same step with u(q-1) and u(q-3) supplied by the caller (kernels that keep the input rows in a
  // shared-memory ring re-read them there instead of spending 15 registers per pencil on a delay line).
  __device__ __forceinline__ void advance(const real u[5], const real um1[5], const real um3[5], const BCell<real>& B,
                                          real gamma, real hdt, real qdt, real out[5]) {
    real R0[5], G0[5];
    right_left(u, B, gamma, R0, G0);                 // Alg. 1 step 4 at cell q
    real uh[5], d1[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      d1[k] = R0_[k] - G0[k];                        // step 5: 2 * first-order flux at face (q-1)+1/2
      uh[k] = fnma_(d1[k] - d1_[k], qdt, um1[k]);    // step 6: u^{t+dt/2}(q-1), eq (16)
    }
    real Rc[5], Gc[5];
    right_left(uh, B1_, gamma, Rc, Gc);              // step 7 at cell q-1 (same B_c)
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      // step 8, eqs (11)-(15): right-going value at face (q-2)+1/2 from cells q-3,q-2,q-1;
      // left-going value at face (q-3)+1/2 from the same cells (mirror image)
      const real dRb = Rc[k] - Rb_[k];
      const real Rp = vl_add(Rb_[k], dRa_[k], dRb);
      const real dGb = Gb_[k] - Gc[k];
      const real Gp = vl_add(Gb_[k], dGb, dGa_[k]);
      const real phi2 = Rp_[k] - Gp;                 // 2 * flux at face (q-3)+1/2
      out[k] = fnma_(phi2 - phi2_[k], hdt, um3[k]);  // step 9, eq (17) at cell q-3
      // shift the window by one cell
      phi2_[k] = phi2;
      Rp_[k] = Rp;
      dRa_[k] = dRb; Rb_[k] = Rc[k];
      dGa_[k] = dGb; Gb_[k] = Gc[k];
      d1_[k] = d1[k];
      R0_[k] = R0[k];
    }
    hb2_out_ = hb2_3_;
    hb2_3_ = hb2_2_; hb2_2_ = B1_.hb2;
    B1_ = B;
  }
};

// ---------------------------------------------------------------------------------------------
// Register pipeline of B_{t->d} for one row of faces (Algorithm 2; eqs (20)-(22)
// PAPER.md:147-158).  push(vt(q), B_t(q)) produces the second-order edge flux f*dt at face
// (q-4)+1/2 (fhi); flo() is the previous one (face (q-4)-1/2) and bold() is B_t(q-4).
// Valid after 9 pushes.
// ---------------------------------------------------------------------------------------------
template <class real>
struct BPipe {
  real vt1_, vt2_;        // vt(q-1), vt(q-2)
  real vg2_;              // vg(q-2)
  real w02_;              // vg*B_t at q-2 (first-order)
  real f1_;               // first-order flux at face (q-3)+1/2
  real b1_, b2_, b3_, b4_;// B_t at q-1..q-4
  real wA_, wB_, wC_;     // vg*B_t^{t+dt/2} at q-5, q-4, q-3
  real vhA_, vhB_;        // 2 * face velocity at (q-4)+1/2, (q-3)+1/2 (only the sign is used)
  real f_, flo_, bold_;

  __device__ __forceinline__ void init() {
    vt1_ = vt2_ = vg2_ = w02_ = f1_ = b1_ = b2_ = b3_ = b4_ = wA_ = wB_ = wC_ = vhA_ = vhB_ = f_ = flo_ = bold_ = real(0);
  }

  __device__ __forceinline__ void push(real vt, real bt, real dt, real hdt) {
    const real vg1 = real(0.25) * fma_(real(2), vt1_, vt2_ + vt);      // eq (20) at q-1
    const real w01 = vg1 * b1_;
    const real vh = vg2_ + vg1;                                         // 2 * eq (22) at face (q-2)+1/2
    const real f1 = pick_pos(vh, w02_, w01);                            // eq (21)
    const real bh = fnma_(f1 - f1_, hdt, b2_);                          // Alg. 2 step 7: B_t^{t+dt/2}(q-2)
    const real wD = vg2_ * bh;
    // Alg. 2 step 8: second-order TVD flux at face (q-4)+1/2, upwinded by the sign of vhA_
    const real x = pick_pos(vhA_, wB_, wC_), y = pick_pos(vhA_, wA_, wD), z = pick_pos(vhA_, wC_, wB_);
    const real f = vl_add(x, x - y, z - x);
    flo_ = f_;
    f_ = f * dt;
    bold_ = b4_;
    // shift
    vt2_ = vt1_; vt1_ = vt;
    vg2_ = vg1; w02_ = w01; f1_ = f1;
    b4_ = b3_; b3_ = b2_; b2_ = b1_; b1_ = bt;
    wA_ = wB_; wB_ = wC_; wC_ = wD;
    vhA_ = vhB_; vhB_ = vh;
  }
  __device__ __forceinline__ real fhi() const { return f_; }
  __device__ __forceinline__ real flo() const { return flo_; }
  __device__ __forceinline__ real bold() const { return bold_; }
};

// Register pipeline of B_{t->d} for one row of faces (Algorithm 2; eqs (20)-(22)
// PAPER.md:147-158) with all delay lines as circular arrays indexed by the march step modulo 4 (K is a
// compile-time constant inside the 4x unrolled loop).  push<K>(vt(k), B_t(k)) finishes the second-order
// edge flux f*dt at face (k-4)+1/2 and returns B_t'(k-4); flo is the flux at face (k-4)-1/2, fhi the new one.
template <class real>
struct BPipe4 {
  real vt[2];        // vt(k-2), vt(k-1)            slot = step & 1
  real b[4];         // B_t(k-4..k-1)               slot = step & 3
  real w1[2];        // vg*B_t^{t+dt/2}(k-4), (k-3)  slot = step & 1
  real vh[2];        // 2 * face velocity at (k-4)+1/2, (k-3)+1/2 (only the sign is used)
  real vg, w0, f1, f;   // vg(k-2), vg*B_t(k-2), first-order flux at (k-3)+1/2, second-order flux*dt at (k-5)+1/2
  real dw, sl;       // w1(k-3) - w1(k-4), and the limited slope of w1 at cell k-4 (see push)

  __device__ __forceinline__ void init() {
    vt[0] = vt[1] = vh[0] = vh[1] = vg = w0 = f1 = f = dw = sl = w1[0] = w1[1] = real(0);
#pragma unroll
    for (int j = 0; j < 4; ++j) b[j] = real(0);
  }
  __device__ __forceinline__ real fhi() const { return f; }     // after push: flux*dt at face (k-4)+1/2

  template <int K>
  __device__ __forceinline__ void push(real vtn, real btn, real dt, real hdt, real& bnew, real& flo) {
    const real vg1 = real(0.25) * fma_(real(2), vt[(K + 1) & 1], vt[K & 1] + vtn);   // eq (20) at k-1
    const real w01 = vg1 * b[(K + 3) & 3];
    const real vh2 = vg + vg1;                                                       // 2 * eq (22) at face (k-2)+1/2
    const real f1n = pick_pos(vh2, w0, w01);                                         // eq (21)
    const real bh = fnma_(f1n - f1, hdt, b[(K + 2) & 3]);                            // Alg. 2 step 7: B_t^{t+dt/2}(k-2)
    const real wD = vg * bh;
    // Alg. 2 step 8: second-order TVD flux at face (k-4)+1/2 between the cells k-4 (wB) and k-3 (wC), upwinded by
    // the sign of the face velocity there:  wB + vl(wB - wA, wC - wB)  or  wC + vl(wC - wD, wB - wC).
    // vl(a, b) = ab / (a + b) is symmetric and odd under a common sign change, so the second form is wC - s(k-3)
    // with s(c) = vl(w(c) - w(c-1), w(c+1) - w(c)), the limited slope AT a cell: s(k-3) is computed once here and
    // serves the next face as s(k-4) (same products, same sums: the result has the same bits as selecting the three
    // operands first, with one reciprocal per step as before and two selects fewer).
    const real wB = w1[K & 1], wC = w1[(K + 1) & 1];
    const real dn = wD - wC;
    const real sn = vl_full(dw, dn);                                                 // s(k-3)
    const real fn = pick_pos(vh[K & 1], wB + sl, wC - sn) * dt;
    bnew = b[K & 3] - (fn - f);                                                      // Alg. 2 step 9 at cell k-4
    flo = f;
    f = fn; f1 = f1n; vg = vg1; w0 = w01; dw = dn; sl = sn;
    vt[K & 1] = vtn; b[K & 3] = btn; w1[K & 1] = wD; vh[K & 1] = vh2;
  }
};

}  // namespace mhd
