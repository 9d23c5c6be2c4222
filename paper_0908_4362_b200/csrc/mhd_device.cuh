// mhd_device.cuh -- per-cell arithmetic of the relaxing-TVD scheme, shared by all CUDA kernels.
// PRODUCT code (CUDA path); shares nothing with oracle/.
//
// Citations are to /root/reference/PAPER.md (arxiv/paper_0908_4362), section 3.
#pragma once
#include <cuda_runtime.h>

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

template <class real> __device__ __forceinline__ real rabs(real x);
template <> __device__ __forceinline__ float rabs<float>(float x) { return fabsf(x); }
template <> __device__ __forceinline__ double rabs<double>(double x) { return fabs(x); }
template <class real> __device__ __forceinline__ real rsqrt_(real x);
template <> __device__ __forceinline__ float rsqrt_<float>(float x) { return sqrtf(x); }
template <> __device__ __forceinline__ double rsqrt_<double>(double x) { return sqrt(x); }

// van Leer limiter, eq (14); zero unless both half-differences have the same sign
// (reading R8: strictly a*b > 0).
template <class real>
__device__ __forceinline__ real vanleer(real a, real b) {
  const real ab = a * b;
  return ab > real(0) ? (real(2) * ab) / (a + b) : real(0);
}

// Right- and left-going fluxes R = c u + F, G = c u - F (2c u^R and 2c u^L of eqs (9)-(10),
// PAPER.md:85-89) for one cell.  u = (rho, m1, m2, m3, E) in sweep roles, b = cell-centred field
// in sweep roles (held fixed).  F is eq (6), the freezing speed
// c = |v| + sqrt(|gamma p + B^2| / rho) is PAPER.md:126.
template <class real>
__device__ __forceinline__ void right_left(const real u[5], const real b[3], real gamma, real R[5], real G[5]) {
  const real rho = u[0], m1 = u[1], m2 = u[2], m3 = u[3], E = u[4];
  const real inv = real(1) / rho;
  const real v = m1 * inv;
  const real b2 = b[0] * b[0] + b[1] * b[1] + b[2] * b[2];
  const real ke = real(0.5) * (m1 * m1 + m2 * m2 + m3 * m3) * inv;
  const real p = (gamma - real(1)) * (E - ke - real(0.5) * b2);
  const real ps = p + real(0.5) * b2;
  const real bdotv = (b[0] * m1 + b[1] * m2 + b[2] * m3) * inv;
  real F[5];
  F[0] = m1;
  F[1] = m1 * v + ps - b[0] * b[0];
  F[2] = m2 * v - b[1] * b[0];
  F[3] = m3 * v - b[2] * b[0];
  F[4] = (E + ps) * v - b[0] * bdotv;
  const real c = rabs(v) + rsqrt_(rabs(gamma * p + b2) * inv);
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    R[k] = c * u[k] + F[k];
    G[k] = c * u[k] - F[k];
  }
}

// c of eq (18): max(|vx|,|vy|,|vz|) + sqrt(|gamma p + B^2| / rho)
template <class real>
__device__ __forceinline__ real cfl_speed(real rho, real mx, real my, real mz, real E, real bx, real by, real bz,
                                          real gamma) {
  const real inv = real(1) / rho;
  const real b2 = bx * bx + by * by + bz * bz;
  const real ke = real(0.5) * (mx * mx + my * my + mz * mz) * inv;
  const real p = (gamma - real(1)) * (E - ke - real(0.5) * b2);
  const real vmax = fmax(fmax(rabs(mx * inv), rabs(my * inv)), rabs(mz * inv));
  return vmax + rsqrt_(rabs(gamma * p + b2) * inv);
}

// ---------------------------------------------------------------------------------------------
// Register pipeline of fluid_d for one pencil, fed one cell per call in sweep order.
// Algorithm 1: first-order upwind half step eq (16), then the second-order TVD
// full step eqs (11)-(15),(17) from u^{t+dt/2}.  After push() of cell q the updated u of cell q-3
// is returned (valid once at least 7 cells have been pushed).
// ---------------------------------------------------------------------------------------------
template <class real>
struct FluidPipe {
  real u1_[5], u2_[5], u3_[5];   // u(q-1), u(q-2), u(q-3)
  real bc1_[3];                  // B_c(q-1)
  real R0_[5];                   // R of u^t at q-1
  real phi1_[5];                 // first-order flux at face (q-2)+1/2
  real Ra_[5], Rb_[5];           // R of u^{t+dt/2} at q-3, q-2
  real Ga_[5], Gb_[5];           // G of u^{t+dt/2} at q-3, q-2
  real Rp_[5];                   // limited right-going face value at (q-3)+1/2
  real phi2_[5];                 // second-order flux at face (q-4)+1/2

  __device__ __forceinline__ void init() {
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      u1_[k] = u2_[k] = u3_[k] = real(1);
      R0_[k] = phi1_[k] = Ra_[k] = Rb_[k] = Ga_[k] = Gb_[k] = Rp_[k] = phi2_[k] = real(0);
    }
    bc1_[0] = bc1_[1] = bc1_[2] = real(0);
  }

  // u, b: cell q.  out: updated u of cell q-3.
  __device__ __forceinline__ void push(const real u[5], const real b[3], real gamma, real dt, real out[5]) {
    real R0[5], G0[5];
    right_left(u, b, gamma, R0, G0);                 // Alg. 1 step 4 at cell q
    real uh[5], phi1[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      phi1[k] = real(0.5) * (R0_[k] - G0[k]);        // step 5: first-order flux at face (q-1)+1/2
      uh[k] = u1_[k] - (phi1[k] - phi1_[k]) * (dt * real(0.5));   // step 6: u^{t+dt/2}(q-1), eq (16)
    }
    real Rc[5], Gc[5];
    right_left(uh, bc1_, gamma, Rc, Gc);             // step 7 at cell q-1 (same B_c)
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      // step 8, eqs (11)-(15): right-going value at face (q-2)+1/2 from cells q-3,q-2,q-1;
      // left-going value at face (q-3)+1/2 from cells q-3,q-2,q-1 (mirror image)
      const real Rp = Rb_[k] + vanleer(real(0.5) * (Rb_[k] - Ra_[k]), real(0.5) * (Rc[k] - Rb_[k]));
      const real Gp = Gb_[k] + vanleer(real(0.5) * (Gb_[k] - Gc[k]), real(0.5) * (Ga_[k] - Gb_[k]));
      const real phi2 = real(0.5) * (Rp_[k] - Gp);   // flux at face (q-3)+1/2
      out[k] = u3_[k] - (phi2 - phi2_[k]) * dt;      // step 9, eq (17) at cell q-3
      // shift the window by one cell
      phi2_[k] = phi2;
      Rp_[k] = Rp;
      Ra_[k] = Rb_[k]; Rb_[k] = Rc[k];
      Ga_[k] = Gb_[k]; Gb_[k] = Gc[k];
      phi1_[k] = phi1[k];
      R0_[k] = R0[k];
      u3_[k] = u2_[k]; u2_[k] = u1_[k]; u1_[k] = u[k];
    }
    bc1_[0] = b[0]; bc1_[1] = b[1]; bc1_[2] = b[2];
  }
};

// ---------------------------------------------------------------------------------------------
// Register pipeline of B_{t->d} for one row of faces (Algorithm 2; eqs (20)-(22)
// PAPER.md:147-158).  push(vt(q), B_t(q)) returns the second-order edge flux f*dt at face (q-4)+1/2;
// flo() is the previous one (face (q-4)-1/2) and bold() is B_t(q-4).  Valid after 9 pushes.
// ---------------------------------------------------------------------------------------------
template <class real>
struct BPipe {
  real vt1_, vt2_;        // vt(q-1), vt(q-2)
  real vg2_;              // vg(q-2)
  real w02_;              // vg*B_t at q-2 (first-order)
  real f1_;               // first-order flux at face (q-3)+1/2
  real b1_, b2_, b3_, b4_;// B_t at q-1..q-4
  real wA_, wB_, wC_;     // vg*B_t^{t+dt/2} at q-5, q-4, q-3
  real vhA_, vhB_;        // face velocity at (q-4)+1/2, (q-3)+1/2
  real f_, flo_, bold_;

  __device__ __forceinline__ void init() {
    vt1_ = vt2_ = vg2_ = w02_ = f1_ = b1_ = b2_ = b3_ = b4_ = wA_ = wB_ = wC_ = vhA_ = vhB_ = f_ = flo_ = bold_ = real(0);
  }

  __device__ __forceinline__ void push(real vt, real bt, real dt) {
    const real vg1 = real(0.25) * ((vt2_ + vt) + real(2) * vt1_);      // eq (20) at q-1
    const real w01 = vg1 * b1_;
    const real vh = real(0.5) * (vg2_ + vg1);                           // eq (22) at face (q-2)+1/2
    const real f1 = vh > real(0) ? w02_ : w01;                          // eq (21)
    const real bh = b2_ - (f1 - f1_) * (dt * real(0.5));                // Alg. 2 step 7: B_t^{t+dt/2}(q-2)
    const real wD = vg2_ * bh;
    // Alg. 2 step 8: second-order TVD flux at face (q-4)+1/2, upwinded by vhA_
    const bool up = vhA_ > real(0);
    const real x = up ? wB_ : wC_, y = up ? wA_ : wD, z = up ? wC_ : wB_;
    const real f = x + vanleer(real(0.5) * (x - y), real(0.5) * (z - x));
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

}  // namespace mhd
