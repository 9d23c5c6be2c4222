// mhd_generic.cuh -- direction-agnostic marching kernels (any extents, any direction, both BCs).
// One thread owns one pencil segment along the sweep axis d and marches along it with the register
// pipelines of mhd_device.cuh; direction enters only through strides.  These kernels are the
// always-correct path (and the fast path for y/z sweeps, where the threads of a warp span the
// contiguous x axis, so every load and store is coalesced and no transpose is ever needed).
#pragma once
#include "mhd_device.cuh"

namespace mhd {

template <class real>
struct SweepGeom {
  int nd, na, nb;          // extents along d, t1, t2
  long long sd, sa, sb;    // element strides along d, t1, t2
  int bc;
  int seg;                 // cells per thread along d
  int nseg;                // segments per pencil
  int a_fast;              // 1: consecutive threads walk t1 first, 0: t2 first (pick the stride-1 axis)
  real gamma;
};

template <class real>
struct FluidArgs {
  const real* u[5];        // in : rho, m_d, m_t1, m_t2, E (sweep roles)
  real* uo[5];             // out: same roles
  const real *bd, *bt1, *bt2;
  const double* dt;
  SweepGeom<real> g;
};

template <class real>
struct BPairArgs {
  const real *rho, *md;    // updated fluid (held fixed, Alg. 2 step 1)
  const real *bd, *bt1, *bt2;
  real *bdo, *bt1o, *bt2o;
  const double* dt;
  int t2_first;            // reverse sweeps apply B_{t2->d} before B_{t1->d}
  SweepGeom<real> g;
};

template <class real>
__device__ __forceinline__ bool thread_to_pencil(const SweepGeom<real>& g, int& a, int& b, int& s) {
  const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const long long npencil = (long long)g.na * g.nb;
  if (tid >= npencil * g.nseg) return false;
  const long long pen = tid % npencil;
  s = (int)(tid / npencil);
  if (g.a_fast) { a = (int)(pen % g.na); b = (int)(pen / g.na); }
  else          { b = (int)(pen % g.nb); a = (int)(pen / g.nb); }
  return true;
}

// fluid_d, Algorithm 1
template <class real>
__global__ void __launch_bounds__(256) fluid_march_kernel(const FluidArgs<real> A) {
  const SweepGeom<real>& g = A.g;
  int a, b, s;
  if (!thread_to_pencil(g, a, b, s)) return;
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt, qdt = real(0.25) * dt;
  const long long oab = a * g.sa + b * g.sb;
  const long long oa1 = map_index(a + 1, g.na, g.bc) * g.sa + b * g.sb;   // row a+1 (for B_t1 at its +face)
  const long long ob1 = a * g.sa + map_index(b + 1, g.nb, g.bc) * g.sb;   // row b+1 (for B_t2 at its +face)
  const int n0 = s * g.seg;
  const int n1 = min(n0 + g.seg, g.nd);

  FluidPipe<real> pipe;
  pipe.init();
  real bd_lo = A.bd[map_index(n0 - 3, g.nd, g.bc) * g.sd + oab];
  for (int q = n0 - 3; q < n1 + 3; ++q) {
    const long long od = map_index(q, g.nd, g.bc) * g.sd;
    real u[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) u[k] = A.u[k][od + oab];
    const real bd_hi = A.bd[map_index(q + 1, g.nd, g.bc) * g.sd + oab];
    BCell<real> B;                                                     // eq (19): faces -> centre
    B.set(real(0.5) * (bd_lo + bd_hi), real(0.5) * (A.bt1[od + oab] + A.bt1[od + oa1]),
          real(0.5) * (A.bt2[od + oab] + A.bt2[od + ob1]));
    bd_lo = bd_hi;
    real out[5];
    pipe.push(u, B, g.gamma, hdt, qdt, out);
    const int m = q - 3;
    if (m >= n0) {
      const long long o = (long long)m * g.sd + oab;
#pragma unroll
      for (int k = 0; k < 5; ++k) A.uo[k][o] = out[k];
    }
  }
}

// B_{t1->d} and B_{t2->d} in one pass (Algorithm 2).  Each thread runs four
// flux pipelines: rows tau and tau+1 for both transverse components; the tau+1 rows supply the
// constraint update of B_d.
template <class real>
__global__ void __launch_bounds__(256) bpair_march_kernel(const BPairArgs<real> A) {
  const SweepGeom<real>& g = A.g;
  int a, b, s;
  if (!thread_to_pencil(g, a, b, s)) return;
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt;
  const int am = map_index(a - 1, g.na, g.bc), ap = map_index(a + 1, g.na, g.bc);
  const int bm = map_index(b - 1, g.nb, g.bc), bp = map_index(b + 1, g.nb, g.bc);
  const long long o00 = a * g.sa + b * g.sb;
  const long long om0 = am * g.sa + b * g.sb, op0 = ap * g.sa + b * g.sb;
  const long long o0m = a * g.sa + bm * g.sb, o0p = a * g.sa + bp * g.sb;
  const int n0 = s * g.seg;
  const int n1 = min(n0 + g.seg, g.nd);

  BPipe<real> p1, p1p, p2, p2p;    // t1 rows a, a+1;  t2 rows b, b+1
  p1.init(); p1p.init(); p2.init(); p2p.init();
  for (int q = n0 - 4; q < n1 + 4; ++q) {
    const long long od = map_index(q, g.nd, g.bc) * g.sd;
    const real r00 = A.rho[od + o00], m00 = A.md[od + o00];
    // Alg. 2 step 4: velocity at the transverse face = momentum sum / density sum of the two cells
    // sharing it (reading R5).  Row tau uses cells tau-1, tau; row tau+1 uses the MAPPED tau and tau+1.
    const real rm0 = A.rho[od + om0], mm0 = A.md[od + om0];
    const real rp0 = A.rho[od + op0], mp0 = A.md[od + op0];
    const real r0m = A.rho[od + o0m], m0m = A.md[od + o0m];
    const real r0p = A.rho[od + o0p], m0p = A.md[od + o0p];
    p1.push((mm0 + m00) * rcp_(rm0 + r00), A.bt1[od + o00], dt, hdt);
    p2.push((m0m + m00) * rcp_(r0m + r00), A.bt2[od + o00], dt, hdt);
    // the "+1" rows: row tau+1 uses cells map(tau), map(tau+1).  map(tau) = tau always; with clamping at
    // the last row map(tau+1) = tau too, so the same expression covers both boundary rules.
    p1p.push((m00 + mp0) * rcp_(r00 + rp0), A.bt1[od + op0], dt, hdt);
    p2p.push((m00 + m0p) * rcp_(r00 + r0p), A.bt2[od + o0p], dt, hdt);
    const int m = q - 4;
    if (m >= n0) {
      const long long o = (long long)m * g.sd + o00;
      A.bt1o[o] = p1.bold() - (p1.fhi() - p1.flo());       // Alg. 2 step 9: advect B_t
      A.bt2o[o] = p2.bold() - (p2.fhi() - p2.flo());
      real bdv = A.bd[o];
      const real c1 = p1p.flo() - p1.flo();                // constraint: same flux, face m-1/2
      const real c2 = p2p.flo() - p2.flo();
      if (A.t2_first) { bdv = bdv + c2; bdv = bdv + c1; }
      else            { bdv = bdv + c1; bdv = bdv + c2; }
      A.bdo[o] = bdv;
    }
  }
}

// B_{t1->d}, B_{t2->d} along an axis of extent 1 (the z sweeps of a 2-D problem, the y and z sweeps of a 1-D one).
// Every index along d maps to the only cell under both boundary rules (reading R10), so in Algorithm 2
// the smoothed velocity is vg = (vt + vt + 2 vt) / 4 = vt (exact), both first-order fluxes of a row are the same vg B_t,
// the half step leaves B_t as it is, the limited differences vanish (a b = 0 is not > 0), and the edge flux is
// f = (vg B_t) dt on both faces: B_t - (f - f) = B_t exactly, and only the constraint term f(tau+1) - f(tau) changes B_d
// -- the d-derivative-free part of the induction equation that a 2-D run still needs.  One thread per
// cell, no march, no warm-up; writes B_d only (the caller swaps that one field).
template <class real>
__global__ void __launch_bounds__(256) bpair_flat_kernel(const BPairArgs<real> A) {
  const SweepGeom<real>& g = A.g;
  int a, b, s;
  if (!thread_to_pencil(g, a, b, s)) return;
  const real dt = (real)(*A.dt);
  const int am = map_index(a - 1, g.na, g.bc), ap = map_index(a + 1, g.na, g.bc);
  const int bm = map_index(b - 1, g.nb, g.bc), bp = map_index(b + 1, g.nb, g.bc);
  const long long o00 = a * g.sa + b * g.sb;
  const long long om0 = am * g.sa + b * g.sb, op0 = ap * g.sa + b * g.sb;
  const long long o0m = a * g.sa + bm * g.sb, o0p = a * g.sa + bp * g.sb;
  const real r00 = A.rho[o00], m00 = A.md[o00];
  // Alg. 2 step 4 (reading R5) for the rows tau and tau+1 of either transverse component, as in bpair_march_kernel
  const real f1 = (((A.md[om0] + m00) * rcp_(A.rho[om0] + r00)) * A.bt1[o00]) * dt;
  const real f1p = (((m00 + A.md[op0]) * rcp_(r00 + A.rho[op0])) * A.bt1[op0]) * dt;
  const real f2 = (((A.md[o0m] + m00) * rcp_(A.rho[o0m] + r00)) * A.bt2[o00]) * dt;
  const real f2p = (((m00 + A.md[o0p]) * rcp_(r00 + A.rho[o0p])) * A.bt2[o0p]) * dt;
  const real c1 = f1p - f1, c2 = f2p - f2;
  real bdv = A.bd[o00];
  if (A.t2_first) { bdv = bdv + c2; bdv = bdv + c1; }
  else            { bdv = bdv + c1; bdv = bdv + c2; }
  A.bdo[o00] = bdv;
}

// ---------------------------------------------------------------------------------------------
// c_max reduction, eq (18) PAPER.md:128-132.  c >= 0, and non-negative IEEE doubles order like
// unsigned integers, so an integer atomicMax on the bit pattern is exact and order independent;
// NaN patterns compare above +Inf, so a poisoned state surfaces instead of being skipped.
// ---------------------------------------------------------------------------------------------
template <class real>
struct CflArgs {
  const real* f[8];
  int nx, ny, nz, bc;
  real gamma;
  unsigned long long* cmax_bits;
};

template <class real>
__global__ void __launch_bounds__(256) cfl_kernel(const CflArgs<real> A) {
  const long long N = (long long)A.nx * A.ny * A.nz;
  const long long sy = A.nx, sz = (long long)A.nx * A.ny;
  unsigned long long best = 0ull;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < N;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx % A.nx);
    const int j = (int)((idx / A.nx) % A.ny);
    const int k = (int)(idx / sz);
    const long long ip = map_index(i + 1, A.nx, A.bc) + j * sy + k * sz;
    const long long jp = i + map_index(j + 1, A.ny, A.bc) * sy + k * sz;
    const long long kp = i + j * sy + map_index(k + 1, A.nz, A.bc) * sz;
    const real bx = real(0.5) * (A.f[5][idx] + A.f[5][ip]);
    const real by = real(0.5) * (A.f[6][idx] + A.f[6][jp]);
    const real bz = real(0.5) * (A.f[7][idx] + A.f[7][kp]);
    const real c = cfl_speed(A.f[0][idx], A.f[1][idx], A.f[2][idx], A.f[3][idx], A.f[4][idx], bx, by, bz, A.gamma);
    const unsigned long long bits = (unsigned long long)__double_as_longlong((double)c);
    best = bits > best ? bits : best;
  }
  best = warp_max_u64(best);
  __shared__ unsigned long long sm[8];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = best;
  __syncthreads();
  if (threadIdx.x < 32) {
    best = threadIdx.x < (blockDim.x >> 5) ? sm[threadIdx.x] : 0ull;
    best = warp_max_u64(best);
    if (threadIdx.x == 0) atomicMax(A.cmax_bits, best);
  }
}

// Scalar block kept on the device so that no host round trip is needed between steps
// (the paper reads dt back every step; we do not).
struct Scalars {
  double dt;                       // current time step
  double t_total;                  // time since set_state
  double t_call;                   // time advanced by the current mhd_step call
  double cmax;                     // last c_max
  unsigned long long cmax_bits;    // reduction target
  int nonfinite;                   // sticky flag: a reduction saw NaN/Inf or c_max <= 0
  int pad;
  double t_end;                    // target time of mhd_run_until (time since set_state); unused unless clip = 1
  double dt_last;                  // last positive dt (the host sizes the next batch of mhd_run_until from it)
  long long steps_real;            // steps of the current mhd_run_until call that advanced time (dt > 0)
};

// one thread: dt = cfl / c_max, t += 2 dt; re-arms the reduction
// reuse = 0: finalize the reduction (cmax <- accumulator, accumulator re-armed); 1: s->cmax is already final
// clip = 1 (mhd_run_until): dt = min(cfl / c_max, (t_end - t) / 2) (reading R14: the loop of PAPER.md:233-243 stops
// at a given time, the last step is shortened to land on it); a clipped step sets t = t_end exactly, and once
// t >= t_end every further step gets dt = 0, which makes all six operators exact no-ops (u - 0 * flux = u).
__global__ void dt_from_cmax_kernel(Scalars* s, double cfl, int advance, int reuse, int clip) {
  double cm = s->cmax;
  if (!reuse) {
    cm = __longlong_as_double((long long)s->cmax_bits);
    s->cmax = cm;
    s->cmax_bits = 0ull;
  }
  double dt = 0.0;
  if (!(cm > 0.0) || isinf(cm) || isnan(cm)) s->nonfinite = 1;
  else dt = cfl / cm;
  if (clip && advance) {
    const double rem = 0.5 * (s->t_end - s->t_total);
    if (!(rem > 0.0)) dt = 0.0;
    else if (dt >= rem) {
      s->dt = rem;
      s->dt_last = rem;
      s->t_call += s->t_end - s->t_total;
      s->t_total = s->t_end;
      s->steps_real += 1;
      return;
    }
    if (dt > 0.0) { s->steps_real += 1; s->dt_last = dt; }
  }
  s->dt = dt;
  if (advance) { s->t_total += 2.0 * dt; s->t_call += 2.0 * dt; }
}

__global__ void begin_run_kernel(Scalars* s, double t_end) { s->t_call = 0.0; s->t_end = t_end; s->steps_real = 0; }

__global__ void set_dt_kernel(Scalars* s, double dt, int nsteps) {
  s->dt = dt;
  s->t_total += 2.0 * dt * nsteps;
  s->t_call += 2.0 * dt * nsteps;
}

__global__ void reset_call_kernel(Scalars* s) { s->t_call = 0.0; }

// ---------------------------------------------------------------------------------------------
// diagnostics (not on the timed path): field sums and max |div B|
// ---------------------------------------------------------------------------------------------
template <class real>
__global__ void __launch_bounds__(256) diag_kernel(const CflArgs<real> A, double* sums /*8*/, unsigned long long* divb_bits) {
  const long long N = (long long)A.nx * A.ny * A.nz;
  const long long sy = A.nx, sz = (long long)A.nx * A.ny;
  double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  unsigned long long best = 0ull;
  for (long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x; idx < N;
       idx += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(idx % A.nx);
    const int j = (int)((idx / A.nx) % A.ny);
    const int k = (int)(idx / sz);
#pragma unroll
    for (int c = 0; c < 8; ++c) acc[c] += (double)A.f[c][idx];
    const bool skip = (A.bc == BC_OUTFLOW) && ((i + 1 >= A.nx && A.nx > 1) || (j + 1 >= A.ny && A.ny > 1) || (k + 1 >= A.nz && A.nz > 1));
    if (!skip) {
      const long long ip = map_index(i + 1, A.nx, A.bc) + j * sy + k * sz;
      const long long jp = i + map_index(j + 1, A.ny, A.bc) * sy + k * sz;
      const long long kp = i + j * sy + map_index(k + 1, A.nz, A.bc) * sz;
      const double dv = ((double)A.f[5][ip] - (double)A.f[5][idx]) + ((double)A.f[6][jp] - (double)A.f[6][idx]) +
                        ((double)A.f[7][kp] - (double)A.f[7][idx]);
      const unsigned long long bits = (unsigned long long)__double_as_longlong(fabs(dv));
      best = bits > best ? bits : best;
    }
  }
#pragma unroll
  for (int c = 0; c < 8; ++c) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) acc[c] += __shfl_xor_sync(0xffffffffu, acc[c], o);
    if ((threadIdx.x & 31) == 0) atomicAdd(&sums[c], acc[c]);
  }
  best = warp_max_u64(best);
  if ((threadIdx.x & 31) == 0) atomicMax(divb_bits, best);
}

}  // namespace mhd
