// mhd_yz.cuh -- marching kernels for sweeps along y and z (the axes that are NOT contiguous).
//
// Layout is x fastest, so for a sweep along y or z the 32 lanes of a warp sit on 32 consecutive x:
// every load and store of the march is one fully coalesced 128-byte (fp32) line per field, and the
// sweep needs no transpose at all (the paper's z-fastest layout made two of its three sweeps
// uncoalesced; the Fortran code it follows transposes instead).
// Each thread owns one pencil segment: it walks n along the sweep axis, holds the +-3 (fluid) or +-4
// (B) stencil in registers (FluidPipe / BPipe) and writes each result once.  HBM traffic is therefore
// the algorithmic minimum of the two-kernel split: fluid reads 5 u + 3 B and writes 5 u; the B pair
// reads rho, m_d, 3 B and writes 3 B (transverse +-1 neighbours come out of L1/L2).
//
// Requirements (else the generic kernels of mhd_generic.cuh run): extent along the sweep >= 8 and
// N < 2^31 (32-bit element offsets).
#pragma once
#include "mhd_device.cuh"

namespace mhd {

template <class real>
struct YZArgs {
  // fluid: u[5] in / uo[5] out in sweep roles (rho, m_d, m_t1, m_t2, E);  B pair: u[0] = rho, u[1] = m_d
  const real* u[5];
  real* uo[5];
  const real *bd, *bx, *bo;     // B along the sweep, Bx (transverse, +1 neighbour is the next lane), B along the other axis
  real *bdo, *bxo, *boo;        // B-pair outputs
  const double* dt;
  unsigned long long* cmax_bits;   // != nullptr: also reduce c of eq (18) over the UPDATED cells (last operator of a step)
  int nx, nd, no;               // extents: x, sweep axis, other transverse axis
  int sd, so;                   // element strides of the sweep axis and of the other transverse axis
  int bc, seg;
  int x_is_t1;                  // sweep z: (t1,t2) = (x,y) -> 1;  sweep y: (t1,t2) = (z,x) -> 0
  int t2_first;                 // B pair in a reverse sweep
  real gamma;
};

template <class real>
struct FluidIn {
  real u[5];
  real bd_hi, bxa, bxb, boa, bob;
};

template <class real>
__device__ __forceinline__ void load_fluid(const YZArgs<real>& A, int q, int base, int xp_off, int op_off, FluidIn<real>& c) {
  const int off = map_index1(q, A.nd, A.bc) * A.sd + base;
#pragma unroll
  for (int k = 0; k < 5; ++k) c.u[k] = __ldg(A.u[k] + off);
  c.bd_hi = __ldg(A.bd + map_index1(q + 1, A.nd, A.bc) * A.sd + base);
  c.bxa = __ldg(A.bx + off);
  c.bxb = __ldg(A.bx + off + xp_off);
  c.boa = __ldg(A.bo + off);
  c.bob = __ldg(A.bo + off + op_off);
}

// fluid_y / fluid_z, Algorithm 1
#ifndef MHD_YZ_MINB
#define MHD_YZ_MINB 4
#endif
#ifndef MHD_YZ_UNROLL
#define MHD_YZ_UNROLL 3
#endif
#ifndef MHD_YZ_PREFETCH
#define MHD_YZ_PREFETCH 1
#endif
#define MHD_STR2(x) #x
#define MHD_STR(x) MHD_STR2(x)

template <class real, int BLOCK>
__global__ void __launch_bounds__(BLOCK, MHD_YZ_MINB) fluid_yz_kernel(const YZArgs<real> A) {
  int i = blockIdx.x * BLOCK + threadIdx.x;
  const bool live = i < A.nx;
  if (!live) i = A.nx - 1;                     // stay in step for the warp reduction; stores are masked
  const int o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = live ? min(n0 + A.seg, A.nd) : n0 - 6;   // dead threads run no iteration
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt, qdt = real(0.25) * dt;
  const int base = i + o * A.so;
  const int xp_off = map_index1(i + 1, A.nx, A.bc) - i;              // to the +x neighbour
  const int op_off = (map_index1(o + 1, A.no, A.bc) - o) * A.so;     // to the + neighbour along the other axis

  FluidPipe<real> pipe;
  pipe.init();
  real bd_lo = __ldg(A.bd + map_index1(n0 - 3, A.nd, A.bc) * A.sd + base);
  FluidIn<real> cur, nxt;
  load_fluid(A, n0 - 3, base, xp_off, op_off, cur);
  unsigned long long cbest = 0ull;
_Pragma(MHD_STR(unroll MHD_YZ_UNROLL))
  for (int q = n0 - 3; q < n1 + 3; ++q) {
#if MHD_YZ_PREFETCH
    if (q + 1 < n1 + 3) load_fluid(A, q + 1, base, xp_off, op_off, nxt);   // prefetch the next cell
#else
    if (q > n0 - 3) load_fluid(A, q, base, xp_off, op_off, cur);
#endif
    BCell<real> B;                                                           // eq (19): faces -> centre
    const real bxc = real(0.5) * (cur.bxa + cur.bxb), boc = real(0.5) * (cur.boa + cur.bob);
    if (A.x_is_t1) B.set(real(0.5) * (bd_lo + cur.bd_hi), bxc, boc);
    else           B.set(real(0.5) * (bd_lo + cur.bd_hi), boc, bxc);
    bd_lo = cur.bd_hi;
    real out[5];
    pipe.push(cur.u, B, A.gamma, hdt, qdt, out);
    const int m = q - 3;
    if (m >= n0) {
      const int off = m * A.sd + base;
#pragma unroll
      for (int k = 0; k < 5; ++k) A.uo[k][off] = out[k];
      if (A.cmax_bits) {          // last operator of a step: c of eq (18) from the updated cell (B unchanged)
        const unsigned long long b = speed_bits(cfl_speed_hb2(out, pipe.hb2_out(), A.gamma));
        cbest = b > cbest ? b : cbest;
      }
    }
#if MHD_YZ_PREFETCH
    cur = nxt;
#endif
  }
  if (A.cmax_bits) {
    cbest = warp_max_u64(cbest);
    if ((threadIdx.x & 31) == 0) publish_max(A.cmax_bits, cbest);
  }
}

// ---------------------------------------------------------------------------------------------
// B_{t1->d} and B_{t2->d} in one pass for d = y, z (Algorithm 2).
// ---------------------------------------------------------------------------------------------
template <class real>
struct BIn {
  real r00, m00, rxm, mxm, rxp, mxp, rom, mom, rop, mop;   // rho, m_d at the cell and its x-1, x+1, o-1, o+1 neighbours
  real bx0, bxp, bo0, bop;                                   // transverse B at the cell and at its + neighbour
};

template <class real>
__device__ __forceinline__ void load_b(const YZArgs<real>& A, int q, int base, int xm, int xp, int om, int op, BIn<real>& c) {
  const int off = map_index1(q, A.nd, A.bc) * A.sd + base;
  const real* rho = A.u[0];
  const real* md = A.u[1];
  c.r00 = __ldg(rho + off);      c.m00 = __ldg(md + off);
  c.rxm = __ldg(rho + off + xm); c.mxm = __ldg(md + off + xm);
  c.rxp = __ldg(rho + off + xp); c.mxp = __ldg(md + off + xp);
  c.rom = __ldg(rho + off + om); c.mom = __ldg(md + off + om);
  c.rop = __ldg(rho + off + op); c.mop = __ldg(md + off + op);
  c.bx0 = __ldg(A.bx + off);     c.bxp = __ldg(A.bx + off + xp);
  c.bo0 = __ldg(A.bo + off);     c.bop = __ldg(A.bo + off + op);
}

template <class real, int BLOCK>
__global__ void __launch_bounds__(BLOCK) bpair_yz_kernel(const YZArgs<real> A) {
  const int i = blockIdx.x * BLOCK + threadIdx.x;
  if (i >= A.nx) return;
  const int o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt;
  const int base = i + o * A.so;
  const int xm = map_index1(i - 1, A.nx, A.bc) - i, xp = map_index1(i + 1, A.nx, A.bc) - i;
  const int om = (map_index1(o - 1, A.no, A.bc) - o) * A.so, op = (map_index1(o + 1, A.no, A.bc) - o) * A.so;

  BPipe<real> px, pxp, po, pop;      // Bx rows i, i+1;  B_other rows o, o+1
  px.init(); pxp.init(); po.init(); pop.init();
  BIn<real> cur, nxt;
  load_b(A, n0 - 4, base, xm, xp, om, op, cur);
#pragma unroll 2
  for (int q = n0 - 4; q < n1 + 4; ++q) {
    if (q + 1 < n1 + 4) load_b(A, q + 1, base, xm, xp, om, op, nxt);
    // Alg. 2 step 4: velocity at the transverse face = momentum sum / density sum of the two cells
    // sharing it (reading R5); row tau uses cells tau-1, tau and row tau+1 cells map(tau), map(tau+1).
    px.push((cur.mxm + cur.m00) * rcp_(cur.rxm + cur.r00), cur.bx0, dt, hdt);
    pxp.push((cur.m00 + cur.mxp) * rcp_(cur.r00 + cur.rxp), cur.bxp, dt, hdt);
    po.push((cur.mom + cur.m00) * rcp_(cur.rom + cur.r00), cur.bo0, dt, hdt);
    pop.push((cur.m00 + cur.mop) * rcp_(cur.r00 + cur.rop), cur.bop, dt, hdt);
    const int m = q - 4;
    if (m >= n0) {
      const int off = m * A.sd + base;
      A.bxo[off] = px.bold() - (px.fhi() - px.flo());        // Alg. 2 step 9: advect B_t
      A.boo[off] = po.bold() - (po.fhi() - po.flo());
      real bdv = __ldg(A.bd + off);
      const real cx = pxp.flo() - px.flo();                  // constraint: same flux, face m-1/2
      const real co = pop.flo() - po.flo();
      // forward sweeps apply t1 then t2, reverse sweeps t2 then t1
      const bool x_first = (A.x_is_t1 != 0) != (A.t2_first != 0);
      if (x_first) { bdv = bdv + cx; bdv = bdv + co; }
      else         { bdv = bdv + co; bdv = bdv + cx; }
      A.bdo[off] = bdv;
    }
    cur = nxt;
  }
}

}  // namespace mhd
