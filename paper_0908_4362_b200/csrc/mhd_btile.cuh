// mhd_btile.cuh -- B_{t1->d}, B_{t2->d} for sweeps along y and z as a "tile march".
//
// Algorithm 2 needs, for the constraint update of B_d in cell (i,o), the edge
// fluxes of the rows i+1 and o+1 as well, and, for the face velocities, rho and m_d
// of the cells i-1 and o-1.  Instead of every thread recomputing its neighbours' flux pipelines and
// re-reading their rho, m_d from global memory (mhd_yz.cuh: 4 pipelines, 15 loads per cell), a block
// owns a TX x TO tile of pencils in the (x, o) plane and marches along d in lock step:
//   * every thread loads only its own cell (rho, m_d, B_x, B_o, B_d: 5 coalesced loads, prefetched one
//     march step ahead) and runs only its own two pipelines (B_x row i, B_o row o),
//   * rho, m_d and the finished fluxes are exchanged through double-buffered shared memory with one
//     block barrier per march step,
//   * one extra "halo" row of threads runs the B_o pipelines of row o0+TO and, in its first TO lanes,
//     the B_x pipelines of column x0+TX; its next TO lanes fetch column x0-1 (overhead 1/TO).
// The loop is unrolled by 4 with the pipeline state held in circular register arrays (BPipe4), so the
// delay lines cost no register moves: ncu on the first version of this kernel showed 264 instructions
// per cell of which 46 were moves and ~100 address arithmetic (profiles/r01_c4_step_ncu_full.md).
//
// Requirements (else bpair_yz_kernel runs): nx % TX == 0, no % TO == 0, extent along the sweep >= 8.
#pragma once
#include <type_traits>
#include "mhd_yz.cuh"

namespace mhd {

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

template <class real, int TX, int TO>
struct BTile {
  static constexpr int TW = TX + 2, TH = TO + 2;
  static constexpr int NU = TH * TW;                     // rho / m_d tile incl. one-cell halo, slot (o_local+1)*TW + x_local+1
  static constexpr int NFX = TO * (TX + 1) + 1;          // B_x-row fluxes at (o_local, x_local <= TX); +1 dummy
  static constexpr int NFO = (TO + 1) * TX;              // B_o-row fluxes at (o_local <= TO, x_local)
  static constexpr int BUF = 2 * NU + NFX + NFO;         // reals per buffer
  static constexpr int NT = (TO + 1) * TX;
};

// keeps a per-thread constant in a register: without it ptxas rematerialises these few-instruction
// index expressions inside the march loop, every step
__device__ __forceinline__ void pin_reg(int& v) { asm volatile("" : "+r"(v)); }

#ifndef MHD_BTILE_L2PF
#define MHD_BTILE_L2PF 4
#endif
__device__ __forceinline__ void l2_prefetch(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }

#ifndef MHD_BTILE_MINB
#define MHD_BTILE_MINB 3
#endif

// One thread's march.  ROLE 0: interior tile rows 1..TO-1; 1: tile row 0 (also fetches row o0-1);
// 2: the halo row.  Roles are warp uniform, so every warp runs exactly one instantiation; all of them
// meet at the same hardware barrier (bar.sync 0) once per march step.
template <class real, int TX, int TO, int ROLE>
__device__ __forceinline__ void bpair_tile_march(const YZArgs<real>& A, real* sm, const int row, const int col) {
  using T = BTile<real, TX, TO>;
  constexpr int TW = T::TW;
  constexpr bool halo = ROLE == 2;
  const int x0 = blockIdx.x * TX, o0 = blockIdx.y * TO;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt;

  // my O position (B_o pipeline; rho, m_d, B_d of my own cell) and X position (B_x pipeline).
  // interior thread: both are my cell.  halo row: O = (x0+col, o0+TO); X = lanes < TO: (x0+TX, o0+col),
  // lanes TO..2TO-1: (x0-1, o0+col-TO) (fetch only), other lanes idle in the X role.
  const int xrole = !halo ? 0 : (col < TO ? 1 : (col < 2 * TO ? 2 : 3));
  const int oO = halo ? map_index1(o0 + TO, A.no, A.bc) : o0 + row;
  int offO = x0 + col + oO * A.so;
  const int xr_row = xrole == 2 ? col - TO : (xrole == 1 ? col : 0);
  const int iX = xrole == 1 ? map_index1(x0 + TX, A.nx, A.bc) : map_index1(x0 - 1, A.nx, A.bc);
  int offX = halo ? iX + (o0 + xr_row) * A.so : offO;                  // halo: my X cell; row 0: the cell in row o0-1
  if (ROLE == 1) offX = x0 + col + map_index1(o0 - 1, A.no, A.bc) * A.so;
  // tile slots (in reals, relative to the buffer)
  int tO = (halo ? TO + 1 : row + 1) * TW + col + 1;
  int tX = xrole == 1 ? (xr_row + 1) * TW + TX + 1 : (xrole == 2 ? (xr_row + 1) * TW : (ROLE == 1 ? col + 1 : tO));
  int fXw = T::NU * 2 + (halo ? (xrole == 1 ? xr_row * (TX + 1) + TX : TO * (TX + 1)) : row * (TX + 1) + col);
  int fOw = T::NU * 2 + T::NFX + (halo ? TO : row) * TX + col;
  pin_reg(offO); pin_reg(offX); pin_reg(tO); pin_reg(tX); pin_reg(fXw); pin_reg(fOw);
  const int nbO = tO - TW;                                            // cell o-1 of the O pipeline
  const int nbX = (halo ? tX : tO) - 1;                               // cell x-1 of the X pipeline
  const int fXr = fXw + 1, fOr = fOw + TX;                            // interior only: the rows i+1 and o+1
  const bool xload = xrole <= 2;                                      // halo: fetches rho, m_d, B_x at its X cell
  const bool x_first = (A.x_is_t1 != 0) != (A.t2_first != 0);         // forward: t1 then t2; reverse: t2 then t1

  const real* __restrict__ rho = A.u[0];
  const real* __restrict__ md = A.u[1];
  const real* __restrict__ bxp = A.bx;
  const real* __restrict__ bop = A.bo;
  const real* __restrict__ bdp = A.bd;

  struct In { real rO, mO, rX, mX, bX, bO, bD; };
  In cur, nxt;
  cur.rX = cur.mX = real(1);
  cur.bX = cur.bD = real(0);
  nxt = cur;
  int qn = n0 - 4;                                                    // next cell to load
  int off = (n0 - 8) * A.sd + offO;                                   // output cell m = q - 4 = n0 + it - 8
  // loads of march step `it+1` (cell qn) and B_d of the cell that step finishes, issued one step ahead
  auto load = [&](In& c, int it_next) {
    const int od = map_index1(qn, A.nd, A.bc) * A.sd;                 // index mapped by the boundary rule (reading R9)
    const int iO = od + offO;
    c.rO = __ldg(rho + iO); c.mO = __ldg(md + iO); c.bO = __ldg(bop + iO);
    if (halo) {
      if (xload) { const int iXx = od + offX; c.rX = __ldg(rho + iXx); c.mX = __ldg(md + iXx); c.bX = __ldg(bxp + iXx); }
    } else {
      c.bX = __ldg(bxp + iO);
      if (ROLE == 1) { const int iR = od + offX; c.rX = __ldg(rho + iR); c.mX = __ldg(md + iR); }
      const int mn = n0 + it_next - 8;
      if (it_next >= 8 && mn < n1) c.bD = __ldg(bdp + (off + A.sd));
    }
    ++qn;
#if MHD_BTILE_L2PF > 0
    {   // the loads above have one march step to arrive; pull the lines of a later step from HBM into L2 now
      const int ip = map_index1(qn + MHD_BTILE_L2PF - 1, A.nd, A.bc) * A.sd + offO;
      l2_prefetch(rho + ip); l2_prefetch(md + ip); l2_prefetch(bop + ip);
      if (!halo) { l2_prefetch(bxp + ip); l2_prefetch(bdp + ip); }
    }
#endif
  };

  BPipe4<real> px, po;
  px.init(); po.init();
  load(cur, 0);
  const int niter = n1 - n0 + 8;                                      // cells n0-4 .. n1+3

  auto step = [&](auto Ktag, int it) {
    constexpr int K = decltype(Ktag)::value;
    real* buf = sm + (K & 1) * T::BUF;
    load(nxt, it + 1);
    // publish rho, m_d of this march step and the fluxes finished in the previous one
    buf[tO] = cur.rO; buf[T::NU + tO] = cur.mO;
    if (halo) { if (xload) { buf[tX] = cur.rX; buf[T::NU + tX] = cur.mX; } }
    else if (ROLE == 1) { buf[tX] = cur.rX; buf[T::NU + tX] = cur.mX; }
    buf[fXw] = px.fhi();
    buf[fOw] = po.fhi();
    asm volatile("bar.sync 0;" ::: "memory");
    // Alg. 2 step 4: face velocity = momentum sum / density sum of the two cells sharing the face (reading R5)
    const real rXc = halo ? cur.rX : cur.rO, mXc = halo ? cur.mX : cur.mO;
    const real vtX = (buf[T::NU + nbX] + mXc) * rcp_(buf[nbX] + rXc);
    const real vtO = (buf[T::NU + nbO] + cur.mO) * rcp_(buf[nbO] + cur.rO);
    real bxn, bon, fxlo, folo;
    px.template push<K>(vtX, cur.bX, dt, hdt, bxn, fxlo);
    po.template push<K>(vtO, cur.bO, dt, hdt, bon, folo);
    if (!halo) {
      const int m = n0 + it - 8;
      if (it >= 8 && m < n1) {
        A.bxo[off] = bxn;                                             // Alg. 2 step 9: advected B_t
        A.boo[off] = bon;
        // constraint with the same fluxes at face m-1/2: the neighbours published theirs above
        const real cx = buf[fXr] - fxlo;
        const real co = buf[fOr] - folo;
        real bdv = cur.bD;
        if (x_first) { bdv = bdv + cx; bdv = bdv + co; }
        else         { bdv = bdv + co; bdv = bdv + cx; }
        A.bdo[off] = bdv;
      }
    }
    off += A.sd;
    cur = nxt;
  };
  for (int it = 0; it < niter; it += 4) {
    step(std::integral_constant<int, 0>{}, it);
    step(std::integral_constant<int, 1>{}, it + 1);
    step(std::integral_constant<int, 2>{}, it + 2);
    step(std::integral_constant<int, 3>{}, it + 3);
  }
}

template <class real, int TX, int TO>
__global__ void __launch_bounds__((TO + 1) * TX, (TO + 1) * TX <= 320 ? MHD_BTILE_MINB : 1) bpair_tile_kernel(const YZArgs<real> A) {
  static_assert(2 * TO <= TX && TX % 32 == 0, "tile shape");
  using T = BTile<real, TX, TO>;
  __shared__ real sm[2 * T::BUF];
  const int tid = threadIdx.x;
  const int row = tid / TX, col = tid - row * TX;
  if (row == TO) bpair_tile_march<real, TX, TO, 2>(A, sm, row, col);
  else if (row == 0) bpair_tile_march<real, TX, TO, 1>(A, sm, row, col);
  else bpair_tile_march<real, TX, TO, 0>(A, sm, row, col);
}

}  // namespace mhd
