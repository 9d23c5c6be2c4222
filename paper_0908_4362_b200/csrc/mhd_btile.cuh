// mhd_btile.cuh -- B_{t1->d}, B_{t2->d} for sweeps along y and z as a "tile march".
//
// Algorithm 2 needs, for the constraint update of B_d in cell (i,o), the edge
// fluxes of the rows i+1 and o+1 as well, and, for the face velocities, rho and m_d
// of the cells i-1 and o-1.  Instead of every thread recomputing its neighbours' flux pipelines and
// re-reading their rho, m_d from global memory (mhd_yz.cuh: 4 pipelines, 15 loads per cell), a block
// owns a TX x TO tile of pencils in the (x, o) plane and marches along d in lock step:
//   * every thread runs only its own two pipelines (B_x row i, B_o row o),
//   * rho, m_d and the finished fluxes are exchanged through double-buffered shared memory with one
//     __syncthreads per march step,
//   * one extra "halo" row of threads runs the B_o pipelines of row o0+TO and, in its first TO lanes,
//     the B_x pipelines of column x0+TX, so nothing else is recomputed (overhead 1/TO).
// Per cell: 5 global loads (rho, m_d, B_x, B_o, B_d) + 3 stores, 2 pipelines.
//
// Requirements (else bpair_yz_kernel runs): nx % TX == 0, no % TO == 0, extent along the sweep >= 8.
#pragma once
#include "mhd_yz.cuh"

namespace mhd {

template <class real, int TX, int TO>
__global__ void __launch_bounds__((TO + 1) * TX) bpair_tile_kernel(const YZArgs<real> A) {
  static_assert(TO <= 32 && TX % 32 == 0, "tile shape");
  constexpr int TW = TX + 2, TH = TO + 2;
  __shared__ real sR[2][TH * TW], sM[2][TH * TW];      // rho, m_d at tile coords (o_local+1, x_local+1)
  __shared__ real sFX[2][TO * (TX + 1) + 1];           // B_x-row fluxes at (o_local, x_local), x_local <= TX; +1 dummy
  __shared__ real sFO[2][(TO + 1) * TX];               // B_o-row fluxes at (o_local <= TO, x_local)

  const int tid = threadIdx.x;
  const int row = tid / TX, col = tid - row * TX;
  const bool halo = row == TO;
  const int x0 = blockIdx.x * TX, o0 = blockIdx.y * TO;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt;

  // ---- where my two pipelines sit (global, index-mapped) and where they live in the tiles --------
  const int iO = x0 + col;
  const int oO = halo ? map_index1(o0 + TO, A.no, A.bc) : o0 + row;
  const bool hasX = !halo || col < TO;
  const int iX = halo ? map_index1(x0 + TX, A.nx, A.bc) : iO;
  const int oX = halo ? o0 + (hasX ? col : 0) : oO;
  const int offO = iO + oO * A.so, offX = iX + oX * A.so;
  const int tO = (halo ? TO + 1 : row + 1) * TW + col + 1;          // tile slot of the O position
  const int tX = halo ? (hasX ? (col + 1) * TW + TX + 1 : tO) : tO;  // tile slot of the X position
  const int nbX = tX - 1;                                            // cell x-1 of the X pipeline
  const int nbO = tO - TW;                                           // cell o-1 of the O pipeline
  const int fXw = halo ? (hasX ? col * (TX + 1) + TX : TO * (TX + 1)) : row * (TX + 1) + col;   // dummy slot for idle lanes
  const int fOw = (halo ? TO : row) * TX + col;
  const int fXr = row * (TX + 1) + col + 1, fOr = (row + 1) * TX + col;      // interior only
  // extra tile cells loaded by interior threads: row o0-1 (by row 0) and column x0-1 (by column 0)
  const bool exR = !halo && row == 0, exC = !halo && col == 0;
  const int offR = iO + map_index1(o0 - 1, A.no, A.bc) * A.so;
  const int offC = map_index1(x0 - 1, A.nx, A.bc) + oO * A.so;
  const int tR = col + 1, tC = (row + 1) * TW;

  const real* __restrict__ rho = A.u[0];
  const real* __restrict__ md = A.u[1];

  struct In { real rO, mO, rX, mX, rE, mE, rF, mF, bX, bO; };
  auto load = [&](int q, In& c) {
    const int od = map_index1(q, A.nd, A.bc) * A.sd;
    c.rO = __ldg(rho + od + offO); c.mO = __ldg(md + od + offO);
    if (halo) { c.rX = __ldg(rho + od + offX); c.mX = __ldg(md + od + offX); }
    else { c.rX = c.rO; c.mX = c.mO; }
    if (exR) { c.rE = __ldg(rho + od + offR); c.mE = __ldg(md + od + offR); }
    if (exC) { c.rF = __ldg(rho + od + offC); c.mF = __ldg(md + od + offC); }
    c.bX = __ldg(A.bx + od + offX);
    c.bO = __ldg(A.bo + od + offO);
  };

  BPipe<real> px, po;
  px.init(); po.init();
  In cur, nxt;
  cur.rE = cur.mE = cur.rF = cur.mF = real(1);
  nxt = cur;
  load(n0 - 4, cur);
  for (int q = n0 - 4; q < n1 + 4; ++q) {
    const int buf = q & 1;
    const int m = q - 4;
    real bdv = real(0);
    if (!halo && m >= n0) bdv = __ldg(A.bd + m * A.sd + offO);
    if (q + 1 < n1 + 4) load(q + 1, nxt);
    // publish rho, m_d of this march step and the fluxes finished in the previous one
    sR[buf][tO] = cur.rO; sM[buf][tO] = cur.mO;
    if (halo && hasX) { sR[buf][tX] = cur.rX; sM[buf][tX] = cur.mX; }
    if (exR) { sR[buf][tR] = cur.rE; sM[buf][tR] = cur.mE; }
    if (exC) { sR[buf][tC] = cur.rF; sM[buf][tC] = cur.mF; }
    sFX[buf][fXw] = px.fhi();
    sFO[buf][fOw] = po.fhi();
    __syncthreads();
    // Alg. 2 step 4: face velocity = momentum sum / density sum of the two cells sharing the face (reading R5)
    const real vtX = (sM[buf][nbX] + cur.mX) * rcp_(sR[buf][nbX] + cur.rX);
    const real vtO = (sM[buf][nbO] + cur.mO) * rcp_(sR[buf][nbO] + cur.rO);
    px.push(vtX, cur.bX, dt, hdt);
    po.push(vtO, cur.bO, dt, hdt);
    if (!halo && m >= n0) {
      const int off = m * A.sd + offO;
      A.bxo[off] = px.bold() - (px.fhi() - px.flo());        // Alg. 2 step 9: advect B_t
      A.boo[off] = po.bold() - (po.fhi() - po.flo());
      // constraint with the same fluxes at face m-1/2: the neighbours published theirs above
      const real cx = sFX[buf][fXr] - px.flo();
      const real co = sFO[buf][fOr] - po.flo();
      const bool x_first = (A.x_is_t1 != 0) != (A.t2_first != 0);   // forward: t1 then t2; reverse: t2 then t1
      if (x_first) { bdv = bdv + cx; bdv = bdv + co; }
      else         { bdv = bdv + co; bdv = bdv + cx; }
      A.bdo[off] = bdv;
    }
    cur = nxt;
  }
}

}  // namespace mhd
