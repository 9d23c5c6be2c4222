// mhd_btma.cuh -- B_{t1->d}, B_{t2->d} for sweeps along y and z: tile march fed by a TMA bulk-copy ring.
//
// Same dataflow as mhd_btile.cuh (a block owns a TX x TO tile of pencils in the (x, o) plane and marches
// along d in lock step; every thread runs only its own two flux pipelines; one extra row of threads runs
// the pipelines of row o0+TO and column x0+TX; finished edge fluxes are exchanged through double-buffered
// shared memory), but no consumer thread ever forms a global LOAD address: a producer warp brings, for
// every march step, the rows of rho, m_d (tile + one-cell halo), B_x, B_o and B_d into a D-stage
// shared-memory ring with cp.async.bulk (SASS UBLKCP), one contiguous row per copy, the copies spread over
// the 32 producer lanes, completion on an mbarrier per stage.  Consumers read their operands with
// LDS [thread offset + immediate].  ncu on the register/LDG version showed 264 instructions per cell of
// which ~65 floating point (profiles/r01_c4_step_ncu_full.md): the rest was 64-bit address arithmetic.
//
// Algorithm 2, eqs (20)-(22) PAPER.md:147-158; constraint step PAPER.md:160.
//
// Requirements (else bpair_tile_kernel / bpair_yz_kernel run): nx % TX == 0, no % TO == 0,
// nx*sizeof(real) % 16 == 0, TX*sizeof(real) % 16 == 0.
#pragma once
#include "mhd_async.cuh"
#include "mhd_yz.cuh"

namespace mhd {

template <class real, int TX, int TO>
struct BRing {
  static constexpr int CH = 16 / sizeof(real);          // elements in one 16-byte chunk
  static constexpr int P = TX + 2 * CH;                  // row pitch: [left chunk][TX cells][right chunk]
  // row blocks of one stage
  static constexpr int R_RHO = 0;                        // TO+2 rows: o0-1 .. o0+TO
  static constexpr int R_MD = R_RHO + TO + 2;            // TO+2 rows
  static constexpr int R_BX = R_MD + TO + 2;             // TO rows (+ right chunk: column x0+TX)
  static constexpr int R_BO = R_BX + TO;                 // TO+1 rows: o0 .. o0+TO
  static constexpr int R_BD = R_BO + TO + 1;             // TO rows, of the cell 4 steps behind
  static constexpr int ROWS = R_BD + TO;
  static constexpr int STAGE = ROWS * P;                 // reals per stage
  static constexpr int NCHUNK = 5 * TO;                  // rho, m_d: left+right for the TO tile rows; B_x: right
  static constexpr int NCOPY = ROWS + NCHUNK;
  static constexpr int KPL = (NCOPY + 31) / 32;          // copies per producer lane
  static constexpr uint32_t BYTES = ROWS * TX * sizeof(real) + NCHUNK * 16;
  static constexpr int NT = (TO + 1) * TX;               // consumer threads
  static size_t smem_bytes(int D) {
    return (size_t)D * STAGE * sizeof(real) + 2 * D * sizeof(uint64_t) +
           2 * (size_t)(TO * (TX + 1) + 1 + (TO + 1) * TX) * sizeof(real);
  }
};

template <class real, int TX, int TO, int D>
__global__ void __launch_bounds__((TO + 1) * TX + 32) bpair_tma_kernel(const YZArgs<real> A) {
  using RG = BRing<real, TX, TO>;
  constexpr int CH = RG::CH, P = RG::P, NT = RG::NT;
  constexpr int MD = (RG::R_MD - RG::R_RHO) * P;        // rho slot -> m_d slot
  constexpr int NFX = TO * (TX + 1) + 1, NFO = (TO + 1) * TX;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;
  real* sFX = reinterpret_cast<real*>(empty + D);        // [2][NFX]  B_x-row fluxes at (o_local, x_local <= TX)
  real* sFO = sFX + 2 * NFX;                             // [2][NFO]  B_o-row fluxes at (o_local <= TO, x_local)

  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TX, o0 = blockIdx.y * TO;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = n1 - n0 + 8;                         // cells n0-4 .. n1+3
  const int xl = map_index1(x0 - 1, A.nx, A.bc), xr = map_index1(x0 + TX, A.nx, A.bc);
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], 1); }
    mbar_fence_init();
  }
  __syncthreads();

  if (tid >= NT) {
    // ---------------- producer warp: lane l issues copies l, l+32, ... of every stage ----------------
    const int lane = tid - NT;
    const real* src[RG::KPL];
    int dst[RG::KPL], nbytes[RG::KPL], late[RG::KPL];
#pragma unroll
    for (int k = 0; k < RG::KPL; ++k) {
      const int c = lane + 32 * k;
      src[k] = nullptr; dst[k] = 0; nbytes[k] = 0; late[k] = 0;
      if (c >= RG::NCOPY) continue;
      int r, xoff, doff, nb;                             // stage row, source x offset, destination offset in the row, bytes
      if (c < RG::ROWS) { r = c; xoff = x0; doff = CH; nb = TX * (int)sizeof(real); }
      else {
        const int e = c - RG::ROWS;
        int side;
        if (e < 2 * TO)      { r = RG::R_RHO + 1 + (e >> 1); side = e & 1; }
        else if (e < 4 * TO) { r = RG::R_MD + 1 + ((e - 2 * TO) >> 1); side = e & 1; }
        else                 { r = RG::R_BX + (e - 4 * TO); side = 1; }
        xoff = ((side ? xr : xl) / CH) * CH;
        doff = side ? CH + TX : 0;
        nb = 16;
      }
      const real* f; int orow;
      if (r < RG::R_MD)      { f = A.u[0]; orow = o0 - 1 + (r - RG::R_RHO); }
      else if (r < RG::R_BX) { f = A.u[1]; orow = o0 - 1 + (r - RG::R_MD); }
      else if (r < RG::R_BO) { f = A.bx;   orow = o0 + (r - RG::R_BX); }
      else if (r < RG::R_BD) { f = A.bo;   orow = o0 + (r - RG::R_BO); }
      else                   { f = A.bd;   orow = o0 + (r - RG::R_BD); late[k] = 1; }
      src[k] = f + (size_t)map_index1(orow, A.no, A.bc) * A.so + xoff;
      dst[k] = r * P + doff;
      nbytes[k] = nb;
    }
    for (int it = 0; it < niter; ++it) {
      const int s = it % D;
      if (it >= D) mbar_wait(&empty[s], ((it / D) & 1) ^ 1);
      const int q = n0 - 4 + it;
      const int od = map_index1(q, A.nd, A.bc) * A.sd;
      const int od4 = map_index1(q - 4, A.nd, A.bc) * A.sd;          // B_d of the cell finished this step (nd >= 8)
      real* st = ring + s * RG::STAGE;
      if (lane == 0) mbar_expect_tx(&full[s], RG::BYTES);
      __syncwarp();
#pragma unroll
      for (int k = 0; k < RG::KPL; ++k)
        if (nbytes[k]) bulk_g2s(st + dst[k], src[k] + (late[k] ? od4 : od), (uint32_t)nbytes[k], &full[s]);
    }
    return;
  }

  // ---------------- consumers ----------------
  const int row = tid / TX, col = tid - row * TX;
  const bool halo = row == TO;
  const bool hasX = !halo || col < TO;
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt;
  const int xlm = xl % CH, xrm = xr % CH;
  // slot of rho at tile coordinates (c, r), c in -1..TX, r in -1..TO
  auto slotU = [&](int c, int r) { return (RG::R_RHO + r + 1) * P + (c < 0 ? xlm : (c >= TX ? CH + TX + xrm : CH + c)); };
  // my two pipelines: O = B_o row (interior: my cell; halo: row o0+TO), X = B_x row (interior: my cell; halo lanes < TO: column x0+TX)
  const int cOc = slotU(col, halo ? TO : row), cOn = cOc - P;
  const int cXc = halo ? slotU(TX, hasX ? col : 0) : cOc;
  const int cXn = halo ? slotU(TX - 1, hasX ? col : 0) : slotU(col - 1, row);
  const int bXs = halo ? (RG::R_BX + (hasX ? col : 0)) * P + CH + TX + xrm : (RG::R_BX + row) * P + CH + col;
  const int bOs = (RG::R_BO + (halo ? TO : row)) * P + CH + col;
  const int bDs = (RG::R_BD + (halo ? 0 : row)) * P + CH + col;
  const int fXw = halo ? (hasX ? col * (TX + 1) + TX : TO * (TX + 1)) : row * (TX + 1) + col;   // dummy slot for idle lanes
  const int fOw = (halo ? TO : row) * TX + col;
  const int fXr = (halo ? 0 : row) * (TX + 1) + col + 1, fOr = ((halo ? 0 : row) + 1) * TX + col;
  const int offO = x0 + col + (o0 + (halo ? 0 : row)) * A.so;
  const bool x_first = (A.x_is_t1 != 0) != (A.t2_first != 0);        // forward: t1 then t2; reverse: t2 then t1

  BPipe<real> px, po;
  px.init(); po.init();
  int s = 0;
  uint32_t ph = 0;
  int off = (n0 - 8) * A.sd + offO;                                    // output cell m = q-4 = n0 + it - 8
  for (int it = 0; it < niter; ++it) {
    const real* st = ring + s * RG::STAGE;
    const int buf = it & 1;
    mbar_wait(&full[s], ph);
    const real rOc = st[cOc], rOn = st[cOn], mOc = st[cOc + MD], mOn = st[cOn + MD];
    const real rXc = st[cXc], rXn = st[cXn], mXc = st[cXc + MD], mXn = st[cXn + MD];
    const real bX = st[bXs], bO = st[bOs], bdv0 = st[bDs];
    // publish the fluxes finished in the previous step (= this step's flux at face m-1/2)
    sFX[buf * NFX + fXw] = px.fhi();
    sFO[buf * NFO + fOw] = po.fhi();
    asm volatile("bar.sync 1, %0;" ::"n"(NT) : "memory");            // consumers only (the producer warp never joins)
    if (tid == 0) mbar_arrive(&empty[s]);                            // every consumer has read stage s
    if (++s == D) { s = 0; ph ^= 1; }
    // Alg. 2 step 4: face velocity = momentum sum / density sum of the two cells sharing the face (reading R5)
    const real vtX = (mXn + mXc) * rcp_(rXn + rXc);
    const real vtO = (mOn + mOc) * rcp_(rOn + rOc);
    px.push(vtX, bX, dt, hdt);
    po.push(vtO, bO, dt, hdt);
    if (!halo && it >= 8) {
      A.bxo[off] = px.bold() - (px.fhi() - px.flo());                // Alg. 2 step 9: advect B_t
      A.boo[off] = po.bold() - (po.fhi() - po.flo());
      // constraint with the same fluxes at face m-1/2: the neighbours published theirs above
      const real cx = sFX[buf * NFX + fXr] - px.flo();
      const real co = sFO[buf * NFO + fOr] - po.flo();
      real bdv = bdv0;
      if (x_first) { bdv = bdv + cx; bdv = bdv + co; }
      else         { bdv = bdv + co; bdv = bdv + cx; }
      A.bdo[off] = bdv;
    }
    off += A.sd;
  }
}

}  // namespace mhd
