// mhd_bring.cuh -- B_{t1->d}, B_{t2->d} for sweeps along y and z: a march with NO block barrier.
//
// Algorithm 2, eqs (20)-(22) PAPER.md:147-158; constraint step PAPER.md:160.
//
// A block owns one row of TXB pencils (fixed o, x0 <= x < x0+TXB) and marches along d.  The warp on duty
// brings, for every march step, the ten rows the step needs (rho and m_d of the rows o-1, o, o+1; B_x of
// row o; B_o of rows o, o+1; B_d of the cell that is finished in this step, four cells behind) plus the
// 16-byte chunks holding the columns x0-1 and x0+TXB into a D-stage shared-memory ring with
// cp.async.bulk (SASS UBLKCP), one copy per lane, completion on an mbarrier per stage.
// A consumer thread owns L adjacent pencils (L = 2 in packed f2 arithmetic for fp32, mhd_pack.cuh;
// L = 1 for fp64) and runs every flux pipeline its own cells need:
//     pxA  B_x rows (faces) of its own L columns        pxE  B_x row of the column to its right (scalar)
//     po   B_o row o                                     pop  B_o row o+1
// The +1 rows (pxE, pop) supply the constraint update of B_d and are recomputed instead of
// exchanged: compared with a tile march that exchanges fluxes behind a block barrier (round 1: 1.11 ms) that costs arithmetic (which packed f2
// instructions make cheap) and buys a kernel with no __syncthreads, no shared-memory flux exchange, no
// global LOAD address arithmetic in the consumers, and warps that drift freely up to the ring depth.
// A stage is released as soon as its rows are in registers, so the producer runs D-1 march steps ahead
// (ncu on a first version that re-read B_t(k-4) from the ring and so kept stages four steps longer showed
// the consumers waiting on the full-barriers: 4 stages in flight do not cover the HBM latency).
//
// Requirements (else bpair_march_kernel of mhd_generic.cuh runs): nx a multiple of 16 bytes (a narrower last tile per row
// is allowed, as in mhd_yz2.cuh), extent along d >= 8.
#pragma once
#include <type_traits>
#include "mhd_args.cuh"
#include "mhd_async.cuh"
#include "mhd_pack_io.cuh"

namespace mhd {

template <class real, int TXB>
struct BRowRing {
  static constexpr int CH = 16 / sizeof(real);           // elements in one 16-byte chunk
  static constexpr int P = TXB + 2 * CH;                 // row pitch: [left chunk][TXB cells][right chunk]
  enum { R_RHO = 0, R_MD = 3, R_BX = 6, R_BO = 7, R_BD = 9, ROWS = 10, NCHUNK = 5, NCOPY = ROWS + NCHUNK };
  static constexpr int STAGE = ROWS * P;
  static constexpr uint32_t BYTES = ROWS * TXB * sizeof(real) + NCHUNK * 16;
  static size_t smem_bytes(int D) { return (size_t)D * STAGE * sizeof(real) + 2 * D * sizeof(uint64_t); }
};

// Measured at 512^3 fp32 (ms per launch; tile march with a block barrier: 1.11): dedicated producer warp,
// 2 blocks/SM 1.17; rotating duty, 3 blocks/SM, 6-7 stages: no slack 1.05, slack 1-2 0.87; 2 blocks/SM,
// 10 stages, slack 3 1.04; 4 blocks/SM (128 registers, spills) 1.55.
#ifndef MHD_BRING_MINB
#define MHD_BRING_MINB 3
#endif
#ifndef MHD_BRING_STAGES
#define MHD_BRING_STAGES 7
#endif
// the warp on duty refills a stage that every warp released SLACK+1 steps ago: with no slack the duty
// warp waits for the slowest warp every step, which couples the warps like a block barrier
#ifndef MHD_BRING_SLACK
#define MHD_BRING_SLACK 1
#endif

// real: element type in memory (float/double).  T: arithmetic pack (f2 for float, double for double).
// No producer warp: the warps take turns (march step modulo the warp count) at issuing the copies of the
// stage PF steps ahead, one copy per lane (see mhd_yz2.cuh for why).
template <class real, class T, int TXB, int D, bool RAG = false>
__global__ void __launch_bounds__(TXB / PackOf<T>::L, MHD_BRING_MINB) bpair_ring_kernel(const YZArgs<real> A) {
  using RG = BRowRing<real, TXB>;
  constexpr int L = PackOf<T>::L;
  constexpr int NC = TXB / L;                             // threads (all consumers)
  constexpr int NW = NC / 32;
  constexpr int PF = D - 1 - MHD_BRING_SLACK;            // the stage of step it+PF was last read at step it-1-SLACK
  constexpr int CH = RG::CH, P = RG::P;
  static_assert(NW >= 1 && (NW & (NW - 1)) == 0 && NW <= 4, "block shape");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;

  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // the same value, warp-uniform for the compiler too
  const int x0 = blockIdx.x * TXB, o = blockIdx.y;
  const int w = RAG ? min(TXB, A.nx - x0) : TXB;          // columns of this tile (RAG: the row ends in a narrower one)
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = (n1 - n0 + 8 + 3) & ~3;               // cells n0-4 .. n1+3, rounded up to the 4x unrolled march
  const int xl = map_index1(x0 - 1, A.nx, A.bc), xr = map_index1(x0 + w, A.nx, A.bc);
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NW); }
    mbar_fence_init();
  }
  __syncthreads();

  // ---- producer duty: one elected lane of the warp on duty issues the NCOPY copies of a stage; every operand is
  // warp-uniform (block indices, kernel parameters, the march step), so they are straight-line UBLKCPs (mhd_async.cuh).
  // Sources are  rho + (march offset) + (row / chunk byte offset of this block) + A.src[field]  (A.src in the constant bank)
  constexpr long long ES = (long long)sizeof(real);
  const long long om_b = (long long)(map_index1(o - 1, A.no, A.bc) * A.so + x0) * ES, o_b = (long long)(o * A.so + x0) * ES,
                  op_b = (long long)(map_index1(o + 1, A.no, A.bc) * A.so + x0) * ES;
  const long long cl_b = o_b + (long long)((xl / CH) * CH - x0) * ES, cr_b = o_b + (long long)((xr / CH) * CH - x0) * ES;   // the 16-byte chunks holding columns x0-1, x0+TXB of row o
  auto produce = [&](int itp) {                           // called by one whole, converged warp
    const unsigned s = (unsigned)itp % D;
    if (itp >= D) mbar_wait(&empty[s], (((unsigned)itp / D) & 1) ^ 1);
    if (elect_one()) {
      const int od = map_index1(n0 - 4 + itp, A.nd, A.bc) * A.sd;
      const int odl = map_index1(n0 - 8 + itp, A.nd, A.bc) * A.sd;        // B_d of the cell finished at this step
      real* st = ring + s * RG::STAGE;
      uint64_t* bar = &full[s];
      const uint32_t RB = (uint32_t)w * sizeof(real);
      const char* rho = reinterpret_cast<const char*>(A.u[0] + od);
      const char* md = rho + A.src[1];
      mbar_expect_tx(bar, (uint32_t)RG::ROWS * RB + RG::NCHUNK * 16u);
      bulk_g2s(st + 0 * P + CH, rho + om_b, RB, bar);
      bulk_g2s(st + 1 * P + CH, rho + o_b, RB, bar);
      bulk_g2s(st + 2 * P + CH, rho + op_b, RB, bar);
      bulk_g2s(st + 3 * P + CH, md + om_b, RB, bar);
      bulk_g2s(st + 4 * P + CH, md + o_b, RB, bar);
      bulk_g2s(st + 5 * P + CH, md + op_b, RB, bar);
      bulk_g2s(st + 6 * P + CH, rho + A.src[7] + o_b, RB, bar);
      bulk_g2s(st + 7 * P + CH, rho + A.src[6] + o_b, RB, bar);
      bulk_g2s(st + 8 * P + CH, rho + A.src[6] + op_b, RB, bar);
      bulk_g2s(st + 9 * P + CH, reinterpret_cast<const char*>(A.u[0] + odl) + A.src[5] + o_b, RB, bar);
      bulk_g2s(st + 1 * P, rho + cl_b, 16, bar);
      bulk_g2s(st + 1 * P + CH + w, rho + cr_b, 16, bar);
      bulk_g2s(st + 4 * P, md + cl_b, 16, bar);
      bulk_g2s(st + 4 * P + CH + w, md + cr_b, 16, bar);
      bulk_g2s(st + 6 * P + CH + w, rho + A.src[7] + cr_b, 16, bar);
    }
    __syncwarp();
  };
  for (int itp = warp; itp < PF && itp < niter; itp += NW) produce(itp);

  // ---------------- consumers: L adjacent pencils each ----------------
  typedef typename PackOf<T>::scalar S;
  const int cx = CH + L * tid;                            // my first column inside a stage row
  const int iL = tid == 0 ? xl % CH : cx - 1;             // column to my left / right (the chunks at the row ends)
  const int iR = L * tid + L == w ? CH + w + xr % CH : cx + L;
  const bool active = L * tid < w;                        // threads beyond a narrow last tile store nothing
  const S dts = (S)(*A.dt);
  const T dt(dts), hdt(S(0.5) * dts);
  const bool x_first = (A.x_is_t1 != 0) != (A.t2_first != 0);     // forward: t1 then t2; reverse: t2 then t1

  BPipe4<T> pxA, po, pop;
  BPipe4<S> pxE;
  pxA.init(); po.init(); pop.init(); pxE.init();
  int off = (n0 - 8) * A.sd + x0 + L * tid + o * A.so;    // output cell m = q - 4 = n0 + it - 8
  int stg = 0;                                            // ring stage of this march step and its phase parity
  uint32_t ph = 0;

  auto step = [&](auto Ktag, int it) {
    constexpr int K = decltype(Ktag)::value;
    if ((K & (NW - 1)) == warp && it + PF < niter) produce(it + PF);
    const real* st = ring + stg * RG::STAGE;
    mbar_wait(&full[stg], ph);
    T* tag = nullptr;
    const T rm = ld_pack(st + 0 * P + cx, tag), r0 = ld_pack(st + 1 * P + cx, tag), rp = ld_pack(st + 2 * P + cx, tag);
    const T mm = ld_pack(st + 3 * P + cx, tag), m0 = ld_pack(st + 4 * P + cx, tag), mp = ld_pack(st + 5 * P + cx, tag);
    const S rl = st[1 * P + iL], rr = st[1 * P + iR], ml = st[4 * P + iL], mr = st[4 * P + iR];
    const T bx = ld_pack(st + 6 * P + cx, tag);
    const S bxr = st[6 * P + iR];
    const T bo = ld_pack(st + 7 * P + cx, tag), bop = ld_pack(st + 8 * P + cx, tag);
    const T bd = ld_pack(st + 9 * P + cx, tag);             // B_d of the cell finished now (copied 4 cells behind)
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[stg]);                // this warp's reads of the stage are done
    if (++stg == D) { stg = 0; ph ^= 1; }
    // Alg. 2 step 4: face velocity = momentum sum / density sum of the two cells sharing the face (reading R5)
    const T vtA = (shift_in_left(m0, ml) + m0) * rcp_(shift_in_left(r0, rl) + r0);
    const S vtE = (last_lane(m0) + mr) * rcp_(last_lane(r0) + rr);
    const T vtO = (mm + m0) * rcp_(rm + r0);
    const T vtP = (m0 + mp) * rcp_(r0 + rp);
    T bxn, bon, bpn, fxlo, folo, fplo;
    S ben, felo;
    pxA.template push<K>(vtA, bx, dt, hdt, bxn, fxlo);
    pxE.template push<K>(vtE, bxr, dts, S(0.5) * dts, ben, felo);
    po.template push<K>(vtO, bo, dt, hdt, bon, folo);
    pop.template push<K>(vtP, bop, dt, hdt, bpn, fplo);
    const int m = n0 + it - 8;
    if (it >= 8 && m < n1 && active) {
      st_pack(A.bxo + off, bxn);                            // Alg. 2 step 9: advected B_t
      st_pack(A.boo + off, bon);
      // constraint with the same fluxes at face m-1/2: rows x+1 and o+1
      const T cxv = shift_in_right(fxlo, felo) - fxlo;
      const T cov = fplo - folo;
      T bdv = bd;
      if (x_first) { bdv = bdv + cxv; bdv = bdv + cov; }
      else         { bdv = bdv + cov; bdv = bdv + cxv; }
      st_pack(A.bdo + off, bdv);
    }
    off += A.sd;
  };
  for (int it = 0; it < niter; it += 4) {
    step(std::integral_constant<int, 0>{}, it);
    step(std::integral_constant<int, 1>{}, it + 1);
    step(std::integral_constant<int, 2>{}, it + 2);
    step(std::integral_constant<int, 3>{}, it + 3);
  }
}

// ---------------------------------------------------------------------------------------------------------------
// The same march with TWO rows (o, o+1) per thread.  The flux row o+1 that the constraint step of row o needs (pop above)
// is the thread's own row-o+1 pipeline, and the two scalar edge pipelines (pxE of either row) share ONE packed pipeline
// whose lanes are the two rows: six packed pipelines for four pencils instead of eight, fifteen row copies per stage for two
// rows instead of twenty, and every per-step cost (barrier waits, producer duty, loop, store offsets) once for two rows.
// The price is registers: six pipelines are 192 registers of state, so two blocks of four warps per SM, each thread
// with six independent dependency chains.  Requirements as above plus an even extent along o; fp32 (T = f2) only.
//   stage rows: 0-3 rho(o-1..o+2)  4-7 m_d(o-1..o+2)  8,9 B_x(o, o+1)  10-12 B_o(o..o+2)  13,14 B_d(o, o+1) four cells behind
//   chunks (columns x0-1 / x0+TXB): rho and m_d of rows o, o+1 (left and right), B_x of rows o, o+1 (right)
// ---------------------------------------------------------------------------------------------------------------
template <class real, int TXB>
struct BRowRing2 {
  static constexpr int CH = 16 / sizeof(real);
  static constexpr int P = TXB + 2 * CH;
  enum { ROWS = 15, NCHUNK = 10 };
  static constexpr int STAGE = ROWS * P;
  static constexpr uint32_t BYTES = ROWS * TXB * sizeof(real) + NCHUNK * 16;
  static size_t smem_bytes(int D) { return (size_t)D * STAGE * sizeof(real) + 2 * D * sizeof(uint64_t); }
};

#ifndef MHD_BRING2_STAGES
#define MHD_BRING2_STAGES 7
#endif
#ifndef MHD_BRING2_SLACK
#define MHD_BRING2_SLACK 1
#endif

template <int TXB, int D, bool RAG = false>
__global__ void __launch_bounds__(TXB / 2, TXB == 256 ? 2 : 4) bpair_ring2_kernel(const YZArgs<float> A) {
  typedef float real;
  typedef f2 T;
  typedef float S;
  using RG = BRowRing2<real, TXB>;
  constexpr int L = 2;
  constexpr int NC = TXB / L;
  constexpr int NW = NC / 32;
  constexpr int PF = D - 1 - MHD_BRING2_SLACK;
  constexpr int CH = RG::CH, P = RG::P;
  static_assert(NW >= 1 && (NW & (NW - 1)) == 0 && NW <= 4, "block shape");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;

  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int x0 = blockIdx.x * TXB, o = 2 * blockIdx.y;
  const int w = RAG ? min(TXB, A.nx - x0) : TXB;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = (n1 - n0 + 8 + 3) & ~3;
  const int xl = map_index1(x0 - 1, A.nx, A.bc), xr = map_index1(x0 + w, A.nx, A.bc);
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NW); }
    mbar_fence_init();
  }
  __syncthreads();

  constexpr long long ES = (long long)sizeof(real);
  const long long om_b = (long long)(map_index1(o - 1, A.no, A.bc) * A.so + x0) * ES, o_b = (long long)(o * A.so + x0) * ES,
                  o1_b = (long long)((o + 1) * A.so + x0) * ES, o2_b = (long long)(map_index1(o + 2, A.no, A.bc) * A.so + x0) * ES;
  const long long cl_b = (long long)((xl / CH) * CH - x0) * ES, cr_b = (long long)((xr / CH) * CH - x0) * ES;   // chunk offsets inside a row
  auto produce = [&](int itp) {
    const unsigned s = (unsigned)itp % D;
    if (itp >= D) mbar_wait(&empty[s], (((unsigned)itp / D) & 1) ^ 1);
    if (elect_one()) {
      const int od = map_index1(n0 - 4 + itp, A.nd, A.bc) * A.sd;
      const int odl = map_index1(n0 - 8 + itp, A.nd, A.bc) * A.sd;
      real* st = ring + s * RG::STAGE;
      uint64_t* bar = &full[s];
      const uint32_t RB = (uint32_t)w * sizeof(real);
      const char* rho = reinterpret_cast<const char*>(A.u[0] + od);
      const char* md = rho + A.src[1];
      const char* bx = rho + A.src[7];
      const char* bo = rho + A.src[6];
      const char* bd = reinterpret_cast<const char*>(A.u[0] + odl) + A.src[5];
      mbar_expect_tx(bar, (uint32_t)RG::ROWS * RB + RG::NCHUNK * 16u);
      bulk_g2s(st + 0 * P + CH, rho + om_b, RB, bar);
      bulk_g2s(st + 1 * P + CH, rho + o_b, RB, bar);
      bulk_g2s(st + 2 * P + CH, rho + o1_b, RB, bar);
      bulk_g2s(st + 3 * P + CH, rho + o2_b, RB, bar);
      bulk_g2s(st + 4 * P + CH, md + om_b, RB, bar);
      bulk_g2s(st + 5 * P + CH, md + o_b, RB, bar);
      bulk_g2s(st + 6 * P + CH, md + o1_b, RB, bar);
      bulk_g2s(st + 7 * P + CH, md + o2_b, RB, bar);
      bulk_g2s(st + 8 * P + CH, bx + o_b, RB, bar);
      bulk_g2s(st + 9 * P + CH, bx + o1_b, RB, bar);
      bulk_g2s(st + 10 * P + CH, bo + o_b, RB, bar);
      bulk_g2s(st + 11 * P + CH, bo + o1_b, RB, bar);
      bulk_g2s(st + 12 * P + CH, bo + o2_b, RB, bar);
      bulk_g2s(st + 13 * P + CH, bd + o_b, RB, bar);
      bulk_g2s(st + 14 * P + CH, bd + o1_b, RB, bar);
      bulk_g2s(st + 1 * P, rho + o_b + cl_b, 16, bar);
      bulk_g2s(st + 1 * P + CH + w, rho + o_b + cr_b, 16, bar);
      bulk_g2s(st + 2 * P, rho + o1_b + cl_b, 16, bar);
      bulk_g2s(st + 2 * P + CH + w, rho + o1_b + cr_b, 16, bar);
      bulk_g2s(st + 5 * P, md + o_b + cl_b, 16, bar);
      bulk_g2s(st + 5 * P + CH + w, md + o_b + cr_b, 16, bar);
      bulk_g2s(st + 6 * P, md + o1_b + cl_b, 16, bar);
      bulk_g2s(st + 6 * P + CH + w, md + o1_b + cr_b, 16, bar);
      bulk_g2s(st + 8 * P + CH + w, bx + o_b + cr_b, 16, bar);
      bulk_g2s(st + 9 * P + CH + w, bx + o1_b + cr_b, 16, bar);
    }
    __syncwarp();
  };
  for (int itp = warp; itp < PF && itp < niter; itp += NW) produce(itp);

  const int cx = CH + L * tid;
  const int iL = tid == 0 ? xl % CH : cx - 1;
  const int iR = L * tid + L == w ? CH + w + xr % CH : cx + L;
  const bool active = L * tid < w;
  const S dts = (S)(*A.dt);
  const T dt(dts), hdt(S(0.5) * dts);
  const bool x_first = (A.x_is_t1 != 0) != (A.t2_first != 0);

  BPipe4<T> pxA0, pxA1, pxE, po0, po1, po2;
  pxA0.init(); pxA1.init(); pxE.init(); po0.init(); po1.init(); po2.init();
  int off = (n0 - 8) * A.sd + x0 + L * tid + o * A.so;    // output cell m = q - 4 = n0 + it - 8, row o (row o+1: + A.so)
  int stg = 0;
  uint32_t ph = 0;

  auto step = [&](auto Ktag, int it) {
    constexpr int K = decltype(Ktag)::value;
    if ((K & (NW - 1)) == warp && it + PF < niter) produce(it + PF);
    const real* st = ring + stg * RG::STAGE;
    mbar_wait(&full[stg], ph);
    T* tag = nullptr;
    const T r0 = ld_pack(st + 0 * P + cx, tag), r1 = ld_pack(st + 1 * P + cx, tag), r2 = ld_pack(st + 2 * P + cx, tag), r3 = ld_pack(st + 3 * P + cx, tag);
    const T m0 = ld_pack(st + 4 * P + cx, tag), m1 = ld_pack(st + 5 * P + cx, tag), m2 = ld_pack(st + 6 * P + cx, tag), m3 = ld_pack(st + 7 * P + cx, tag);
    const T rl(st[1 * P + iL], st[2 * P + iL]), rr(st[1 * P + iR], st[2 * P + iR]);      // lanes: rows o, o+1
    const T ml(st[5 * P + iL], st[6 * P + iL]), mr(st[5 * P + iR], st[6 * P + iR]);
    const T bx0 = ld_pack(st + 8 * P + cx, tag), bx1 = ld_pack(st + 9 * P + cx, tag);
    const T bxr(st[8 * P + iR], st[9 * P + iR]);
    const T bo0 = ld_pack(st + 10 * P + cx, tag), bo1 = ld_pack(st + 11 * P + cx, tag), bo2 = ld_pack(st + 12 * P + cx, tag);
    const T bd0 = ld_pack(st + 13 * P + cx, tag), bd1 = ld_pack(st + 14 * P + cx, tag);
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[stg]);
    if (++stg == D) { stg = 0; ph ^= 1; }
    // Alg. 2 step 4 (reading R5): face velocity = momentum sum / density sum of the two cells sharing the face
    const T vtA0 = (shift_in_left(m1, ml.v.x) + m1) * rcp_(shift_in_left(r1, rl.v.x) + r1);
    const T vtA1 = (shift_in_left(m2, ml.v.y) + m2) * rcp_(shift_in_left(r2, rl.v.y) + r2);
    const T vtE = (T(m1.v.y, m2.v.y) + mr) * rcp_(T(r1.v.y, r2.v.y) + rr);       // the column right of my pack, rows o and o+1
    const T vtO0 = (m0 + m1) * rcp_(r0 + r1);
    const T vtO1 = (m1 + m2) * rcp_(r1 + r2);
    const T vtO2 = (m2 + m3) * rcp_(r2 + r3);
    T bxn0, bxn1, ben, bon0, bon1, bon2, fx0, fx1, fe, fo0, fo1, fo2;
    pxA0.template push<K>(vtA0, bx0, dt, hdt, bxn0, fx0);
    pxA1.template push<K>(vtA1, bx1, dt, hdt, bxn1, fx1);
    pxE.template push<K>(vtE, bxr, dt, hdt, ben, fe);
    po0.template push<K>(vtO0, bo0, dt, hdt, bon0, fo0);
    po1.template push<K>(vtO1, bo1, dt, hdt, bon1, fo1);
    po2.template push<K>(vtO2, bo2, dt, hdt, bon2, fo2);
    const int m = n0 + it - 8;
    if (it >= 8 && m < n1 && active) {
      st_pack(A.bxo + off, bxn0);                           // Alg. 2 step 9: advected B_t, rows o and o+1
      st_pack(A.boo + off, bon0);
      st_pack(A.bxo + off + A.so, bxn1);
      st_pack(A.boo + off + A.so, bon1);
      // constraint with the same fluxes at face m-1/2: columns x+1 and rows +1
      const T cx0 = shift_in_right(fx0, fe.v.x) - fx0, cx1 = shift_in_right(fx1, fe.v.y) - fx1;
      const T co0 = fo1 - fo0, co1 = fo2 - fo1;
      T b0 = bd0, b1 = bd1;
      if (x_first) { b0 = b0 + cx0; b0 = b0 + co0; b1 = b1 + cx1; b1 = b1 + co1; }
      else         { b0 = b0 + co0; b0 = b0 + cx0; b1 = b1 + co1; b1 = b1 + cx1; }
      st_pack(A.bdo + off, b0);
      st_pack(A.bdo + off + A.so, b1);
    }
    off += A.sd;
  };
  for (int it = 0; it < niter; it += 4) {
    step(std::integral_constant<int, 0>{}, it);
    step(std::integral_constant<int, 1>{}, it + 1);
    step(std::integral_constant<int, 2>{}, it + 2);
    step(std::integral_constant<int, 3>{}, it + 3);
  }
}

}  // namespace mhd
