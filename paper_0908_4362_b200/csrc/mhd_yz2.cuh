// mhd_yz2.cuh -- fluid_y / fluid_z march on a TMA ring; fp32 with two pencils per thread in packed f2
// arithmetic (T = f2), fp64 with one (T = double).
//
// Same march as fluid_yz_tma_kernel (mhd_yz_tma.cuh): the 10 input rows of each march step (5 u, B_d at
// the next face, B_o at o and o+1, B_x and the 16-byte chunk holding B_x at x0+TXB) are brought into a
// D-stage shared-memory ring with cp.async.bulk, full/empty mbarriers per stage.  What changes:
//   * a thread owns L adjacent columns (L = 2: one 8-byte LDS per row, ONE FluidPipe<f2> whose
//     FADD2/FMUL2/FFMA2 advance both pencils per issued instruction, 8-byte stores; mhd_pack.cuh);
//   * u(q-1) and u(q-3) are re-read from the ring instead of being carried in registers
//     (FluidPipe::advance), so a stage is released three march steps after it is first consumed;
//   * there is no producer warp: every warp is a consumer and the warps take turns (march step modulo
//     the warp count) at issuing the copies of the stage PF steps ahead, one copy per lane.  A
//     dedicated producer warp costs a fifth of the block's registers for a thread that issues ten
//     instructions per step, and five-warp blocks leave one scheduler with three warps, which caps
//     every thread at 168 registers.
//
// Requirements (else fluid_yz_tma_kernel / fluid_yz_kernel run): nx % TXB == 0.
#pragma once
#include "mhd_yz_tma.cuh"
#include "mhd_pack_io.cuh"

namespace mhd {

// Resident blocks per SM the register budget is cut for.  Measured at 512^3 fp32 (ms per launch), current kernel
// (elected-lane producer, c_max as a template switch): 2 blocks / 184 registers 1.17, 3 blocks / 168 registers, no
// spills, 1.11 (8 stages x 9.2 KB x 3 blocks = 222 KB of shared memory: the most that fits); 7 stages 1.13.
// Earlier producer-warp version: 168 registers 1.28; 128 registers with spills 1.94; 96 registers 3.3.
#ifndef MHD_YZ2_MINB
#define MHD_YZ2_MINB 3
#endif
#ifndef MHD_YZ2_UNROLL
#define MHD_YZ2_UNROLL 3      // march steps per unrolled loop body
#endif
#ifndef MHD_YZ2_STAGES
#define MHD_YZ2_STAGES 8
#endif
// the warp on duty refills a stage that every warp released SLACK+1 steps ago: with no slack the duty
// warp waits for the slowest warp every step, which couples the warps like a block barrier
#ifndef MHD_YZ2_SLACK
#define MHD_YZ2_SLACK 1
#endif

// real: element type in memory.  T: arithmetic pack (f2 for float, double for double).
// D ring stages, PF = D - 4 - SLACK steps of prefetch.
// CM: also reduce c of eq (18) over the updated cells (the last operator of a step); a compile-time switch keeps the
// reduction out of the instruction stream and the register allocation of the other five launches of a step
template <class real, class T, int TXB, int D, bool XT1, bool CM>
__global__ void __launch_bounds__(TXB / PackOf<T>::L, MHD_YZ2_MINB) fluid_yz_ring_kernel(const YZArgs<real> A) {
  using RG = FluidRing<real, TXB>;
  typedef typename PackOf<T>::scalar S;
  constexpr int L = PackOf<T>::L;
  constexpr int NT = TXB / L;                            // threads (all consumers)
  constexpr int NW = NT / 32;                            // warps
  constexpr int PF = D - 4 - MHD_YZ2_SLACK;              // the stage of step it+PF was released at step it+PF-D+3 = it-1-SLACK
  static_assert(NW >= 1 && (NW & (NW - 1)) == 0 && PF >= 1, "block shape");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;

  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // the same value, warp-uniform for the compiler too
  const int x0 = blockIdx.x * TXB;
  const int o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = n1 - n0 + 6;                         // cells n0-3 .. n1+2
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NW); }
    mbar_fence_init();
  }
  __syncthreads();

  // ---- producer duty: one elected lane of the warp on duty issues the 10 copies of a stage; every operand is
  // warp-uniform (block indices, kernel parameters, the march step), so the copies are straight-line UBLKCPs ------
#ifdef MHD_EXP_L2FEED
  const int rowbase = x0 + (o & 7) * A.so;       // experiment: inputs out of L2 (results are wrong on purpose)
#else
  const int rowbase = x0 + o * A.so;
#endif
  const int op_off = (map_index1(o + 1, A.no, A.bc) - o) * A.so;
  const int xchunk = (map_index1(x0 + TXB, A.nx, A.bc) / RG::CH) * RG::CH + o * A.so;   // B_x at x0+TXB lives in this 16-byte chunk
  auto produce = [&](int itp) {                          // called by one whole, converged warp
    const unsigned s = (unsigned)itp % D;
    if (itp >= D) mbar_wait(&empty[s], (((unsigned)itp / D) & 1) ^ 1);
    if (elect_one()) {
      const int q = n0 - 3 + itp;
#ifdef MHD_EXP_L2FEED
      const int od = (map_index1(q, A.nd, A.bc) & 15) * A.sd;
      const int od1 = (map_index1(q + 1, A.nd, A.bc) & 15) * A.sd;
#else
      const int od = map_index1(q, A.nd, A.bc) * A.sd;
      const int od1 = map_index1(q + 1, A.nd, A.bc) * A.sd;
#endif
      real* st = ring + s * RG::STAGE;
      constexpr uint32_t RB = TXB * sizeof(real);
      mbar_expect_tx(&full[s], RG::BYTES);
#ifdef MHD_EXP_CHEAPPROD
      {   // experiment: ten copies from one base pointer with constant strides (same bytes, wrong rows)
        const real* b0 = A.u[0] + od + rowbase;
#pragma unroll
        for (int k = 0; k < 9; ++k) bulk_g2s(st + k * RG::ROW, b0 + k * 1024, RB, &full[s]);
        bulk_g2s(st + 9 * RG::ROW, b0 + 9 * 1024, 16, &full[s]);
        (void)od1; (void)op_off; (void)xchunk;
      }
      if (false)
#endif
#pragma unroll
      for (int k = 0; k < 5; ++k) bulk_g2s(st + k * RG::ROW, A.u[k] + od + rowbase, RB, &full[s]);
#ifndef MHD_EXP_CHEAPPROD
      bulk_g2s(st + 5 * RG::ROW, A.bd + od1 + rowbase, RB, &full[s]);
      bulk_g2s(st + 6 * RG::ROW, A.bo + od + rowbase, RB, &full[s]);
      bulk_g2s(st + 7 * RG::ROW, A.bo + od + rowbase + op_off, RB, &full[s]);
      bulk_g2s(st + 8 * RG::ROW, A.bx + od + rowbase, RB, &full[s]);
      bulk_g2s(st + 9 * RG::ROW, A.bx + od + xchunk, 16, &full[s]);
#endif
    }
    __syncwarp();
  };
  for (int itp = warp; itp < PF && itp < niter; itp += NW) produce(itp);

  // ---- consumers: L adjacent pencils each -------------------------------------------------------------
  const int c2 = L * tid;
  const int base = x0 + c2 + o * A.so;
  const S dts = (S)(*A.dt);
  const T hdt(S(0.5) * dts), qdt(S(0.25) * dts), gamma(A.gamma);
  const int xn = map_index1(x0 + TXB, A.nx, A.bc);
  const int xp_idx = 8 * RG::ROW + (c2 + L < TXB ? c2 + L : TXB + (xn % RG::CH));   // B_x at column c2+L
  T* tag = nullptr;

  FluidPipe<T> pipe;
  pipe.init();
  T bd_lo = ld_pack(A.bd + map_index1(n0 - 3, A.nd, A.bc) * A.sd + base, tag);
  decltype(pack_speed_key((const T*)nullptr, T(), S())) cbest = 0;
  // During the first three steps the re-reads of u(q-1), u(q-3) return whatever the ring holds: it only
  // feeds warm-up state that is flushed before the first stored cell, like the dummy values of
  // FluidPipe::init().
  constexpr int UNR = MHD_YZ2_UNROLL;
#pragma unroll UNR
  for (int it = 0; it < niter; ++it) {
    if (((unsigned)it & (NW - 1)) == (unsigned)warp && it + PF < niter) produce(it + PF);
    const unsigned s = (unsigned)it % D;
    const real* st = ring + s * RG::STAGE;
    const real* st1 = ring + ((unsigned)(it + D - 1) % D) * RG::STAGE;
    const real* st3 = ring + ((unsigned)(it + D - 3) % D) * RG::STAGE;
    mbar_wait(&full[s], ((unsigned)it / D) & 1);
    T u[5], um1[5], um3[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      u[k] = ld_pack(st + k * RG::ROW + c2, tag);
      um1[k] = ld_pack(st1 + k * RG::ROW + c2, tag);
      um3[k] = ld_pack(st3 + k * RG::ROW + c2, tag);
    }
    const T bd_hi = ld_pack(st + 5 * RG::ROW + c2, tag);
    const T boa = ld_pack(st + 6 * RG::ROW + c2, tag);
    const T bob = ld_pack(st + 7 * RG::ROW + c2, tag);
    const T bxa = ld_pack(st + 8 * RG::ROW + c2, tag);
    const S bxn = st[xp_idx];
    if (it >= 3) {                                       // stage it-3 is no longer needed by this warp
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[(unsigned)(it + D - 3) % D]);
    }
    const T half(S(0.5));
    const T boc = half * (boa + bob);
    const T bxc = half * (bxa + shift_in_right(bxa, bxn));   // eq (19): faces -> centre
    const T bdc = half * (bd_lo + bd_hi);
    BCell<T> B;
    if (XT1) B.set(bdc, bxc, boc);       // sweep z: (t1,t2) = (x,y);  sweep y: (t1,t2) = (z,x)
    else     B.set(bdc, boc, bxc);
    bd_lo = bd_hi;
    T out[5];
    pipe.advance(u, um1, um3, B, gamma, hdt, qdt, out);
    const int m = n0 - 6 + it;                           // cell q-3
    if (m >= n0) {
      const int off = m * A.sd + base;
#pragma unroll
      for (int k = 0; k < 5; ++k) st_pack(A.uo[k] + off, out[k]);
      if (CM) {                   // last operator of a step: c of eq (18) from the updated cells (B unchanged)
        const auto b = pack_speed_key(out, pipe.hb2_out(), (S)A.gamma);
        cbest = b > cbest ? b : cbest;
      }
    }
  }
  if (CM) {
    const unsigned long long cw = warp_max_u64(key_bits(cbest));
    if (lane == 0) publish_max(A.cmax_bits, cw);
  }
}

}  // namespace mhd
