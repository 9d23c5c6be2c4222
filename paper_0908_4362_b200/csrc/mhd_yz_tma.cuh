// mhd_yz_tma.cuh -- fluid_y / fluid_z as a march fed by a TMA bulk-copy ring (sm_100a).
//
// Same register pipeline as fluid_yz_kernel (mhd_yz.cuh), but the 10 input rows of each march step
// (5 u, B_d at the next face, B_x at x and x+1, B_o at o and o+1) are brought into a D-stage
// shared-memory ring by cp.async.bulk copies that one producer thread issues D-1 steps ahead; each
// copy is one contiguous TXB-element row, completion is signalled on an mbarrier per stage, and the
// consumer threads release a stage through a second mbarrier, so warps may drift up to D-1 steps
// apart without a block-wide barrier.  The consumers spend no registers on prefetch and no
// instructions on global addresses.
//
// Requirements (else fluid_yz_kernel runs): nx % TXB == 0, 16-byte row alignment (nx*sizeof(real) % 16 == 0).
#pragma once
#include "mhd_async.cuh"
#include "mhd_yz.cuh"

namespace mhd {

template <class real, int TXB>
struct FluidRing {
  static constexpr int CH = 16 / sizeof(real);            // elements in one 16-byte chunk
  static constexpr int ROW = TXB;
  static constexpr int STAGE = 9 * ROW + CH;              // u0..u4, bd(q+1), bo(o), bo(o+1), bx, bx chunk at x0+TXB
  static constexpr uint32_t BYTES = STAGE * sizeof(real);
  static size_t smem_bytes(int D) { return (size_t)D * STAGE * sizeof(real) + 2 * D * sizeof(uint64_t); }
};

#ifndef MHD_TMA_MINB
#define MHD_TMA_MINB 4
#endif

template <class real, int TXB, int D>
__global__ void __launch_bounds__(TXB + 32, (TXB == 128 && sizeof(real) == 4) ? MHD_TMA_MINB : 1) fluid_yz_tma_kernel(const YZArgs<real> A) {
  using RG = FluidRing<real, TXB>;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;

  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TXB;
  const int o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = n1 - n0 + 6;                       // cells n0-3 .. n1+2
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], TXB); }
    mbar_fence_init();
  }
  __syncthreads();

  if (tid >= TXB) {
    // ---------------- producer warp: one thread issues all copies ----------------
    if (tid == TXB) {
      const int rowbase = x0 + o * A.so;
      const int op_off = (map_index1(o + 1, A.no, A.bc) - o) * A.so;
      // 16-byte chunk holding B_x at x0+TXB (index-mapped); xp_idx of the consumers picks the element
      const int xn = map_index1(x0 + TXB, A.nx, A.bc);
      const int chunk = (xn / RG::CH) * RG::CH + o * A.so;
      for (int it = 0; it < niter; ++it) {
        const int s = it % D;
        if (it >= D) mbar_wait(&empty[s], ((it / D) & 1) ^ 1);
        const int q = n0 - 3 + it;
        const int od = map_index1(q, A.nd, A.bc) * A.sd;
        const int od1 = map_index1(q + 1, A.nd, A.bc) * A.sd;
        real* st = ring + s * RG::STAGE;
        mbar_expect_tx(&full[s], RG::BYTES);
        constexpr uint32_t RB = TXB * sizeof(real);
#pragma unroll
        for (int k = 0; k < 5; ++k) bulk_g2s(st + k * RG::ROW, A.u[k] + od + rowbase, RB, &full[s]);
        bulk_g2s(st + 5 * RG::ROW, A.bd + od1 + rowbase, RB, &full[s]);
        bulk_g2s(st + 6 * RG::ROW, A.bo + od + rowbase, RB, &full[s]);
        bulk_g2s(st + 7 * RG::ROW, A.bo + od + rowbase + op_off, RB, &full[s]);
        bulk_g2s(st + 8 * RG::ROW, A.bx + od + rowbase, RB, &full[s]);
        bulk_g2s(st + 9 * RG::ROW, A.bx + od + chunk, 16, &full[s]);
      }
    }
    return;
  }

  // ---------------- consumers: one pencil each ----------------
  const int col = tid;
  const int base = x0 + col + o * A.so;
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt, qdt = real(0.25) * dt;
  // where B_x(x+1) sits in the stage: next column, or inside the extra chunk for the last column
  const int xn = map_index1(x0 + TXB, A.nx, A.bc);
  const int xp_idx = 8 * RG::ROW + (col + 1 < TXB ? col + 1 : TXB + (xn % RG::CH));

  FluidPipe<real> pipe;
  pipe.init();
  real bd_lo = __ldg(A.bd + map_index1(n0 - 3, A.nd, A.bc) * A.sd + base);
  unsigned long long cbest = 0ull;
  int s = 0;
  uint32_t ph = 0;
#pragma unroll 3
  for (int it = 0; it < niter; ++it) {
    const real* st = ring + s * RG::STAGE;
    mbar_wait(&full[s], ph);
    real u[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) u[k] = st[k * RG::ROW + col];
    const real bd_hi = st[5 * RG::ROW + col];
    const real boc = real(0.5) * (st[6 * RG::ROW + col] + st[7 * RG::ROW + col]);
    const real bxc = real(0.5) * (st[8 * RG::ROW + col] + st[xp_idx]);
    mbar_arrive(&empty[s]);                            // my reads of this stage are done
    if (++s == D) { s = 0; ph ^= 1; }
    BCell<real> B;                                     // eq (19): faces -> centre
    if (A.x_is_t1) B.set(real(0.5) * (bd_lo + bd_hi), bxc, boc);
    else           B.set(real(0.5) * (bd_lo + bd_hi), boc, bxc);
    bd_lo = bd_hi;
    real out[5];
    pipe.push(u, B, A.gamma, hdt, qdt, out);
    const int m = n0 - 6 + it;                         // cell q-3
    if (m >= n0) {
      const int off = m * A.sd + base;
#pragma unroll
      for (int k = 0; k < 5; ++k) A.uo[k][off] = out[k];
      if (A.cmax_bits) {          // last operator of a step: c of eq (18) from the updated cell (B unchanged)
        const unsigned long long b = speed_bits(cfl_speed_hb2(out, pipe.hb2_out(), A.gamma));
        cbest = b > cbest ? b : cbest;
      }
    }
  }
  if (A.cmax_bits) {
    cbest = warp_max_u64(cbest);
    if ((tid & 31) == 0) publish_max(A.cmax_bits, cbest);
  }
}

}  // namespace mhd
