// mhd_yz2.cuh -- fluid_y / fluid_z for fp32 with two pencils per thread in packed f2 arithmetic.
//
// Same march and the same TMA bulk-copy ring as fluid_yz_tma_kernel (mhd_yz_tma.cuh): one producer
// thread brings the 10 input rows of each march step (5 u, B_d at the next face, B_o at o and o+1,
// B_x and the 16-byte chunk holding B_x at x0+TXB) into a D-stage shared-memory ring with
// cp.async.bulk, full/empty mbarriers per stage.  What changes is the consumer: a thread owns the
// two adjacent columns x0+2c, x0+2c+1, reads them with one 8-byte LDS per row, runs ONE
// FluidPipe<f2> whose FADD2/FMUL2/FFMA2 advance both pencils per issued instruction (mhd_pack.cuh),
// and writes 8-byte stores.  Per cell that is about half the issue slots of the scalar kernel.
//
// Requirements (else fluid_yz_tma_kernel / fluid_yz_kernel run): fp32, nx % TXB == 0.
#pragma once
#include "mhd_yz_tma.cuh"

namespace mhd {

// Resident blocks per SM the register budget is cut for (TXB = 256, 128).  Measured at 512^3 (ms per
// launch): 168 registers (256:2 or 128:3, 6-8 consumer warps per SM) 1.28; 214 registers, no spills
// (256:1) 1.96; 128 registers with spills (256:3) 1.94; 96 registers (256:4) 3.3.  The scalar kernel: 1.60.
#ifndef MHD_YZ2_MINB256
#define MHD_YZ2_MINB256 2
#endif
#ifndef MHD_YZ2_MINB128
#define MHD_YZ2_MINB128 3
#endif

template <int TXB, int D, bool XT1>
__global__ void __launch_bounds__(TXB / 2 + 32, TXB == 256 ? MHD_YZ2_MINB256 : MHD_YZ2_MINB128) fluid_yz_p2_kernel(const YZArgs<float> A) {
  using RG = FluidRing<float, TXB>;
  constexpr int NC = TXB / 2;                            // consumer threads
  extern __shared__ __align__(128) unsigned char smem_raw[];
  float* ring = reinterpret_cast<float*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;

  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TXB;
  const int o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = n1 - n0 + 6;                         // cells n0-3 .. n1+2
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NC); }
    mbar_fence_init();
  }
  __syncthreads();

  if (tid >= NC) {
    // ---------------- producer warp: one thread issues all copies ----------------
    if (tid == NC) {
      const int rowbase = x0 + o * A.so;
      const int op_off = (map_index1(o + 1, A.no, A.bc) - o) * A.so;
      const int xn = map_index1(x0 + TXB, A.nx, A.bc);   // B_x at x0+TXB lives in this 16-byte chunk
      const int chunk = (xn / RG::CH) * RG::CH + o * A.so;
      for (int it = 0; it < niter; ++it) {
        const int s = it % D;
        if (it >= D) mbar_wait(&empty[s], ((it / D) & 1) ^ 1);
        const int q = n0 - 3 + it;
        const int od = map_index1(q, A.nd, A.bc) * A.sd;
        const int od1 = map_index1(q + 1, A.nd, A.bc) * A.sd;
        float* st = ring + s * RG::STAGE;
        mbar_expect_tx(&full[s], RG::BYTES);
        constexpr uint32_t RB = TXB * sizeof(float);
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

  // ---------------- consumers: two adjacent pencils each ----------------
  const int c2 = 2 * tid;
  const int base = x0 + c2 + o * A.so;
  const float dts = (float)(*A.dt);
  const f2 hdt(0.5f * dts), qdt(0.25f * dts), gamma(A.gamma);
  const int xn = map_index1(x0 + TXB, A.nx, A.bc);
  const int xp_idx = 8 * RG::ROW + (c2 + 2 < TXB ? c2 + 2 : TXB + (xn % RG::CH));   // B_x at column c2+2

  FluidPipe<f2> pipe;
  pipe.init();
  f2 bd_lo(__ldg(reinterpret_cast<const float2*>(A.bd + map_index1(n0 - 3, A.nd, A.bc) * A.sd + base)));
  unsigned long long cbest = 0ull;
  // u(q-1) and u(q-3) are re-read from the ring (stages it-1, it-3) instead of being carried in
  // registers, so a stage is released three march steps after it was first consumed; during the first
  // three steps those reads return whatever the ring holds: it only feeds warm-up state that is
  // flushed before the first stored cell, exactly like the dummy values of FluidPipe::init().
#pragma unroll 3
  for (int it = 0; it < niter; ++it) {
    const unsigned s = (unsigned)it % D;
    const float* st = ring + s * RG::STAGE;
    const float* st1 = ring + ((unsigned)(it + D - 1) % D) * RG::STAGE;
    const float* st3 = ring + ((unsigned)(it + D - 3) % D) * RG::STAGE;
    mbar_wait(&full[s], ((unsigned)it / D) & 1);
    f2 u[5], um1[5], um3[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      u[k] = f2(*reinterpret_cast<const float2*>(st + k * RG::ROW + c2));
      um1[k] = f2(*reinterpret_cast<const float2*>(st1 + k * RG::ROW + c2));
      um3[k] = f2(*reinterpret_cast<const float2*>(st3 + k * RG::ROW + c2));
    }
    const f2 bd_hi(*reinterpret_cast<const float2*>(st + 5 * RG::ROW + c2));
    const f2 boa(*reinterpret_cast<const float2*>(st + 6 * RG::ROW + c2));
    const f2 bob(*reinterpret_cast<const float2*>(st + 7 * RG::ROW + c2));
    const f2 bxa(*reinterpret_cast<const float2*>(st + 8 * RG::ROW + c2));
    const float bxn = st[xp_idx];
    if (it >= 3) mbar_arrive(&empty[(unsigned)(it + D - 3) % D]);   // stage it-3 is no longer needed
    const f2 half(0.5f);
    const f2 boc = half * (boa + bob);
    const f2 bxc = half * (bxa + f2(bxa.v.y, bxn));      // eq (19): faces -> centre
    const f2 bdc = half * (bd_lo + bd_hi);
    BCell<f2> B;
    if (XT1) B.set(bdc, bxc, boc);       // sweep z: (t1,t2) = (x,y);  sweep y: (t1,t2) = (z,x)
    else     B.set(bdc, boc, bxc);
    bd_lo = bd_hi;
    f2 out[5];
    pipe.advance(u, um1, um3, B, gamma, hdt, qdt, out);
    const int m = n0 - 6 + it;                           // cell q-3
    if (m >= n0) {
      const int off = m * A.sd + base;
#pragma unroll
      for (int k = 0; k < 5; ++k) *reinterpret_cast<float2*>(A.uo[k] + off) = out[k].v;
      if (A.cmax_bits) {          // last operator of a step: c of eq (18) from the updated cells (B unchanged)
        const float ua[5] = {out[0].v.x, out[1].v.x, out[2].v.x, out[3].v.x, out[4].v.x};
        const float ub[5] = {out[0].v.y, out[1].v.y, out[2].v.y, out[3].v.y, out[4].v.y};
        const float ca = cfl_speed_hb2(ua, pipe.hb2_out().v.x, A.gamma);
        const float cb = cfl_speed_hb2(ub, pipe.hb2_out().v.y, A.gamma);
        // NaN must win the maximum (it poisons dt): compare the bit patterns, not the floats
        const unsigned long long ba = speed_bits(ca), bb = speed_bits(cb);
        const unsigned long long b = ba > bb ? ba : bb;
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
