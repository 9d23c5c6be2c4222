// mhd_yz2.cuh -- fluid_y / fluid_z march on a TMA ring; fp32 with two pencils per thread in packed f2
// arithmetic (T = f2), fp64 with one (T = double).
//
// Layout is x fastest, so for a sweep along y or z the lanes of a warp sit on consecutive x: every access is
// coalesced and the sweep needs no transpose (the paper's z-fastest layout made two of its three sweeps
// uncoalesced).  A block owns a row of TXB pencils and marches along the sweep axis with
// the +-3 stencil of Algorithm 1 in registers (FluidPipe); the 10 input rows of each march step (5 u, B_d at
// the next face, B_o at o and o+1, B_x and the 16-byte chunk holding B_x at x0+TXB) are brought into a
// D-stage shared-memory ring with cp.async.bulk, full/empty mbarriers per stage, no block barrier:
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
// Requirements (else fluid_march_kernel of mhd_generic.cuh runs): nx a multiple of 16 bytes (the last tile of a row may be
// narrower than TXB: its copies are shorter and the threads beyond it compute on stale shared memory and store nothing),
// extent along the sweep >= 8.
#pragma once
#include "mhd_args.cuh"
#include "mhd_async.cuh"
#include <type_traits>
#include "mhd_pack_io.cuh"
#include <cuda.h>                                         // CUtensorMap (type only; the driver entry point is looked up at run time)

namespace mhd {

// TM: the nine row copies of a stage are tensor-map TMA copies (cp.async.bulk.tensor.3d, SASS UTMALDG), whose shared-memory
// destination must be 128-byte aligned: the stage is padded to a multiple of 128 bytes
template <class real, int TXB, bool TM = false>
struct FluidRing {
  static constexpr int CH = 16 / sizeof(real);            // elements in one 16-byte chunk
  static constexpr int ROW = TXB;
  static constexpr int STAGE = 9 * ROW + (TM ? 128 / (int)sizeof(real) : CH);   // u0..u4, bd(q+1), bo(o), bo(o+1), bx, bx chunk at x0+TXB
  static constexpr uint32_t BYTES = STAGE * sizeof(real);
  static size_t smem_bytes(int D) { return (size_t)D * STAGE * sizeof(real) + 2 * D * sizeof(uint64_t); }
};


// Resident blocks per SM the register budget is cut for.  Measured at 512^3 fp32 (ms per launch), current kernel
// (elected-lane producer, c_max as a template switch): 2 blocks / 184 registers 1.17, 3 blocks / 168 registers, no
// spills, 1.11 (8 stages x 9.2 KB x 3 blocks = 222 KB of shared memory: the most that fits); 7 stages 1.13.
// Earlier producer-warp version: 168 registers 1.28; 128 registers with spills 1.94; 96 registers 3.3.
#ifndef MHD_YZ2_MINB
#define MHD_YZ2_MINB 3
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
// D ring stages (8: two groups of four, so that inside the 4x unrolled march every ring slot, barrier and re-read is a
// compile-time offset from one of two base registers), PF = D - 4 - SLACK steps of prefetch.
// CM: also reduce c of eq (18) over the updated cells (the last operator of a step); a compile-time switch keeps the
// reduction out of the instruction stream and the register allocation of the other five launches of a step.
//
// Instruction budget (the kernel is bound by instruction issue, not by HBM: with all inputs served from L2 it is only 5 %
// faster, and every instruction removed from the march shows up 1:1 in the run time; profiles/r02_*): the producer reads
// its ten source rows as  u[0] + (row offset) + A.src[k]  with the byte offsets A.src[] in the constant bank, the
// consumers keep one running store offset, and the march is unrolled by four with the step number modulo 4 a
// compile-time constant.
// RAG: the row ends in a tile narrower than TXB (else the width is a compile-time constant, as the tuned kernel wants)
struct FluidMaps { CUtensorMap m[8]; };                  // u0..u4 (sweep roles), B_d, B_o, B_x: 3-D maps (x, y, z), box TXB x 1 x 1

__device__ __forceinline__ void tma_g2s_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(smem_u32(dst)),
               "l"(reinterpret_cast<uint64_t>(map)), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
               : "memory");
}

template <class real, class T, int TXB, int D, bool XT1, bool CM, bool RAG, bool TM>
__device__ __forceinline__ void fluid_yz_ring_body(const YZArgs<real>& A, const CUtensorMap* tm) {
  using RG = FluidRing<real, TXB, TM>;
  typedef typename PackOf<T>::scalar S;
  constexpr int L = PackOf<T>::L;
  constexpr int NT = TXB / L;                            // threads (all consumers)
  constexpr int NW = NT / 32;                            // warps
  constexpr int PF = D - 4 - MHD_YZ2_SLACK;              // the stage of step it+PF was released at step it+PF-D+3 = it-1-SLACK
  static_assert(NW >= 1 && (NW & (NW - 1)) == 0 && NW <= 4 && PF >= 1 && PF <= 4 && D == 8, "block shape");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;

  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // the same value, warp-uniform for the compiler too
  const int x0 = blockIdx.x * TXB;
  const int w = RAG ? min(TXB, A.nx - x0) : TXB;         // columns of this tile (a multiple of the 16-byte chunk)
  const int o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = (n1 - n0 + 6 + 3) & ~3;              // cells n0-3 .. n1+2, rounded up to the 4x unrolled march
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NW); }
    mbar_fence_init();
  }
  __syncthreads();

  // ---- producer duty: one elected lane of the warp on duty issues the 10 copies of a stage; every operand is
  // warp-uniform (block indices, kernel parameters, the march step), so the copies are straight-line UBLKCPs ------
  const int rowbase = x0 + o * A.so;
  const long long op_bytes = (long long)((map_index1(o + 1, A.no, A.bc) - o) * A.so) * (long long)sizeof(real);
  const long long xc_bytes = (long long)((map_index1(x0 + w, A.nx, A.bc) / RG::CH) * RG::CH - x0) * (long long)sizeof(real);   // B_x at x0+w lives in this 16-byte chunk
  auto produce = [&](int itp) {                          // called by one whole, converged warp
    const unsigned s = (unsigned)itp % D;
#if defined(MHD_BUG_NO_EMPTY_WAIT) && !defined(MHD_JITTER)
#error "MHD_BUG_NO_EMPTY_WAIT injects a race on purpose: only the jitter build (-DMHD_JITTER, libmhd_jitter.so) may define it"
#endif
#ifndef MHD_BUG_NO_EMPTY_WAIT        // (fault injection, jitter build only: refill a stage without waiting for its readers)
    if (itp >= D) mbar_wait(&empty[s], (((unsigned)itp / D) & 1) ^ 1);
#endif
    if (elect_one()) {
      const int q = n0 - 3 + itp;
      const int od = map_index1(q, A.nd, A.bc) * A.sd;
      const int od1 = map_index1(q + 1, A.nd, A.bc) * A.sd;
      const char* b0 = reinterpret_cast<const char*>(A.u[0] + od + rowbase);     // row (q, o), columns x0.. of field u[0]
      const char* b1 = reinterpret_cast<const char*>(A.u[0] + od1 + rowbase);    // row (q+1, o)
      real* st = ring + s * RG::STAGE;
      const uint32_t RB = (uint32_t)w * sizeof(real);
      mbar_expect_tx(&full[s], 9u * RB + 16u);
      if constexpr (TM) {
        // coordinates (x, y, z) of the rows (q, o), (q+1, o), (q, o+1): the sweep axis is z when x is t1 (XT1), else y
        const int qm = map_index1(q, A.nd, A.bc), q1 = map_index1(q + 1, A.nd, A.bc), op = map_index1(o + 1, A.no, A.bc);
        const int ya = XT1 ? o : qm, za = XT1 ? qm : o;            // row (q, o)
        const int yb = XT1 ? o : q1, zb = XT1 ? q1 : o;            // row (q+1, o)
        const int yc = XT1 ? op : qm, zc = XT1 ? qm : op;          // row (q, o+1)
#pragma unroll
        for (int k = 0; k < 5; ++k) tma_g2s_3d(st + k * RG::ROW, tm + k, x0, ya, za, &full[s]);
        tma_g2s_3d(st + 5 * RG::ROW, tm + 5, x0, yb, zb, &full[s]);
        tma_g2s_3d(st + 6 * RG::ROW, tm + 6, x0, ya, za, &full[s]);
        tma_g2s_3d(st + 7 * RG::ROW, tm + 6, x0, yc, zc, &full[s]);
        tma_g2s_3d(st + 8 * RG::ROW, tm + 7, x0, ya, za, &full[s]);
        bulk_g2s(st + 9 * RG::ROW, b0 + A.src[7] + xc_bytes, 16, &full[s]);
      } else {
#pragma unroll
      for (int k = 0; k < 5; ++k) bulk_g2s(st + k * RG::ROW, b0 + A.src[k], RB, &full[s]);
      bulk_g2s(st + 5 * RG::ROW, b1 + A.src[5], RB, &full[s]);               // B_d at the next face
      bulk_g2s(st + 6 * RG::ROW, b0 + A.src[6], RB, &full[s]);               // B_o at o
      bulk_g2s(st + 7 * RG::ROW, b0 + A.src[6] + op_bytes, RB, &full[s]);    // B_o at o+1
      bulk_g2s(st + 8 * RG::ROW, b0 + A.src[7], RB, &full[s]);               // B_x
      bulk_g2s(st + 9 * RG::ROW, b0 + A.src[7] + xc_bytes, 16, &full[s]);    // the chunk holding B_x at x0+TXB
      }
    }
    __syncwarp();
  };
  for (int itp = warp; itp < PF && itp < niter; itp += NW) produce(itp);

  // ---- consumers: L adjacent pencils each -------------------------------------------------------------
  const int c2 = L * tid;
  const S dts = (S)(*A.dt);
  const T hdt(S(0.5) * dts), qdt(S(0.25) * dts), gamma(A.gamma);
  const int xn = map_index1(x0 + w, A.nx, A.bc);
  const int xp_idx = 8 * RG::ROW + (c2 + L < w ? L : TXB - c2 + (xn % RG::CH));   // B_x at column c2+L, relative to my column
  const bool active = c2 < w;                            // threads beyond a narrow last tile store nothing
  T* tag = nullptr;

  FluidPipe<T> pipe;
  pipe.init();
  T bd_lo = ld_pack(A.bd + map_index1(n0 - 3, A.nd, A.bc) * A.sd + x0 + (active ? c2 : 0) + o * A.so, tag);
  decltype(pack_speed_key((const T*)nullptr, T(), S())) cbest = 0;
  // ring slots of the current group of four march steps and of the previous one (D = 8: the two halves of the ring),
  // as this thread's column inside stage 0 of each half; barrier addresses likewise
  const real* ra = ring + c2;                            // steps 4g .. 4g+3
  const real* rb = ring + 4 * RG::STAGE + c2;            // steps 4g-4 .. 4g-1
  uint64_t* fa = full;
  uint64_t* ea = empty;
  uint64_t* eb = empty + 4;
  uint32_t ph = 0;
  int off = (n0 - 6) * A.sd + x0 + c2 + o * A.so;        // output cell m = q - 3 = n0 - 6 + it
  // During the first three steps the re-reads of u(q-1), u(q-3) return whatever the ring holds: it only
  // feeds warm-up state that is flushed before the first stored cell, like the dummy values of
  // FluidPipe::init().
  auto step = [&](auto Ktag, int it) {
    constexpr int K = decltype(Ktag)::value;
    if ((K & (NW - 1)) == warp && it + PF < niter) produce(it + PF);
    const real* st = ra + K * RG::STAGE;
    const real* st1 = K >= 1 ? ra + (K - 1) * RG::STAGE : rb + 3 * RG::STAGE;
    const real* st3 = K >= 3 ? ra + (K - 3) * RG::STAGE : rb + (K + 1) * RG::STAGE;
    mbar_wait(&fa[K], ph);
    T u[5], um1[5], um3[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      u[k] = ld_pack(st + k * RG::ROW, tag);
      um1[k] = ld_pack(st1 + k * RG::ROW, tag);
      um3[k] = ld_pack(st3 + k * RG::ROW, tag);
    }
    const T bd_hi = ld_pack(st + 5 * RG::ROW, tag);
    const T boa = ld_pack(st + 6 * RG::ROW, tag);
    const T bob = ld_pack(st + 7 * RG::ROW, tag);
    const T bxa = ld_pack(st + 8 * RG::ROW, tag);
    const S bxn = st[xp_idx];
    if (it >= 3) {                                       // stage it-3 is no longer needed by this warp
      __syncwarp();
      if (lane == 0) mbar_arrive(K >= 3 ? &ea[K - 3] : &eb[K + 1]);
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
    if (it >= 6 && it - 6 < n1 - n0 && active) {         // cell q-3 = n0 - 6 + it
#pragma unroll
      for (int k = 0; k < 5; ++k) st_pack(A.uo[k] + off, out[k]);
      if (CM) {                   // last operator of a step: c of eq (18) from the updated cells (B unchanged)
        const auto b = pack_speed_key(out, pipe.hb2_out(), (S)A.gamma);
        cbest = b > cbest ? b : cbest;
      }
    }
    off += A.sd;
  };
  for (int it = 0; it < niter; it += 4) {
    step(std::integral_constant<int, 0>{}, it);
    step(std::integral_constant<int, 1>{}, it + 1);
    step(std::integral_constant<int, 2>{}, it + 2);
    step(std::integral_constant<int, 3>{}, it + 3);
    { const real* t = ra; ra = rb; rb = t; }             // the other half of the ring
    { uint64_t* t = ea; ea = eb; eb = t; }
    fa = (fa == full) ? full + 4 : full;
    if (fa == full) ph ^= 1u;
  }
  if (CM) {
    const unsigned long long cw = warp_max_u64(key_bits(cbest));
    if (lane == 0) publish_max(A.cmax_bits, cw);
  }
}

template <class real, class T, int TXB, int D, bool XT1, bool CM, bool RAG = false>
__global__ void __launch_bounds__(TXB / PackOf<T>::L, MHD_YZ2_MINB) fluid_yz_ring_kernel(const YZArgs<real> A) {
  fluid_yz_ring_body<real, T, TXB, D, XT1, CM, RAG, false>(A, nullptr);
}
// the same with tensor-map copies (option tmap; whole tiles only)
template <class real, class T, int TXB, int D, bool XT1, bool CM>
__global__ void __launch_bounds__(TXB / PackOf<T>::L, MHD_YZ2_MINB) fluid_yz_ring_tm_kernel(const YZArgs<real> A, const __grid_constant__ FluidMaps M) {
  fluid_yz_ring_body<real, T, TXB, D, XT1, CM, false, true>(A, M.m);
}

}  // namespace mhd
