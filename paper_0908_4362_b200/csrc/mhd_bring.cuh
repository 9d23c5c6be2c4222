// mhd_bring.cuh -- B_{t1->d}, B_{t2->d} for sweeps along y and z: a march with NO block barrier.
//
// Algorithm 2, eqs (20)-(22) PAPER.md:147-158; constraint step PAPER.md:160.
//
// A block owns one row of TXB pencils (fixed o, x0 <= x < x0+TXB) and marches along d.  A producer warp
// brings, for every march step, the ten rows the step needs (rho and m_d of the rows o-1, o, o+1; B_x of
// row o; B_o of rows o, o+1; B_d of the cell that is finished in this step, four cells behind) plus the
// 16-byte chunks holding the columns x0-1 and x0+TXB into a D-stage shared-memory ring with
// cp.async.bulk (SASS UBLKCP), one copy per producer lane, completion on an mbarrier per stage.
// A consumer thread owns L adjacent pencils (L = 2 in packed f2 arithmetic for fp32, mhd_pack.cuh;
// L = 1 for fp64) and runs every flux pipeline its own cells need:
//     pxA  B_x rows (faces) of its own L columns        pxE  B_x row of the column to its right (scalar)
//     po   B_o row o                                     pop  B_o row o+1
// The +1 rows (pxE, pop) supply the constraint update of B_d and are recomputed instead of
// exchanged: compared with the tile march of mhd_btile.cuh that costs arithmetic (which packed f2
// instructions make cheap) and buys a kernel with no __syncthreads, no shared-memory flux exchange, no
// global LOAD address arithmetic in the consumers, and warps that drift freely up to the ring depth.
// B_t(k-4), needed when the cell is finished, is re-read from the ring (stage it-4) instead of being
// carried through a register delay line, so a stage is released four steps after it is first read.
//
// Requirements (else bpair_tile_kernel / bpair_yz_kernel run): nx % TXB == 0, extent along d >= 8.
#pragma once
#include <type_traits>
#include "mhd_async.cuh"
#include "mhd_btile.cuh"

namespace mhd {

// lane-pack plumbing: T = double (1 cell) or f2 (2 cells)
template <class T> struct PackOf;
template <> struct PackOf<double> { typedef double scalar; enum { L = 1 }; };
template <> struct PackOf<float> { typedef float scalar; enum { L = 1 }; };
template <> struct PackOf<f2> { typedef float scalar; enum { L = 2 }; };

__device__ __forceinline__ double ld_pack(const double* p, double*) { return *p; }
__device__ __forceinline__ float ld_pack(const float* p, float*) { return *p; }
__device__ __forceinline__ f2 ld_pack(const float* p, f2*) { return f2(*reinterpret_cast<const float2*>(p)); }
__device__ __forceinline__ void st_pack(double* p, double v) { *p = v; }
__device__ __forceinline__ void st_pack(float* p, float v) { *p = v; }
__device__ __forceinline__ void st_pack(float* p, f2 v) { *reinterpret_cast<float2*>(p) = v.v; }
// (s, a[0..L-2]): the pack one column to the left;  a[L-1]: the last lane
__device__ __forceinline__ double shift_in_left(double, double s) { return s; }
__device__ __forceinline__ float shift_in_left(float, float s) { return s; }
__device__ __forceinline__ f2 shift_in_left(f2 a, float s) { return f2(s, a.v.x); }
__device__ __forceinline__ double shift_in_right(double, double s) { return s; }
__device__ __forceinline__ float shift_in_right(float, float s) { return s; }
__device__ __forceinline__ f2 shift_in_right(f2 a, float s) { return f2(a.v.y, s); }
__device__ __forceinline__ double last_lane(double a) { return a; }
__device__ __forceinline__ float last_lane(float a) { return a; }
__device__ __forceinline__ float last_lane(f2 a) { return a.v.y; }

// BPipe4 (mhd_btile.cuh) with the B_t delay line cut to two cells: B_t(k-4) is supplied by the caller.
template <class real>
struct BPipe4R {
  real vt[2];        // vt(k-2), vt(k-1)            slot = step & 1
  real b[2];         // B_t(k-2), B_t(k-1)           slot = step & 1
  real w1[4];        // vg*B_t^{t+dt/2}(k-5..k-2)    slot = step & 3
  real vh[2];        // 2 * face velocity at (k-4)+1/2, (k-3)+1/2 (only the sign is used)
  real vg, w0, f1, f;   // vg(k-2), vg*B_t(k-2), first-order flux at (k-3)+1/2, second-order flux*dt at (k-5)+1/2

  __device__ __forceinline__ void init() {
    vt[0] = vt[1] = vh[0] = vh[1] = b[0] = b[1] = vg = w0 = f1 = f = real(0);
#pragma unroll
    for (int j = 0; j < 4; ++j) w1[j] = real(0);
  }
  // push<K>(vt(k), B_t(k), B_t(k-4)): finishes the flux*dt at face (k-4)+1/2; returns B_t'(k-4) and the
  // flux at face (k-4)-1/2 (flo); fhi() is the new one.
  template <int K>
  __device__ __forceinline__ void push(real vtn, real btn, real bold, real dt, real hdt, real& bnew, real& flo) {
    const real vg1 = real(0.25) * fma_(real(2), vt[(K + 1) & 1], vt[K & 1] + vtn);   // eq (20) at k-1
    const real w01 = vg1 * b[(K + 1) & 1];
    const real vh2 = vg + vg1;                                                       // 2 * eq (22) at face (k-2)+1/2
    const real f1n = pick_pos(vh2, w0, w01);                                         // eq (21)
    const real bh = fnma_(f1n - f1, hdt, b[K & 1]);                                  // Alg. 2 step 7: B_t^{t+dt/2}(k-2)
    const real wD = vg * bh;
    // Alg. 2 step 8: second-order TVD flux at face (k-4)+1/2, upwinded by the sign of the face velocity there
    const real up = vh[K & 1];
    const real wA = w1[(K + 3) & 3], wB = w1[K & 3], wC = w1[(K + 1) & 3];           // at k-5, k-4, k-3
    const real x = pick_pos(up, wB, wC), y = pick_pos(up, wA, wD), z = pick_pos(up, wC, wB);
    const real fn = (x + vl_full(x - y, z - x)) * dt;
    bnew = bold - (fn - f);                                                          // Alg. 2 step 9 at cell k-4
    flo = f;
    f = fn; f1 = f1n; vg = vg1; w0 = w01;
    vt[K & 1] = vtn; b[K & 1] = btn; w1[(K + 2) & 3] = wD; vh[K & 1] = vh2;
  }
  __device__ __forceinline__ real fhi() const { return f; }
};

template <class real, int TXB>
struct BRowRing {
  static constexpr int CH = 16 / sizeof(real);           // elements in one 16-byte chunk
  static constexpr int P = TXB + 2 * CH;                 // row pitch: [left chunk][TXB cells][right chunk]
  enum { R_RHO = 0, R_MD = 3, R_BX = 6, R_BO = 7, R_BD = 9, ROWS = 10, NCHUNK = 5, NCOPY = ROWS + NCHUNK };
  static constexpr int STAGE = ROWS * P;
  static constexpr uint32_t BYTES = ROWS * TXB * sizeof(real) + NCHUNK * 16;
  static size_t smem_bytes(int D) { return (size_t)D * STAGE * sizeof(real) + 2 * D * sizeof(uint64_t); }
};

#ifndef MHD_BRING_MINB
#define MHD_BRING_MINB 2
#endif

// real: element type in memory (float/double).  T: arithmetic pack (f2 for float, double for double).
template <class real, class T, int TXB, int D>
__global__ void __launch_bounds__(TXB / PackOf<T>::L + 32, MHD_BRING_MINB) bpair_ring_kernel(const YZArgs<real> A) {
  using RG = BRowRing<real, TXB>;
  constexpr int L = PackOf<T>::L;
  constexpr int NC = TXB / L;                             // consumer threads
  constexpr int CH = RG::CH, P = RG::P;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* ring = reinterpret_cast<real*>(smem_raw);
  uint64_t* full = reinterpret_cast<uint64_t*>(ring + D * RG::STAGE);
  uint64_t* empty = full + D;

  const int tid = threadIdx.x;
  const int x0 = blockIdx.x * TXB, o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  const int niter = (n1 - n0 + 8 + 3) & ~3;               // cells n0-4 .. n1+3, rounded up to the 4x unrolled march
  const int xl = map_index1(x0 - 1, A.nx, A.bc), xr = map_index1(x0 + TXB, A.nx, A.bc);
  if (tid == 0) {
    for (int s = 0; s < D; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], NC); }
    mbar_fence_init();
  }
  __syncthreads();

  if (tid >= NC) {
    // ---------------- producer warp: lane c issues copy c of every stage ----------------
    const int c = tid - NC;
    if (c >= RG::NCOPY) return;
    const int om = map_index1(o - 1, A.no, A.bc), op = map_index1(o + 1, A.no, A.bc);
    const real* src;
    int dst, nbytes = TXB * (int)sizeof(real), late = 0, xoff = x0;
    switch (c) {
      case 0: src = A.u[0] + (size_t)om * A.so; dst = 0 * P + CH; break;
      case 1: src = A.u[0] + (size_t)o * A.so;  dst = 1 * P + CH; break;
      case 2: src = A.u[0] + (size_t)op * A.so; dst = 2 * P + CH; break;
      case 3: src = A.u[1] + (size_t)om * A.so; dst = 3 * P + CH; break;
      case 4: src = A.u[1] + (size_t)o * A.so;  dst = 4 * P + CH; break;
      case 5: src = A.u[1] + (size_t)op * A.so; dst = 5 * P + CH; break;
      case 6: src = A.bx + (size_t)o * A.so;    dst = 6 * P + CH; break;
      case 7: src = A.bo + (size_t)o * A.so;    dst = 7 * P + CH; break;
      case 8: src = A.bo + (size_t)op * A.so;   dst = 8 * P + CH; break;
      case 9: src = A.bd + (size_t)o * A.so;    dst = 9 * P + CH; late = 1; break;
      case 10: src = A.u[0] + (size_t)o * A.so; dst = 1 * P;            xoff = (xl / CH) * CH; nbytes = 16; break;
      case 11: src = A.u[0] + (size_t)o * A.so; dst = 1 * P + CH + TXB; xoff = (xr / CH) * CH; nbytes = 16; break;
      case 12: src = A.u[1] + (size_t)o * A.so; dst = 4 * P;            xoff = (xl / CH) * CH; nbytes = 16; break;
      case 13: src = A.u[1] + (size_t)o * A.so; dst = 4 * P + CH + TXB; xoff = (xr / CH) * CH; nbytes = 16; break;
      default: src = A.bx + (size_t)o * A.so;   dst = 6 * P + CH + TXB; xoff = (xr / CH) * CH; nbytes = 16; break;
    }
    src += xoff;
    for (int it = 0; it < niter; ++it) {
      const int s = it % D;
      if (it >= D) mbar_wait(&empty[s], ((it / D) & 1) ^ 1);
      const int q = n0 - 4 + it;
      const int od = map_index1(late ? q - 4 : q, A.nd, A.bc) * A.sd;
      if (c == 0) mbar_expect_tx(&full[s], RG::BYTES);
      __syncwarp((1u << RG::NCOPY) - 1u);
      bulk_g2s(ring + s * RG::STAGE + dst, src + od, (uint32_t)nbytes, &full[s]);
    }
    return;
  }

  // ---------------- consumers: L adjacent pencils each ----------------
  typedef typename PackOf<T>::scalar S;
  const int cx = CH + L * tid;                            // my first column inside a stage row
  const int iL = tid == 0 ? xl % CH : cx - 1;             // column to my left / right (the chunks at the row ends)
  const int iR = tid == NC - 1 ? CH + TXB + xr % CH : cx + L;
  const S dts = (S)(*A.dt);
  const T dt(dts), hdt(S(0.5) * dts);
  const bool x_first = (A.x_is_t1 != 0) != (A.t2_first != 0);     // forward: t1 then t2; reverse: t2 then t1

  BPipe4R<T> pxA, po, pop;
  BPipe4R<S> pxE;
  pxA.init(); po.init(); pop.init(); pxE.init();
  int off = (n0 - 8) * A.sd + x0 + L * tid + o * A.so;    // output cell m = q - 4 = n0 + it - 8

  auto step = [&](auto Ktag, int it) {
    constexpr int K = decltype(Ktag)::value;
    const real* st = ring + ((unsigned)it % D) * RG::STAGE;
    const real* st4 = ring + ((unsigned)(it + D - 4) % D) * RG::STAGE;
    mbar_wait(&full[(unsigned)it % D], ((unsigned)it / D) & 1);
    T* tag = nullptr;
    const T rm = ld_pack(st + 0 * P + cx, tag), r0 = ld_pack(st + 1 * P + cx, tag), rp = ld_pack(st + 2 * P + cx, tag);
    const T mm = ld_pack(st + 3 * P + cx, tag), m0 = ld_pack(st + 4 * P + cx, tag), mp = ld_pack(st + 5 * P + cx, tag);
    const S rl = st[1 * P + iL], rr = st[1 * P + iR], ml = st[4 * P + iL], mr = st[4 * P + iR];
    const T bx = ld_pack(st + 6 * P + cx, tag);
    const S bxr = st[6 * P + iR];
    const T bo = ld_pack(st + 7 * P + cx, tag), bop = ld_pack(st + 8 * P + cx, tag);
    const T bd = ld_pack(st + 9 * P + cx, tag);             // B_d of the cell finished now (copied 4 cells behind)
    // B_t of the cell finished now: four march steps back in the ring
    const T bx4 = ld_pack(st4 + 6 * P + cx, tag), bo4 = ld_pack(st4 + 7 * P + cx, tag), bop4 = ld_pack(st4 + 8 * P + cx, tag);
    const S bxr4 = st4[6 * P + iR];
    if (it >= 4) mbar_arrive(&empty[(unsigned)(it + D - 4) % D]);   // stage it-4 is no longer needed
    // Alg. 2 step 4: face velocity = momentum sum / density sum of the two cells sharing the face (reading R5)
    const T vtA = (shift_in_left(m0, ml) + m0) * rcp_(shift_in_left(r0, rl) + r0);
    const S vtE = (last_lane(m0) + mr) * rcp_(last_lane(r0) + rr);
    const T vtO = (mm + m0) * rcp_(rm + r0);
    const T vtP = (m0 + mp) * rcp_(r0 + rp);
    T bxn, bon, bpn, fxlo, folo, fplo;
    S ben, felo;
    pxA.template push<K>(vtA, bx, bx4, dt, hdt, bxn, fxlo);
    pxE.template push<K>(vtE, bxr, bxr4, dts, S(0.5) * dts, ben, felo);
    po.template push<K>(vtO, bo, bo4, dt, hdt, bon, folo);
    pop.template push<K>(vtP, bop, bop4, dt, hdt, bpn, fplo);
    const int m = n0 + it - 8;
    if (it >= 8 && m < n1) {
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

}  // namespace mhd
