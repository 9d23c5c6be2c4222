// mhd_lrev.cuh -- fused operators for sweeps along y and z, periodic boundaries:
//
//   NP = 1, FL      reverse L_d = B pair (t2 first), then fluid_d          16 words / cell instead of 21
//   NP = 2, FL      the middle pair of a step: forward B pair, reverse B pair, fluid_d            16 instead of 29
//   NP = 2, !FL     the two adjacent B pairs of the middle pair alone                              8 instead of 16
//
// Every step's third and fourth operator share a direction (eqs (23)-(25) PAPER.md:164-170: L_z L_z, L_y L_y, L_x L_x), so
// the forward operator's B pair is followed at once by the reverse operator's B pair on the same rho, m_d, and that by the
// reverse operator's fluid update ("temporal fusion of the middle pair").
//
// One block owns a row of TXB pencils (fixed o, x0 <= x < x0 + TXB) and marches along d like the ring kernels of
// mhd_yz2.cuh / mhd_bring.cuh, but its warps are SPECIALISED and chained through shared memory:
//
//   TMA rings (cp.async.bulk) --> P1 warps --X1--> P2 warps (NP = 2) --X2--> F warps --> global u
//                                                  '--> global B (the last pass stores the field)
//
//   P1, P2   Algorithm 2 exactly as bpair_ring_kernel runs it: four flux pipelines per thread (B_x of its
//            own columns and of the column to the right, B_o of rows o and o+1).  The "+1" pipelines exist for the constraint
//            step -- and their ADVECTED values are B_x' of the next column and B_o' of row o+1, which is
//            everything the next stage needs from the neighbouring pencils: the cell-centred field of the fluid update
//            (eq (19)) and the +1 rows of the next B pair.  So no stage reads a row this block does not
//            compute, and the intermediate field never touches global memory.
//   F        Algorithm 1 exactly as fluid_yz_ring_kernel runs it, with the updated faces taken from
//            the X2 ring instead of global memory.
//
// Each stage trails the one before by its stencil (4 cells per B pass, 1 + 3 for the fluid update); the stages hand rows
// over through small shared-memory rings guarded by full/empty mbarriers (generic-proxy writes, release on arrive,
// acquire on wait), so there is still no block barrier and every warp drifts freely within the ring depths.
// A chained stage consumes its predecessor's values at ghost positions (cells outside the segment, and outside the grid);
// those equal the mapped values of the predecessor's OUTPUT only for periodic boundaries (reading R9 maps the INPUTS of
// every operator), hence: periodic only.  Outflow grids run the unfused kernels.
//
// Requirements: periodic BC, nx % TXB == 0, extent along d >= 16, N < 2^31.
#pragma once
#include <type_traits>
#include "mhd_async.cuh"
#include "mhd_bring.cuh"
#include "mhd_yz2.cuh"

namespace mhd {

template <class real>
struct LRevArgs {
  const real* u[5];             // rho, m_d, m_t1, m_t2, E (sweep roles), current state
  real* uo[5];                  // fluid outputs (FL)
  const real *bd, *bx, *bo;
  real *bdo, *bxo, *boo;
  const double* dt;
  unsigned long long* cmax_bits;
  int nx, nd, no;
  int sd, so;
  int seg;
  int x_is_t1;
  int t2_first[2];              // per B pass: reverse sweeps apply B_{t2->d} first
  real gamma;
};

template <class real, int TXB, int NP, bool FL>
struct LRevLayout {
  static constexpr int CH = 16 / sizeof(real);
  static constexpr int P = TXB + 2 * CH;                  // row pitch: [left chunk][TXB cells][right chunk]
  static constexpr int DA = NP == 2 ? 12 : 8;             // rho, m_d rows o-1, o, o+1 (P2 reads them 4 steps after P1)
  static constexpr int DB = 8;                            // B_x, B_o (o, o+1), B_d four cells behind: P1 only
  static constexpr int DX1 = NP == 2 ? 8 : 0;             // P1 -> P2: B_x' (+ edge), B_o'(o), B_o'(o+1), B_d'; P2 re-reads B_d' 4 steps later
  static constexpr int DX2 = FL ? 4 : 0;                  // last pass -> F
  static constexpr int DU = FL ? 8 : 0;                   // u rows of the fluid stage (re-read 1 and 3 steps later)
  static constexpr int A_STAGE = 6 * P, B_STAGE = 4 * P, X_STAGE = 4 * P, U_STAGE = 5 * TXB;
  static constexpr int A_OFF = 0;
  static constexpr int B_OFF = A_OFF + DA * A_STAGE;
  static constexpr int X1_OFF = B_OFF + DB * B_STAGE;
  static constexpr int X2_OFF = X1_OFF + DX1 * X_STAGE;
  static constexpr int U_OFF = X2_OFF + DX2 * X_STAGE;
  static constexpr int REALS = U_OFF + DU * U_STAGE;
  static constexpr int NBAR = 2 * (DA + DB + DX1 + DX2 + DU);
  static constexpr uint32_t A_BYTES = 6 * TXB * sizeof(real) + 4 * 16;
  static constexpr uint32_t B_BYTES = 4 * TXB * sizeof(real) + 16;
  static constexpr uint32_t U_BYTES = 5 * TXB * sizeof(real);
  static size_t smem_bytes() { return (size_t)REALS * sizeof(real) + NBAR * sizeof(uint64_t); }
};

#ifndef MHD_LREV_PF
#define MHD_LREV_PF 5          // march steps of TMA prefetch for the A/B rings (depth 8: consumed at 0, slack 2)
#endif
#ifndef MHD_LREV_PFU
#define MHD_LREV_PFU 3         // for the U ring (depth 8, stages live three steps)
#endif
#ifndef MHD_LREV_MINB
#define MHD_LREV_MINB(NP, FL) ((NP) == 2 && (FL) ? 2 : 3)
#endif

// slot of a ring with D stages (D a multiple of 4) for march step 4*g + K, K a compile-time constant: base + K, where
// base = (4*g) % D is carried in a register and advanced once per four steps
__device__ __forceinline__ void adv4(int& base, uint32_t& phase, int D) { base += 4; if (base == D) { base = 0; phase ^= 1u; } }

template <class real, class T, int TXB, int NP, bool FL, bool XT1, bool CM>
__global__ void __launch_bounds__((NP + (FL ? 1 : 0)) * (TXB / PackOf<T>::L), MHD_LREV_MINB(NP, FL))
lrev_ring_kernel(const LRevArgs<real> A) {
  using LY = LRevLayout<real, TXB, NP, FL>;
  typedef typename PackOf<T>::scalar S;
  constexpr int L = PackOf<T>::L;
  constexpr int NR = TXB / L;                              // threads per role
  constexpr int NWG = NR / 32;                             // warps per role
  constexpr int CH = LY::CH, P = LY::P;
  constexpr int DA = LY::DA, DB = LY::DB, DX1 = LY::DX1, DX2 = LY::DX2, DU = LY::DU;
  constexpr int PF = MHD_LREV_PF, PFU = MHD_LREV_PFU;
  static_assert(NWG >= 1 && (NWG & (NWG - 1)) == 0 && NWG <= 4, "role shape");
  static_assert(DA % 4 == 0 && DB % 4 == 0 && DX1 % 4 == 0 && DX2 % 4 == 0 && DU % 4 == 0, "ring depths are multiples of the unroll");
  extern __shared__ __align__(128) unsigned char smem_raw[];
  real* sm = reinterpret_cast<real*>(smem_raw);
  real* ringA = sm + LY::A_OFF;
  real* ringB = sm + LY::B_OFF;
  real* ringX1 = sm + LY::X1_OFF;
  real* ringX2 = sm + LY::X2_OFF;
  real* ringU = sm + LY::U_OFF;
  uint64_t* bars = reinterpret_cast<uint64_t*>(sm + LY::REALS);
  uint64_t* fullA = bars;            uint64_t* emptyA = fullA + DA;
  uint64_t* fullB = emptyA + DA;     uint64_t* emptyB = fullB + DB;
  uint64_t* fullX1 = emptyB + DB;    uint64_t* emptyX1 = fullX1 + DX1;
  uint64_t* fullX2 = emptyX1 + DX1;  uint64_t* emptyX2 = fullX2 + DX2;
  uint64_t* fullU = emptyX2 + DX2;   uint64_t* emptyU = fullU + DU;

  const int tid = threadIdx.x, lane = tid & 31;
  const int role = __shfl_sync(0xffffffffu, tid / NR, 0);          // warp-uniform, and known to be so
  const int rt = tid - role * NR;                                   // thread index inside the role
  const int wr = __shfl_sync(0xffffffffu, rt >> 5, 0);              // warp index inside the role
  const int x0 = blockIdx.x * TXB, o = blockIdx.y;
  const int n0 = blockIdx.z * A.seg;
  const int n1 = min(n0 + A.seg, A.nd);
  // iteration counts, from the last stage backwards (all multiples of 4; see the header for the lags)
  const int nF = (n1 - n0 + 6 + 3) & ~3;                            // F pushes cells n0-3 ..
  const int cB = FL ? n0 - 3 : n0;                                  // first cell the LAST pass must deliver
  const int nOutL = FL ? nF + 1 : n1 - n0;                          // how many (F also reads B_d of the next cell)
  const int nPL = (nOutL + 8 + 3) & ~3;                             // iterations of the last pass
  const int nP1 = NP == 2 ? nPL + 8 : nPL;                          // P1 must deliver every input cell of P2
  const int a0 = cB - 4 * NP;                                       // first input cell of P1 = ordinal 0 of the A/B rings
  if (tid == 0) {
    for (int s = 0; s < DA; ++s) { mbar_init(&fullA[s], 1); mbar_init(&emptyA[s], NWG * NP); }
    for (int s = 0; s < DB; ++s) { mbar_init(&fullB[s], 1); mbar_init(&emptyB[s], NWG); }
    for (int s = 0; s < DX1; ++s) { mbar_init(&fullX1[s], NWG); mbar_init(&emptyX1[s], NWG); }
    for (int s = 0; s < DX2; ++s) { mbar_init(&fullX2[s], NWG); mbar_init(&emptyX2[s], NWG); }
    for (int s = 0; s < DU; ++s) { mbar_init(&fullU[s], 1); mbar_init(&emptyU[s], NWG); }
    mbar_fence_init();
  }
  __syncthreads();

  const S dts = (S)(*A.dt);
  const int xl = x0 == 0 ? A.nx - 1 : x0 - 1, xr = x0 + TXB == A.nx ? 0 : x0 + TXB;     // periodic neighbours of the tile
  auto wrap = [](int q, int n) { return q < 0 ? q + n : (q >= n ? q - n : q); };        // one wrap: |halo| <= 16 <= n
  T* tag = nullptr;

  if (role < NP) {
    // =========================================== B passes ===========================================================
    const bool first = role == 0, last = role == NP - 1;
    const int om_off = wrap(o - 1, A.no) * A.so, o_off = o * A.so, op_off = wrap(o + 1, A.no) * A.so;
    const int cl = (xl / CH) * CH + o_off, cr = (xr / CH) * CH + o_off;
    // ---- P1 warps take turns at feeding the A and B rings: one elected lane, warp-uniform operands (mhd_async.cuh) ----
    auto produce = [&](int ord) {
      const int sa = ord % DA, sb = ord % DB;
      if (ord >= DA) mbar_wait(&emptyA[sa], (((unsigned)ord / DA) & 1) ^ 1);
      if (ord >= DB) mbar_wait(&emptyB[sb], (((unsigned)ord / DB) & 1) ^ 1);
      if (elect_one()) {
        const int od = wrap(a0 + ord, A.nd) * A.sd;
        const int odl = wrap(a0 + ord - 4, A.nd) * A.sd;            // B_d of the cell P1 finishes at this step
        real* sa_ = ringA + sa * LY::A_STAGE;
        real* sb_ = ringB + sb * LY::B_STAGE;
        constexpr uint32_t RB = TXB * sizeof(real);
        const real* rho = A.u[0] + od;
        const real* md = A.u[1] + od;
        mbar_expect_tx(&fullA[sa], LY::A_BYTES);
        bulk_g2s(sa_ + 0 * P + CH, rho + om_off + x0, RB, &fullA[sa]);
        bulk_g2s(sa_ + 1 * P + CH, rho + o_off + x0, RB, &fullA[sa]);
        bulk_g2s(sa_ + 2 * P + CH, rho + op_off + x0, RB, &fullA[sa]);
        bulk_g2s(sa_ + 3 * P + CH, md + om_off + x0, RB, &fullA[sa]);
        bulk_g2s(sa_ + 4 * P + CH, md + o_off + x0, RB, &fullA[sa]);
        bulk_g2s(sa_ + 5 * P + CH, md + op_off + x0, RB, &fullA[sa]);
        bulk_g2s(sa_ + 1 * P, rho + cl, 16, &fullA[sa]);
        bulk_g2s(sa_ + 1 * P + CH + TXB, rho + cr, 16, &fullA[sa]);
        bulk_g2s(sa_ + 4 * P, md + cl, 16, &fullA[sa]);
        bulk_g2s(sa_ + 4 * P + CH + TXB, md + cr, 16, &fullA[sa]);
        mbar_expect_tx(&fullB[sb], LY::B_BYTES);
        bulk_g2s(sb_ + 0 * P + CH, A.bx + od + o_off + x0, RB, &fullB[sb]);
        bulk_g2s(sb_ + 0 * P + CH + TXB, A.bx + od + cr, 16, &fullB[sb]);
        bulk_g2s(sb_ + 1 * P + CH, A.bo + od + o_off + x0, RB, &fullB[sb]);
        bulk_g2s(sb_ + 2 * P + CH, A.bo + od + op_off + x0, RB, &fullB[sb]);
        bulk_g2s(sb_ + 3 * P + CH, A.bd + odl + o_off + x0, RB, &fullB[sb]);
      }
      __syncwarp();
    };
    if (first) {
      for (int ord = wr; ord < PF && ord < nP1; ord += NWG) produce(ord);
    } else if (lane == 0) {
      // P2 never reads the A stages of ordinals 0..3 (its first input cell is ordinal 4): release them now
      for (int s = 0; s < 4; ++s) mbar_arrive(&emptyA[s]);
    }

    const int cx = CH + L * rt;                                      // my first column inside a row
    const int iL = rt == 0 ? xl % CH : cx - 1;                       // rho, m_d of the column to my left / right
    const int iR = rt == NR - 1 ? CH + TXB + xr % CH : cx + L;
    const int iRb = first ? iR : (rt == NR - 1 ? CH + TXB : cx + L); // B_x of the column to my right: TMA chunk (P1) or edge slot (X1)
    const T dt(dts), hdt(S(0.5) * dts);
    const int niter = first ? nP1 : nPL;
    const int t2f = A.t2_first[role];
    const bool x_first = (A.x_is_t1 != 0) != (t2f != 0);             // forward: t1 then t2; reverse: t2 then t1
    // my output cells: ordinal j = it - 8 of the next ring <-> cell c_out0 + j
    const int c_out0 = first ? a0 + 4 : cB;
    int off = c_out0 * A.sd + x0 + L * rt + o * A.so;                // global offset of output ordinal 0 (may be a ghost cell: only used in range)

    BPipe4<T> pxA, po, pop;
    BPipe4<S> pxE;
    pxA.init(); po.init(); pop.init(); pxE.init();
    // ring positions for step 4*g + K: A (P2 runs 4 ordinals behind its own step count: it reads ordinal it + 4)
    int a4 = first ? 0 : 4; uint32_t aph = 0;
    int b4 = 0; uint32_t bph = 0;                                    // P1: B ring; P2: X1 ring as input
    int b4prev = 0; uint32_t bphprev = 0;                            // P2: the X1 slots of four steps ago (B_d' of the finishing cell)
    int w4 = 0; uint32_t wph = 0;                                    // output ring (X1 for P1 when NP = 2, X2 for the last pass when FL)
    real* ringIn = first ? ringB : ringX1;
    uint64_t* fullIn = first ? fullB : fullX1;
    constexpr int IN_STAGE = LY::B_STAGE;                            // = X_STAGE
    static_assert(LY::B_STAGE == LY::X_STAGE, "P1 and P2 share the input row layout");
    const bool to_ring = (NP == 2 && first) || (FL && last);
    real* ringOut = (NP == 2 && first) ? ringX1 : ringX2;
    uint64_t* fullOut = (NP == 2 && first) ? fullX1 : fullX2;
    uint64_t* emptyOut = (NP == 2 && first) ? emptyX1 : emptyX2;
    const int DOUT = (NP == 2 && first) ? DX1 : DX2;
    const int nOut = first && NP == 2 ? nPL : nOutL;                  // output ordinals the next stage reads

    auto step = [&](auto Ktag, int it) {
      constexpr int K = decltype(Ktag)::value;
      if (first) { if ((K & (NWG - 1)) == wr && it + PF < niter) produce(it + PF); }
      const real* sa = ringA + (a4 + K) * LY::A_STAGE;
      const real* sb = ringIn + (b4 + K) * IN_STAGE;
      mbar_wait(&fullA[a4 + K], aph);
      mbar_wait(&fullIn[b4 + K], bph);
      const T rm = ld_pack(sa + 0 * P + cx, tag), r0 = ld_pack(sa + 1 * P + cx, tag), rp = ld_pack(sa + 2 * P + cx, tag);
      const T mm = ld_pack(sa + 3 * P + cx, tag), m0 = ld_pack(sa + 4 * P + cx, tag), mp = ld_pack(sa + 5 * P + cx, tag);
      const S rl = sa[1 * P + iL], rr = sa[1 * P + iR], ml = sa[4 * P + iL], mr = sa[4 * P + iR];
      const T bx = ld_pack(sb + 0 * P + cx, tag);
      const S bxr = sb[0 * P + iRb];
      const T bo = ld_pack(sb + 1 * P + cx, tag), bop = ld_pack(sb + 2 * P + cx, tag);
      T bd;
      if (first) bd = ld_pack(sb + 3 * P + cx, tag);                 // TMA copied B_d four cells behind
      else bd = ld_pack(ringX1 + (b4prev + K) * IN_STAGE + 3 * P + cx, tag);   // B_d' of the cell finishing now: X1 ordinal it - 4
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&emptyA[a4 + K]);
        if (first) mbar_arrive(&emptyB[b4 + K]);
        else if (it >= 4) mbar_arrive(&emptyX1[b4prev + K]);        // ordinal it - 4 is no longer needed
      }
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
      const int j = it - 8;                                          // output ordinal
      if (j >= 0) {
        // constraint with the same fluxes at face m-1/2: rows x+1 and o+1
        const T cxv = shift_in_right(fxlo, felo) - fxlo;
        const T cov = fplo - folo;
        T bdv = bd;
        if (x_first) { bdv = bdv + cxv; bdv = bdv + cov; }
        else         { bdv = bdv + cov; bdv = bdv + cxv; }
        if (to_ring && j < nOut) {
          real* so = ringOut + (w4 + K) * LY::X_STAGE;
          if (j >= DOUT) mbar_wait(&emptyOut[w4 + K], wph ^ 1);
          st_pack(so + 0 * P + cx, bxn);
          if (rt == NR - 1) so[0 * P + CH + TXB] = ben;              // B_x' of column x0 + TXB
          st_pack(so + 1 * P + cx, bon);
          st_pack(so + 2 * P + cx, bpn);
          st_pack(so + 3 * P + cx, bdv);
          __syncwarp();
          if (lane == 0) mbar_arrive(&fullOut[w4 + K]);
        }
        if (last) {
          const int m = c_out0 + j;
          if (m >= n0 && m < n1) {
            st_pack(A.bxo + off, bxn);                               // Alg. 2 step 9: advected B_t
            st_pack(A.boo + off, bon);
            st_pack(A.bdo + off, bdv);
          }
        }
        off += A.sd;
      }
    };
    for (int it = 0; it < niter; it += 4) {
      step(std::integral_constant<int, 0>{}, it);
      step(std::integral_constant<int, 1>{}, it + 1);
      step(std::integral_constant<int, 2>{}, it + 2);
      step(std::integral_constant<int, 3>{}, it + 3);
      adv4(a4, aph, DA);
      b4prev = b4; bphprev = bph;
      adv4(b4, bph, first ? DB : DX1);
      if (it >= 8) adv4(w4, wph, DOUT);
    }
    (void)bphprev;
  } else if constexpr (FL) {
    // =========================================== fluid update ========================================================
    const int rowbase = x0 + o * A.so;
    auto produceU = [&](int ord) {
      const int s = ord % DU;
      if (ord >= DU) mbar_wait(&emptyU[s], (((unsigned)ord / DU) & 1) ^ 1);
      if (elect_one()) {
        const int od = wrap(n0 - 3 + ord, A.nd) * A.sd;
        real* st = ringU + s * LY::U_STAGE;
        constexpr uint32_t RB = TXB * sizeof(real);
        mbar_expect_tx(&fullU[s], LY::U_BYTES);
#pragma unroll
        for (int k = 0; k < 5; ++k) bulk_g2s(st + k * TXB, A.u[k] + od + rowbase, RB, &fullU[s]);
      }
      __syncwarp();
    };
    for (int ord = wr; ord < PFU && ord < nF; ord += NWG) produceU(ord);

    const int c2 = L * rt;
    const int cx = CH + c2;
    const int iRb = rt == NR - 1 ? CH + TXB : cx + L;                // B_x'' of the column to my right
    const int base = x0 + c2 + o * A.so;
    const T hdt(S(0.5) * dts), qdt(S(0.25) * dts), gamma(A.gamma);
    FluidPipe<T> pipe;
    pipe.init();
    decltype(pack_speed_key((const T*)nullptr, T(), S())) cbest = 0;
    int u4 = 0, u4p = DU - 4; uint32_t uph = 0;                      // U slots of this group of four steps and of the previous one
    uint32_t xph = 0;                                                // X2 has exactly four slots: slot = K
    static_assert(!FL || DX2 == 4, "the fluid stage indexes X2 by the step modulo 4");
    mbar_wait(&fullX2[0], 0);
    T bd_lo = ld_pack(ringX2 + 3 * P + cx, tag);                     // B_d'' at the lower face of cell n0-3

    auto step = [&](auto Ktag, int it) {
      constexpr int K = decltype(Ktag)::value;
      if ((K & (NWG - 1)) == wr && it + PFU < nF) produceU(it + PFU);
      const real* st = ringU + (u4 + K) * LY::U_STAGE;
      const real* st1 = ringU + (K >= 1 ? u4 + K - 1 : u4p + 3) * LY::U_STAGE;
      const real* st3 = ringU + (K >= 3 ? u4 + K - 3 : u4p + K + 1) * LY::U_STAGE;
      const real* sx = ringX2 + K * LY::X_STAGE;
      const real* sxn = ringX2 + ((K + 1) & 3) * LY::X_STAGE;
      mbar_wait(&fullU[u4 + K], uph);
      // X2 ordinal `it` (slot K) was waited for one step ago as the "next" one (ordinal 0: before the loop)
      mbar_wait(&fullX2[(K + 1) & 3], K == 3 ? (xph ^ 1u) : xph);
      T u[5], um1[5], um3[5];
#pragma unroll
      for (int k = 0; k < 5; ++k) {
        u[k] = ld_pack(st + k * TXB + c2, tag);
        um1[k] = ld_pack(st1 + k * TXB + c2, tag);
        um3[k] = ld_pack(st3 + k * TXB + c2, tag);
      }
      const T bxa = ld_pack(sx + 0 * P + cx, tag);
      const S bxn = sx[0 * P + iRb];
      const T boa = ld_pack(sx + 1 * P + cx, tag), bob = ld_pack(sx + 2 * P + cx, tag);
      const T bd_hi = ld_pack(sxn + 3 * P + cx, tag);
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&emptyX2[K]);
        if (it >= 3) mbar_arrive(&emptyU[K >= 3 ? u4 + K - 3 : u4p + K + 1]);
      }
      const T half(S(0.5));
      const T boc = half * (boa + bob);
      const T bxc = half * (bxa + shift_in_right(bxa, bxn));         // eq (19): faces -> centre
      const T bdc = half * (bd_lo + bd_hi);
      BCell<T> B;
      if (XT1) B.set(bdc, bxc, boc);
      else     B.set(bdc, boc, bxc);
      bd_lo = bd_hi;
      T out[5];
      pipe.advance(u, um1, um3, B, gamma, hdt, qdt, out);
      const int m = n0 - 6 + it;                                     // cell q-3
      if (m >= n0 && m < n1) {
        const int offo = m * A.sd + base;
#pragma unroll
        for (int k = 0; k < 5; ++k) st_pack(A.uo[k] + offo, out[k]);
        if (CM) {                  // last operator of a step: c of eq (18) from the updated cells (B is final here too)
          const auto b = pack_speed_key(out, pipe.hb2_out(), (S)A.gamma);
          cbest = b > cbest ? b : cbest;
        }
      }
    };
    for (int it = 0; it < nF; it += 4) {
      step(std::integral_constant<int, 0>{}, it);
      step(std::integral_constant<int, 1>{}, it + 1);
      step(std::integral_constant<int, 2>{}, it + 2);
      step(std::integral_constant<int, 3>{}, it + 3);
      u4p = u4;
      adv4(u4, uph, DU);
      xph ^= 1u;
    }
    if (CM) {
      const unsigned long long cw = warp_max_u64(key_bits(cbest));
      if (lane == 0) publish_max(A.cmax_bits, cw);
    }
  }
}

}  // namespace mhd
