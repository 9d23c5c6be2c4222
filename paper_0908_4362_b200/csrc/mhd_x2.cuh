// mhd_x2.cuh -- sweeps along x (the contiguous axis), periodic boundaries, in lane-pack arithmetic, and the
// fused reverse operator L_x^rev = B_{z->x}, B_{y->x}, fluid_x in ONE kernel.
//
// Along x the stencil runs along the lanes, so instead of marching a thread owns V consecutive cells of a row
// (V = 4 floats or 2 doubles: every global access is one aligned 16-byte vector) and a group of nx/V threads
// covers the whole row, so the periodic wrap is the group's own ring; the few stencil values a thread needs from
// its neighbours go through shared memory, one barrier per stage, and no halo cell is recomputed.  Two refinements:
//
//  * T = f2 (mhd_pack.cuh): a thread owns the same V columns of TWO adjacent rows (j, j+1) and advances
//    both with packed fp32 instructions (FADD2/FMUL2/FFMA2): the scalar x kernels are issue-bound
//    (round-1 ncu capture: 273 and 194 issued instructions per cell, 65-68 % issue
//    utilisation), and about 60 % of what they issue is FADD/FMUL/FFMA.  The shared-memory exchange moves
//    8-byte packs (LDS.64/STS.64), so those instructions halve per cell as well.
//  * the reverse operator needs no second pass over the state: in a reverse sweep the B pair runs BEFORE
//    the fluid update, and everything fluid_x needs from the updated field is already in the
//    registers of the thread that ran the four flux rows of Algorithm 2: B_y' of rows j and j+1 (the row
//    j+1 pipeline exists for the constraint step, and its advected value is B_y'(j+1)),
//    B_z' of planes k and k+1 likewise, B_x' of its own faces; only B_x' of the next thread's first face
//    crosses threads.  One kernel then reads 8 fields and writes 8 (16 words per cell instead of 21).
//    The FORWARD operator cannot be fused this way: its B pair needs the UPDATED rho, m_x of the four
//    transverse neighbour rows, i.e. the fluid update of rows this block does not own.
//
// Requirements (else the generic kernels of mhd_generic.cuh run): nx % V == 0, a row (plus its ghost threads under
// outflow boundaries, see ghost_fix) within 512 threads, i.e. nx <= 2048 (fp32) / 1024 (fp64), N < 2^31; the packed (f2)
// and fused variants additionally need periodic boundaries, nx <= 512 and (f2) an even ny.
#pragma once
#include "mhd_args.cuh"
#include "mhd_pack_io.cuh"

namespace mhd {

// threads per block (maximum) = shared-memory slot stride: a compile-time constant keeps every exchange
// address an immediate offset from three base registers (own slot, left and right neighbour)
// NT is also a template parameter of the kernels: rows longer than NT * V cells (512) run in blocks of 2 NT or 4 NT
// threads (the paper's own 2-D sizes reach 1024^2, Table 2), at proportionally fewer blocks per SM
template <class real> struct X2Block { static constexpr int NT = sizeof(real) == 4 ? 128 : 256; static constexpr int NT_MAX = sizeof(real) == 4 ? 512 : 512; };
// blocks per SM for a block of NT threads, given the count tuned for the base block
template <class real> constexpr int x2_minb(int base, int NT) { return base * X2Block<real>::NT / NT > 0 ? base * X2Block<real>::NT / NT : 1; }

// ---- V-cell vectors of L rows <-> packs ------------------------------------------------------------
// f2: the two rows arrive as two 16-byte vectors, and a pack must sit in an aligned register PAIR.  ptxas
// re-forms such a pair with two MOVs at EVERY use of a value that came straight out of a vector load (46 MOVs
// per cell in a first version of fluid_x: 208 issued instructions per cell against 164 now, ncu SASS page).  A value produced by a scalar
// instruction, however, is allocated directly into its half of the pair, so each loaded value is passed
// through ONE exact scalar multiplication by a run-time 1.0f (XArgs::one; a literal would be folded away).
__device__ __forceinline__ void xload(const float* f, int oa, int ob, f2 (&v)[4], float one) {
  const float4 a = __ldg(reinterpret_cast<const float4*>(f + oa));
  const float4 b = __ldg(reinterpret_cast<const float4*>(f + ob));
  v[0] = f2(a.x * one, b.x * one); v[1] = f2(a.y * one, b.y * one);
  v[2] = f2(a.z * one, b.z * one); v[3] = f2(a.w * one, b.w * one);
}
__device__ __forceinline__ void xload(const double* f, int oa, int, double (&v)[2], double) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(f + oa));
  v[0] = a.x; v[1] = a.y;
}
__device__ __forceinline__ void xload(const float* f, int oa, int, float (&v)[4], float) {
  const float4 a = __ldg(reinterpret_cast<const float4*>(f + oa));
  v[0] = a.x; v[1] = a.y; v[2] = a.z; v[3] = a.w;
}
__device__ __forceinline__ void xstore(float* f, int oa, int ob, const f2 (&v)[4]) {
  *reinterpret_cast<float4*>(f + oa) = make_float4(v[0].v.x, v[1].v.x, v[2].v.x, v[3].v.x);
  *reinterpret_cast<float4*>(f + ob) = make_float4(v[0].v.y, v[1].v.y, v[2].v.y, v[3].v.y);
}
__device__ __forceinline__ void xstore(double* f, int oa, int, const double (&v)[2]) {
  *reinterpret_cast<double2*>(f + oa) = make_double2(v[0], v[1]);
}
__device__ __forceinline__ void xstore(float* f, int oa, int, const float (&v)[4]) {
  *reinterpret_cast<float4*>(f + oa) = make_float4(v[0], v[1], v[2], v[3]);
}
// one element per row
__device__ __forceinline__ f2 xload1(const float* f, int oa, int ob, f2*) { return f2(__ldg(f + oa), __ldg(f + ob)); }   // scalar loads land in place
__device__ __forceinline__ double xload1(const double* f, int oa, int, double*) { return __ldg(f + oa); }
__device__ __forceinline__ float xload1(const float* f, int oa, int, float*) { return __ldg(f + oa); }

// Where the rows of one thread live.  Lane l of a pack is row j+l of plane k (L = 1 or 2).
struct XRows {
  int t, tl, tr;            // my thread index in the row group; block-local thread ids of my left / right neighbour
  int col;                  // first column
  int o[4];                 // offsets of rows j-1, j, j+1, j+2 of plane k (j+2 only used for L = 2)
  int okm[2], okp[2];       // rows j, j+1 of planes k-1 and k+1
  int onext[2];             // B_x face of the next thread's first column, rows j and j+1
  int mode;                 // outflow kernels: 0 interior thread, 1 left ghost (every cell = column 0), 2 right ghost (column nx-1)
  bool live;
};

// Outflow along x (reading R9: every out-of-range read of an operator INPUT is clamped, intermediates at ghost positions
// are computed from the clamped inputs): a row group is widened by A.ghost threads = 4 cells on either side whose loads
// return the edge column and whose results are not stored.  A kept cell depends on inputs at most 3 (fluid) or 4 (B pair)
// cells away, all of them true ghost values; what the ring of the exchange joins beyond them (the other end's ghosts) never
// reaches it.
template <int V, class T>
__device__ __forceinline__ void ghost_fix(T (&v)[V], int mode) {     // selects, no branch: the edge warps stay in step
  const T lo = v[0], hi = v[V - 1];
#pragma unroll
  for (int i = 0; i < V; ++i) v[i] = mode == 1 ? lo : (mode == 2 ? hi : v[i]);
}

template <class real, int L, bool OUT = false>
__device__ __forceinline__ XRows x_rows(const XArgs<real>& A) {
  constexpr int V = VecOf<real>::V;
  XRows r;
  const int tid = threadIdx.x;
  const int lr = A.tpr_shift >= 0 ? (tid >> A.tpr_shift) : tid / A.tpr;
  r.t = tid - lr * A.tpr;
  const int gpp = A.ny / L;                           // row groups per plane; blockIdx.y is the plane
  int g = blockIdx.x * A.rpb + lr;
  r.live = g < gpp;
  if (!r.live) g = gpp - 1;                           // keep the thread in step for the barriers
  const int k = blockIdx.y, j = g * L;
  r.mode = 0;
  int kp, km, jm, j1, j2, i_next;
  if (OUT) {
    int col = (r.t - A.ghost) * V;
    if (col < 0) { r.mode = 1; col = 0; }
    else if (col >= A.nx) { r.mode = 2; col = A.nx - V; }
    r.col = col;
    kp = min(k + 1, A.nz - 1); km = max(k - 1, 0);
    jm = max(j - 1, 0); j1 = min(j + 1, A.ny - 1); j2 = min(j1 + 1, A.ny - 1);
    i_next = r.mode == 1 ? 0 : (r.mode == 2 ? A.nx - 1 : min(col + V, A.nx - 1));
    r.live = r.live && r.mode == 0;
  } else {
    r.col = r.t * V;
    kp = (k + 1 == A.nz) ? 0 : k + 1; km = (k == 0) ? A.nz - 1 : k - 1;
    jm = (j == 0) ? A.ny - 1 : j - 1;
    j1 = (j + 1 == A.ny) ? 0 : j + 1;                 // L = 2: j is even and ny is even, so j1 = j + 1
    j2 = (j1 + 1 == A.ny) ? 0 : j1 + 1;
    i_next = (r.t == A.tpr - 1) ? 0 : (r.t + 1) * V;
  }
  auto row = [&](int jj, int kk) { return (kk * A.ny + jj) * A.nx + r.col; };
  r.o[0] = row(jm, k); r.o[1] = row(j, k); r.o[2] = row(j1, k); r.o[3] = row(j2, k);
  const int jb = (L == 2) ? j1 : j;
  r.okm[0] = row(j, km); r.okm[1] = row(jb, km);
  r.okp[0] = row(j, kp); r.okp[1] = row(jb, kp);
  r.onext[0] = (k * A.ny + j) * A.nx + i_next;
  r.onext[1] = (k * A.ny + jb) * A.nx + i_next;
  r.tl = lr * A.tpr + (r.t == 0 ? A.tpr - 1 : r.t - 1);
  r.tr = lr * A.tpr + (r.t == A.tpr - 1 ? 0 : r.t + 1);
  return r;
}

// right_left of the V cells of a thread.  One row per thread in fp32 (T = float, V = 4): the flux evaluation is cell by cell
// (no stencil), so cells (0,1) and (2,3) run as two f2 packs: FADD2 / FMUL2 / FFMA2 for what was two scalar streams, with
// the SAME registers (a float4 load puts neighbours in an aligned pair, scalar producers write into their half of a pair), so
// unlike packing two rows it costs no occupancy.  Results per cell are the same operations in the same order.
template <class T, int V>
__device__ __forceinline__ void right_left_cells(const T (&u)[V][5], const BCell<T> (&B)[V], T gamma, T (&R)[V][5], T (&G)[V][5]) {
#pragma unroll
  for (int v = 0; v < V; ++v) right_left(u[v], B[v], gamma, R[v], G[v]);
}
#ifndef MHD_X2_NO_CELLPACK
template <>
__device__ __forceinline__ void right_left_cells<float, 4>(const float (&u)[4][5], const BCell<float> (&B)[4], float gamma,
                                                           float (&R)[4][5], float (&G)[4][5]) {
#pragma unroll
  for (int v = 0; v < 4; v += 2) {
    f2 uu[5], RR[5], GG[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) uu[c] = f2(u[v][c], u[v + 1][c]);
    BCell<f2> BB;
    BB.b0 = f2(B[v].b0, B[v + 1].b0); BB.b1 = f2(B[v].b1, B[v + 1].b1); BB.b2 = f2(B[v].b2, B[v + 1].b2);
    BB.hb2 = f2(B[v].hb2, B[v + 1].hb2);
    right_left(uu, BB, f2(gamma), RR, GG);
#pragma unroll
    for (int c = 0; c < 5; ++c) { R[v][c] = RR[c].v.x; R[v + 1][c] = RR[c].v.y; G[v][c] = GG[c].v.x; G[v + 1][c] = GG[c].v.y; }
  }
}
#endif

// x[v] - d[v] * s for the V cells of a thread (the two update steps of Algorithm 1); fp32 one row per thread: two packs
template <class T, int V>
__device__ __forceinline__ void axpy_cells(const T (&d)[V], T s, const T (&x)[V], T (&y)[V]) {
#pragma unroll
  for (int v = 0; v < V; ++v) y[v] = fnma_(d[v], s, x[v]);
}
#ifndef MHD_X2_NO_CELLPACK
template <>
__device__ __forceinline__ void axpy_cells<float, 4>(const float (&d)[4], float s, const float (&x)[4], float (&y)[4]) {
#pragma unroll
  for (int v = 0; v < 4; v += 2) {
    const f2 r = fnma_(f2(d[v], d[v + 1]), f2(s), f2(x[v], x[v + 1]));
    y[v] = r.v.x; y[v + 1] = r.v.y;
  }
}
#endif

// ---------------------------------------------------------------------------------------------
// fluid_x of the V cells of one thread, Algorithm 1, in pack arithmetic.
// sm: 7 groups x 5 components x NT packs.  u[c][v], B[v] in; un[v][c] out.  Contains three barriers;
// the caller guarantees that nobody still reads sm when it is entered.
// ---------------------------------------------------------------------------------------------
template <class T, int V, int NT>
__device__ __forceinline__ void fluid_x_core(T* sm, int tid, int tl, int tr, const T (&u)[5][V],
                                             const BCell<T> (&B)[V], T gamma, T hdt, T qdt, T (&un)[V][5]) {
  auto S = [&](int group, int comp, int thr) -> T& { return sm[(group * 5 + comp) * NT + thr]; };
  // stage 0: R, G of u^t (Alg. 1 step 4)
  T R[V][5], G[V][5];
  {
    T uc[V][5];
#pragma unroll
    for (int v = 0; v < V; ++v)
#pragma unroll
      for (int c = 0; c < 5; ++c) uc[v][c] = u[c][v];
    right_left_cells<T, V>(uc, B, gamma, R, G);
  }
#pragma unroll
  for (int c = 0; c < 5; ++c) { S(0, c, tid) = R[V - 1][c]; S(1, c, tid) = G[0][c]; }
  __syncthreads();
  // steps 5-6: first-order fluxes at the V+1 faces of my cells, half step (eq (16))
  T uh[V][5];
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    T d1[V + 1];
    d1[0] = S(0, c, tl) - G[0][c];
#pragma unroll
    for (int v = 1; v < V; ++v) d1[v] = R[v - 1][c] - G[v][c];
    d1[V] = R[V - 1][c] - S(1, c, tr);
    {
      T dd[V], y[V];
#pragma unroll
      for (int v = 0; v < V; ++v) dd[v] = d1[v + 1] - d1[v];
      axpy_cells<T, V>(dd, qdt, u[c], y);
#pragma unroll
      for (int v = 0; v < V; ++v) uh[v][c] = y[v];
    }
  }
  // stage 1: R, G of u^{t+dt/2} (step 7), same B_c
  right_left_cells<T, V>(uh, B, gamma, R, G);
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    S(2, c, tid) = R[V - 1][c];      // my last R  -> right neighbour's R[-1]
    S(3, c, tid) = R[0][c];          // my first R -> left neighbour's R[V]
    S(4, c, tid) = G[0][c];          // my first two G -> left neighbour's G[V], G[V+1]
    S(5, c, tid) = G[1][c];
  }
  __syncthreads();
  // step 8: second-order TVD flux (twice its value) at the right face of each of my cells
  T phi[V + 1][5];
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    T r[V + 2], g[V + 2];            // r[v+1] = R at cell v (v = -1..V);  g[v] = G at cell v (v = 0..V+1)
    r[0] = S(2, c, tl);
#pragma unroll
    for (int v = 0; v < V; ++v) { r[v + 1] = R[v][c]; g[v] = G[v][c]; }
    r[V + 1] = S(3, c, tr);
    g[V] = S(4, c, tr);
    g[V + 1] = S(5, c, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const T Rp = vl_add(r[v + 1], r[v + 1] - r[v], r[v + 2] - r[v + 1]);        // eqs (11)-(15)
      const T Gp = vl_add(g[v + 1], g[v + 1] - g[v + 2], g[v] - g[v + 1]);        // mirror image
      phi[v + 1][c] = Rp - Gp;
    }
    S(6, c, tid) = phi[V][c];        // my last face -> right neighbour's left face
  }
  __syncthreads();
  // step 9: full step (eq (17))
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    phi[0][c] = S(6, c, tl);
    {
      T dd[V], y[V];
#pragma unroll
      for (int v = 0; v < V; ++v) dd[v] = phi[v + 1][c] - phi[v][c];
      axpy_cells<T, V>(dd, hdt, u[c], y);
#pragma unroll
      for (int v = 0; v < V; ++v) un[v][c] = y[v];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// B_{y->x} and B_{z->x} of the V cells of one thread (Algorithm 2; eqs (20)-(22)
// PAPER.md:147-158).  Four flux rows in lock step: p = 0: B_y row j, 1: B_y row j+1, 2: B_z plane k,
// 3: B_z plane k+1 (the +1 rows supply the constraint update of B_x).
// In: vt[p][v] face velocities, b[p][v] the transverse component of each row.  Out: f[p][0..V] = flux*dt at
// the faces v-1/2 (index v) of the V cells plus the right face of the last one.
// sm: 2 sets x 12 slots x NT packs.  Five barriers.
// ---------------------------------------------------------------------------------------------
template <class T, int V, int NT>
__device__ __forceinline__ void bpair_x_core(T* sm, int tid, int tl, int tr, const T (&vt)[4][V],
                                             const T (&b)[4][V], T dt, T hdt, T (&f)[4][V + 1]) {
  auto S = [&](int set, int slot, int thr) -> T& { return sm[(set * 12 + slot) * NT + thr]; };
  // stage A: eq (20), 1-2-1 smoothing along x
#pragma unroll
  for (int p = 0; p < 4; ++p) { S(0, p, tid) = vt[p][V - 1]; S(0, 4 + p, tid) = vt[p][0]; }
  __syncthreads();
  T vg[4][V + 1], w[4][V + 2];
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    T e[V + 2];
    e[0] = S(0, p, tl);
#pragma unroll
    for (int v = 0; v < V; ++v) e[v + 1] = vt[p][v];
    e[V + 1] = S(0, 4 + p, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      vg[p][v] = T(0.25) * fma_(T(2), e[v + 1], e[v] + e[v + 2]);
      w[p][v] = vg[p][v] * b[p][v];
    }
    S(1, p, tid) = vg[p][0]; S(1, 4 + p, tid) = w[p][0];
  }
  __syncthreads();
  // stage B: eqs (21),(22): first-order upwind flux at the right face of each cell
  T vh[4][V], f1[4][V + 1];
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    vg[p][V] = S(1, p, tr);
    w[p][V] = S(1, 4 + p, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      vh[p][v] = vg[p][v] + vg[p][v + 1];
      f1[p][v + 1] = pick_pos(vh[p][v], w[p][v], w[p][v + 1]);
    }
    S(0, 8 + p, tid) = f1[p][V];
  }
  __syncthreads();
  // stage C: half step (Alg. 2 step 7) and vg * B^{t+dt/2}
  T w1[4][V + 3];        // w1[p][v+1] = value at cell v, v = -1..V+1
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    f1[p][0] = S(0, 8 + p, tl);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const T bh = fnma_(f1[p][v + 1] - f1[p][v], hdt, b[p][v]);
      w1[p][v + 1] = vg[p][v] * bh;
    }
    S(1, 8 + p, tid) = w1[p][V];       // last  -> right neighbour's cell -1
    S(0, p, tid) = w1[p][1];           // first two -> left neighbour's cells V, V+1   (set 0 slots 0..7 are free again)
    S(0, 4 + p, tid) = w1[p][2];
  }
  __syncthreads();
  // stage D: second-order TVD flux at the right face of each cell (Alg. 2 step 8)
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    w1[p][0] = S(1, 8 + p, tl);
    w1[p][V + 1] = S(0, p, tr);
    w1[p][V + 2] = S(0, 4 + p, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const T x = pick_pos(vh[p][v], w1[p][v + 1], w1[p][v + 2]);
      const T y = pick_pos(vh[p][v], w1[p][v], w1[p][v + 3]);
      const T z = pick_pos(vh[p][v], w1[p][v + 2], w1[p][v + 1]);
      f[p][v + 1] = vl_add(x, x - y, z - x) * dt;
    }
    S(1, p, tid) = f[p][V];
  }
  __syncthreads();
#pragma unroll
  for (int p = 0; p < 4; ++p) f[p][0] = S(1, p, tl);
}

// Alg. 2 step 4 (reading R5) for the V cells of a thread: (ma + mb) / (ra + rb) cell by cell (packing these over cell pairs,
// like right_left_cells, and likewise the cell-by-cell parts of bpair_x_core, was measured: no gain / 7 % slower)
template <class T, int V>
__device__ __forceinline__ void face_velocity(const T (&ma)[V], const T (&mb)[V], const T (&ra)[V], const T (&rb)[V], T (&vt)[V]) {
#pragma unroll
  for (int v = 0; v < V; ++v) vt[v] = (ma[v] + mb[v]) * rcp_(ra[v] + rb[v]);
}

// face velocities and transverse fields of the four flux rows of one thread (Alg. 2 step 4, reading R5:
// momentum sum over density sum of the two cells sharing the face).  r0, m0: rho, m_x of the thread's own cells.
template <class real, class T, int V, bool OUT = false>
__device__ __forceinline__ void bpair_x_inputs(const XArgs<real>& A, const XRows& q, T (&r0)[V], T (&m0)[V],
                                               T (&vt)[4][V], T (&b)[4][V]) {
  T r[V], m[V];
  auto ld = [&](const real* f, int oa, int ob, T (&v)[V]) { xload(f, oa, ob, v, A.one); };
  ld(A.u[0], q.o[1], q.o[2], r0); ld(A.u[1], q.o[1], q.o[2], m0);
  ld(A.u[0], q.o[0], q.o[1], r); ld(A.u[1], q.o[0], q.o[1], m);                  // rows j-1 (, j)
  face_velocity<T, V>(m, m0, r, r0, vt[0]);
  ld(A.u[0], q.o[2], q.o[3], r); ld(A.u[1], q.o[2], q.o[3], m);                  // rows j+1 (, j+2)
  face_velocity<T, V>(m0, m, r0, r, vt[1]);
  ld(A.u[0], q.okm[0], q.okm[1], r); ld(A.u[1], q.okm[0], q.okm[1], m);
  face_velocity<T, V>(m, m0, r, r0, vt[2]);
  ld(A.u[0], q.okp[0], q.okp[1], r); ld(A.u[1], q.okp[0], q.okp[1], m);
  face_velocity<T, V>(m0, m, r0, r, vt[3]);
  ld(A.by, q.o[1], q.o[2], b[0]);
  ld(A.by, q.o[2], q.o[3], b[1]);
  ld(A.bz, q.o[1], q.o[2], b[2]);
  ld(A.bz, q.okp[0], q.okp[1], b[3]);
  if (OUT) {      // ghost threads: every cell is the edge column.  vt is computed column by column, so fixing the results is
                  // the same as fixing the loads, and it leaves the loads free to be issued back to back
#pragma unroll
    for (int p = 0; p < 4; ++p) { ghost_fix<V>(vt[p], q.mode); ghost_fix<V>(b[p], q.mode); }
  }
}

// cell-centred field of my V cells from face values (eq (19))
template <class T, int V>
__device__ __forceinline__ void x_centre(const T (&bxe)[V + 1], const T (&bya)[V], const T (&byb)[V], const T (&bza)[V],
                                         const T (&bzb)[V], BCell<T> (&B)[V]) {
  const T half(0.5);
#pragma unroll
  for (int v = 0; v < V; ++v)
    B[v].set(half * (bxe[v] + bxe[v + 1]), half * (bya[v] + byb[v]), half * (bza[v] + bzb[v]));
}
#ifndef MHD_X2_NO_CELLPACK
template <>
__device__ __forceinline__ void x_centre<float, 4>(const float (&bxe)[5], const float (&bya)[4], const float (&byb)[4], const float (&bza)[4],
                                                   const float (&bzb)[4], BCell<float> (&B)[4]) {
  const f2 half(0.5f);
#pragma unroll
  for (int v = 0; v < 4; v += 2) {           // cells (v, v+1) as one pack (see right_left_cells)
    BCell<f2> BB;
    BB.set(half * (f2(bxe[v], bxe[v + 1]) + f2(bxe[v + 1], bxe[v + 2])), half * (f2(bya[v], bya[v + 1]) + f2(byb[v], byb[v + 1])),
           half * (f2(bza[v], bza[v + 1]) + f2(bzb[v], bzb[v + 1])));
    B[v].b0 = BB.b0.v.x; B[v + 1].b0 = BB.b0.v.y; B[v].b1 = BB.b1.v.x; B[v + 1].b1 = BB.b1.v.y;
    B[v].b2 = BB.b2.v.x; B[v + 1].b2 = BB.b2.v.y; B[v].hb2 = BB.hb2.v.x; B[v + 1].hb2 = BB.hb2.v.y;
  }
}
#endif

template <class real, class T, int V>
__device__ __forceinline__ void x_store_u_and_cmax(const XArgs<real>& A, const XRows& q, const T (&un)[V][5],
                                                   const BCell<T> (&B)[V]) {
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    T o[V];
#pragma unroll
    for (int v = 0; v < V; ++v) o[v] = un[v][c];
    if (q.live) xstore(A.uo[c], q.o[1], q.o[2], o);
  }
  if (A.cmax_bits) {            // last operator of a step: c of eq (18) from the updated cells (B unchanged by fluid_x)
    typedef typename PackOf<T>::scalar S;
    decltype(pack_speed_key((const T*)nullptr, T(), S())) cbest = 0;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const auto bts = pack_speed_key(un[v], B[v].hb2, (S)A.gamma);
      cbest = bts > cbest ? bts : cbest;
    }
    const unsigned long long cw = warp_max_u64(q.live ? key_bits(cbest) : 0ull);
    if ((threadIdx.x & 31) == 0) publish_max(A.cmax_bits, cw);
  }
}

#ifndef MHD_X2_MINB2
#define MHD_X2_MINB2 3     // blocks per SM the register budget is cut for, two rows per thread (f2)
#endif
#ifndef MHD_X2_MINB1
#define MHD_X2_MINB1 6     // one row per thread (fluid_x scalar fp32: 80 registers 1.21 ms at 512^3; 5: 96 registers 1.29; 7: spills 1.24)
#endif
#ifndef MHD_X2_MINB64
#define MHD_X2_MINB64 2    // fp64: 256-thread blocks
#endif
#define MHD_X2_MINB(real, T) (sizeof(real) == 8 ? MHD_X2_MINB64 : (PackOf<T>::L == 2 ? MHD_X2_MINB2 : MHD_X2_MINB1))
// the scalar fp32 B pair and fused reverse L_x have their own budgets
#ifndef MHD_X2_MINB1_B
#define MHD_X2_MINB1_B 5
#endif
#ifndef MHD_X2_MINB1_L
#define MHD_X2_MINB1_L 6     // 80 registers: 2.09 ms at 512^3 (5: 96 registers 2.17; 7: 72 registers, spills, 2.15; 8: 2.43)
#endif
#define MHD_X2_MINB_B(real, T) (sizeof(real) == 8 ? MHD_X2_MINB64 : (PackOf<T>::L == 2 ? MHD_X2_MINB2 : MHD_X2_MINB1_B))
#define MHD_X2_MINB_L(real, T) (sizeof(real) == 8 ? MHD_X2_MINB64 : (PackOf<T>::L == 2 ? MHD_X2_MINB2 : MHD_X2_MINB1_L))

// ---- fluid_x --------------------------------------------------------------------------------------
// OUT: outflow boundaries (ghost threads, see ghost_fix); one row per thread only
template <class real, class T, int NT = X2Block<real>::NT, bool OUT = false>
__global__ void __launch_bounds__(NT, x2_minb<real>(MHD_X2_MINB(real, T), NT)) fluid_x2_kernel(const XArgs<real> A) {
  constexpr int V = VecOf<real>::V;
  constexpr int L = PackOf<T>::L;
  typedef typename PackOf<T>::scalar S;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  const XRows q = x_rows<real, L, OUT>(A);
  const S dts = (S)(*A.dt);
  const T hdt(S(0.5) * dts), qdt(S(0.25) * dts), gamma(A.gamma);
  T u[5][V];
#pragma unroll
  for (int c = 0; c < 5; ++c) xload(A.u[c], q.o[1], q.o[2], u[c], A.one);
  T bxf[V], bya[V], byb[V], bza[V], bzb[V], bxe[V + 1];
  xload(A.bx, q.o[1], q.o[2], bxf, A.one);
  xload(A.by, q.o[1], q.o[2], bya, A.one); xload(A.by, q.o[2], q.o[3], byb, A.one);
  xload(A.bz, q.o[1], q.o[2], bza, A.one); xload(A.bz, q.okp[0], q.okp[1], bzb, A.one);
  bxe[V] = xload1(A.bx, q.onext[0], q.onext[1], (T*)nullptr);
  if (OUT) {          // after ALL loads are issued (a fix behind each load keeps only two or three of them in flight)
#pragma unroll
    for (int c = 0; c < 5; ++c) ghost_fix<V>(u[c], q.mode);
    ghost_fix<V>(bxf, q.mode); ghost_fix<V>(bya, q.mode); ghost_fix<V>(byb, q.mode); ghost_fix<V>(bza, q.mode); ghost_fix<V>(bzb, q.mode);
  }
#pragma unroll
  for (int v = 0; v < V; ++v) bxe[v] = bxf[v];
  BCell<T> B[V];
  x_centre<T, V>(bxe, bya, byb, bza, bzb, B);
  T un[V][5];
  fluid_x_core<T, V, NT>(sm, threadIdx.x, q.tl, q.tr, u, B, gamma, hdt, qdt, un);
  x_store_u_and_cmax<real, T, V>(A, q, un, B);
}

// ---- B_{y->x}, B_{z->x} ------------------------------------------------------------------------------
template <class real, class T, int NT = X2Block<real>::NT, bool OUT = false>
__global__ void __launch_bounds__(NT, x2_minb<real>(MHD_X2_MINB_B(real, T), NT)) bpair_x2_kernel(const XArgs<real> A) {
  constexpr int V = VecOf<real>::V;
  constexpr int L = PackOf<T>::L;
  typedef typename PackOf<T>::scalar S;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  const XRows q = x_rows<real, L, OUT>(A);
  const S dts = (S)(*A.dt);
  const T dt(dts), hdt(S(0.5) * dts);
  T r0[V], m0[V], vt[4][V], b[4][V], f[4][V + 1];
  bpair_x_inputs<real, T, V, OUT>(A, q, r0, m0, vt, b);
  bpair_x_core<T, V, NT>(sm, threadIdx.x, q.tl, q.tr, vt, b, dt, hdt, f);
  // advect B_y, B_z (Alg. 2 step 9) and constrain B_x with the same fluxes
  T bxv[V], byn[V], bzn[V];
  xload(A.bx, q.o[1], q.o[2], bxv, A.one);
#pragma unroll
  for (int v = 0; v < V; ++v) {
    byn[v] = b[0][v] - (f[0][v + 1] - f[0][v]);
    bzn[v] = b[2][v] - (f[2][v + 1] - f[2][v]);
    const T cy = f[1][v] - f[0][v];          // face v-1/2, rows j+1 and j
    const T cz = f[3][v] - f[2][v];
    if (A.t2_first) { bxv[v] = bxv[v] + cz; bxv[v] = bxv[v] + cy; }
    else            { bxv[v] = bxv[v] + cy; bxv[v] = bxv[v] + cz; }
  }
  if (q.live) {
    xstore(A.byo, q.o[1], q.o[2], byn);
    xstore(A.bzo, q.o[1], q.o[2], bzn);
    xstore(A.bxo, q.o[1], q.o[2], bxv);
  }
}

// ---- reverse L_x in one pass: B_{z->x}, B_{y->x} (t2 first), then fluid_x with the UPDATED field ----
// Shared memory: 35 slots x NT packs (the B pair uses slots 0..23, the B_x' exchange slot 34,
// fluid_x slots 0..34; slot 34 is rewritten by fluid_x only two barriers after it was read).
template <class real, class T, int NT = X2Block<real>::NT>
__global__ void __launch_bounds__(NT, x2_minb<real>(MHD_X2_MINB_L(real, T), NT)) lrev_x2_kernel(const XArgs<real> A) {
  constexpr int V = VecOf<real>::V;
  constexpr int L = PackOf<T>::L;
  typedef typename PackOf<T>::scalar S;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  T* sm = reinterpret_cast<T*>(smem_raw);
  const int tid = threadIdx.x;
  const XRows q = x_rows<real, L>(A);
  const S dts = (S)(*A.dt);
  const T dt(dts), hdt(S(0.5) * dts), qdt(S(0.25) * dts), gamma(A.gamma);
  T u[5][V];
  BCell<T> B[V];
  {
    T vt[4][V], b[4][V], f[4][V + 1];
    bpair_x_inputs<real, T, V>(A, q, u[0], u[1], vt, b);
    bpair_x_core<T, V, NT>(sm, tid, q.tl, q.tr, vt, b, dt, hdt, f);
    // Alg. 2 step 9 on all four rows: rows j and k are this thread's own B_y', B_z'; rows j+1 and k+1 are
    // the neighbour rows' updated values, which the cell-centred field of my cells needs (eq (19))
    T bxe[V + 1], bya[V], byb[V], bza[V], bzb[V];
    {
      T bxv[V];
      xload(A.bx, q.o[1], q.o[2], bxv, A.one);
#pragma unroll
      for (int v = 0; v < V; ++v) {
        bya[v] = b[0][v] - (f[0][v + 1] - f[0][v]);
        byb[v] = b[1][v] - (f[1][v + 1] - f[1][v]);
        bza[v] = b[2][v] - (f[2][v + 1] - f[2][v]);
        bzb[v] = b[3][v] - (f[3][v + 1] - f[3][v]);
        const T cy = f[1][v] - f[0][v];        // constraint on B_x: face v-1/2, rows j+1 and j
        const T cz = f[3][v] - f[2][v];
        if (A.t2_first) { bxv[v] = bxv[v] + cz; bxv[v] = bxv[v] + cy; }
        else            { bxv[v] = bxv[v] + cy; bxv[v] = bxv[v] + cz; }
        bxe[v] = bxv[v];
      }
      if (q.live) {
        xstore(A.byo, q.o[1], q.o[2], bya);
        xstore(A.bzo, q.o[1], q.o[2], bza);
        xstore(A.bxo, q.o[1], q.o[2], bxv);
      }
    }
    sm[34 * NT + tid] = bxe[0];              // my first updated B_x face -> left neighbour's face V
    __syncthreads();
    bxe[V] = sm[34 * NT + q.tr];
    x_centre<T, V>(bxe, bya, byb, bza, bzb, B);
  }
#pragma unroll
  for (int c = 2; c < 5; ++c) xload(A.u[c], q.o[1], q.o[2], u[c], A.one);
  T un[V][5];
  fluid_x_core<T, V, NT>(sm, tid, q.tl, q.tr, u, B, gamma, hdt, qdt, un);
  x_store_u_and_cmax<real, T, V>(A, q, un, B);
}

}  // namespace mhd
