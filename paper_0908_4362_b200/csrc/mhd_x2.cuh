// mhd_x2.cuh -- sweeps along x (the contiguous axis), periodic boundaries, in lane-pack arithmetic, and the
// fused reverse operator L_x^rev = B_{z->x}, B_{y->x}, fluid_x in ONE kernel.
//
// Same decomposition as mhd_x.cuh (a thread owns V consecutive cells of a row, a group of nx/V threads
// covers the whole row so the periodic wrap is the group's own ring, neighbour values go through shared
// memory, one barrier per stage, no halo cell recomputed), with two changes:
//
//  * T = f2 (mhd_pack.cuh): a thread owns the same V columns of TWO adjacent rows (j, j+1) and advances
//    both with packed fp32 instructions (FADD2/FMUL2/FFMA2): the x kernels of mhd_x.cuh are issue-bound
//    (profiles/r01_c4_step_ncu_full_b.md: 273 and 194 issued instructions per cell, 65-68 % issue
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
// Requirements (else the kernels of mhd_x.cuh / mhd_generic.cuh run): periodic BC, nx % V == 0,
// nx / V <= 256, N < 2^31, and for T = f2 an even ny.
#pragma once
#include "mhd_pack_io.cuh"
#include "mhd_x.cuh"

namespace mhd {

// ---- V-cell vectors of L rows <-> packs ------------------------------------------------------------
__device__ __forceinline__ void xload(const float* f, int oa, int ob, f2 (&v)[4]) {
  const float4 a = __ldg(reinterpret_cast<const float4*>(f + oa));
  const float4 b = __ldg(reinterpret_cast<const float4*>(f + ob));
  v[0] = f2(a.x, b.x); v[1] = f2(a.y, b.y); v[2] = f2(a.z, b.z); v[3] = f2(a.w, b.w);
}
__device__ __forceinline__ void xload(const double* f, int oa, int, double (&v)[2]) {
  const double2 a = __ldg(reinterpret_cast<const double2*>(f + oa));
  v[0] = a.x; v[1] = a.y;
}
__device__ __forceinline__ void xload(const float* f, int oa, int, float (&v)[4]) {
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
__device__ __forceinline__ f2 xload1(const float* f, int oa, int ob, f2*) { return f2(__ldg(f + oa), __ldg(f + ob)); }
__device__ __forceinline__ double xload1(const double* f, int oa, int, double*) { return __ldg(f + oa); }
__device__ __forceinline__ float xload1(const float* f, int oa, int, float*) { return __ldg(f + oa); }

// Where the rows of one thread live.  Lane l of a pack is row j+l of plane k (L = 1 or 2).
struct XRows {
  int t, tl, tr;            // my thread index in the row group; block-local thread ids of my left / right neighbour
  int col;                  // first column
  int o[4];                 // offsets of rows j-1, j, j+1, j+2 of plane k (j+2 only used for L = 2)
  int okm[2], okp[2];       // rows j, j+1 of planes k-1 and k+1
  int onext[2];             // B_x face of the next thread's first column, rows j and j+1
  bool live;
};

template <class real, int L>
__device__ __forceinline__ XRows x_rows(const XArgs<real>& A) {
  constexpr int V = VecOf<real>::V;
  XRows r;
  const int tid = threadIdx.x;
  const int lr = tid / A.tpr;
  r.t = tid - lr * A.tpr;
  const int ngroups = (A.ny / L) * A.nz;
  int g = blockIdx.x * A.rpb + lr;
  r.live = g < ngroups;
  if (!r.live) g = ngroups - 1;                       // keep the thread in step for the barriers
  const int gpp = A.ny / L;                           // row groups per plane
  const int k = g / gpp, j = (g - k * gpp) * L;
  const int kp = (k + 1 == A.nz) ? 0 : k + 1, km = (k == 0) ? A.nz - 1 : k - 1;
  r.col = r.t * V;
  auto row = [&](int jj, int kk) { return (kk * A.ny + jj) * A.nx + r.col; };
  const int jm = (j == 0) ? A.ny - 1 : j - 1;
  const int j1 = (j + 1 == A.ny) ? 0 : j + 1;         // L = 2: j is even and ny is even, so j1 = j + 1
  const int j2 = (j1 + 1 == A.ny) ? 0 : j1 + 1;
  r.o[0] = row(jm, k); r.o[1] = row(j, k); r.o[2] = row(j1, k); r.o[3] = row(j2, k);
  const int jb = (L == 2) ? j1 : j;
  r.okm[0] = row(j, km); r.okm[1] = row(jb, km);
  r.okp[0] = row(j, kp); r.okp[1] = row(jb, kp);
  const int i_next = (r.t == A.tpr - 1) ? 0 : (r.t + 1) * V;
  r.onext[0] = (k * A.ny + j) * A.nx + i_next;
  r.onext[1] = (k * A.ny + jb) * A.nx + i_next;
  r.tl = lr * A.tpr + (r.t == 0 ? A.tpr - 1 : r.t - 1);
  r.tr = lr * A.tpr + (r.t == A.tpr - 1 ? 0 : r.t + 1);
  return r;
}

// ---------------------------------------------------------------------------------------------
// fluid_x of the V cells of one thread, Algorithm 1, in pack arithmetic.
// sm: 7 groups x 5 components x nthr packs.  u[c][v], B[v] in; un[v][c] out.  Contains three barriers;
// the caller guarantees that nobody still reads sm when it is entered.
// ---------------------------------------------------------------------------------------------
template <class T, int V>
__device__ __forceinline__ void fluid_x_core(T* sm, int nthr, int tid, int tl, int tr, const T (&u)[5][V],
                                             const BCell<T> (&B)[V], T gamma, T hdt, T qdt, T (&un)[V][5]) {
  auto S = [&](int group, int comp, int thr) -> T& { return sm[(group * 5 + comp) * nthr + thr]; };
  // stage 0: R, G of u^t (Alg. 1 step 4)
  T R[V][5], G[V][5];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    T uu[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) uu[c] = u[c][v];
    right_left(uu, B[v], gamma, R[v], G[v]);
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
#pragma unroll
    for (int v = 0; v < V; ++v) uh[v][c] = fnma_(d1[v + 1] - d1[v], qdt, u[c][v]);
  }
  // stage 1: R, G of u^{t+dt/2} (step 7), same B_c
#pragma unroll
  for (int v = 0; v < V; ++v) right_left(uh[v], B[v], gamma, R[v], G[v]);
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
      const T Rp = r[v + 1] + vl_full(r[v + 1] - r[v], r[v + 2] - r[v + 1]);      // eqs (11)-(15)
      const T Gp = g[v + 1] + vl_full(g[v + 1] - g[v + 2], g[v] - g[v + 1]);      // mirror image
      phi[v + 1][c] = Rp - Gp;
    }
    S(6, c, tid) = phi[V][c];        // my last face -> right neighbour's left face
  }
  __syncthreads();
  // step 9: full step (eq (17))
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    phi[0][c] = S(6, c, tl);
#pragma unroll
    for (int v = 0; v < V; ++v) un[v][c] = fnma_(phi[v + 1][c] - phi[v][c], hdt, u[c][v]);
  }
}
