// mhd_x.cuh -- kernels for sweeps along x (the contiguous axis), periodic boundaries.
//
// Along x the stencil runs along the lanes, so instead of marching each thread owns V consecutive
// cells of one row (V = 4 floats or 2 doubles: every global access is one aligned 16-byte vector,
// a warp reads 512 contiguous bytes per field) and a group of nx/V threads covers a whole row, so the
// periodic wrap is just "thread 0's left neighbour is the last thread": no halo cells are recomputed.
// The few stencil values a thread needs from its neighbours (the R/G of one or two edge cells per
// stage) go through shared memory, one __syncthreads per stage.
//
// Requirements (else the generic kernels run): periodic BC, nx % V == 0, nx/V <= 256, N < 2^31.
#pragma once
#include "mhd_device.cuh"

namespace mhd {

template <class real> struct VecOf;
template <> struct VecOf<float> { typedef float4 type; enum { V = 4 }; };
template <> struct VecOf<double> { typedef double2 type; enum { V = 2 }; };

template <class real>
__device__ __forceinline__ void vload(const real* p, real (&v)[VecOf<real>::V]);
template <>
__device__ __forceinline__ void vload<float>(const float* p, float (&v)[4]) {
  const float4 t = __ldg(reinterpret_cast<const float4*>(p));
  v[0] = t.x; v[1] = t.y; v[2] = t.z; v[3] = t.w;
}
template <>
__device__ __forceinline__ void vload<double>(const double* p, double (&v)[2]) {
  const double2 t = __ldg(reinterpret_cast<const double2*>(p));
  v[0] = t.x; v[1] = t.y;
}
__device__ __forceinline__ void vstore(float* p, const float (&v)[4]) {
  *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]);
}
__device__ __forceinline__ void vstore(double* p, const double (&v)[2]) {
  *reinterpret_cast<double2*>(p) = make_double2(v[0], v[1]);
}

template <class real>
struct XArgs {
  const real* u[5];        // fluid: rho, mx, my, mz, E;  B pair: u[0] = rho, u[1] = mx
  real* uo[5];
  const real *bx, *by, *bz;
  real *bxo, *byo, *bzo;
  const double* dt;
  unsigned long long* cmax_bits;   // != nullptr: also reduce c of eq (18) over the updated cells
  int nx, ny, nz;
  int tpr;                 // threads per row = nx / V
  int tpr_shift;           // log2(tpr) if tpr is a power of two, else -1 (mhd_x2.cuh)
  int rpb;                 // rows per block
  int t2_first;
  real gamma;
  real one;                // 1.0 at run time (mhd_x2.cuh, xload)
};

// fluid_x, Algorithm 1.  Shared memory: 7 groups x 5 components x blockDim.x reals.
template <class real>
__global__ void __launch_bounds__(256) fluid_x_kernel(const XArgs<real> A) {
  constexpr int V = VecOf<real>::V;
  extern __shared__ unsigned char smem_raw[];
  real* sm = reinterpret_cast<real*>(smem_raw);
  const int nthr = blockDim.x;
  const int tid = threadIdx.x;
  const int lr = tid / A.tpr, t = tid - lr * A.tpr;
  const int nrows = A.ny * A.nz;
  int row = blockIdx.x * A.rpb + lr;
  const bool live = row < nrows;
  if (!live) row = nrows - 1;                       // keep the thread in step for the barriers
  const int k = row / A.ny, j = row - k * A.ny;
  const int jp = (j + 1 == A.ny) ? 0 : j + 1, kp = (k + 1 == A.nz) ? 0 : k + 1;
  const int off = row * A.nx + t * V;
  const int off_jp = (k * A.ny + jp) * A.nx + t * V;
  const int off_kp = (kp * A.ny + j) * A.nx + t * V;
  const int tl = lr * A.tpr + (t == 0 ? A.tpr - 1 : t - 1);          // periodic neighbours in the row
  const int tr = lr * A.tpr + (t == A.tpr - 1 ? 0 : t + 1);
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt, qdt = real(0.25) * dt;
  auto S = [&](int group, int comp, int thr) -> real& { return sm[(group * 5 + comp) * nthr + thr]; };

  // ---- load: 5 u vectors, Bx faces i..i+V, By at j and j+1, Bz at k and k+1 --------------------
  real u[5][V];
#pragma unroll
  for (int c = 0; c < 5; ++c) vload(A.u[c] + off, u[c]);
  real bxf[V], bya[V], byb[V], bza[V], bzb[V];
  vload(A.bx + off, bxf);
  vload(A.by + off, bya); vload(A.by + off_jp, byb);
  vload(A.bz + off, bza); vload(A.bz + off_kp, bzb);
  const int i_next = (t == A.tpr - 1) ? 0 : (t + 1) * V;
  const real bx_next = __ldg(A.bx + row * A.nx + i_next);
  real bxe[V + 1];
#pragma unroll
  for (int v = 0; v < V; ++v) bxe[v] = bxf[v];
  bxe[V] = bx_next;
  BCell<real> B[V];
#pragma unroll
  for (int v = 0; v < V; ++v)                                          // eq (19): faces -> centre
    B[v].set(real(0.5) * (bxe[v] + bxe[v + 1]), real(0.5) * (bya[v] + byb[v]), real(0.5) * (bza[v] + bzb[v]));

  // ---- stage 0: R, G of u^t (Alg. 1 step 4) ----------------------------------------------------
  real R[V][5], G[V][5];
#pragma unroll
  for (int v = 0; v < V; ++v) {
    real uu[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) uu[c] = u[c][v];
    right_left(uu, B[v], A.gamma, R[v], G[v]);
  }
#pragma unroll
  for (int c = 0; c < 5; ++c) { S(0, c, tid) = R[V - 1][c]; S(1, c, tid) = G[0][c]; }
  __syncthreads();
  // steps 5-6: first-order fluxes at the V+1 faces of my cells, half step (eq (16))
  real uh[V][5];
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    real d1[V + 1];
    d1[0] = S(0, c, tl) - G[0][c];
#pragma unroll
    for (int v = 1; v < V; ++v) d1[v] = R[v - 1][c] - G[v][c];
    d1[V] = R[V - 1][c] - S(1, c, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) uh[v][c] = u[c][v] - (d1[v + 1] - d1[v]) * qdt;
  }
  // ---- stage 1: R, G of u^{t+dt/2} (step 7) ----------------------------------------------------
#pragma unroll
  for (int v = 0; v < V; ++v) right_left(uh[v], B[v], A.gamma, R[v], G[v]);
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    S(2, c, tid) = R[V - 1][c];      // my last R  -> right neighbour's R[-1]
    S(3, c, tid) = R[0][c];          // my first R -> left neighbour's R[V]
    S(4, c, tid) = G[0][c];          // my first two G -> left neighbour's G[V], G[V+1]
    S(5, c, tid) = G[1][c];
  }
  __syncthreads();
  // step 8: second-order TVD flux (twice its value) at the right face of each of my cells
  real phi[V + 1][5];
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    real r[V + 2], g[V + 2];         // r[v+1] = R at cell v (v = -1..V);  g[v] = G at cell v (v = 0..V+1)
    r[0] = S(2, c, tl);
#pragma unroll
    for (int v = 0; v < V; ++v) { r[v + 1] = R[v][c]; g[v] = G[v][c]; }
    r[V + 1] = S(3, c, tr);
    g[V] = S(4, c, tr);
    g[V + 1] = S(5, c, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const real Rp = r[v + 1] + vl_full(r[v + 1] - r[v], r[v + 2] - r[v + 1]);      // eqs (11)-(15)
      const real Gp = g[v + 1] + vl_full(g[v + 1] - g[v + 2], g[v] - g[v + 1]);      // mirror image
      phi[v + 1][c] = Rp - Gp;
    }
    S(6, c, tid) = phi[V][c];        // my last face -> right neighbour's left face
  }
  __syncthreads();
  // step 9: full step (eq (17)) and store
  real un[V][5];
#pragma unroll
  for (int c = 0; c < 5; ++c) {
    phi[0][c] = S(6, c, tl);
    real o[V];
#pragma unroll
    for (int v = 0; v < V; ++v) { o[v] = u[c][v] - (phi[v + 1][c] - phi[v][c]) * hdt; un[v][c] = o[v]; }
    if (live) vstore(A.uo[c] + off, o);
  }
  if (A.cmax_bits) {            // last operator of a step: c of eq (18) from the updated cells (B unchanged)
    unsigned long long cbest = 0ull;
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const unsigned long long b = speed_bits(cfl_speed_hb2(un[v], B[v].hb2, A.gamma));
      cbest = b > cbest ? b : cbest;
    }
    cbest = warp_max_u64(live ? cbest : 0ull);
    if ((tid & 31) == 0) publish_max(A.cmax_bits, cbest);
  }
}

// ---------------------------------------------------------------------------------------------
// B_{y->x} and B_{z->x} in one pass (Algorithm 2; eqs (20)-(22) PAPER.md:147-158).
// Four flux rows per thread, in lock step: p = 0: By row j, 1: By row j+1, 2: Bz row k, 3: Bz row k+1
// (the +1 rows supply the constraint update of Bx).
// Shared memory: 2 sets x 12 values x blockDim.x reals (the sets alternate between stages).
// ---------------------------------------------------------------------------------------------
template <class real>
__global__ void __launch_bounds__(256) bpair_x_kernel(const XArgs<real> A) {
  constexpr int V = VecOf<real>::V;
  extern __shared__ unsigned char smem_raw[];
  real* sm = reinterpret_cast<real*>(smem_raw);
  const int nthr = blockDim.x;
  const int tid = threadIdx.x;
  const int lr = tid / A.tpr, t = tid - lr * A.tpr;
  const int nrows = A.ny * A.nz;
  int row = blockIdx.x * A.rpb + lr;
  const bool live = row < nrows;
  if (!live) row = nrows - 1;
  const int k = row / A.ny, j = row - k * A.ny;
  const int jp = (j + 1 == A.ny) ? 0 : j + 1, kp = (k + 1 == A.nz) ? 0 : k + 1;
  const int jm = (j == 0) ? A.ny - 1 : j - 1, km = (k == 0) ? A.nz - 1 : k - 1;
  const int col = t * V;
  const int off = row * A.nx + col;
  const int off_jp = (k * A.ny + jp) * A.nx + col, off_jm = (k * A.ny + jm) * A.nx + col;
  const int off_kp = (kp * A.ny + j) * A.nx + col, off_km = (km * A.ny + j) * A.nx + col;
  const int tl = lr * A.tpr + (t == 0 ? A.tpr - 1 : t - 1);
  const int tr = lr * A.tpr + (t == A.tpr - 1 ? 0 : t + 1);
  const real dt = (real)(*A.dt);
  const real hdt = real(0.5) * dt;
  auto S = [&](int set, int slot, int thr) -> real& { return sm[(set * 12 + slot) * nthr + thr]; };

  real vt[4][V], b[4][V];
  {
    real r0[V], m0[V], r[V], m[V];
    vload(A.u[0] + off, r0); vload(A.u[1] + off, m0);
    // Alg. 2 step 4: face velocity = momentum sum / density sum of the two cells sharing the face (reading R5)
    vload(A.u[0] + off_jm, r); vload(A.u[1] + off_jm, m);
#pragma unroll
    for (int v = 0; v < V; ++v) vt[0][v] = (m[v] + m0[v]) * rcp_(r[v] + r0[v]);
    vload(A.u[0] + off_jp, r); vload(A.u[1] + off_jp, m);
#pragma unroll
    for (int v = 0; v < V; ++v) vt[1][v] = (m0[v] + m[v]) * rcp_(r0[v] + r[v]);
    vload(A.u[0] + off_km, r); vload(A.u[1] + off_km, m);
#pragma unroll
    for (int v = 0; v < V; ++v) vt[2][v] = (m[v] + m0[v]) * rcp_(r[v] + r0[v]);
    vload(A.u[0] + off_kp, r); vload(A.u[1] + off_kp, m);
#pragma unroll
    for (int v = 0; v < V; ++v) vt[3][v] = (m0[v] + m[v]) * rcp_(r0[v] + r[v]);
  }
  vload(A.by + off, b[0]); vload(A.by + off_jp, b[1]);
  vload(A.bz + off, b[2]); vload(A.bz + off_kp, b[3]);

  // stage A: eq (20), 1-2-1 smoothing along x
#pragma unroll
  for (int p = 0; p < 4; ++p) { S(0, p, tid) = vt[p][V - 1]; S(0, 4 + p, tid) = vt[p][0]; }
  __syncthreads();
  real vg[4][V + 1], w[4][V + 2];
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    real e[V + 2];
    e[0] = S(0, p, tl);
#pragma unroll
    for (int v = 0; v < V; ++v) e[v + 1] = vt[p][v];
    e[V + 1] = S(0, 4 + p, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      vg[p][v] = real(0.25) * ((e[v] + e[v + 2]) + real(2) * e[v + 1]);
      w[p][v] = vg[p][v] * b[p][v];
    }
    S(1, p, tid) = vg[p][0]; S(1, 4 + p, tid) = w[p][0];
  }
  __syncthreads();
  // stage B: eqs (21),(22): first-order upwind flux at the right face of each cell
  real vh[4][V], f1[4][V + 1];
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    vg[p][V] = S(1, p, tr);
    w[p][V] = S(1, 4 + p, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      vh[p][v] = vg[p][v] + vg[p][v + 1];
      f1[p][v + 1] = vh[p][v] > real(0) ? w[p][v] : w[p][v + 1];
    }
    S(0, 8 + p, tid) = f1[p][V];
  }
  __syncthreads();
  // stage C: half step (Alg. 2 step 7) and vg * B^{t+dt/2}
  real w1[4][V + 3];     // w1[p][v+1] = value at cell v, v = -1..V+1
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    f1[p][0] = S(0, 8 + p, tl);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const real bh = b[p][v] - (f1[p][v + 1] - f1[p][v]) * hdt;
      w1[p][v + 1] = vg[p][v] * bh;
    }
    S(1, 8 + p, tid) = w1[p][V];       // last  -> right neighbour's cell -1
    S(0, p, tid) = w1[p][1];           // first two -> left neighbour's cells V, V+1   (set 0 slots 0..7 are free again)
    S(0, 4 + p, tid) = w1[p][2];
  }
  __syncthreads();
  // stage D: second-order TVD flux at the right face of each cell (Alg. 2 step 8)
  real f[4][V + 1];      // f[p][v+1] = flux*dt at face v+1/2, f[p][0] at face -1/2
#pragma unroll
  for (int p = 0; p < 4; ++p) {
    w1[p][0] = S(1, 8 + p, tl);
    w1[p][V + 1] = S(0, p, tr);
    w1[p][V + 2] = S(0, 4 + p, tr);
#pragma unroll
    for (int v = 0; v < V; ++v) {
      const bool up = vh[p][v] > real(0);
      const real x = up ? w1[p][v + 1] : w1[p][v + 2];
      const real y = up ? w1[p][v] : w1[p][v + 3];
      const real z = up ? w1[p][v + 2] : w1[p][v + 1];
      f[p][v + 1] = (x + vl_full(x - y, z - x)) * dt;
    }
    S(1, p, tid) = f[p][V];
  }
  __syncthreads();
  // stage E: advect By, Bz (Alg. 2 step 9) and constrain Bx with the same fluxes
#pragma unroll
  for (int p = 0; p < 4; ++p) f[p][0] = S(1, p, tl);
  real bxv[V], byn[V], bzn[V];
  vload(A.bx + off, bxv);
#pragma unroll
  for (int v = 0; v < V; ++v) {
    byn[v] = b[0][v] - (f[0][v + 1] - f[0][v]);
    bzn[v] = b[2][v] - (f[2][v + 1] - f[2][v]);
    const real cy = f[1][v] - f[0][v];       // face v-1/2, rows j+1 and j
    const real cz = f[3][v] - f[2][v];
    if (A.t2_first) { bxv[v] = bxv[v] + cz; bxv[v] = bxv[v] + cy; }
    else            { bxv[v] = bxv[v] + cy; bxv[v] = bxv[v] + cz; }
  }
  if (live) {
    vstore(A.byo + off, byn);
    vstore(A.bzo + off, bzn);
    vstore(A.bxo + off, bxv);
  }
}

}  // namespace mhd
