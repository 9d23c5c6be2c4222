// oracle/mhd_oracle.cpp  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// Plain, slow, serial-in-spirit CPU restatement of the relaxing-TVD ideal-MHD update of
// arxiv/paper_0908_4362 ("GPU-MHD", Wong, Wong, Feng & Tang), written from PAPER.md section 3
// for the arithmetic and section 4.2-4.3 for the sequencing.
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may use it.
// It shares no code, header, table or helper with paper_0908_4362_b200/csrc (the CUDA path) and
// neither side includes or imports the other.
//
// What it is: the algorithm itself, step by step, as scalar gather loops over ghost-padded 1-D
// pencils (the method is an explicit iteration, not a shortcut to a closed form).  The optional
// "#pragma omp parallel for" lines only distribute independent pencils over host threads; every
// pencil is computed by exactly the same scalar code, so results are bitwise identical for any
// thread count (checked in tests/test_oracle_pins.py).
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): conservation, div B, second-order
// convergence of linear Alfven / fast / slow eigenmodes to their closed-form solution, Sod tube
// against the exact Riemann solution (B = 0), Orszag-Tang rotation symmetry, uniform-state fixed
// point, 1-D replication, cyclic-permutation equivariance, Brio-Wu invariants, constant-velocity
// linear advection of the scalar B scheme, brute-force NumPy restatement on tiny grids, and c_max of
// eq (18) against hand-computed values (uniform state, one moving cell per velocity component, face
// pattern whose centred average differs from either face, last cell under both boundary rules).
// Parity unpinned by the paper: PAPER.md prints no numerical field values (figures only), so no
// golden values from the paper exist; the pins above are mathematical.
//
// Conventions: grid units (cells have unit width); fields
// 0..7 = rho, m_x, m_y, m_z, E, Bx, By, Bz; x fastest: idx = i + nx*(j + ny*k); staggered B,
// eq (19): Bx[i,j,k] sits on face (i-1/2,j,k) etc.  For a sweep along d the
// cyclic triple is (d,t1,t2): x->(x,y,z), y->(y,z,x), z->(z,x,y).
// Boundary rule (paper silent; reading R9): every read of an INPUT array of an operator
// at an out-of-range index is mapped, index by index, by wrap (periodic) or clamp (outflow);
// intermediates at ghost positions are computed from those mapped inputs.

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

enum { BC_PERIODIC = 0, BC_OUTFLOW = 1 };

template <class real>
struct Grid {
  int n[3];      // nx, ny, nz
  real gamma;
  int bc;
  real* f[8];    // rho, mx, my, mz, E, Bx, By, Bz

  // index map of the boundary rule (reading R9)
  int map(int q, int axis) const {
    const int m = n[axis];
    if (bc == BC_PERIODIC) { q %= m; return q < 0 ? q + m : q; }
    return q < 0 ? 0 : (q >= m ? m - 1 : q);
  }
  // linear index of the cell whose (unmapped) coordinates along axes (d,t1,t2) are (q,a,b)
  size_t at(int d, int q, int a, int b) const {
    int c[3];
    c[d] = map(q, d);
    c[(d + 1) % 3] = map(a, (d + 1) % 3);
    c[(d + 2) % 3] = map(b, (d + 2) % 3);
    return (size_t)c[0] + (size_t)n[0] * ((size_t)c[1] + (size_t)n[1] * (size_t)c[2]);
  }
};

// van Leer limiter, eq (14); "when the corrections have opposite signs, there is no
// second-order correction" PAPER.md:103  (reading R8: active iff a*b > 0 strictly)
template <class real>
inline real vanleer(real a, real b) {
  const real ab = a * b;
  return ab > real(0) ? real(2) * ab / (a + b) : real(0);
}

// Flux vector F(u) of eq (6) PAPER.md:76 with the cell-centred field (b1,b2,b3) held fixed, and the
// freezing speed c = |v| + sqrt(gamma p/rho + B^2/rho).   u = (rho, m1, m2, m3, E) in
// sweep roles (1 = sweep direction).  P* = P + B^2/2,  P = (gamma-1)(E - rho v^2/2 - B^2/2).
template <class real>
inline void flux(const real u[5], const real b[3], real gamma, real F[5], real& c) {
  const real rho = u[0], m1 = u[1], m2 = u[2], m3 = u[3], E = u[4];
  const real v = m1 / rho;
  const real b2 = b[0] * b[0] + b[1] * b[1] + b[2] * b[2];
  const real ke = real(0.5) * (m1 * m1 + m2 * m2 + m3 * m3) / rho;
  const real p = (gamma - real(1)) * (E - ke - real(0.5) * b2);   // gas pressure
  const real ps = p + real(0.5) * b2;                              // total pressure P*
  const real bdotm = b[0] * m1 + b[1] * m2 + b[2] * m3;            // rho * (B.v)
  F[0] = m1;
  F[1] = m1 * v + ps - b[0] * b[0];
  F[2] = m2 * v - b[1] * b[0];
  F[3] = m3 * v - b[2] * b[0];
  F[4] = (E + ps) * v - b[0] * bdotm / rho;
  c = std::fabs(v) + std::sqrt(std::fabs(gamma * p + b2) / rho);   // |.|: reading R3
}

// ---------------------------------------------------------------------------------------------
// O1  c_max of eq (18), B cell-centred (reading R4)
// ---------------------------------------------------------------------------------------------
template <class real>
real cmax(const Grid<real>& g) {
  real best = real(0);
  int sawnan = 0;
  const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
#pragma omp parallel for collapse(2) reduction(max : best) reduction(| : sawnan)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        const size_t o = g.at(0, i, j, k);
        const real bx = real(0.5) * (g.f[5][o] + g.f[5][g.at(0, i + 1, j, k)]);
        const real by = real(0.5) * (g.f[6][o] + g.f[6][g.at(0, i, j + 1, k)]);
        const real bz = real(0.5) * (g.f[7][o] + g.f[7][g.at(0, i, j, k + 1)]);
        const real rho = g.f[0][o];
        const real vx = g.f[1][o] / rho, vy = g.f[2][o] / rho, vz = g.f[3][o] / rho;
        const real b2 = bx * bx + by * by + bz * bz;
        const real ke = real(0.5) * (g.f[1][o] * g.f[1][o] + g.f[2][o] * g.f[2][o] + g.f[3][o] * g.f[3][o]) / rho;
        const real p = (g.gamma - real(1)) * (g.f[4][o] - ke - real(0.5) * b2);
        const real vmax = std::max(std::fabs(vx), std::max(std::fabs(vy), std::fabs(vz)));
        const real c = vmax + std::sqrt(std::fabs(g.gamma * p + b2) / rho);
        if (c != c) sawnan = 1;            // NaN must surface, not be skipped by max()
        else best = std::max(best, c);
      }
  return sawnan ? std::nan("") : best;
}

// ---------------------------------------------------------------------------------------------
// O3  fluid_d : Algorithm 1.  B interpolated to cell centres (step 3) and held
//     fixed through both stages; first-order upwind half step, eq (16); second-
//     order TVD full step from u^{t+dt/2}, eqs (11)-(15),(17).
// ---------------------------------------------------------------------------------------------
template <class real>
void fluid(Grid<real>& g, int d, real dt) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  const int nd = g.n[d], na = g.n[t1], nb = g.n[t2];
  const int P = 3;                       // ghost cells per side
  const int W = nd + 2 * P;              // padded pencil length; padded index p <-> cell q = p - P
  real* U[5] = {g.f[0], g.f[1 + d], g.f[1 + t1], g.f[1 + t2], g.f[4]};   // sweep roles
  const real *Bd = g.f[5 + d], *Bt1 = g.f[5 + t1], *Bt2 = g.f[5 + t2];

#pragma omp parallel
  {
    std::vector<real> u(5 * W), bc(3 * W), R(5 * W), G(5 * W), u1(5 * W), phi(5 * W);
#pragma omp for collapse(2)
    for (int b = 0; b < nb; ++b)
      for (int a = 0; a < na; ++a) {
        // step 1+3: gather u and the cell-centred B (faces averaged, eq (19))
        for (int p = 0; p < W; ++p) {
          const int q = p - P;
          const size_t o = g.at(d, q, a, b);
          for (int c = 0; c < 5; ++c) u[c * W + p] = U[c][o];
          bc[0 * W + p] = real(0.5) * (Bd[o] + Bd[g.at(d, q + 1, a, b)]);
          bc[1 * W + p] = real(0.5) * (Bt1[o] + Bt1[g.at(d, q, a + 1, b)]);
          bc[2 * W + p] = real(0.5) * (Bt2[o] + Bt2[g.at(d, q, a, b + 1)]);
        }
        // step 4: F, c from u^t;  right/left-going R = c u + F, G = c u - F  (2c u^R, 2c u^L of eqs (9),(10))
        for (int p = 0; p < W; ++p) {
          real uu[5], bb[3], F[5], c;
          for (int k = 0; k < 5; ++k) uu[k] = u[k * W + p];
          for (int k = 0; k < 3; ++k) bb[k] = bc[k * W + p];
          flux(uu, bb, g.gamma, F, c);
          for (int k = 0; k < 5; ++k) { R[k * W + p] = c * uu[k] + F[k]; G[k * W + p] = c * uu[k] - F[k]; }
        }
        // step 5: first-order upwind flux at face p+1/2: right-going from cell p, left-going from p+1
        for (int k = 0; k < 5; ++k)
          for (int p = 0; p + 1 < W; ++p) phi[k * W + p] = real(0.5) * (R[k * W + p] - G[k * W + p + 1]);
        // step 6: u^{t+dt/2}, eq (16)
        for (int k = 0; k < 5; ++k)
          for (int p = 1; p + 1 < W; ++p)
            u1[k * W + p] = u[k * W + p] - (phi[k * W + p] - phi[k * W + p - 1]) * (dt * real(0.5));
        // step 7: F, c from u^{t+dt/2} (same cell-centred B)
        for (int p = 1; p + 1 < W; ++p) {
          real uu[5], bb[3], F[5], c;
          for (int k = 0; k < 5; ++k) uu[k] = u1[k * W + p];
          for (int k = 0; k < 3; ++k) bb[k] = bc[k * W + p];
          flux(uu, bb, g.gamma, F, c);
          for (int k = 0; k < 5; ++k) { R[k * W + p] = c * uu[k] + F[k]; G[k * W + p] = c * uu[k] - F[k]; }
        }
        // step 8: second-order TVD flux at face p+1/2, eqs (11)-(15); left-going is the mirror image
        for (int k = 0; k < 5; ++k) {
          const real *r = &R[k * W], *l = &G[k * W];
          for (int p = 2; p + 3 < W; ++p) {   // faces -1/2 .. nd-1/2; needs R at p-1..p+1, G at p..p+2
            const real rp = r[p] + vanleer(real(0.5) * (r[p] - r[p - 1]), real(0.5) * (r[p + 1] - r[p]));
            const real lp = l[p + 1] + vanleer(real(0.5) * (l[p + 1] - l[p + 2]), real(0.5) * (l[p] - l[p + 1]));
            phi[k * W + p] = real(0.5) * (rp - lp);
          }
        }
        // step 9: u^{t+dt}, eq (17) applied to u^t; scatter the interior back
        for (int q = 0; q < nd; ++q) {
          const int p = q + P;
          const size_t o = g.at(d, q, a, b);
          for (int k = 0; k < 5; ++k) U[k][o] = u[k * W + p] - (phi[k * W + p] - phi[k * W + p - 1]) * dt;
        }
      }
  }
}

// ---------------------------------------------------------------------------------------------
// O4  B_{t->d}: advect the transverse component B_t along d and apply the same edge flux to B_d
//     (constraint step).  Eqs (19)-(22) PAPER.md:134-160, Algorithm 2 PAPER.md:293-311.
//     edge_flux() returns f at faces q+1/2, q = -1..nd-1, of the pencil whose (unmapped) index
//     along t is tau; f lives on the edge (q+1/2, tau-1/2).
// ---------------------------------------------------------------------------------------------
template <class real>
void edge_flux(const Grid<real>& g, int d, int t, int tau, int sig, real dt, real* fout /* nd+1 */,
               std::vector<real>& wk) {
  const int nd = g.n[d];
  const int P = 4, W = nd + 2 * P;
  wk.resize(6 * (size_t)W);
  real *vt = &wk[0], *vg = &wk[W], *b = &wk[2 * W], *b1 = &wk[3 * W], *w = &wk[4 * W], *f1 = &wk[5 * W];
  const real *rho = g.f[0], *md = g.f[1 + d], *Bt = g.f[5 + t];
  const bool t_is_t1 = (t == (d + 1) % 3);
  auto cell = [&](int q, int tt) { return t_is_t1 ? g.at(d, q, tt, sig) : g.at(d, q, sig, tt); };

  // Alg. 2 step 4: velocity at the B_t face = the two cells sharing it (reading R5: mass weighted)
  for (int p = 0; p < W; ++p) {
    const size_t lo = cell(p - P, tau - 1), hi = cell(p - P, tau);
    vt[p] = (md[lo] + md[hi]) / (rho[lo] + rho[hi]);
    b[p] = Bt[hi];
  }
  // step 5: eq (20), 1-2-1 smoothing along d
  for (int p = 1; p + 1 < W; ++p) vg[p] = real(0.25) * ((vt[p - 1] + vt[p + 1]) + real(2) * vt[p]);
  // step 6: first-order upwind flux at face p+1/2, eqs (21),(22)
  for (int p = 1; p + 1 < W; ++p) w[p] = vg[p] * b[p];
  for (int p = 1; p + 2 < W; ++p) {
    const real vh = real(0.5) * (vg[p] + vg[p + 1]);
    f1[p] = vh > real(0) ? w[p] : w[p + 1];
  }
  // step 7: half step, eq (16) applied to B_t
  for (int p = 2; p + 2 < W; ++p) b1[p] = b[p] - (f1[p] - f1[p - 1]) * (dt * real(0.5));
  // step 8: second-order TVD flux from B_t^{t+dt/2}, same velocities (fluid held fixed)
  for (int p = 2; p + 2 < W; ++p) w[p] = vg[p] * b1[p];
  for (int q = -1; q < nd; ++q) {
    const int p = q + P;
    const real vh = real(0.5) * (vg[p] + vg[p + 1]);
    real f;
    if (vh > real(0)) f = w[p] + vanleer(real(0.5) * (w[p] - w[p - 1]), real(0.5) * (w[p + 1] - w[p]));
    else f = w[p + 1] + vanleer(real(0.5) * (w[p + 1] - w[p + 2]), real(0.5) * (w[p] - w[p + 1]));
    fout[q + 1] = f * dt;
  }
}

template <class real>
void badvect(Grid<real>& g, int d, int t, real dt) {
  const int s = 3 - d - t;                       // the third axis
  const int nd = g.n[d], nt = g.n[t], ns = g.n[s];
  const bool t_is_t1 = (t == (d + 1) % 3);
  real *Bt = g.f[5 + t], *Bd = g.f[5 + d];
  const size_t L = (size_t)nd + 1;
  // all edge fluxes first, from the pre-update B_t of this call: own row tau and row tau+1
  std::vector<real> fown(L * nt * ns), fplus(L * nt * ns);
#pragma omp parallel
  {
    std::vector<real> wk;
#pragma omp for collapse(2)
    for (int sig = 0; sig < ns; ++sig)
      for (int tau = 0; tau < nt; ++tau) {
        const size_t o = L * ((size_t)tau + (size_t)nt * sig);
        edge_flux(g, d, t, tau, sig, dt, &fown[o], wk);
        edge_flux(g, d, t, tau + 1, sig, dt, &fplus[o], wk);
      }
  }
#pragma omp parallel for collapse(2)
  for (int sig = 0; sig < ns; ++sig)
    for (int tau = 0; tau < nt; ++tau) {
      const size_t o = L * ((size_t)tau + (size_t)nt * sig);
      for (int q = 0; q < nd; ++q) {
        const size_t c = t_is_t1 ? g.at(d, q, tau, sig) : g.at(d, q, sig, tau);
        // step 9: advection of B_t, flux difference along d ...
        Bt[c] = Bt[c] - (fown[o + q + 1] - fown[o + q]);
        // ... and the constraint step: the same flux updates B_d; B_d[q] sits on face q-1/2
        Bd[c] = Bd[c] + (fplus[o + q] - fown[o + q]);
      }
    }
}

// O5  L_d: forward = fluid_d, B_{t1->d}, B_{t2->d}; reverse = mirror image.
template <class real>
void sweep(Grid<real>& g, int d, bool reverse, real dt) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  if (!reverse) { fluid(g, d, dt); badvect(g, d, t1, dt); badvect(g, d, t2, dt); }
  else          { badvect(g, d, t2, dt); badvect(g, d, t1, dt); fluid(g, d, dt); }
}

// O6  one double sweep, eqs (23)-(25) PAPER.md:164-170 (operators act right to left)
template <class real>
void step(Grid<real>& g, long long s, real dt) {
  static const int order[3][3] = {{0, 1, 2}, {2, 0, 1}, {1, 2, 0}};
  const int* o = order[((s % 3) + 3) % 3];
  for (int i = 0; i < 3; ++i) sweep(g, o[i], false, dt);
  for (int i = 2; i >= 0; --i) sweep(g, o[i], true, dt);
}

template <class real>
Grid<real> make(int nx, int ny, int nz, double gamma, int bc, void* const fields[8]) {
  Grid<real> g;
  g.n[0] = nx; g.n[1] = ny; g.n[2] = nz; g.gamma = (real)gamma; g.bc = bc;
  for (int c = 0; c < 8; ++c) g.f[c] = (real*)fields[c];
  return g;
}

bool bad(int prec, int nx, int ny, int nz, double gamma, int bc, void* const fields[8]) {
  if (prec != 0 && prec != 1) return true;
  if (nx < 1 || ny < 1 || nz < 1 || !(gamma > 1.0) || (bc != 0 && bc != 1) || !fields) return true;
  for (int c = 0; c < 8; ++c) if (!fields[c]) return true;
  return false;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// C entry points for ctypes (oracle/__init__.py).  prec: 0 = float, 1 = double.  All arrays are
// caller-owned host memory, updated in place.  Return 0, or -1 on invalid arguments.
// ---------------------------------------------------------------------------------------------
#define DISPATCH(EXPR32, EXPR64) do { if (prec == 0) { auto g = make<float>(nx, ny, nz, gamma, bc, fields); EXPR32; } \
                                      else { auto g = make<double>(nx, ny, nz, gamma, bc, fields); EXPR64; } } while (0)

extern "C" {

int mhdo_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void mhdo_set_num_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
#else
  (void)n;
#endif
}

int mhdo_cmax(int prec, int nx, int ny, int nz, double gamma, int bc, void* const fields[8], double* out) {
  if (bad(prec, nx, ny, nz, gamma, bc, fields) || !out) return -1;
  DISPATCH(*out = (double)cmax(g), *out = (double)cmax(g));
  return 0;
}

int mhdo_fluid(int prec, int nx, int ny, int nz, double gamma, int bc, void* const fields[8], int d, double dt) {
  if (bad(prec, nx, ny, nz, gamma, bc, fields) || d < 0 || d > 2) return -1;
  DISPATCH(fluid(g, d, (float)dt), fluid(g, d, dt));
  return 0;
}

// t is an absolute axis (0,1,2), t != d
int mhdo_badvect(int prec, int nx, int ny, int nz, double gamma, int bc, void* const fields[8], int d, int t, double dt) {
  if (bad(prec, nx, ny, nz, gamma, bc, fields) || d < 0 || d > 2 || t < 0 || t > 2 || t == d) return -1;
  DISPATCH(badvect(g, d, t, (float)dt), badvect(g, d, t, dt));
  return 0;
}

int mhdo_sweep(int prec, int nx, int ny, int nz, double gamma, int bc, void* const fields[8], int d, int reverse, double dt) {
  if (bad(prec, nx, ny, nz, gamma, bc, fields) || d < 0 || d > 2) return -1;
  DISPATCH(sweep(g, d, reverse != 0, (float)dt), sweep(g, d, reverse != 0, dt));
  return 0;
}

// one double sweep with step index s and the caller's dt
int mhdo_step_fixed(int prec, int nx, int ny, int nz, double gamma, int bc, void* const fields[8], long long s, double dt) {
  if (bad(prec, nx, ny, nz, gamma, bc, fields)) return -1;
  DISPATCH(step(g, s, (float)dt), step(g, s, dt));
  return 0;
}

// program flow steps 4-9: n times { c_max; dt = cfl/c_max; six L_i; t += 2 dt }.
// dt is formed in double from the c_max computed in the run precision and rounded to the run
// precision where it is used.  *t_advanced (optional) accumulates 2 dt in double.
int mhdo_run(int prec, int nx, int ny, int nz, double gamma, int bc, void* const fields[8], long long s0, int nsteps,
             double cfl, double* t_advanced) {
  if (bad(prec, nx, ny, nz, gamma, bc, fields) || nsteps < 0 || !(cfl > 0.0)) return -1;
  double t = 0.0;
  for (int it = 0; it < nsteps; ++it) {
    double cm;
    DISPATCH(cm = (double)cmax(g), cm = (double)cmax(g));
    if (!(cm > 0.0) || !std::isfinite(cm)) return -4;
    const double dt = cfl / cm;
    DISPATCH(step(g, s0 + it, (float)dt), step(g, s0 + it, dt));
    t += 2.0 * dt;
  }
  if (t_advanced) *t_advanced = t;
  return 0;
}

}  // extern "C"
