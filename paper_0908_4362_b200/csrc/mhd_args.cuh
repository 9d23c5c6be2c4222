// mhd_args.cuh -- kernel argument blocks of the specialised sweep kernels.
#pragma once
#include "mhd_device.cuh"

namespace mhd {

// sweeps along y and z (mhd_yz2.cuh, mhd_bring.cuh): lanes span x, a block marches along the sweep axis d
template <class real>
struct YZArgs {
  // fluid: u[5] in / uo[5] out in sweep roles (rho, m_d, m_t1, m_t2, E);  B pair: u[0] = rho, u[1] = m_d
  const real* u[5];
  real* uo[5];
  const real *bd, *bx, *bo;     // B along the sweep, Bx (transverse, +1 neighbour is the next lane), B along the other axis
  real *bdo, *bxo, *boo;        // B-pair outputs
  const double* dt;
  unsigned long long* cmax_bits;   // != nullptr: also reduce c of eq (18) over the UPDATED cells (last operator of a step)
  int nx, nd, no;               // extents: x, sweep axis, other transverse axis
  int sd, so;                   // element strides of the sweep axis and of the other transverse axis
  int bc, seg;
  int x_is_t1;                  // sweep z: (t1,t2) = (x,y) -> 1;  sweep y: (t1,t2) = (z,x) -> 0
  int t2_first;                 // B pair in a reverse sweep
  real gamma;
  // byte offsets of the source rows of a ring stage relative to u[0] (host-computed, read straight from the constant
  // bank by the elected producer lane: one 64-bit add per copy instead of a pointer load plus index arithmetic)
  long long src[8];
};

// sweeps along x (mhd_x2.cuh): a thread owns V consecutive cells (one 16-byte vector) of one or two rows
template <class real> struct VecOf;
template <> struct VecOf<float> { typedef float4 type; enum { V = 4 }; };
template <> struct VecOf<double> { typedef double2 type; enum { V = 2 }; };

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
  int tpr_shift;           // log2(tpr) if tpr is a power of two, else -1
  int rpb;                 // row groups per block
  int t2_first;
  int ghost;               // outflow along x: ghost threads on either side of a row (4 clamped cells), else 0; tpr counts them
  real gamma;
  real one;                // 1.0 at run time (xload)
};

}  // namespace mhd
