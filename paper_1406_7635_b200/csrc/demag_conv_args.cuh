// demag_conv_args.cuh - argument block of the convolution kernels
#pragma once
#include "common.cuh"

struct ConvArgs {
  Geometry g;
  AxisPlan px, py, pz;
  const float2* twx;
  const float2* twy;
  const float2* twz;
  float2* spec;          // [3][rowsS][pitch]
  long long cstride;     // rowsS * pitch
  int rowsS;             // Ny (Pz == 1) or Nz * Py
  const float* K;        // [6 or 4][Hz][Hy][Cx] real symmetric kernel spectrum, comps xx,yy,zz,xy,xz,yz
  long long kstride;     // Hz * Hy * Cx
  const uint8_t* regions;
  const Luts* luts;
  DevState* st;
};

// argument block of the fast 2D path (fast2d.cuh)
struct Fast2DArgs {
  int Nx, Ny, Cx;        // transform lengths (powers of two >= the physical sizes); Cx = Nx + 1 stored kx
  int nxp, nyp;          // physical cells along x and y (rows/columns beyond are implicit zeros)
  int nsm;               // SMs of the device (look-ahead distance of the L2 prefetches)
  long long ncell;       // nxp * nyp
  float2* spec;          // [3][Cx][Ny]
  long long cstride;     // Cx * Ny
  const float* Kt;       // [4][Cx][Ny + 1]: per (component, kx) the even-ky entries ky = 0,2,..,Ny
                         // (Ny/2 + 1) followed by the odd ones ky = 1,3,..,Ny-1; comps xx, yy, zz, xy
  long long kstride;     // Cx * (Ny + 1)
  const float2 *twx, *twx_r;   // plan tables, length Nx: forward plan / reversed plan
  const float2 *twy, *twy_r;   // same for length Ny
  const float2 *twox, *twoy;   // exp(-2 pi i n / (2Nx)), n < Nx ; same for y
  const uint8_t* regions;
  const Luts* luts;
  DevState* st;
};

// argument block of the register-FFT stages of open 3D boxes (fast3d.cuh)
struct Fast3DArgs {
  Geometry g;
  int mode[3];                     // per axis: 0 generic kernels, 1 open axis (padded x2, pruned), 2 periodic axis
  const float2 *twx, *twx_r, *twox;   // x plan (length Nxt)
  const uint8_t* regions;
  const Luts* luts;
  float2* spec;                    // [3][Nz][Py][pitch]
  long long cstride;               // Nz * Py * pitch
  const float* K3;                 // [Hy][kx tiles][6][Nz + 1][C]: the kernel spectrum (xx, yy, zz, xy, xz, yz over the
                                   // non-negative octant) cut into the tiles of the z stage: the (Nz + 1) x C values of
                                   // the six components at one ky and C neighbouring kx are one contiguous block
  const float2 *twy, *twy_r, *twoy;   // y plan (length Ny): forward table, reversed-plan table, exp(-i pi n / Ny)
  const float2 *twz, *twz_r, *twoz;   // z plan (length Nz)
  DevState* st;
};

