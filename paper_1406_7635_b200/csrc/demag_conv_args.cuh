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
