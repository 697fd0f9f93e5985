// demag_setup.cuh - demagnetising kernel set-up on the device, fp64:
//   1. cell-averaged demagnetising tensor N_ij(R) between two uniformly magnetised cuboid cells on
//      the zero-padded displacement grid (periodic axes: wrapped sum of the images, L175-L177);
//   2. fp64 FFT of K = -N along every axis (global-memory Stockham passes; set-up only);
//   3. the spectra are real and mirror-(anti)symmetric (L145), so only the real part of
//      kx <= Px/2, ky <= Py/2, kz <= Pz/2 is kept, scaled by 1/(Px Py Pz) and truncated to fp32.
// Near field: closed form of the six-fold integral (second difference of the auxiliary functions
// f, g of the prism-prism interaction). Far field (|R| >= 12 largest cell edges): the closed form
// cancels catastrophically in fp64 there, so the point-dipole tensor is integrated over the
// difference variable s = u - u' of the two cells, whose density per axis is the triangle
// (d - |s|) on [-d, d], by Gauss-Legendre on each half interval.
#pragma once
#include "common.cuh"

namespace setup {

__device__ __forceinline__ double f_aux(double x, double y, double z) {
  x = fabs(x); y = fabs(y); z = fabs(z);
  const double x2 = x * x, y2 = y * y, z2 = z * z;
  const double R = sqrt(x2 + y2 + z2);
  double r = (2.0 * x2 - y2 - z2) * R * (1.0 / 6.0);
  const double p1 = 0.5 * y * (z2 - x2), p2 = 0.5 * z * (y2 - x2), p3 = x * y * z;
  if (p1 != 0.0) r += p1 * asinh(y / sqrt(x2 + z2));
  if (p2 != 0.0) r += p2 * asinh(z / sqrt(x2 + y2));
  if (p3 != 0.0) r -= p3 * atan(y * z / (x * R));
  return r;
}

__device__ __forceinline__ double g_aux(double x, double y, double z) {
  const double sg = ((x < 0.0) != (y < 0.0)) ? -1.0 : 1.0;
  x = fabs(x); y = fabs(y); z = fabs(z);
  const double x2 = x * x, y2 = y * y, z2 = z * z;
  const double R = sqrt(x2 + y2 + z2);
  double r = -x * y * R * (1.0 / 3.0);
  const double p1 = x * y * z;
  const double p2 = y * (3.0 * z2 - y2) * (1.0 / 6.0), p3 = x * (3.0 * z2 - x2) * (1.0 / 6.0);
  if (p1 != 0.0) r += p1 * asinh(z / sqrt(x2 + y2));
  if (p2 != 0.0 && x != 0.0) r += p2 * asinh(x / sqrt(y2 + z2));
  if (p3 != 0.0 && y != 0.0) r += p3 * asinh(y / sqrt(x2 + z2));
  if (z != 0.0 && x != 0.0 && y != 0.0) {
    r -= z * z2 * (1.0 / 6.0) * atan(x * y / (z * R));
    r -= z * y2 * 0.5 * atan(x * z / (y * R));
    r -= z * x2 * 0.5 * atan(y * z / (x * R));
  }
  return sg * r;
}

template <bool G>
__device__ double second_difference(double X, double Y, double Z, double dx, double dy, double dz) {
  double acc = 0.0;
#pragma unroll
  for (int a = -1; a <= 1; ++a)
#pragma unroll
    for (int b = -1; b <= 1; ++b)
#pragma unroll
      for (int c = -1; c <= 1; ++c) {
        const double w = (a == 0 ? 2.0 : -1.0) * (b == 0 ? 2.0 : -1.0) * (c == 0 ? 2.0 : -1.0);
        acc += w * (G ? g_aux(X + a * dx, Y + b * dy, Z + c * dz) : f_aux(X + a * dx, Y + b * dy, Z + c * dz));
      }
  return acc;
}

// N_ij, components xx, yy, zz, xy, xz, yz
__device__ void tensor_near(double X, double Y, double Z, double dx, double dy, double dz, double* out) {
  const double c = 1.0 / (4.0 * 3.14159265358979323846 * dx * dy * dz);
  out[0] = c * second_difference<false>(X, Y, Z, dx, dy, dz);
  out[1] = c * second_difference<false>(Y, X, Z, dy, dx, dz);
  out[2] = c * second_difference<false>(Z, Y, X, dz, dy, dx);
  out[3] = c * second_difference<true>(X, Y, Z, dx, dy, dz);
  out[4] = c * second_difference<true>(X, Z, Y, dx, dz, dy);
  out[5] = c * second_difference<true>(Y, Z, X, dy, dz, dx);
}

// Gauss-Legendre nodes / weights on [0, 1]
__constant__ double GL_X[2][4] = {{0.21132486540518711775, 0.78867513459481288225, 0.0, 0.0},
                                  {0.06943184420297371239, 0.33000947820757186760, 0.66999052179242813240,
                                   0.93056815579702628761}};
__constant__ double GL_W[2][4] = {{0.5, 0.5, 0.0, 0.0},
                                  {0.17392742256872692869, 0.32607257743127307131, 0.32607257743127307131,
                                   0.17392742256872692869}};

// far field: N_ij = -(1/V) * int T_ij(R + s) prod_a (d_a - |s_a|) d3s,  T = (3 r_i r_j - r^2 delta_ij)/(4 pi r^5)
__device__ void tensor_far(double X, double Y, double Z, double dx, double dy, double dz, int rule, double* out) {
  const int n = rule == 0 ? 2 : 4;
  double acc[6] = {0, 0, 0, 0, 0, 0};
  for (int ia = 0; ia < 2 * n; ++ia) {
    const double ua = GL_X[rule][ia % n], sa = (ia < n ? ua : -ua) * dx, wa = GL_W[rule][ia % n] * (1.0 - ua);
    for (int ib = 0; ib < 2 * n; ++ib) {
      const double ub = GL_X[rule][ib % n], sb = (ib < n ? ub : -ub) * dy, wb = GL_W[rule][ib % n] * (1.0 - ub);
      for (int ic = 0; ic < 2 * n; ++ic) {
        const double uc = GL_X[rule][ic % n], sc = (ic < n ? uc : -uc) * dz, wc = GL_W[rule][ic % n] * (1.0 - uc);
        const double x = X + sa, y = Y + sb, z = Z + sc;
        const double r2 = x * x + y * y + z * z;
        const double w = wa * wb * wc / (r2 * r2 * sqrt(r2));
        acc[0] += w * (3.0 * x * x - r2); acc[1] += w * (3.0 * y * y - r2); acc[2] += w * (3.0 * z * z - r2);
        acc[3] += w * 3.0 * x * y; acc[4] += w * 3.0 * x * z; acc[5] += w * 3.0 * y * z;
      }
    }
  }
  // each axis integral carries d_a^2 (sum of weights = 1/2 per half => total 1); 1/V and 1/(4 pi)
  const double c = -(dx * dy * dz) / (4.0 * 3.14159265358979323846);
  for (int k = 0; k < 6; ++k) out[k] = c * acc[k];
}

__device__ void tensor_any(double X, double Y, double Z, double dx, double dy, double dz, double* out) {
  const double dmax = fmax(dx, fmax(dy, dz));
  const double rr = sqrt(X * X + Y * Y + Z * Z) / dmax;
  if (rr < 12.0) tensor_near(X, Y, Z, dx, dy, dz, out);
  else if (rr < 40.0) tensor_far(X, Y, Z, dx, dy, dz, 1, out);
  else tensor_far(X, Y, Z, dx, dy, dz, 0, out);
}

struct TensorGrid {
  int N[3];      // cells (x, y, z)
  int P[3];      // padded lengths
  int rep[3];    // PBC repeats (0 = open)
  int E[3];      // evaluated extent per axis: indices 0..E-1 (non-negative displacements)
  double d[3];
};

// K = -N on the non-negative octant of the (wrapped) displacement grid: out[comp][iz][iy][ix],
// ix < E[0] etc. For a periodic axis the entry i holds sum over images D = i + n*N, |D| <= N*rep - 1.
__global__ void k_tensor_octant(TensorGrid tg, double* __restrict__ out) {
  const long long total = (long long)tg.E[0] * tg.E[1] * tg.E[2];
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= total) return;
  const int ix = (int)(id % tg.E[0]);
  const int iy = (int)((id / tg.E[0]) % tg.E[1]);
  const int iz = (int)(id / ((long long)tg.E[0] * tg.E[1]));
  int lo[3], hi[3];
  const int idx[3] = {ix, iy, iz};
  for (int a = 0; a < 3; ++a) {
    if (tg.rep[a] > 0) {
      const int lim = tg.N[a] * tg.rep[a] - 1;            // |D| <= lim
      // images n with |idx + n N| <= lim
      int nlo = -((lim + idx[a]) / tg.N[a]);
      int nhi = (lim - idx[a]) / tg.N[a];
      lo[a] = nlo; hi[a] = nhi;
    } else { lo[a] = 0; hi[a] = 0; }
  }
  double acc[6] = {0, 0, 0, 0, 0, 0};
  for (int nz = lo[2]; nz <= hi[2]; ++nz)
    for (int ny = lo[1]; ny <= hi[1]; ++ny)
      for (int nx = lo[0]; nx <= hi[0]; ++nx) {
        double t[6];
        tensor_any((ix + nx * tg.N[0]) * tg.d[0], (iy + ny * tg.N[1]) * tg.d[1], (iz + nz * tg.N[2]) * tg.d[2],
                   tg.d[0], tg.d[1], tg.d[2], t);
        for (int k = 0; k < 6; ++k) acc[k] += t[k];
      }
  for (int k = 0; k < 6; ++k) out[(size_t)k * total + id] = -acc[k];
}

// Expand one component from the octant to the full padded grid as complex fp64 (imag = 0), with the
// parity of the component: xx,yy,zz even; xy odd in x,y; xz odd in x,z; yz odd in y,z.
__global__ void k_expand(TensorGrid tg, const double* __restrict__ oct, int comp, double2* __restrict__ full) {
  const long long total = (long long)tg.P[0] * tg.P[1] * tg.P[2];
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= total) return;
  const int i[3] = {(int)(id % tg.P[0]), (int)((id / tg.P[0]) % tg.P[1]), (int)(id / ((long long)tg.P[0] * tg.P[1]))};
  const int odd[6][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 1, 1}};
  int j[3];
  double sg = 1.0;
  bool zero = false;
  for (int a = 0; a < 3; ++a) {
    int v = i[a];
    int neg = 0;
    if (tg.rep[a] > 0) {                 // periodic, P == N: displacement v or v - N (same wrapped sum)
      if (v > tg.N[a] / 2) { v = tg.N[a] - v; neg = 1; }
    } else {
      if (v >= tg.N[a]) {                // negative displacement v - P, or inside the zero padding
        v = tg.P[a] - v; neg = 1;
        if (v >= tg.N[a]) zero = true;
      }
    }
    if (v >= tg.E[a]) zero = true;
    if (neg && odd[comp][a]) sg = -sg;
    j[a] = v;
  }
  double val = 0.0;
  if (!zero) val = sg * oct[(size_t)comp * tg.E[0] * tg.E[1] * tg.E[2] + ((size_t)j[2] * tg.E[1] + j[1]) * tg.E[0] + j[0]];
  full[id] = make_double2(val, 0.0);
}

// One Stockham pass (radix R in {2,3,4,5,8} done as a plain O(R^2) DFT - set-up only) along an axis
// with element stride `s` (s = product of the faster dimensions), length P.
__global__ void k_fft_pass_f64(const double2* __restrict__ src, double2* __restrict__ dst, long long total_bf, int P,
                               int R, int Ns, long long s) {
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= total_bf) return;
  const int nb = P / R;
  const long long inner = id % s;
  const int j = (int)((id / s) % nb);
  const long long outer = id / (s * nb);
  const size_t base = (size_t)outer * P * s + inner;
  const int k = j % Ns;
  double2 v[8];
  for (int r = 0; r < R; ++r) {
    double2 x = src[base + (size_t)(j + r * nb) * s];
    double sn, cs;
    sincospi(-2.0 * (double)r * (double)k / ((double)Ns * (double)R), &sn, &cs);
    v[r] = make_double2(x.x * cs - x.y * sn, x.x * sn + x.y * cs);
  }
  const int j0 = (j - k) * R + k;
  for (int q = 0; q < R; ++q) {
    double2 acc = make_double2(0.0, 0.0);
    for (int r = 0; r < R; ++r) {
      double sn, cs;
      sincospi(-2.0 * (double)((r * q) % R) / (double)R, &sn, &cs);
      acc.x += v[r].x * cs - v[r].y * sn;
      acc.y += v[r].x * sn + v[r].y * cs;
    }
    dst[base + (size_t)(j0 + q * Ns) * s] = acc;
  }
}

// keep Re K~ on kx <= Px/2, ky <= Py/2, kz <= Pz/2, scaled, as fp32; track max |Im| as a self-check
__global__ void k_pack_spectrum(TensorGrid tg, const double2* __restrict__ full, float* __restrict__ out, int Cx, int Hy,
                                int Hz, double scale, double* __restrict__ max_imag) {
  const long long total = (long long)Cx * Hy * Hz;
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= total) return;
  const int kx = (int)(id % Cx), ky = (int)((id / Cx) % Hy), kz = (int)(id / ((long long)Cx * Hy));
  const double2 v = full[((size_t)kz * tg.P[1] + ky) * tg.P[0] + kx];
  out[id] = (float)(v.x * scale);
  const double im = fabs(v.y * scale);
  if (im > 1e-9) atomicMax((unsigned long long*)max_imag, (unsigned long long)__double_as_longlong(im));
}

// 2D fast-path layout (fast2d.cuh): out[kx][pos], pos = even ky (0,2,..,Ny) then odd ky (1,3,..,Ny-1)
__global__ void k_pack_spectrum_2dfast(TensorGrid tg, const double2* __restrict__ full, float* __restrict__ out, int Cx,
                                       int Ny, double scale) {
  const long long total = (long long)Cx * (Ny + 1);
  const long long id = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (id >= total) return;
  const int kx = (int)(id / (Ny + 1)), pos = (int)(id % (Ny + 1));
  const int ky = pos <= Ny / 2 ? 2 * pos : 2 * (pos - Ny / 2 - 1) + 1;
  out[id] = (float)(full[(size_t)ky * tg.P[0] + kx].x * scale);
}

}  // namespace setup
