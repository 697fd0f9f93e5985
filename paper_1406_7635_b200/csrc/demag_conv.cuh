// demag_conv.cuh - generic (any 5-smooth size, 2D/3D, open/periodic) demagnetising convolution
//   B_demag,i = K_ij * (Bsat m_j)      (Eq. 3)
// as: x forward (two real rows packed in one complex line) -> [y forward] -> last axis forward +
// multiply by the real symmetric kernel spectrum + last axis inverse (one kernel) -> [y inverse]
// -> x inverse.  Zero padding is implicit (never stored); the padded half of an open axis is never
// read and the outputs that fall in the padding are never written (L509, L531).
#pragma once
#include "common.cuh"
#include "fft_generic.cuh"
#include "demag_conv_args.cuh"


__device__ __forceinline__ int spec_row(const Geometry& g, int r) {
  // physical row r = z * Ny + y  ->  spectrum row
  if (g.Pz == 1) return r;
  int z = r / g.Ny, y = r - z * g.Ny;
  return z * g.Py + y;
}

// ---- x forward: L row pairs per block
__global__ void k_x_fwd(ConvArgs a, int src_role, int L) {
  if (a.st->skip) return;
  extern __shared__ float2 smem[];
  const Geometry& g = a.g;
  const int P = g.Px, c = blockIdx.y;
  const int rows = g.Ny * g.Nz;
  const int pair0 = blockIdx.x * L;
  float2* bufA = smem;
  float2* bufB = smem + (size_t)L * P;
  const float* __restrict__ src = a.st->ptr[src_role] + (size_t)c * g.N;
  const float* __restrict__ bsat = a.luts->Bsat;
  for (int idx = threadIdx.x; idx < L * P; idx += blockDim.x) {
    int l = idx / P, x = idx - l * P;
    int r0 = 2 * (pair0 + l), r1 = r0 + 1;
    float2 v = make_float2(0.f, 0.f);
    if (x < g.Nx) {
      if (r0 < rows) { size_t i = (size_t)r0 * g.Nx + x; v.x = src[i] * bsat[a.regions[i]]; }
      if (r1 < rows) { size_t i = (size_t)r1 * g.Nx + x; v.y = src[i] * bsat[a.regions[i]]; }
    }
    bufA[idx] = v;
  }
  __syncthreads();
  float2* res = stockham_fft(bufA, bufB, a.px, L, P, a.twx);
  const int Cx = g.Cx;
  for (int idx = threadIdx.x; idx < L * Cx; idx += blockDim.x) {
    int l = idx / Cx, k = idx - l * Cx;
    int r0 = 2 * (pair0 + l), r1 = r0 + 1;
    if (r0 >= rows) continue;
    float2 zk = res[l * P + k];
    float2 zm = res[l * P + (k == 0 ? 0 : P - k)];
    float2 A = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));
    float2 B = make_float2(0.5f * (zk.y + zm.y), -0.5f * (zk.x - zm.x));
    a.spec[(size_t)c * a.cstride + (size_t)spec_row(g, r0) * g.pitch + k] = A;
    if (r1 < rows) a.spec[(size_t)c * a.cstride + (size_t)spec_row(g, r1) * g.pitch + k] = B;
  }
}

// ---- x inverse: writes B_demag rows (real part -> first row of the pair, imaginary -> second)
__global__ void k_x_inv(ConvArgs a, int dst_role, int L) {
  if (a.st->skip) return;
  extern __shared__ float2 smem[];
  const Geometry& g = a.g;
  const int P = g.Px, c = blockIdx.y, Cx = g.Cx;
  const int rows = g.Ny * g.Nz;
  const int pair0 = blockIdx.x * L;
  float2* bufA = smem;
  float2* bufB = smem + (size_t)L * P;
  for (int idx = threadIdx.x; idx < L * P; idx += blockDim.x) {
    int l = idx / P, k = idx - l * P;
    int r0 = 2 * (pair0 + l), r1 = r0 + 1;
    float2 v = make_float2(0.f, 0.f);
    if (r0 < rows) {
      int kk = (k < Cx) ? k : P - k;           // Hermitian partner for k > P/2
      float2 A = a.spec[(size_t)c * a.cstride + (size_t)spec_row(g, r0) * g.pitch + kk];
      float2 B = make_float2(0.f, 0.f);
      if (r1 < rows) B = a.spec[(size_t)c * a.cstride + (size_t)spec_row(g, r1) * g.pitch + kk];
      if (k >= Cx) { A.y = -A.y; B.y = -B.y; }
      // Z = A + i B, conjugated for the inverse transform
      v = make_float2(A.x - B.y, -(A.y + B.x));
    }
    bufA[idx] = v;
  }
  __syncthreads();
  float2* res = stockham_fft(bufA, bufB, a.px, L, P, a.twx);
  float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * g.N;
  for (int idx = threadIdx.x; idx < L * g.Nx; idx += blockDim.x) {
    int l = idx / g.Nx, x = idx - l * g.Nx;
    int r0 = 2 * (pair0 + l), r1 = r0 + 1;
    if (r0 >= rows) continue;
    float2 z = res[l * P + x];                  // conj(z) = (z.x, -z.y)
    dst[(size_t)r0 * g.Nx + x] = z.x;
    if (r1 < rows) dst[(size_t)r1 * g.Nx + x] = -z.y;
  }
}

// ---- y stage of 3D problems: lines along y at fixed (comp, z < Nz, kx); in place
__global__ void k_y_axis(ConvArgs a, int inverse, int C) {
  if (a.st->skip) return;
  extern __shared__ float2 smem[];
  const Geometry& g = a.g;
  const int P = g.Py;
  const int kx0 = blockIdx.x * C, z = blockIdx.y, c = blockIdx.z;
  const int nc = min(C, g.Cx - kx0);
  const int n_in = inverse ? P : g.Ny, n_out = inverse ? g.Ny : P;
  float2* bufA = smem;
  float2* bufB = smem + (size_t)C * P;
  float2* base = a.spec + (size_t)c * a.cstride + (size_t)z * g.Py * g.pitch + kx0;
  const float sgn = inverse ? -1.f : 1.f;
  for (int idx = threadIdx.x; idx < C * P; idx += blockDim.x) {
    int i = idx / C, cc = idx - i * C;
    float2 v = make_float2(0.f, 0.f);
    if (cc < nc && i < n_in) { v = base[(size_t)i * g.pitch + cc]; v.y *= sgn; }
    bufA[cc * P + i] = v;
  }
  __syncthreads();
  float2* res = stockham_fft(bufA, bufB, a.py, C, P, a.twy);
  for (int idx = threadIdx.x; idx < C * n_out; idx += blockDim.x) {
    int i = idx / C, cc = idx - i * C;
    if (cc >= nc) continue;
    float2 v = res[cc * P + i];
    v.y *= sgn;
    base[(size_t)i * g.pitch + cc] = v;
  }
}

// ---- last axis: forward + kernel multiply + inverse, in place on the spectrum.
// mode 0: 2D, components (x, y) coupled by K_xx, K_xy, K_yy;  mode 1: 2D, component z with K_zz;
// mode 2: 3D, all three components, six kernel components; lines along z at fixed (ky, kx).
template <int NC>
__global__ void k_last_fused(ConvArgs a, int mode, int C) {
  if (a.st->skip) return;
  extern __shared__ float2 smem[];
  const Geometry& g = a.g;
  const bool alongz = (mode == 2);
  const AxisPlan& pl = alongz ? a.pz : a.py;
  const float2* tw = alongz ? a.twz : a.twy;
  const int P = pl.P, n = pl.N;
  const int kx0 = blockIdx.x * C;
  const int nc = min(C, g.Cx - kx0);
  const int ky = alongz ? blockIdx.y : 0;
  const size_t lstride = alongz ? (size_t)g.Py * g.pitch : (size_t)g.pitch;
  const size_t base0 = (alongz ? (size_t)ky * g.pitch : 0) + kx0;
  const int c0 = (mode == 1) ? 2 : 0;
  float2* buf[NC + 1];
#pragma unroll
  for (int i = 0; i <= NC; ++i) buf[i] = smem + (size_t)i * C * P;
  // forward transforms
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    const float2* src = a.spec + (size_t)(c0 + i) * a.cstride + base0;
    for (int idx = threadIdx.x; idx < C * P; idx += blockDim.x) {
      int j = idx / C, cc = idx - j * C;
      float2 v = make_float2(0.f, 0.f);
      if (cc < nc && j < n) v = src[(size_t)j * lstride + cc];
      buf[i][cc * P + j] = v;
    }
    __syncthreads();
    float2* res = stockham_fft(buf[i], buf[NC], pl, C, P, tw);
    if (res != buf[i]) { buf[NC] = buf[i]; buf[i] = res; }
  }
  // multiply by the real symmetric kernel spectrum; leave conj(result) for the inverse transform
  {
    const int Hy = g.Hy, Cx = g.Cx;
    const int kyf = (ky <= g.Py / 2) ? ky : g.Py - ky;
    const float sy_line = (ky <= g.Py / 2) ? 1.f : -1.f;
    for (int idx = threadIdx.x; idx < C * P; idx += blockDim.x) {
      int k = idx / C, cc = idx - k * C;
      if (cc >= nc) continue;
      int kf = (k <= P / 2) ? k : P - k;
      float sk = (k <= P / 2) ? 1.f : -1.f;
      int e = cc * P + k;
      if (mode == 2) {
        size_t ki = ((size_t)kf * Hy + kyf) * Cx + kx0 + cc;
        float kxx = a.K[ki], kyy = a.K[a.kstride + ki], kzz = a.K[2 * a.kstride + ki];
        float kxy = a.K[3 * a.kstride + ki] * sy_line;
        float kxz = a.K[4 * a.kstride + ki] * sk;
        float kyz = a.K[5 * a.kstride + ki] * sy_line * sk;
        float2 mx = buf[0][e], my = buf[NC > 1 ? 1 : 0][e], mz = buf[NC > 2 ? 2 : 0][e];
        buf[0][e] = make_float2(kxx * mx.x + kxy * my.x + kxz * mz.x, -(kxx * mx.y + kxy * my.y + kxz * mz.y));
        if (NC > 1) buf[NC > 1 ? 1 : 0][e] = make_float2(kxy * mx.x + kyy * my.x + kyz * mz.x, -(kxy * mx.y + kyy * my.y + kyz * mz.y));
        if (NC > 2) buf[NC > 2 ? 2 : 0][e] = make_float2(kxz * mx.x + kyz * my.x + kzz * mz.x, -(kxz * mx.y + kyz * my.y + kzz * mz.y));
      } else if (mode == 0) {
        size_t ki = (size_t)kf * Cx + kx0 + cc;
        float kxx = a.K[ki], kyy = a.K[a.kstride + ki], kxy = a.K[3 * a.kstride + ki] * sk;
        float2 mx = buf[0][e], my = buf[NC > 1 ? 1 : 0][e];
        buf[0][e] = make_float2(kxx * mx.x + kxy * my.x, -(kxx * mx.y + kxy * my.y));
        if (NC > 1) buf[NC > 1 ? 1 : 0][e] = make_float2(kxy * mx.x + kyy * my.x, -(kxy * mx.y + kyy * my.y));
      } else {
        size_t ki = (size_t)kf * Cx + kx0 + cc;
        float kzz = a.K[2 * a.kstride + ki];
        float2 mz = buf[0][e];
        buf[0][e] = make_float2(kzz * mz.x, -kzz * mz.y);
      }
    }
    __syncthreads();
  }
  // inverse transforms, first n outputs only
#pragma unroll
  for (int i = 0; i < NC; ++i) {
    float2* res = stockham_fft(buf[i], buf[NC], pl, C, P, tw);
    float2* dst = a.spec + (size_t)(c0 + i) * a.cstride + base0;
    for (int idx = threadIdx.x; idx < C * n; idx += blockDim.x) {
      int j = idx / C, cc = idx - j * C;
      if (cc >= nc) continue;
      float2 v = res[cc * P + j];
      v.y = -v.y;
      dst[(size_t)j * lstride + cc] = v;
    }
    if (res != buf[i]) { buf[NC] = buf[i]; buf[i] = res; }
    __syncthreads();
  }
}
