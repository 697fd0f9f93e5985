// fast3d.cuh - y and z stages of the demagnetising convolution of open 3D boxes on the register-FFT engine
// (Eq. 3; zero padding x2 per open axis L509; 3D costs about 1.5x 2D per cell, L507).
//
// The spectrum keeps the natural layout spec[c][z][ky][kx] (kx fastest). Lines along y or z are strided, so a
// CTA takes C lines that are neighbours in kx: thread (t, g) holds sixteen points of line g, and for every point
// index the C lines of the CTA touch one contiguous piece of 8 C bytes. As in the 2D path a line of N samples
// zero-padded to 2N is two length-N transforms (even bins: FFT_N(z), odd bins: FFT_N(z w^n)) that run in
// lockstep in the two lanes of the packed-fp32 instructions (fft_reg.cuh); the padded half is never read, stored
// or transformed. All lines of a CTA run in lockstep, so the exchanges use the CTA barrier and shared buffers
// laid out [point][line]: a quarter-warp always reads or writes 128 contiguous bytes (no padding, no conflicts).
//
//   k3_y   : y forward (rows y < Ny -> bins ky < 2Ny) or y inverse (bins -> rows), in place, one component
//   k3_z   : z forward of the three components, product with the six-component real symmetric kernel spectrum
//            (Eq. 3; K real and even/odd under the mirrors, L145), z inverse; in place, only the Nz physical layers
//            are stored. The three components of a line are three thread groups that hand their spectra to one
//            another through the exchange buffer, so nothing is parked and each thread forms one output component.
#pragma once
#include "common.cuh"
#include "fft_reg.cuh"

struct Fast3DArgs {
  Geometry g;
  float2* spec;                    // [3][Nz][Py][pitch]
  long long cstride;               // Nz * Py * pitch
  const float* K;                  // [6][Hz][Hy][Cx]: xx, yy, zz, xy, xz, yz over the non-negative octant
  long long kstride;               // Hz * Hy * Cx
  const float2 *twy, *twy_r, *twoy;   // y plan (length Ny): forward table, reversed-plan table, exp(-i pi n / Ny)
  const float2 *twz, *twz_r, *twoz;   // z plan (length Nz)
  DevState* st;
};

namespace f3 {
using rf::C2;

// exchange between two passes through a [point][line] buffer with LS lines; xb already points at this thread's line
template <class P, int R, int RN, int MP, int LS>
__device__ __forceinline__ void exchange(C2* v, float4* xb, int t) {
  constexpr int MN = MP / RN;
  static_assert(P::T % MN == 0, "threads of a line must cover whole butterflies of the next pass");
  const int rbase = (t / MN) * MP + (t % MN);
  constexpr int RB_STEP = (P::T / MN) * MP;
  __syncthreads();
#pragma unroll
  for (int b = 0; b < P::E / R; ++b)
#pragma unroll
    for (int s = 0; s < R; ++s) xb[(size_t)(t + P::T * b + (P::N / R) * s) * LS] = rf::pack(v[b * R + s]);
  __syncthreads();
#pragma unroll
  for (int b = 0; b < P::E / RN; ++b)
#pragma unroll
    for (int s = 0; s < RN; ++s) v[b * RN + s] = rf::unpack(xb[(size_t)(rbase + RB_STEP * b + s * MN) * LS]);
}

// the transform of rf::fft with the exchange above. The first exchange starts with a CTA barrier, so xb may still
// be read until then; after the call it is safe to reuse only after another barrier.
template <class P, int DIR, int LS>
__device__ __forceinline__ void fft(C2* v, float4* xb, int t, const float2* __restrict__ tw) {
  rf::pass_butterflies<P, P::RA, DIR>(v);
  {
    float2 w[(P::RA - 1) * (P::E / P::RA)];
    rf::load_twiddles<P, P::RA>(w, t, tw);
    rf::apply_twiddles<P, P::RA, DIR>(v, w);
  }
  exchange<P, P::RA, P::RB, P::M1, LS>(v, xb, t);
  rf::pass_butterflies<P, P::RB, DIR>(v);
  if constexpr (P::NPASS == 3) {
    {
      float2 w[(P::RB - 1) * (P::E / P::RB)];
      rf::load_twiddles<P, P::RB>(w, t, tw + P::TW1);
      rf::apply_twiddles<P, P::RB, DIR>(v, w);
    }
    exchange<P, P::RB, P::RC, P::M2, LS>(v, xb, t);
    rf::pass_butterflies<P, P::RC, DIR>(v);
  }
}

// samples z[n], n = t + (N/16) e (zero beyond nphys), of a strided line -> lanes (z, z w_2N^n) -> both forward transforms
template <class P, int LS>
__device__ __forceinline__ void load_fwd(const float2* __restrict__ line, size_t stride, int nphys, float2 wt, C2* v, float4* xb,
                                         int t, const float2* __restrict__ tw) {
  static_assert(P::RA == 16 && P::E == 16, "sixteen points per thread at stride N/16 on the sample side");
#pragma unroll
  for (int e = 0; e < 16; ++e) {
    const int n = t + (P::N / 16) * e;
    const float2 z = n < nphys ? line[(size_t)n * stride] : make_float2(0.f, 0.f);
    const float2 zw = rf::cmul_tw1<-1>(z, rf::half_twiddle(wt, e));
    v[e] = {make_float2(z.x, zw.x), make_float2(z.y, zw.y)};
  }
  fft<P, -1, LS>(v, xb, t, tw);
}
// both inverse transforms -> first N samples: even part + conj(w)^n odd part -> strided line (n < nphys, if live)
template <class P, int LS>
__device__ __forceinline__ void inv_store(float2* __restrict__ line, size_t stride, int nphys, bool live, float2 wt, C2* v,
                                          float4* xb, int t, const float2* __restrict__ tw_r) {
  using PI = typename P::Reversed;
  static_assert(PI::RLAST == 16, "sixteen points per thread at stride N/16 on the sample side");
  fft<PI, +1, LS>(v, xb, t, tw_r);
#pragma unroll
  for (int e = 0; e < 16; ++e) {
    const int n = t + (P::N / 16) * e;
    const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), rf::half_twiddle(wt, e));
    if (live && n < nphys) line[(size_t)n * stride] = make_float2(v[e].re.x + u.x, v[e].im.x + u.y);
  }
}

}  // namespace f3

// ---------------------------------------------------------------------------------- y stage
// grid (kx tiles, z < Nz, component); block P::T * C threads; shared memory N * C float4
template <class P, int C, bool INV>
__global__ void __launch_bounds__(P::T * C) k3_y(Fast3DArgs a) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, g = tid % C, t = tid / C;
  const int kx = blockIdx.x * C + g;
  const bool live = kx < a.g.Cx;
  const size_t ps = (size_t)a.g.pitch;
  float2* __restrict__ line = a.spec + (size_t)blockIdx.z * a.cstride + (size_t)blockIdx.y * a.g.Py * ps + (live ? kx : a.g.Cx - 1);
  float4* xb = smem4 + g;
  const float2 wt = __ldg(&a.twoy[t]);
  rf::C2 v[E];
  if (!INV) {
    f3::load_fwd<P, C>(line, ps, a.g.Ny, wt, v, xb, t, a.twy);
    if (live) {
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const int j = rf::slot_index<P, P::RLAST>(t, e);            // lanes: bins 2j and 2j + 1
        line[(size_t)(2 * j) * ps] = make_float2(v[e].re.x, v[e].im.x);
        line[(size_t)(2 * j + 1) * ps] = make_float2(v[e].re.y, v[e].im.y);
      }
    }
  } else {
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int j = rf::slot_index<PI, PI::RA>(t, e);
      const float2 lo = line[(size_t)(2 * j) * ps], hi = line[(size_t)(2 * j + 1) * ps];
      v[e] = {make_float2(lo.x, hi.x), make_float2(lo.y, hi.y)};
    }
    f3::inv_store<P, C>(line, ps, a.g.Ny, live, wt, v, xb, t, a.twy_r);
  }
}

// ---------------------------------------------------------------------------------- z stage, fused
// index of kernel component (i, j) in K: xx, yy, zz, xy, xz, yz
__host__ __device__ constexpr int k3_comp(int i, int j) { return i == j ? i : (i + j == 1 ? 3 : (i + j == 2 ? 4 : 5)); }

// grid (kx tiles, Py); block 3 * P::T * C threads (component-major inside a point); shared memory N * 3C float4.
// blockIdx.y walks ky as 0, 1, Py-1, 2, Py-2, ..: a line and its mirror read the same kernel rows back to back.
template <class P, int C>
__global__ void __launch_bounds__(3 * P::T * C) k3_z(Fast3DArgs a) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E, LS = 3 * C;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, g = tid % C, comp = (tid / C) % 3, t = tid / LS;
  const int Py = a.g.Py, i = blockIdx.y;
  const int ky = i == 0 ? 0 : ((i & 1) ? (i + 1) / 2 : Py - i / 2);
  const int kyf = ky <= Py / 2 ? ky : Py - ky;
  const float sy = ky <= Py / 2 ? 1.f : -1.f;
  const int kx = blockIdx.x * C + g;
  const bool live = kx < a.g.Cx;
  const int kxc = live ? kx : a.g.Cx - 1;
  const size_t zs = (size_t)Py * a.g.pitch;
  float2* __restrict__ line = a.spec + (size_t)comp * a.cstride + (size_t)ky * a.g.pitch + kxc;
  float4* xb = smem4 + comp * C + g;
  const float2 wt = __ldg(&a.twoz[t]);
  rf::C2 v[E];
  f3::load_fwd<P, LS>(line, zs, a.g.Nz, wt, v, xb, t, a.twz);
  // hand the spectrum to the other two components of this line (same t, same slots)
  __syncthreads();
#pragma unroll
  for (int e = 0; e < E; ++e) xb[(size_t)rf::slot_index<P, P::RLAST>(t, e) * LS] = rf::pack(v[e]);
  __syncthreads();
  {
    const int o1 = (comp + 1) % 3, o2 = (comp + 2) % 3;
    const float4* x1 = smem4 + o1 * C + g;
    const float4* x2 = smem4 + o2 * C + g;
    // mirror signs: a component pair that contains y is odd under ky -> -ky, one that contains z under kz -> -kz
    const float y1 = (comp == 1 || o1 == 1) ? sy : 1.f, y2 = (comp == 1 || o2 == 1) ? sy : 1.f;
    const bool z1 = comp == 2 || o1 == 2, z2 = comp == 2 || o2 == 2;
    const float* __restrict__ K0 = a.K + (size_t)comp * a.kstride + (size_t)kyf * a.g.Cx + kxc;
    const float* __restrict__ K1 = a.K + (size_t)k3_comp(comp, o1) * a.kstride + (size_t)kyf * a.g.Cx + kxc;
    const float* __restrict__ K2 = a.K + (size_t)k3_comp(comp, o2) * a.kstride + (size_t)kyf * a.g.Cx + kxc;
    const size_t ks = (size_t)a.g.Hy * a.g.Cx;                      // stride of kz in K
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int j = rf::slot_index<P, P::RLAST>(t, e);
      const int b0 = 2 * j, b1 = 2 * j + 1;                         // bins of the two lanes; Pz / 2 = N
      const int f0 = b0 <= N ? b0 : 2 * N - b0, f1 = b1 <= N ? b1 : 2 * N - b1;
      const float s0 = b0 <= N ? 1.f : -1.f, s1 = b1 <= N ? 1.f : -1.f;
      const float2 kd = make_float2(__ldg(K0 + f0 * ks), __ldg(K0 + f1 * ks));
      float2 k1 = make_float2(__ldg(K1 + f0 * ks) * y1, __ldg(K1 + f1 * ks) * y1);
      float2 k2 = make_float2(__ldg(K2 + f0 * ks) * y2, __ldg(K2 + f1 * ks) * y2);
      if (z1) { k1.x *= s0; k1.y *= s1; }
      if (z2) { k2.x *= s0; k2.y *= s1; }
      const rf::C2 A = rf::unpack(x1[(size_t)j * LS]), B = rf::unpack(x2[(size_t)j * LS]);
      v[e].re = __ffma2_rn(k2, B.re, __ffma2_rn(k1, A.re, __fmul2_rn(kd, v[e].re)));
      v[e].im = __ffma2_rn(k2, B.im, __ffma2_rn(k1, A.im, __fmul2_rn(kd, v[e].im)));
    }
  }
  // (the first exchange of the inverse starts with a barrier: all reads of the handed-over spectra are done by then)
  f3::inv_store<P, LS>(line, zs, a.g.Nz, live, wt, v, xb, t, a.twz_r);
}
