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
//   k3_xfwd: rows -> x spectrum. Two real rows a, b form one complex line z = a + i b (lanes: even / odd bins of the
//            padded transform); the spectra of a and b are separated by Hermitian symmetry (partner values through
//            shared memory) and stored as rows spec[c][z][y][kx], kx = 0 .. Nx, 16 bytes (two bins) per store.
//   k3_xinv: x spectrum -> rows of B_demag (only the Nx physical outputs are formed).
//   k3_y   : y forward (rows y < Ny -> bins ky < 2Ny) or y inverse (bins -> rows), in place, one component
//   k3_z   : z forward of the three components, product with the six-component real symmetric kernel spectrum
//            (Eq. 3; K real and even/odd under the mirrors, L145), z inverse; in place, only the Nz physical layers
//            are stored. The three components of a line are three thread groups that hand their spectra to one
//            another through the exchange buffer, so nothing is parked and each thread forms one output component.
#pragma once
#include "common.cuh"
#include "fft_reg.cuh"
#include "tma_util.cuh"
#include <type_traits>
#include "demag_conv_args.cuh"

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

// ---- rows: the T threads of a line are neighbours (coalesced 4-byte accesses along x); one padded buffer per line
__device__ __forceinline__ int xp(int a) { return a + (a >> 4); }
template <class P> __host__ __device__ constexpr int row_pitch() { return P::N + P::N / 16 + 1; }      // float4 units, odd

template <class P, int R, int RN, int MP>
__device__ __forceinline__ void exchange_rows(C2* v, float4* xb, int t) {
  constexpr int MN = MP / RN;
  static_assert(P::T % MN == 0, "threads of a line must cover whole butterflies of the next pass");
  const int rbase = (t / MN) * MP + (t % MN);
  constexpr int RB_STEP = (P::T / MN) * MP;
  __syncthreads();
#pragma unroll
  for (int b = 0; b < P::E / R; ++b)
#pragma unroll
    for (int s = 0; s < R; ++s) xb[xp(t + P::T * b + (P::N / R) * s)] = rf::pack(v[b * R + s]);
  __syncthreads();
#pragma unroll
  for (int b = 0; b < P::E / RN; ++b)
#pragma unroll
    for (int s = 0; s < RN; ++s) v[b * RN + s] = rf::unpack(xb[xp(rbase + RB_STEP * b + s * MN)]);
}
template <class P, int DIR>
__device__ __forceinline__ void fft_rows(C2* v, float4* xb, int t, const float2* __restrict__ tw) {
  rf::pass_butterflies<P, P::RA, DIR>(v);
  {
    float2 w[(P::RA - 1) * (P::E / P::RA)];
    rf::load_twiddles<P, P::RA>(w, t, tw);
    rf::apply_twiddles<P, P::RA, DIR>(v, w);
  }
  exchange_rows<P, P::RA, P::RB, P::M1>(v, xb, t);
  rf::pass_butterflies<P, P::RB, DIR>(v);
  if constexpr (P::NPASS == 3) {
    {
      float2 w[(P::RB - 1) * (P::E / P::RB)];
      rf::load_twiddles<P, P::RB>(w, t, tw + P::TW1);
      rf::apply_twiddles<P, P::RB, DIR>(v, w);
    }
    exchange_rows<P, P::RB, P::RC, P::M2>(v, xb, t);
    rf::pass_butterflies<P, P::RC, DIR>(v);
  }
}

__device__ __forceinline__ float ldg_f(const float* p) {
  float v;
  asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void stg_f(float* p, float v) { asm volatile("st.global.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }

}  // namespace f3

// ---------------------------------------------------------------------------------- x stage
// grid (row pairs / G, component); block G * P::T threads (t fastest); shared memory G * row_pitch float4.
// (The forward kernel waits mostly on its row loads: three CTAs per SM at 80 registers beat two at 96, 0.276 -> 0.222 ms
// at 256^3; the same bound makes the inverse kernel and the y stage slower.)
template <class P, int G>
__global__ void __launch_bounds__(P::T * G, 3) k3_xfwd(Fast3DArgs a, int src_role) {
  if (a.st->skip) return;
  constexpr int N = P::N, T = P::T, E = P::E;
  static_assert(P::RA == 16 && E == 16, "sixteen points per thread at stride N/16 on the sample side");
  extern __shared__ float4 smem4[];
  __shared__ float bsat_s[MM_MAX_REGIONS];
  const int tid = threadIdx.x, t = tid % T, gi = tid / T;
  const int c = blockIdx.y;
  const int pair = blockIdx.x * G + gi, npairs = a.g.Ny * a.g.Nz / 2;      // Ny is even: a pair never straddles z
  const bool live = pair < npairs;
  const int r0 = 2 * (live ? pair : 0);                                      // flattened (z, y) row index
  const int z = r0 / a.g.Ny, y = r0 - z * a.g.Ny;
  float4* xb = smem4 + (size_t)gi * f3::row_pitch<P>();
  const bool uniform = a.luts->nregions == 1;
  const float b0 = a.luts->Bsat[0];
  if (!uniform) {
    for (int i = tid; i < MM_MAX_REGIONS; i += T * G) bsat_s[i] = a.luts->Bsat[i];
    __syncthreads();
  }
  const float* __restrict__ src = a.st->ptr[src_role] + (size_t)c * a.g.N + (size_t)r0 * a.g.Nx;
  const uint8_t* __restrict__ reg = a.regions + (size_t)r0 * a.g.Nx;
  const float2 wt = __ldg(&a.twox[t]);
  rf::C2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int n = t + (N / 16) * e;
    float2 zz = make_float2(0.f, 0.f);                      // M = B_sat m (L121); zero beyond the box (L509)
    if (n < a.g.Nx) {
      zz.x = f3::ldg_f(src + n) * (uniform ? b0 : bsat_s[reg[n]]);
      zz.y = f3::ldg_f(src + a.g.Nx + n) * (uniform ? b0 : bsat_s[reg[a.g.Nx + n]]);
    }
    const float2 zw = rf::cmul_tw1<-1>(zz, rf::half_twiddle(wt, e));
    v[e] = {make_float2(zz.x, zw.x), make_float2(zz.y, zw.y)};
  }
  f3::fft_rows<P, -1>(v, xb, t, a.twx);
  // Hermitian separation: partner of even bin 2j is even bin 2((N - j) mod N), of odd bin 2j + 1 odd bin 2(N - 1 - j) + 1
  __syncthreads();
#pragma unroll
  for (int e = 0; e < E; ++e)
    xb[f3::xp(rf::slot_index<P, P::RLAST>(t, e))] = make_float4(v[e].re.x, v[e].im.x, v[e].re.y, v[e].im.y);
  __syncthreads();
  if (!live) return;
  float2* __restrict__ outA = a.spec + (size_t)c * a.cstride + ((size_t)z * a.g.Py + y) * a.g.pitch;
  float2* __restrict__ outB = outA + a.g.pitch;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int j = rf::slot_index<P, P::RLAST>(t, e);
    if (j > N / 2) continue;                                 // bins above Nx are the mirror images
    const float4 pe = xb[f3::xp((N - j) & (N - 1))], po = xb[f3::xp(N - 1 - j)];
    const float2 ze = make_float2(v[e].re.x, v[e].im.x), zo = make_float2(v[e].re.y, v[e].im.y);
    // A = (Z[k] + conj Z[-k]) / 2, B = (Z[k] - conj Z[-k]) / 2i
    const float4 A = make_float4(0.5f * (ze.x + pe.x), 0.5f * (ze.y - pe.y), 0.5f * (zo.x + po.z), 0.5f * (zo.y - po.w));
    const float4 B = make_float4(0.5f * (ze.y + pe.y), 0.5f * (pe.x - ze.x), 0.5f * (zo.y + po.w), 0.5f * (po.z - zo.x));
    // bins 2j and 2j + 1 side by side (for j = N/2 the second one falls in the padding of the pitch)
    *reinterpret_cast<float4*>(outA + 2 * j) = A;
    *reinterpret_cast<float4*>(outB + 2 * j) = B;
  }
}

template <class P, int G>
__global__ void __launch_bounds__(P::T * G) k3_xinv(Fast3DArgs a, int dst_role) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E;
  static_assert(PI::RLAST == 16, "sixteen points per thread at stride N/16 on the sample side");
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, t = tid % T, gi = tid / T;
  const int c = blockIdx.y;
  const int pair = blockIdx.x * G + gi, npairs = a.g.Ny * a.g.Nz / 2;
  const bool live = pair < npairs;
  const int r0 = 2 * (live ? pair : 0);
  const int z = r0 / a.g.Ny, y = r0 - z * a.g.Ny;
  float4* xb = smem4 + (size_t)gi * f3::row_pitch<P>();
  const float2* __restrict__ inA = a.spec + (size_t)c * a.cstride + ((size_t)z * a.g.Py + y) * a.g.pitch;
  const float2* __restrict__ inB = inA + a.g.pitch;
  const float2 wt = __ldg(&a.twox[t]);
  rf::C2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    // point j of the even-bin transform is Z[2j], of the odd-bin one Z[2j + 1]; Z[b] = A[b] + i B[b] for b <= N,
    // conj(A[2N - b]) + i conj(B[2N - b]) above
    const int j = rf::slot_index<PI, PI::RA>(t, e);
    if (2 * j + 1 <= N) {
      const float4 A = *reinterpret_cast<const float4*>(inA + 2 * j), B = *reinterpret_cast<const float4*>(inB + 2 * j);
      v[e] = {make_float2(A.x - B.y, A.z - B.w), make_float2(A.y + B.x, A.w + B.z)};
    } else if (2 * j == N) {
      const float2 A0 = inA[N], B0 = inB[N], A1 = inA[N - 1], B1 = inB[N - 1];      // bin N itself; bin N + 1 -> N - 1
      v[e] = {make_float2(A0.x - B0.y, A1.x + B1.y), make_float2(A0.y + B0.x, B1.x - A1.y)};
    } else {
      const float2 A0 = inA[2 * N - 2 * j], B0 = inB[2 * N - 2 * j], A1 = inA[2 * N - 2 * j - 1], B1 = inB[2 * N - 2 * j - 1];
      v[e] = {make_float2(A0.x + B0.y, A1.x + B1.y), make_float2(B0.x - A0.y, B1.x - A1.y)};
    }
  }
  f3::fft_rows<PI, +1>(v, xb, t, a.twx_r);
  if (!live) return;
  float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * a.g.N + (size_t)r0 * a.g.Nx;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int n = t + (N / 16) * e;
    const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), rf::half_twiddle(wt, e));
    if (n < a.g.Nx) {
      f3::stg_f(dst + n, v[e].re.x + u.x);
      f3::stg_f(dst + a.g.Nx + n, v[e].im.x + u.y);
    }
  }
}

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

// ---------------------------------------------------------------------------------- periodic axes
// A periodic axis is not padded (the images are folded into the kernel): a plain N-point
// transform per line. The two lanes of the packed engine then carry two different lines.
//
// y stage, periodic: lanes = the lines at kx and kx + 1 (one 16-byte access per point). grid (kx pair tiles, z, c)
template <class P, int C, bool INV>
__global__ void __launch_bounds__(P::T * C) k3_yp(Fast3DArgs a) {
  if (a.st->skip) return;
  using PL = typename std::conditional<INV, typename P::Reversed, P>::type;
  constexpr int T = P::T, E = P::E;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, g = tid % C, t = tid / C;
  const int kx = 2 * (blockIdx.x * C + g);
  const bool live = kx < a.g.Cx;                          // (kx + 1 may be a padding column of the pitch: harmless)
  const size_t ps = (size_t)a.g.pitch;
  float2* __restrict__ line = a.spec + (size_t)blockIdx.z * a.cstride + (size_t)blockIdx.y * a.g.Py * ps + (live ? kx : 0);
  rf::C2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const float4 q = *reinterpret_cast<const float4*>(line + (size_t)rf::slot_index<PL, PL::RA>(t, e) * ps);
    v[e] = {make_float2(q.x, q.z), make_float2(q.y, q.w)};
  }
  f3::fft<PL, INV ? +1 : -1, C>(v, smem4 + g, t, INV ? a.twy_r : a.twy);
  if (live) {
#pragma unroll
    for (int e = 0; e < E; ++e)
      *reinterpret_cast<float4*>(line + (size_t)rf::slot_index<PL, PL::RLAST>(t, e) * ps) =
          make_float4(v[e].re.x, v[e].im.x, v[e].re.y, v[e].im.y);
  }
}

// x stage, periodic: four real rows per line group - lanes = the complex lines (r, r+1) and (r+2, r+3); N-point
// transform, Hermitian separation (partner of bin j is bin (N - j) mod N), bins 0 .. N/2 stored.
template <class P, int G>
__global__ void __launch_bounds__(P::T * G) k3_xfwd_p(Fast3DArgs a, int src_role) {
  if (a.st->skip) return;
  constexpr int N = P::N, T = P::T, E = P::E;
  extern __shared__ float4 smem4[];
  __shared__ float bsat_s[MM_MAX_REGIONS];
  const int tid = threadIdx.x, t = tid % T, gi = tid / T;
  const int c = blockIdx.y;
  const int quad = blockIdx.x * G + gi, nquads = a.g.Ny * a.g.Nz / 4;       // Ny is a multiple of 4
  const bool live = quad < nquads;
  const int r0 = 4 * (live ? quad : 0);
  const int z = r0 / a.g.Ny, y = r0 - z * a.g.Ny;
  float4* xb = smem4 + (size_t)gi * f3::row_pitch<P>();
  const bool uniform = a.luts->nregions == 1;
  const float b0 = a.luts->Bsat[0];
  if (!uniform) {
    for (int i = tid; i < MM_MAX_REGIONS; i += T * G) bsat_s[i] = a.luts->Bsat[i];
    __syncthreads();
  }
  const int nx = a.g.Nx;
  const float* __restrict__ src = a.st->ptr[src_role] + (size_t)c * a.g.N + (size_t)r0 * nx;
  const uint8_t* __restrict__ reg = a.regions + (size_t)r0 * nx;
  rf::C2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int n = rf::slot_index<P, P::RA>(t, e);
    float q[4];
#pragma unroll
    for (int r = 0; r < 4; ++r) q[r] = f3::ldg_f(src + (size_t)r * nx + n) * (uniform ? b0 : bsat_s[reg[(size_t)r * nx + n]]);
    v[e] = {make_float2(q[0], q[2]), make_float2(q[1], q[3])};
  }
  f3::fft_rows<P, -1>(v, xb, t, a.twx);
  __syncthreads();
#pragma unroll
  for (int e = 0; e < E; ++e)
    xb[f3::xp(rf::slot_index<P, P::RLAST>(t, e))] = make_float4(v[e].re.x, v[e].im.x, v[e].re.y, v[e].im.y);
  __syncthreads();
  if (!live) return;
  float2* __restrict__ out = a.spec + (size_t)c * a.cstride + ((size_t)z * a.g.Py + y) * a.g.pitch;
  const size_t ps = (size_t)a.g.pitch;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int j = rf::slot_index<P, P::RLAST>(t, e);
    if (j > N / 2) continue;
    const float4 p = xb[f3::xp((N - j) & (N - 1))];
    const float2 z0 = make_float2(v[e].re.x, v[e].im.x), z1 = make_float2(v[e].re.y, v[e].im.y);
    out[j] = make_float2(0.5f * (z0.x + p.x), 0.5f * (z0.y - p.y));
    out[ps + j] = make_float2(0.5f * (z0.y + p.y), 0.5f * (p.x - z0.x));
    out[2 * ps + j] = make_float2(0.5f * (z1.x + p.z), 0.5f * (z1.y - p.w));
    out[3 * ps + j] = make_float2(0.5f * (z1.y + p.w), 0.5f * (p.z - z1.x));
  }
}

template <class P, int G>
__global__ void __launch_bounds__(P::T * G) k3_xinv_p(Fast3DArgs a, int dst_role) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, t = tid % T, gi = tid / T;
  const int c = blockIdx.y;
  const int quad = blockIdx.x * G + gi, nquads = a.g.Ny * a.g.Nz / 4;
  const bool live = quad < nquads;
  const int r0 = 4 * (live ? quad : 0);
  const int z = r0 / a.g.Ny, y = r0 - z * a.g.Ny;
  float4* xb = smem4 + (size_t)gi * f3::row_pitch<P>();
  const float2* __restrict__ in = a.spec + (size_t)c * a.cstride + ((size_t)z * a.g.Py + y) * a.g.pitch;
  const size_t ps = (size_t)a.g.pitch;
  rf::C2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int j = rf::slot_index<PI, PI::RA>(t, e);
    const bool dir = j <= N / 2;                            // Z[j] = A[j] + i B[j]; above N/2: conj(A[N-j]) + i conj(B[N-j])
    const int k = dir ? j : N - j;
    const float2 A0 = in[k], B0 = in[ps + k], A1 = in[2 * ps + k], B1 = in[3 * ps + k];
    if (dir) v[e] = {make_float2(A0.x - B0.y, A1.x - B1.y), make_float2(A0.y + B0.x, A1.y + B1.x)};
    else v[e] = {make_float2(A0.x + B0.y, A1.x + B1.y), make_float2(B0.x - A0.y, B1.x - A1.y)};
  }
  f3::fft_rows<PI, +1>(v, xb, t, a.twx_r);
  if (!live) return;
  const int nx = a.g.Nx;
  float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * a.g.N + (size_t)r0 * nx;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int n = rf::slot_index<PI, PI::RLAST>(t, e);
    f3::stg_f(dst + n, v[e].re.x);
    f3::stg_f(dst + nx + n, v[e].im.x);
    f3::stg_f(dst + 2 * (size_t)nx + n, v[e].re.y);
    f3::stg_f(dst + 3 * (size_t)nx + n, v[e].im.y);
  }
}

// ---------------------------------------------------------------------------------- z stage, fused
// index of kernel component (i, j) in K: xx, yy, zz, xy, xz, yz
__host__ __device__ constexpr int k3_comp(int i, int j) { return i == j ? i : (i + j == 1 ? 3 : (i + j == 2 ? 4 : 5)); }

// grid (kx tiles, Py); block 3 * P::T * C threads (component-major inside a point); shared memory: N * 3C float4 of
// exchange buffers + the kernel tile 6 (N + 1) C floats, which one bulk copy brings in while the forward transforms
// run. blockIdx.y walks ky as 0, 1, Py-1, 2, Py-2, ..: a line and its mirror read the same kernel tile back to back.
template <class P, int C>
struct K3Z {
  static constexpr int KT = 6 * (P::N + 1) * C;                       // floats of one kernel tile
  static constexpr size_t XB_BYTES = sizeof(float4) * (size_t)P::N * 3 * C;
  static constexpr size_t SMEM = XB_BYTES + sizeof(float) * KT + 16;
};

template <class P, int C, int MINB>
__global__ void __launch_bounds__(3 * P::T * C, MINB) k3_z(Fast3DArgs a) {
  if (a.st->skip) return;
  constexpr int N = P::N, T = P::T, E = P::E, LS = 3 * C;
  extern __shared__ __align__(16) float4 smem4[];
  __shared__ __align__(8) uint64_t kfull;
  float* ksm = reinterpret_cast<float*>(reinterpret_cast<char*>(smem4) + K3Z<P, C>::XB_BYTES);
  const int tid = threadIdx.x, g = tid % C, comp = (tid / C) % 3, t = tid / LS;
  const int Py = a.g.Py, i = blockIdx.y;
  const int ky = i == 0 ? 0 : ((i & 1) ? (i + 1) / 2 : Py - i / 2);
  const int kyf = ky <= Py / 2 ? ky : Py - ky;
  const float sy = ky <= Py / 2 ? 1.f : -1.f;
  if (tid == 0) {
    tma::mbar_init(&kfull, 1);
    tma::fence_barrier_init();
    tma::fence_proxy_async();
    constexpr uint32_t bytes = sizeof(float) * K3Z<P, C>::KT;
    tma::mbar_expect_tx(&kfull, bytes);
    tma::bulk_load(ksm, a.K3 + ((size_t)kyf * gridDim.x + blockIdx.x) * K3Z<P, C>::KT, bytes, &kfull);
  }
  const int kx = blockIdx.x * C + g;
  const bool live = kx < a.g.Cx;
  const int kxc = live ? kx : a.g.Cx - 1;
  const size_t zs = (size_t)Py * a.g.pitch;
  float2* __restrict__ line = a.spec + (size_t)comp * a.cstride + (size_t)ky * a.g.pitch + kxc;
  float4* xb = smem4 + comp * C + g;
  const float2 wt = __ldg(&a.twoz[t]);
  rf::C2 v[E];
  f3::load_fwd<P, LS>(line, zs, a.g.Nz, wt, v, xb, t, a.twz);      // (its barriers also publish the mbarrier's initialisation)
  // hand the spectrum to the other two components of this line (same t, same slots)
  __syncthreads();
#pragma unroll
  for (int e = 0; e < E; ++e) xb[(size_t)rf::slot_index<P, P::RLAST>(t, e) * LS] = rf::pack(v[e]);
  __syncthreads();
  tma::mbar_wait(&kfull, 0);
  {
    const int o1 = (comp + 1) % 3, o2 = (comp + 2) % 3;
    const float4* x1 = smem4 + o1 * C + g;
    const float4* x2 = smem4 + o2 * C + g;
    // mirror signs: a component pair that contains y is odd under ky -> -ky, one that contains z under kz -> -kz
    const float y1 = (comp == 1 || o1 == 1) ? sy : 1.f, y2 = (comp == 1 || o2 == 1) ? sy : 1.f;
    const bool z1 = comp == 2 || o1 == 2, z2 = comp == 2 || o2 == 2;
    const float* K0 = ksm + (size_t)comp * (N + 1) * C + g;
    const float* K1 = ksm + (size_t)k3_comp(comp, o1) * (N + 1) * C + g;
    const float* K2 = ksm + (size_t)k3_comp(comp, o2) * (N + 1) * C + g;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int j = rf::slot_index<P, P::RLAST>(t, e);
      const int b0 = 2 * j, b1 = 2 * j + 1;                         // bins of the two lanes; Pz / 2 = N
      const int f0 = b0 <= N ? b0 : 2 * N - b0, f1 = b1 <= N ? b1 : 2 * N - b1;
      const float s0 = b0 <= N ? 1.f : -1.f, s1 = b1 <= N ? 1.f : -1.f;
      const float2 kd = make_float2(K0[f0 * C], K0[f1 * C]);
      float2 k1 = make_float2(K1[f0 * C] * y1, K1[f1 * C] * y1);
      float2 k2 = make_float2(K2[f0 * C] * y2, K2[f1 * C] * y2);
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

// the kernel spectrum in the tile order of k3_z (see Fast3DArgs::K3), from the generic layout K[6][Hz][Hy][Cx]
__global__ void k3_pack_kernel(const float* __restrict__ K, float* __restrict__ K3, int Cx, int Hy, int Hz, int C, int ntiles) {
  const long long kstride = (long long)Cx * Hy * Hz, total = (long long)Hy * ntiles * 6 * Hz * C;
  for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (long long)gridDim.x * blockDim.x) {
    const int g = (int)(o % C);
    long long r = o / C;
    const int kf = (int)(r % Hz); r /= Hz;
    const int comp = (int)(r % 6); r /= 6;
    const int tile = (int)(r % ntiles);
    const int kyf = (int)(r / ntiles);
    const int kx = tile * C + g;
    K3[o] = kx < Cx ? K[comp * kstride + ((long long)kf * Hy + kyf) * Cx + kx] : 0.f;
  }
}
