// fast2d.cuh - demagnetising convolution of open-boundary 2D films with power-of-two sizes
// (Eq. 3; zero padding x2 per open axis L509; no z transform for one layer L531).
//
// A line of N samples zero-padded to 2N has its even bins = FFT_N(z[n]) and its odd bins =
// FFT_N(z[n] w^n), w = exp(-2 pi i / 2N); conversely the first N samples of the inverse are
// IFFT_N(even)[n] + conj(w)^n IFFT_N(odd)[n]. The two length-N transforms of a line run in
// lockstep in the two lanes of the packed-fp32 engine (fft_reg.cuh), so every line is read once,
// the padded half is never stored, read or transformed, and nothing is parked between halves.
//
//   K_A  k2_xfwd : rows -> x spectrum. Two real rows a, b form one complex line z = a + i b (one
//                  FFT group per row pair); the spectra of a and b are separated (Hermitian
//                  symmetry) on the way out and written TRANSPOSED, spec[c][kx][y], kx = 0..Nx.
//   K_B  k2_ycol : columns (kx fixed, all y; contiguous). XY job: two FFT groups take the x and the
//                  y component of one column, transform forward, swap spectra through shared memory,
//                  each forms its row of the 2x2 symmetric kernel product (K_xx K_xy; K_xy K_yy),
//                  transforms back, stores in place. Z job: one group per column, K_zz only
//                  (K_xz = K_yz = 0 for one layer).
//   K_C  k2_xinv : x spectrum -> rows of B_demag (only the Nx physical outputs are formed).
#pragma once
#include "common.cuh"
#include "fft_reg.cuh"
#include "demag_conv_args.cuh"

// pitch (float4 units) between the exchange buffers of consecutive FFT groups: XB plus a skew that
// spreads the G groups over the 8 16-byte bank groups when one quarter-warp touches several buffers
template <class P, int NT>
struct K2Shape {
  static constexpr int G = NT / P::T;
  static constexpr int GP = P::XB + (G >= 8 ? 1 : 8 / G);
};
template <class P, int NT>
constexpr size_t k2_smem() { return sizeof(float4) * (size_t)K2Shape<P, NT>::G * K2Shape<P, NT>::GP; }

// stage unit = (z0.re, z0.im, z1.re, z1.im): each lane's complex number is one 8-byte half
__device__ __forceinline__ float4 stage_pack(rf::C2 a) { return make_float4(a.re.x, a.im.x, a.re.y, a.im.y); }
__device__ __forceinline__ rf::C2 stage_unpack(float4 q) { return {make_float2(q.x, q.z), make_float2(q.y, q.w)}; }

// Hermitian separation of Z = A + iB (a, b real rows): from Z[k] and Z[-k] -> (A.re, A.im, B.re, B.im)
__device__ __forceinline__ float4 separate(float2 z, float2 zm) {
  return make_float4(0.5f * (z.x + zm.x), 0.5f * (z.y - zm.y), 0.5f * (z.y + zm.y), 0.5f * (zm.x - z.x));
}

// ---------------------------------------------------------------------------------- K_A
template <class P, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) k2_xfwd(Fast2DArgs a, int src_role) {
  if (a.st->skip) return;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T, GP = K2Shape<P, NT>::GP;
  extern __shared__ float4 smem4[];
  __shared__ float bsat_s[MM_MAX_REGIONS];
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float4* xb = smem4 + (size_t)gid * GP;
  const int c = blockIdx.y, r0 = blockIdx.x * 2 * G;
  const float* __restrict__ src = a.st->ptr[src_role] + (size_t)c * a.ncell;
  const uint8_t* __restrict__ reg = a.regions;
  const bool uniform = a.luts->nregions == 1;       // one region: B_sat is a constant
  const float b0 = a.luts->Bsat[0];
  if (!uniform) {
    for (int i = tid; i < MM_MAX_REGIONS; i += NT) bsat_s[i] = a.luts->Bsat[i];
    __syncthreads();
  }
  {
    const size_t rowA = (size_t)(r0 + 2 * gid) * N;
    rf::C2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<P, P::RA>(t, e);
      const size_t iA = rowA + n, iB = iA + N;
      const float sa = uniform ? b0 : bsat_s[reg[iA]], sb = uniform ? b0 : bsat_s[reg[iB]];
      const float2 z = make_float2(src[iA] * sa, src[iB] * sb);            // M = B_sat m (L121)
      const float2 zw = rf::cmul_tw1<-1>(z, __ldg(&a.twox[n]));
      v[e] = {make_float2(z.x, zw.x), make_float2(z.y, zw.y)};
    }
    rf::fft<P, -1, NT>(v, xb, t, gid, a.twx);
    rf::group_sync<T, NT>(gid);
#pragma unroll
    for (int e = 0; e < E; ++e) xb[rf::slot_index<P, P::RLAST>(t, e)] = stage_pack(v[e]);
  }
  __syncthreads();
  // separate the two real rows of every pair and store transposed: lane 0 holds bin kx = 2k,
  // lane 1 bin kx = 2k + 1 of the padded transform; stored kx = 0 .. N
  float2* __restrict__ out = a.spec + (size_t)c * a.cstride;
  for (int w = tid; w < (N / 2 + 1) * G; w += NT) {
    const int p = w % G, k = w / G;
    const float4* st = smem4 + (size_t)p * GP;
    const float2* st2 = reinterpret_cast<const float2*>(st);
    const float4 u = st[k];
    const float2 zm0 = st2[2 * ((N - k) & (N - 1))];
    float2* o = out + (size_t)(2 * k) * a.Ny + r0 + 2 * p;
    *reinterpret_cast<float4*>(o) = separate(make_float2(u.x, u.y), zm0);
    if (k < N / 2) {
      const float2 zm1 = st2[2 * (N - 1 - k) + 1];
      *reinterpret_cast<float4*>(o + a.Ny) = separate(make_float2(u.z, u.w), zm1);
    }
  }
}

// ---------------------------------------------------------------------------------- K_C
template <class P, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) k2_xinv(Fast2DArgs a, int dst_role) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T, GP = K2Shape<P, NT>::GP;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float4* xb = smem4 + (size_t)gid * GP;
  const int c = blockIdx.y, r0 = blockIdx.x * 2 * G;
  float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * a.ncell;
  const float2* __restrict__ in = a.spec + (size_t)c * a.cstride;
  // gather bins of the 2G rows; rebuild Z = A + iB and its Hermitian partner for both halves
  for (int w = tid; w < (N / 2 + 1) * G; w += NT) {
    const int p = w % G, k = w / G;
    float4* st = smem4 + (size_t)p * GP;
    float2* st2 = reinterpret_cast<float2*>(st);
    const float2* src = in + (size_t)(2 * k) * a.Ny + r0 + 2 * p;
    const float4 e = *reinterpret_cast<const float4*>(src);
    const float2 z0 = make_float2(e.x - e.w, e.y + e.z), zm0 = make_float2(e.x + e.w, e.z - e.y);
    if (k < N / 2) {
      const float4 o = *reinterpret_cast<const float4*>(src + a.Ny);
      const float2 z1 = make_float2(o.x - o.w, o.y + o.z), zm1 = make_float2(o.x + o.w, o.z - o.y);
      st[k] = make_float4(z0.x, z0.y, z1.x, z1.y);
      if (k > 0) st2[2 * (N - k)] = zm0;
      st2[2 * (N - 1 - k) + 1] = zm1;
    } else {
      st2[2 * k] = z0;            // k = N/2: its own partner; the odd half has no such bin
    }
  }
  __syncthreads();
  {
    rf::C2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = stage_unpack(xb[rf::slot_index<PI, PI::RA>(t, e)]);
    rf::fft<PI, +1, NT>(v, xb, t, gid, a.twx_r);
    const size_t rowA = (size_t)(r0 + 2 * gid) * N;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RLAST>(t, e);
      const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), __ldg(&a.twox[n]));
      dst[rowA + n] = v[e].re.x + u.x;
      dst[rowA + N + n] = v[e].im.x + u.y;
    }
  }
}

// ---------------------------------------------------------------------------------- K_B
// kernel-table index and mirror sign of bin j: lane 0 = even ky = 2j, lane 1 = odd ky = 2j + 1
template <int N>
__device__ __forceinline__ void k2_kidx(int j, int& i0, int& i1, float& s0, float& s1) {
  i0 = j <= N / 2 ? j : N - j;
  s0 = j > N / 2 ? -1.f : 1.f;
  i1 = N / 2 + 1 + (j < N / 2 ? j : N - 1 - j);
  s1 = j >= N / 2 ? -1.f : 1.f;
}

template <class P, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) k2_ycol(Fast2DArgs a, int nxy) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T, GP = K2Shape<P, NT>::GP;
  static_assert(G % 2 == 0, "XY jobs need an even number of FFT groups");
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float4* xb = smem4 + (size_t)gid * GP;
  const bool xy = (int)blockIdx.x < nxy;
  const int role = gid & 1;
  const int kx_raw = xy ? (int)blockIdx.x * (G / 2) + (gid >> 1) : ((int)blockIdx.x - nxy) * G + gid;
  const bool active = kx_raw < a.Cx;
  const int kx = active ? kx_raw : a.Cx - 1;       // idle groups shadow the last column, store nothing
  const int comp = xy ? role : 2;
  float2* __restrict__ s = a.spec + (size_t)comp * a.cstride + (size_t)kx * a.Ny;
  const float* __restrict__ Kc = a.Kt + (size_t)kx * (N + 1);
  rf::C2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int n = rf::slot_index<P, P::RA>(t, e);
    const float2 z = s[n];
    const float2 zw = rf::cmul_tw1<-1>(z, __ldg(&a.twoy[n]));
    v[e] = {make_float2(z.x, zw.x), make_float2(z.y, zw.y)};
  }
  rf::fft<P, -1, NT>(v, xb, t, gid, a.twy);
  if (xy) {
    // B~_x = K_xx M~_x + K_xy M~_y,  B~_y = K_xy M~_x + K_yy M~_y   (Eq. 3; K real, L145)
    rf::group_sync<T, NT>(gid);
#pragma unroll
    for (int e = 0; e < E; ++e) xb[e * T + t] = rf::pack(v[e]);
    __syncthreads();
    const float4* other = smem4 + (size_t)(gid ^ 1) * GP;
    const float* __restrict__ Kd = Kc + (size_t)role * a.kstride;
    const float* __restrict__ Ko = Kc + (size_t)3 * a.kstride;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      int i0, i1; float s0, s1;
      k2_kidx<N>(rf::slot_index<P, P::RLAST>(t, e), i0, i1, s0, s1);
      const float2 kd = make_float2(__ldg(&Kd[i0]), __ldg(&Kd[i1]));
      const float2 ko = make_float2(s0 * __ldg(&Ko[i0]), s1 * __ldg(&Ko[i1]));
      const rf::C2 o = rf::unpack(other[e * T + t]);
      v[e].re = __ffma2_rn(ko, o.re, __fmul2_rn(kd, v[e].re));
      v[e].im = __ffma2_rn(ko, o.im, __fmul2_rn(kd, v[e].im));
    }
    __syncthreads();
  } else {
    const float* __restrict__ Kz = Kc + (size_t)2 * a.kstride;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      int i0, i1; float s0, s1;
      k2_kidx<N>(rf::slot_index<P, P::RLAST>(t, e), i0, i1, s0, s1);
      const float2 kz = make_float2(__ldg(&Kz[i0]), __ldg(&Kz[i1]));
      v[e].re = __fmul2_rn(kz, v[e].re);
      v[e].im = __fmul2_rn(kz, v[e].im);
    }
  }
  rf::fft<PI, +1, NT>(v, xb, t, gid, a.twy_r);
  if (active) {
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RLAST>(t, e);
      const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), __ldg(&a.twoy[n]));
      s[n] = make_float2(v[e].re.x + u.x, v[e].im.x + u.y);
    }
  }
}
