// fast2d.cuh - demagnetising convolution of open-boundary 2D films with power-of-two sizes
// (Eq. 3; zero padding x2 per open axis L509; no z transform for one layer L531).
//
//   K_A  k2_xfwd : rows -> x spectrum. Two real rows a, b are transformed as one complex line
//                  z = a + i b of padded length 2Nx whose upper half is zero, so the even and the odd
//                  bins are two independent length-Nx transforms (of z[n] and of z[n] w^n); the
//                  spectra of a and b are separated (Hermitian symmetry) on the way out and written
//                  TRANSPOSED, spec[c][kx][y], in 64-byte pieces (8 rows per CTA).
//   K_B  k2_ycol : one contiguous column (kx fixed, all y) per FFT group. Padded length 2Ny, input
//                  half zero, only Ny outputs wanted: even / odd bins again decouple into
//                  length-Ny forward transform -> multiply by the real symmetric kernel spectrum
//                  -> length-Ny inverse; out = inv_even + conj(w)^n inv_odd. In place.
//   K_C  k2_xinv : x spectrum -> rows of B_demag (only the Nx physical outputs are formed).
// The padded halves are never stored, read or transformed.
#pragma once
#include "common.cuh"
#include "fft_reg.cuh"
#include "demag_conv_args.cuh"


constexpr int kStagePad = 8;   // stage row pitch = N + 8 float2: conflict-free separation reads

template <class P, int NT, int RG>
constexpr size_t k2_x_smem() {
  return sizeof(float2) * ((size_t)(RG / 2) * (P::N + kStagePad) + (size_t)(NT / P::T) * P::XB);
}
template <class P, int NT>
constexpr size_t k2_y_smem() {
  return sizeof(float2) * ((size_t)(NT / P::T) * P::XB + (size_t)2 * (NT / P::T) * P::N);
}

// ---------------------------------------------------------------------------------- K_A
template <class P, int NT, int RG>
__global__ void __launch_bounds__(NT) k2_xfwd(Fast2DArgs a, int src_role) {
  if (a.st->skip) return;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T, NPAIR = RG / 2, SP = N + kStagePad;
  static_assert(NPAIR % G == 0, "pairs must divide evenly over the FFT groups");
  extern __shared__ float2 smem[];
  __shared__ float bsat_s[MM_MAX_REGIONS];
  float2* stage = smem;
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float2* xb = smem + (size_t)NPAIR * SP + (size_t)gid * P::XB;
  const int c = blockIdx.y, r0 = blockIdx.x * RG;
  const float* __restrict__ src = a.st->ptr[src_role] + (size_t)c * a.ncell;
  const uint8_t* __restrict__ reg = a.regions;
  for (int i = tid; i < MM_MAX_REGIONS; i += NT) bsat_s[i] = a.luts->Bsat[i];
  __syncthreads();
  float2* __restrict__ out = a.spec + (size_t)c * a.cstride;
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
#pragma unroll 1
    for (int p = gid; p < NPAIR; p += G) {
      const size_t rowA = (size_t)(r0 + 2 * p) * N;
      float2 v[E];
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const int n = rf::slot_index<P, P::RA>(t, e);
        const size_t iA = rowA + n, iB = iA + N;
        v[e] = make_float2(src[iA] * bsat_s[reg[iA]], src[iB] * bsat_s[reg[iB]]);
      }
      if (h) {
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = rf::cmul_tw<-1>(v[e], __ldg(&a.twox[rf::slot_index<P, P::RA>(t, e)]));
      }
      rf::fft<P, -1, NT>(v, xb, t, gid, a.twx);
#pragma unroll
      for (int e = 0; e < E; ++e) stage[p * SP + rf::slot_index<P, P::RLAST>(t, e)] = v[e];
    }
    __syncthreads();
    // separate the two real rows of every pair and store transposed: bins kx = 2k + h
    const int nk = h ? N / 2 : N / 2 + 1;
    const int nkc = (nk + 7) / 8;
    for (int w = tid; w < nkc * 8 * NPAIR; w += NT) {
      const int kl = w & 7, p = (w >> 3) % NPAIR, k = (w / (8 * NPAIR)) * 8 + kl;
      if (k >= nk) continue;
      const int kp = h ? N - 1 - k : (N - k) & (N - 1);
      const float2 z = stage[p * SP + k], zm = stage[p * SP + kp];
      const float4 ab = make_float4(0.5f * (z.x + zm.x), 0.5f * (z.y - zm.y), 0.5f * (z.y + zm.y), 0.5f * (zm.x - z.x));
      *reinterpret_cast<float4*>(out + (size_t)(2 * k + h) * a.Ny + r0 + 2 * p) = ab;
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------- K_C
template <class P, int NT, int RG>
__global__ void __launch_bounds__(NT) k2_xinv(Fast2DArgs a, int dst_role) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T, NPAIR = RG / 2, SP = N + kStagePad;
  extern __shared__ float2 smem[];
  float2* stage = smem;
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float2* xb = smem + (size_t)NPAIR * SP + (size_t)gid * P::XB;
  const int c = blockIdx.y, r0 = blockIdx.x * RG;
  float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * a.ncell;
  const float2* __restrict__ in = a.spec + (size_t)c * a.cstride;
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {
    // gather bins kx = 2k + h of the RG rows; rebuild Z = A + iB and its Hermitian partner
    const int nk = h ? N / 2 : N / 2 + 1;
    const int nkc = (nk + 7) / 8;
    for (int w = tid; w < nkc * 8 * NPAIR; w += NT) {
      const int kl = w & 7, p = (w >> 3) % NPAIR, k = (w / (8 * NPAIR)) * 8 + kl;
      if (k >= nk) continue;
      const int kp = h ? N - 1 - k : (N - k) & (N - 1);
      const float4 ab = *reinterpret_cast<const float4*>(in + (size_t)(2 * k + h) * a.Ny + r0 + 2 * p);
      stage[p * SP + k] = make_float2(ab.x - ab.w, ab.y + ab.z);
      if (kp != k) stage[p * SP + kp] = make_float2(ab.x + ab.w, ab.z - ab.y);
    }
    __syncthreads();
#pragma unroll 1
    for (int p = gid; p < NPAIR; p += G) {
      float2 v[E];
#pragma unroll
      for (int e = 0; e < E; ++e) v[e] = stage[p * SP + rf::slot_index<PI, PI::RA>(t, e)];
      rf::fft<PI, +1, NT>(v, xb, t, gid, a.twx_r);
      const size_t rowA = (size_t)(r0 + 2 * p) * N;
#pragma unroll
      for (int e = 0; e < E; ++e) {
        const int n = rf::slot_index<PI, PI::RLAST>(t, e);
        if (h == 0) {
          dst[rowA + n] = v[e].x;
          dst[rowA + N + n] = v[e].y;
        } else {
          const float2 u = rf::cmul_tw<+1>(v[e], __ldg(&a.twox[n]));
          dst[rowA + n] += u.x;
          dst[rowA + N + n] += u.y;
        }
      }
    }
    __syncthreads();
  }
}

// ---------------------------------------------------------------------------------- K_B
template <class P, int NT>
__global__ void __launch_bounds__(NT) k2_ycol(Fast2DArgs a) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T;
  extern __shared__ float2 smem[];
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float2* xb = smem + (size_t)gid * P::XB;
  float2* park = smem + (size_t)G * P::XB + (size_t)gid * 2 * N;
  const int kx = blockIdx.x * G + gid;
  if (kx >= a.Cx) return;                       // whole group leaves: group barriers stay consistent
  const size_t col = (size_t)kx * a.Ny;
  const float* __restrict__ Kc = a.Kt + (size_t)kx * (N + 1);

  auto load_fwd = [&](int c, int h, float2* v) {
    const float2* __restrict__ s = a.spec + (size_t)c * a.cstride + col;
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = s[rf::slot_index<P, P::RA>(t, e)];
    if (h) {
#pragma unroll
      for (int e = 0; e < E; ++e) v[e] = rf::cmul_tw<-1>(v[e], __ldg(&a.twoy[rf::slot_index<P, P::RA>(t, e)]));
    }
    rf::fft<P, -1, NT>(v, xb, t, gid, a.twy);
  };
  auto inv_out = [&](int c, int h, float2* v, float2* pk) {
    rf::fft<PI, +1, NT>(v, xb, t, gid, a.twy_r);
    float2* __restrict__ d = a.spec + (size_t)c * a.cstride + col;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RLAST>(t, e);
      if (h == 0) pk[n] = v[e];
      else d[n] = rf::cadd(pk[n], rf::cmul_tw<+1>(v[e], __ldg(&a.twoy[n])));
    }
  };
  // kernel table index and mirror sign of bin j of half h
  auto kidx = [&](int h, int j, float& sg) {
    if (h == 0) { sg = j > N / 2 ? -1.f : 1.f; return j <= N / 2 ? j : N - j; }
    sg = j >= N / 2 ? -1.f : 1.f;
    return N / 2 + 1 + (j < N / 2 ? j : N - 1 - j);
  };

#pragma unroll 1
  for (int h = 0; h < 2; ++h) {       // components x, y: coupled by K_xx, K_xy, K_yy
    float2 vx[E], vy[E];
    load_fwd(0, h, vx);
    load_fwd(1, h, vy);
#pragma unroll
    for (int e = 0; e < E; ++e) {
      float sg;
      const int i = kidx(h, rf::slot_index<P, P::RLAST>(t, e), sg);
      const float kxx = __ldg(&Kc[i]), kyy = __ldg(&Kc[a.kstride + i]), kxy = sg * __ldg(&Kc[3 * a.kstride + i]);
      const float2 mx = vx[e], my = vy[e];
      vx[e] = make_float2(kxx * mx.x + kxy * my.x, kxx * mx.y + kxy * my.y);
      vy[e] = make_float2(kxy * mx.x + kyy * my.x, kxy * mx.y + kyy * my.y);
    }
    inv_out(0, h, vx, park);
    inv_out(1, h, vy, park + N);
  }
#pragma unroll 1
  for (int h = 0; h < 2; ++h) {       // component z: K_zz only (K_xz = K_yz = 0 for one layer)
    float2 vz[E];
    load_fwd(2, h, vz);
#pragma unroll
    for (int e = 0; e < E; ++e) {
      float sg;
      const int i = kidx(h, rf::slot_index<P, P::RLAST>(t, e), sg);
      const float kzz = __ldg(&Kc[2 * a.kstride + i]);
      vz[e] = make_float2(kzz * vz[e].x, kzz * vz[e].y);
    }
    inv_out(2, h, vz, park);
  }
}
