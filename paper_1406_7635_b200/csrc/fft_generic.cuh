// fft_generic.cuh - generic in-shared-memory Stockham FFT (any P = 2^a 3^b 5^c), the fallback
// engine of the demag convolution ("FFT-accelerated based on the ... convolution
// theorem"). Always the forward transform exp(-2 pi i jk/P); callers get the inverse by
// conjugating on load and store.
#pragma once
#include "common.cuh"

template <int R>
__device__ __forceinline__ void dft_small(float2* v);

template <>
__device__ __forceinline__ void dft_small<2>(float2* v) {
  float2 a = v[0], b = v[1];
  v[0] = make_float2(a.x + b.x, a.y + b.y);
  v[1] = make_float2(a.x - b.x, a.y - b.y);
}

template <>
__device__ __forceinline__ void dft_small<4>(float2* v) {
  float2 t0 = make_float2(v[0].x + v[2].x, v[0].y + v[2].y);
  float2 t1 = make_float2(v[0].x - v[2].x, v[0].y - v[2].y);
  float2 t2 = make_float2(v[1].x + v[3].x, v[1].y + v[3].y);
  float2 d = make_float2(v[1].x - v[3].x, v[1].y - v[3].y);
  float2 t3 = make_float2(d.y, -d.x);  // -i * d
  v[0] = make_float2(t0.x + t2.x, t0.y + t2.y);
  v[2] = make_float2(t0.x - t2.x, t0.y - t2.y);
  v[1] = make_float2(t1.x + t3.x, t1.y + t3.y);
  v[3] = make_float2(t1.x - t3.x, t1.y - t3.y);
}

template <>
__device__ __forceinline__ void dft_small<8>(float2* v) {
  float2 e[4] = {v[0], v[2], v[4], v[6]};
  float2 o[4] = {v[1], v[3], v[5], v[7]};
  dft_small<4>(e);
  dft_small<4>(o);
  const float h = 0.70710678118654752f;
  float2 o1 = make_float2(h * (o[1].x + o[1].y), h * (o[1].y - o[1].x));    // * (1 - i)/sqrt2
  float2 o2 = make_float2(o[2].y, -o[2].x);                                 // * (-i)
  float2 o3 = make_float2(h * (o[3].y - o[3].x), -h * (o[3].x + o[3].y));   // * (-1 - i)/sqrt2
  v[0] = make_float2(e[0].x + o[0].x, e[0].y + o[0].y);
  v[4] = make_float2(e[0].x - o[0].x, e[0].y - o[0].y);
  v[1] = make_float2(e[1].x + o1.x, e[1].y + o1.y);
  v[5] = make_float2(e[1].x - o1.x, e[1].y - o1.y);
  v[2] = make_float2(e[2].x + o2.x, e[2].y + o2.y);
  v[6] = make_float2(e[2].x - o2.x, e[2].y - o2.y);
  v[3] = make_float2(e[3].x + o3.x, e[3].y + o3.y);
  v[7] = make_float2(e[3].x - o3.x, e[3].y - o3.y);
}

template <>
__device__ __forceinline__ void dft_small<3>(float2* v) {
  const float c = 0.86602540378443865f;  // sin(2 pi / 3)
  float2 s = make_float2(v[1].x + v[2].x, v[1].y + v[2].y);
  float2 d = make_float2(v[1].x - v[2].x, v[1].y - v[2].y);
  float2 a = make_float2(v[0].x - 0.5f * s.x, v[0].y - 0.5f * s.y);
  float2 b = make_float2(c * d.y, -c * d.x);  // -i c d
  v[0] = make_float2(v[0].x + s.x, v[0].y + s.y);
  v[1] = make_float2(a.x + b.x, a.y + b.y);
  v[2] = make_float2(a.x - b.x, a.y - b.y);
}

template <>
__device__ __forceinline__ void dft_small<5>(float2* v) {
  const float c1 = 0.30901699437494742f, c2 = -0.80901699437494742f;  // cos(2pi/5), cos(4pi/5)
  const float s1 = 0.95105651629515357f, s2 = 0.58778525229247313f;   // sin(2pi/5), sin(4pi/5)
  float2 a1 = make_float2(v[1].x + v[4].x, v[1].y + v[4].y), b1 = make_float2(v[1].x - v[4].x, v[1].y - v[4].y);
  float2 a2 = make_float2(v[2].x + v[3].x, v[2].y + v[3].y), b2 = make_float2(v[2].x - v[3].x, v[2].y - v[3].y);
  float2 v0 = v[0];
  float2 p1 = make_float2(v0.x + c1 * a1.x + c2 * a2.x, v0.y + c1 * a1.y + c2 * a2.y);
  float2 p2 = make_float2(v0.x + c2 * a1.x + c1 * a2.x, v0.y + c2 * a1.y + c1 * a2.y);
  // q = -i (s1 b1 + s2 b2),  r = -i (s2 b1 - s1 b2)
  float2 t1 = make_float2(s1 * b1.x + s2 * b2.x, s1 * b1.y + s2 * b2.y);
  float2 t2 = make_float2(s2 * b1.x - s1 * b2.x, s2 * b1.y - s1 * b2.y);
  float2 q1 = make_float2(t1.y, -t1.x), q2 = make_float2(t2.y, -t2.x);
  v[0] = make_float2(v0.x + a1.x + a2.x, v0.y + a1.y + a2.y);
  v[1] = make_float2(p1.x + q1.x, p1.y + q1.y);
  v[4] = make_float2(p1.x - q1.x, p1.y - q1.y);
  v[2] = make_float2(p2.x + q2.x, p2.y + q2.y);
  v[3] = make_float2(p2.x - q2.x, p2.y - q2.y);
}

// One Stockham pass of radix R over `nlines` independent lines of length P held in shared memory
// (line l at src + l * lpitch). tw[k] = exp(-2 pi i k / P), k < P.
template <int R>
__device__ __forceinline__ void stockham_pass(const float2* __restrict__ src, float2* __restrict__ dst, int P, int Ns,
                                              int nlines, int lpitch, const float2* __restrict__ tw) {
  const int nb = P / R;  // butterflies per line
  const int tstride = P / (Ns * R);
  for (int idx = threadIdx.x; idx < nlines * nb; idx += blockDim.x) {
    int l = idx / nb, j = idx - l * nb;
    int k = j % Ns;
    const float2* s = src + (size_t)l * lpitch;
    float2 v[R];
#pragma unroll
    for (int r = 0; r < R; ++r) v[r] = s[j + r * nb];
    if (Ns > 1) {
#pragma unroll
      for (int r = 1; r < R; ++r) v[r] = cmulf(v[r], __ldg(&tw[r * k * tstride]));
    }
    dft_small<R>(v);
    float2* d = dst + (size_t)l * lpitch + (j - k) * R + k;
#pragma unroll
    for (int r = 0; r < R; ++r) d[r * Ns] = v[r];
  }
}

// Full forward FFT of nlines lines; ping-pongs between bufA and bufB; returns where the result is.
__device__ __forceinline__ float2* stockham_fft(float2* bufA, float2* bufB, const AxisPlan& pl, int nlines, int lpitch,
                                                const float2* __restrict__ tw) {
  float2* src = bufA;
  float2* dst = bufB;
  int Ns = 1;
  for (int p = 0; p < pl.npass; ++p) {
    int R = pl.radix[p];
    switch (R) {
      case 8: stockham_pass<8>(src, dst, pl.P, Ns, nlines, lpitch, tw); break;
      case 4: stockham_pass<4>(src, dst, pl.P, Ns, nlines, lpitch, tw); break;
      case 2: stockham_pass<2>(src, dst, pl.P, Ns, nlines, lpitch, tw); break;
      case 3: stockham_pass<3>(src, dst, pl.P, Ns, nlines, lpitch, tw); break;
      default: stockham_pass<5>(src, dst, pl.P, Ns, nlines, lpitch, tw); break;
    }
    Ns *= R;
    __syncthreads();
    float2* t = src; src = dst; dst = t;
  }
  return src;
}
