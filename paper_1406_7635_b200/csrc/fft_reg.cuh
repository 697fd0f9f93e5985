// fft_reg.cuh - register-resident power-of-two FFT engine of the fast demag path (sm_100a).
//
// TWO length-N complex transforms run in lockstep in the two lanes of Blackwell's packed fp32
// instructions (FADD2 / FMUL2 / FFMA2 on 64-bit register pairs): every value is a C2 = (re, im)
// with re = (re of transform 0, re of transform 1), im likewise, so each butterfly instruction
// advances both transforms and every shared-memory exchange moves 16 bytes per point. The fast
// path always has such a pair at hand: the even-bin and the odd-bin half of one zero-padded line
// (fast2d.cuh). Twiddles are the same for both lanes and enter as broadcast scalars.
//
// One pair of transforms is computed by a group of T threads, E = N/T points per thread held in
// registers, in 2 or 3 passes of radix RA, RB[, RC] (N = RA*RB*RC). Between two passes the points
// are exchanged through a (padded, bank-conflict-free) shared-memory buffer; the first pass reads
// and the last pass leaves the data in the striped "natural" layout
//     point index = bf + (N/R) * s,   bf = t + T*b,   register v[b*R + s]
// (R = RA on input, R = last radix on output), so that global loads/stores of consecutive threads
// are contiguous and no digit-reversal pass is ever needed (PAPER.md L123 only asks for "the
// well-known convolution theorem"; how the transforms are organised is ours).
//
// Decomposition (decimation in frequency): n = n1*M1 + n2*M2 + n3, k = k1 + RA*k2 + RA*RB*k3,
// M1 = N/RA, M2 = M1/RB. Pass i transforms digit n_i -> k_i and multiplies by
// w_N^{k_i * (RA..R_{i-1}) * rest_i}, rest_i = the not yet transformed low digits.
#pragma once
#include "common.cuh"

namespace rf {

struct C2 { float2 re, im; };   // two complex numbers: lane x = transform 0, lane y = transform 1

__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }   // folds into the consumer
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ float2 mul2(float2 a, float s) { return __fmul2_rn(a, make_float2(s, s)); }
__device__ __forceinline__ float2 fma2(float2 a, float s, float2 c) { return __ffma2_rn(a, make_float2(s, s), c); }

__device__ __forceinline__ C2 cadd(C2 a, C2 b) { return {add2(a.re, b.re), add2(a.im, b.im)}; }
__device__ __forceinline__ C2 csub(C2 a, C2 b) { return {sub2(a.re, b.re), sub2(a.im, b.im)}; }

// a * w (DIR < 0) or a * conj(w) (DIR > 0): tables hold the forward twiddles w = exp(-i phi)
template <int DIR>
__device__ __forceinline__ C2 cmul_tw(C2 a, float2 w) {
  if (DIR < 0) return {fma2(a.re, w.x, neg2(mul2(a.im, w.y))), fma2(a.re, w.y, mul2(a.im, w.x))};
  return {fma2(a.re, w.x, mul2(a.im, w.y)), fma2(a.im, w.x, neg2(mul2(a.re, w.y)))};
}
// scalar version (one complex number)
template <int DIR>
__device__ __forceinline__ float2 cmul_tw1(float2 a, float2 w) {
  if (DIR < 0) return make_float2(a.x * w.x - a.y * w.y, a.x * w.y + a.y * w.x);
  return make_float2(a.x * w.x + a.y * w.y, a.y * w.x - a.x * w.y);
}

// multiply by exp(DIR * i * pi/4)
template <int DIR>
__device__ __forceinline__ C2 rot45(C2 a) {
  const float h = 0.70710678118654752f;
  if (DIR < 0) return {mul2(add2(a.re, a.im), h), mul2(sub2(a.im, a.re), h)};
  return {mul2(sub2(a.re, a.im), h), mul2(add2(a.re, a.im), h)};
}
// multiply by exp(DIR * i * pi/2): a register renaming plus a sign the consumer absorbs
template <int DIR>
__device__ __forceinline__ C2 rot90(C2 a) {
  if (DIR < 0) return {a.im, neg2(a.re)};
  return {neg2(a.im), a.re};
}
// multiply by exp(DIR * i * 3 pi/4)
template <int DIR>
__device__ __forceinline__ C2 rot135(C2 a) {
  const float h = 0.70710678118654752f;
  if (DIR < 0) return {mul2(sub2(a.im, a.re), h), mul2(add2(a.re, a.im), -h)};
  return {mul2(add2(a.re, a.im), -h), mul2(sub2(a.re, a.im), h)};
}
// multiply by exp(DIR * i * phi) with cos(phi) = C, sin(phi) = S given as literals
template <int DIR>
__device__ __forceinline__ C2 rotcs(C2 a, const float C, const float S) {
  if (DIR < 0) return {fma2(a.re, C, mul2(a.im, S)), fma2(a.im, C, neg2(mul2(a.re, S)))};
  return {fma2(a.re, C, neg2(mul2(a.im, S))), fma2(a.im, C, mul2(a.re, S))};
}

template <int R, int DIR>
struct Bfly;

template <int DIR>
struct Bfly<2, DIR> {
  static __device__ __forceinline__ void run(C2* v) {
    C2 a = v[0], b = v[1];
    v[0] = cadd(a, b);
    v[1] = csub(a, b);
  }
};

template <int DIR>
struct Bfly<4, DIR> {
  static __device__ __forceinline__ void run(C2& v0, C2& v1, C2& v2, C2& v3) {
    const C2 t0 = cadd(v0, v2), t1 = csub(v0, v2), t2 = cadd(v1, v3), d = csub(v1, v3);
    v0 = cadd(t0, t2);
    v2 = csub(t0, t2);
    if (DIR < 0) {   // t3 = -i d = (d.im, -d.re)
      v1 = {add2(t1.re, d.im), sub2(t1.im, d.re)};
      v3 = {sub2(t1.re, d.im), add2(t1.im, d.re)};
    } else {         // t3 = +i d = (-d.im, d.re)
      v1 = {sub2(t1.re, d.im), add2(t1.im, d.re)};
      v3 = {add2(t1.re, d.im), sub2(t1.im, d.re)};
    }
  }
  static __device__ __forceinline__ void run(C2* v) { run(v[0], v[1], v[2], v[3]); }
};

// 8 = 2 x 4: n = 4a + b, k = c + 2d
template <int DIR>
struct Bfly<8, DIR> {
  static __device__ __forceinline__ void run(C2* v) {
    C2 A0[4], A1[4];
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      A0[b] = cadd(v[b], v[b + 4]);
      A1[b] = csub(v[b], v[b + 4]);
    }
    A1[1] = rot45<DIR>(A1[1]);
    A1[2] = rot90<DIR>(A1[2]);
    A1[3] = rot135<DIR>(A1[3]);
    Bfly<4, DIR>::run(A0[0], A0[1], A0[2], A0[3]);
    Bfly<4, DIR>::run(A1[0], A1[1], A1[2], A1[3]);
#pragma unroll
    for (int d = 0; d < 4; ++d) {
      v[2 * d] = A0[d];
      v[2 * d + 1] = A1[d];
    }
  }
};

// 16 = 4 x 4: n = 4a + b, k = c + 4d; twiddles W16^{bc}
template <int DIR>
struct Bfly<16, DIR> {
  static __device__ __forceinline__ void run(C2* v) {
    const float C1 = 0.92387953251128674f, S1 = 0.38268343236508977f;  // cos, sin of pi/8
#pragma unroll
    for (int b = 0; b < 4; ++b) Bfly<4, DIR>::run(v[b], v[b + 4], v[b + 8], v[b + 12]);
    // after the radix-4 over a, element (b, c) sits in v[b + 4c]
    v[1 + 4] = rotcs<DIR>(v[1 + 4], C1, S1);     // W^1
    v[1 + 8] = rot45<DIR>(v[1 + 8]);             // W^2
    v[1 + 12] = rotcs<DIR>(v[1 + 12], S1, C1);   // W^3
    v[2 + 4] = rot45<DIR>(v[2 + 4]);             // W^2
    v[2 + 8] = rot90<DIR>(v[2 + 8]);             // W^4
    v[2 + 12] = rot135<DIR>(v[2 + 12]);          // W^6
    v[3 + 4] = rotcs<DIR>(v[3 + 4], S1, C1);     // W^3
    v[3 + 8] = rot135<DIR>(v[3 + 8]);            // W^6
    v[3 + 12] = rotcs<DIR>(v[3 + 12], -C1, -S1); // W^9
    // radix-4 over b for each c: (v[4c], v[4c+1], v[4c+2], v[4c+3]) -> X[c + 4d] in slot 4c + d
#pragma unroll
    for (int c = 0; c < 4; ++c) Bfly<4, DIR>::run(v[4 * c], v[4 * c + 1], v[4 * c + 2], v[4 * c + 3]);
    // transpose slots (4c + d) -> (c + 4d)
#pragma unroll
    for (int c = 0; c < 4; ++c)
#pragma unroll
      for (int d = c + 1; d < 4; ++d) {
        C2 tmp = v[4 * c + d];
        v[4 * c + d] = v[4 * d + c];
        v[4 * d + c] = tmp;
      }
  }
};

template <int N_, int T_, int RA_, int RB_, int RC_>
struct Plan {
  static constexpr int N = N_, T = T_, E = N_ / T_, RA = RA_, RB = RB_, RC = RC_;
  static constexpr int NPASS = RC_ > 1 ? 3 : 2;
  static constexpr int RLAST = RC_ > 1 ? RC_ : RB_;
  static constexpr int M1 = N_ / RA_, M2 = M1 / RB_;
  static constexpr int XB = N_ + N_ / 16;                       // padded exchange buffer (float4 units)
  static constexpr int TW1 = (RA_ - 1) * (N_ / RA_);            // twiddle entries after pass 1
  static constexpr int TW2 = RC_ > 1 ? (RB_ - 1) * (N_ / RB_) : 0;
  static constexpr int TW = TW1 + TW2;
  static_assert(RA_ * RB_ * RC_ == N_, "radices must multiply to N");
  static_assert(E % RA_ == 0 && E % RB_ == 0 && E % RC_ == 0, "every radix must divide the points per thread");
  typedef Plan<N_, T_, (RC_ > 1 ? RC_ : RB_), (RC_ > 1 ? RB_ : RA_), (RC_ > 1 ? RA_ : 1)> Reversed;
};

// exchange-buffer index of point a: one 16-byte unit per point, one unit of padding per 16, so that
// both the unit-stride writes and the stride-16 reads of the last pass hit 8 different 16-byte bank
// groups per quarter-warp
__device__ __forceinline__ int xpad(int a) { return a + (a >> 4); }

__device__ __forceinline__ float4 pack(C2 a) { return make_float4(a.re.x, a.re.y, a.im.x, a.im.y); }
__device__ __forceinline__ C2 unpack(float4 q) { return {make_float2(q.x, q.y), make_float2(q.z, q.w)}; }

// synchronise the T threads of FFT group `gid` of a CTA with NT threads
template <int T, int NT>
__device__ __forceinline__ void group_sync(int gid) {
  if (T == NT) __syncthreads();
  else if (T >= 32) asm volatile("bar.sync %0, %1;" ::"r"(gid + 1), "r"(T) : "memory");
  else __syncwarp();
}

// point index of register slot e in the striped layout with radix R
template <class P, int R>
__device__ __forceinline__ int slot_index(int t, int e) {
  return t + P::T * (e / R) + (P::N / R) * (e % R);
}

template <class P, int R, int DIR>
__device__ __forceinline__ void pass_butterflies(C2* v) {
#pragma unroll
  for (int b = 0; b < P::E / R; ++b) Bfly<R, DIR>::run(v + b * R);
}

// Twiddles of the pass that follows a radix-R butterfly: w^s, s = 1 .. R-1, of the per-thread base
// w = table entry of s = 1. Only the base is loaded; the powers are formed in registers by a product
// tree of depth <= 4 (about 4 ulp), so the butterfly phases of a warp do not queue behind the
// shared-memory traffic of the other warps in the LSU pipe.
__device__ __forceinline__ float2 csqr(float2 a) { return make_float2(a.x * a.x - a.y * a.y, 2.f * a.x * a.y); }
__device__ __forceinline__ float2 cmul1(float2 a, float2 b) { return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }

// exp(-i pi e / 16), e = 0 .. 15: with 16 points per thread at stride N/16 the half-bin twiddle
// w_2N^n of point n = t + (N/16) e is w_2N^t times this constant, so one table load per thread serves
// all 16 points
__device__ __forceinline__ float2 half_twiddle(float2 wt, int e) {
  constexpr float C[16] = {1.f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f,
                           0.55557023301960218f, 0.38268343236508977f, 0.19509032201612825f, 0.f, -0.19509032201612825f,
                           -0.38268343236508977f, -0.55557023301960218f, -0.70710678118654752f, -0.83146961230254524f,
                           -0.92387953251128674f, -0.98078528040323043f};
  constexpr float S[16] = {0.f, 0.19509032201612825f, 0.38268343236508977f, 0.55557023301960218f, 0.70710678118654752f,
                           0.83146961230254524f, 0.92387953251128674f, 0.98078528040323043f, 1.f, 0.98078528040323043f,
                           0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f, 0.55557023301960218f,
                           0.38268343236508977f, 0.19509032201612825f};
  if (e == 0) return wt;
  if (e == 8) return make_float2(wt.y, -wt.x);                 // times -i
  return make_float2(wt.x * C[e] + wt.y * S[e], wt.y * C[e] - wt.x * S[e]);   // wt * (C - i S)
}

template <class P, int R>
__device__ __forceinline__ void load_twiddles(float2* w, int t, const float2* __restrict__ tw) {
#pragma unroll
  for (int b = 0; b < P::E / R; ++b) {
    float2* p = w + b * (R - 1);                      // p[s - 1] = base^s
    p[0] = __ldg(&tw[t + P::T * b]);
    if (R > 2) { p[1] = csqr(p[0]); p[2] = cmul1(p[1], p[0]); }
    if (R > 4) {
      p[3] = csqr(p[1]);
#pragma unroll
      for (int s = 1; s <= 3; ++s) p[3 + s] = cmul1(p[3], p[s - 1]);
    }
    if (R > 8) {
      p[7] = csqr(p[3]);
#pragma unroll
      for (int s = 1; s <= 7; ++s) p[7 + s] = cmul1(p[7], p[s - 1]);
    }
  }
}

template <class P, int R, int DIR>
__device__ __forceinline__ void apply_twiddles(C2* v, const float2* w) {
#pragma unroll
  for (int b = 0; b < P::E / R; ++b)
#pragma unroll
    for (int s = 1; s < R; ++s) v[b * R + s] = cmul_tw<DIR>(v[b * R + s], w[b * (R - 1) + s - 1]);
}

__host__ __device__ constexpr int xpadc(int c) { return c + c / 16; }

// Write the state after a radix-R pass, read the operands of the next radix-RN pass
// (MP = rest size after the finished pass, MN = MP / RN). All indices are xpad(thread part) plus a
// compile-time constant: the constant parts are multiples of 16 or stay inside one 16-block, so
// xpad is additive over them and every access is base register + immediate.
// PLANES = false: one 16-byte unit per point (xb = XB float4), two group barriers.
// PLANES = true : the re pairs and then the im pairs go through a buffer of 8-byte units (xb = XB
//                 float2, half the shared memory), four group barriers.
template <class P, int R, int RN, int MP, int NT, bool PLANES>
__device__ __forceinline__ void exchange(C2* v, void* xbuf, int t, int gid) {
  constexpr int MN = MP / RN;
  static_assert(MP % 16 == 0 && (MN % 16 == 0 || MP == 16) && P::T % 16 == 0 && P::T % MN == 0,
                "exchange indices must be affine under xpad");
  const int wbase = xpad(t);
  const int rbase = xpad((t / MN) * MP + (t % MN));
  constexpr int RB_STEP = (P::T / MN) * MP;      // read-base step per butterfly index b
  if constexpr (!PLANES) {
    float4* xb = reinterpret_cast<float4*>(xbuf);
    group_sync<P::T, NT>(gid);
#pragma unroll
    for (int b = 0; b < P::E / R; ++b)
#pragma unroll
      for (int s = 0; s < R; ++s) xb[wbase + xpadc(P::T * b + (P::N / R) * s)] = pack(v[b * R + s]);
    group_sync<P::T, NT>(gid);
#pragma unroll
    for (int b = 0; b < P::E / RN; ++b)
#pragma unroll
      for (int s = 0; s < RN; ++s) v[b * RN + s] = unpack(xb[rbase + xpadc(RB_STEP * b + s * MN)]);
  } else {
    float2* xb = reinterpret_cast<float2*>(xbuf);
    group_sync<P::T, NT>(gid);
#pragma unroll
    for (int b = 0; b < P::E / R; ++b)
#pragma unroll
      for (int s = 0; s < R; ++s) xb[wbase + xpadc(P::T * b + (P::N / R) * s)] = v[b * R + s].re;
    group_sync<P::T, NT>(gid);
#pragma unroll
    for (int b = 0; b < P::E / RN; ++b)
#pragma unroll
      for (int s = 0; s < RN; ++s) v[b * RN + s].re = xb[rbase + xpadc(RB_STEP * b + s * MN)];
    group_sync<P::T, NT>(gid);
#pragma unroll
    for (int b = 0; b < P::E / R; ++b)
#pragma unroll
      for (int s = 0; s < R; ++s) xb[wbase + xpadc(P::T * b + (P::N / R) * s)] = v[b * R + s].im;
    group_sync<P::T, NT>(gid);
#pragma unroll
    for (int b = 0; b < P::E / RN; ++b)
#pragma unroll
      for (int s = 0; s < RN; ++s) v[b * RN + s].im = xb[rbase + xpadc(RB_STEP * b + s * MN)];
  }
}

// In-register transform of the group's pair of lines: DIR = -1 forward exp(-i...), +1 inverse
// (unscaled). v: E points in the RA-striped layout on entry, RLAST-striped on exit. xb: the group's
// exchange buffer (P::XB float4, or P::XB float2 with PLANES). tw: P::TW forward twiddles of this plan. t: thread index inside
// the group. The first exchange starts with a group barrier, so xb may still be read by the group
// until then; after the call xb is only safe to reuse after another group barrier.
// first pass (butterflies + twiddles: registers only) and the rest (from the first exchange on) as two calls, for
// kernels that must do something between them (e.g. wait until the exchange buffer is free again)
template <class P, int DIR>
__device__ __forceinline__ void fft_head(C2* v, int t, const float2* __restrict__ tw) {
  pass_butterflies<P, P::RA, DIR>(v);
  float2 w[(P::RA - 1) * (P::E / P::RA)];
  load_twiddles<P, P::RA>(w, t, tw);
  apply_twiddles<P, P::RA, DIR>(v, w);
}
template <class P, int DIR, int NT, bool PLANES = false>
__device__ __forceinline__ void fft_tail(C2* v, void* xb, int t, int gid, const float2* __restrict__ tw) {
  exchange<P, P::RA, P::RB, P::M1, NT, PLANES>(v, xb, t, gid);
  pass_butterflies<P, P::RB, DIR>(v);
  if constexpr (P::NPASS == 3) {
    {
      float2 w[(P::RB - 1) * (P::E / P::RB)];
      load_twiddles<P, P::RB>(w, t, tw + P::TW1);
      apply_twiddles<P, P::RB, DIR>(v, w);
    }
    exchange<P, P::RB, P::RC, P::M2, NT, PLANES>(v, xb, t, gid);
    pass_butterflies<P, P::RC, DIR>(v);
  }
}
template <class P, int DIR, int NT, bool PLANES = false>
__device__ __forceinline__ void fft(C2* v, void* xb, int t, int gid, const float2* __restrict__ tw) {
  fft_head<P, DIR>(v, t, tw);
  fft_tail<P, DIR, NT, PLANES>(v, xb, t, gid, tw);
}

}  // namespace rf
