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
//   K_B  k2_ycol : columns (kx fixed, all y; contiguous), one FFT group per job. XY job: transform the
//                  x component forward and stash it in shared memory, transform y, form the 2x2
//                  symmetric kernel product (K_xx K_xy; K_xy K_yy), transform both back, store in
//                  place. Z job: K_zz only (K_xz = K_yz = 0 for one layer), two columns.
//   K_C  k2_xinv : x spectrum -> rows of B_demag (only the Nx physical outputs are formed).
#pragma once
#include "common.cuh"
#include "fft_reg.cuh"
#include "demag_conv_args.cuh"
#include "tma_util.cuh"

// pitch (float4 units) between the exchange buffers of consecutive FFT groups: XB plus a skew that
// spreads the G groups over the 8 16-byte bank groups when one quarter-warp touches several buffers
template <class P, int NT>
struct K2Shape {
  static_assert(P::E == 16 && P::RA == 16 && P::Reversed::RLAST == 16 && P::T * 16 == P::N,
                "the kernels assume 16 points per thread at stride N/16 on input and output");
  static constexpr int G = NT / P::T;
  static constexpr int GP = P::XB + (G >= 8 ? 1 : 8 / G);
};
template <class P, int NT>
constexpr size_t k2_smem() { return sizeof(float4) * (size_t)K2Shape<P, NT>::G * K2Shape<P, NT>::GP; }

__device__ __forceinline__ void k2_prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" ::"l"(p)); }
__device__ __forceinline__ void k2_prefetch_l1(const void* p) { asm volatile("prefetch.global.L1 [%0];" ::"l"(p)); }

// loads and stores through pointers fetched from DevState::ptr: the compiler cannot see that they are global
__device__ __forceinline__ float k2_ldg(const float* p) {
  float v;
  asm volatile("ld.global.nc.f32 %0, [%1];" : "=f"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void k2_stg(float* p, float v) { asm volatile("st.global.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory"); }

// stage unit = (z0.re, z0.im, z1.re, z1.im): each lane's complex number is one 8-byte half
__device__ __forceinline__ float4 stage_pack(rf::C2 a) { return make_float4(a.re.x, a.im.x, a.re.y, a.im.y); }
__device__ __forceinline__ rf::C2 stage_unpack(float4 q) { return {make_float2(q.x, q.z), make_float2(q.y, q.w)}; }

// Hermitian separation of Z = A + iB (a, b real rows): from Z[k] and Z[-k] -> (A.re, A.im, B.re, B.im)
__device__ __forceinline__ float4 separate(float2 z, float2 zm) {
  return make_float4(0.5f * (z.x + zm.x), 0.5f * (z.y - zm.y), 0.5f * (z.y + zm.y), 0.5f * (zm.x - z.x));
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
  // gather bins of the 2G rows; rebuild Z = A + iB and its Hermitian partner for both halves.
  // (N/2) G items (k, p) over NT threads: exactly 8 per thread, all 16 loads in flight at once
  constexpr int IT = (N / 2) * G / NT;
  static_assert(IT * NT == (N / 2) * G, "items must divide evenly");
  {
    float4 ev[IT], od[IT];
#pragma unroll
    for (int it = 0; it < IT; ++it) {
      const int w = tid + it * NT, p = w % G, k = w / G;
      const float2* src = in + (size_t)(2 * k) * a.Ny + r0 + 2 * p;
      ev[it] = *reinterpret_cast<const float4*>(src);
      od[it] = *reinterpret_cast<const float4*>(src + a.Ny);
    }
#pragma unroll
    for (int it = 0; it < IT; ++it) {
      const int w = tid + it * NT, p = w % G, k = w / G;
      float4* st = smem4 + (size_t)p * GP;
      float2* st2 = reinterpret_cast<float2*>(st);
      const float4 e = ev[it], o = od[it];
      st[k] = make_float4(e.x - e.w, e.y + e.z, o.x - o.w, o.y + o.z);
      if (k > 0) st2[2 * (N - k)] = make_float2(e.x + e.w, e.z - e.y);
      st2[2 * (N - 1 - k) + 1] = make_float2(o.x + o.w, o.z - o.y);
    }
    if (tid < G) {   // bin kx = N (k = N/2 of the even half): its own partner; the odd half has no such bin
      const float4 e = *reinterpret_cast<const float4*>(in + (size_t)N * a.Ny + r0 + 2 * tid);
      reinterpret_cast<float2*>(smem4 + (size_t)tid * GP)[2 * (N / 2)] = make_float2(e.x - e.w, e.y + e.z);
    }
  }
  __syncthreads();
  {
    rf::C2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = stage_unpack(xb[rf::slot_index<PI, PI::RA>(t, e)]);
    const float2 wt = __ldg(&a.twox[t]);      // w_2N^t; the other points follow from constants
    rf::fft<PI, +1, NT>(v, xb, t, gid, a.twx_r);
    const size_t rowA = (size_t)(r0 + 2 * gid) * a.nxp;      // physical row pitch; n >= nxp is zero fill
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RLAST>(t, e);
      const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), rf::half_twiddle(wt, e));
      if (n < a.nxp) {
        k2_stg(dst + rowA + n, v[e].re.x + u.x);
        k2_stg(dst + rowA + a.nxp + n, v[e].im.x + u.y);
      }
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

// shared memory of one FFT group in k2_ycol: plane-wise exchange buffer (XB float2) + stash (N float4)
template <class P>
struct K2YShape {
  static constexpr int GROUP_BYTES = P::XB * 8 + P::N * 16;
};
template <class P, int NT>
constexpr size_t k2_y_smem() { return (size_t)(NT / P::T) * K2YShape<P>::GROUP_BYTES; }


// Every FFT group works on its own: an XY job is one column of the x and y components (coupled by
// the kernel product), a Z job one column of the z component. All code is straight-line (a rolled
// loop over components would carry the 64-register point array around its back edge, which costs
// a register permutation through local memory).
// Two CTAs share an SM: butterflies of one over the exchanges and loads of the other. (Forcing the phases apart - two
// groups per CTA taking turns in their exchanges by named-barrier tokens, or a start offset between the CTAs of an
// SM - was measured and is slower or neutral.)
template <class P, int NT>
struct K2Col {
  using PI = typename P::Reversed;
  static constexpr int N = P::N, T = P::T, E = P::E;

  // column -> lanes (z[n], z[n] w^n) -> forward transforms of the even and the odd bins
  template <bool PLANES>
  static __device__ __forceinline__ void load_fwd(const Fast2DArgs& a, const float2* __restrict__ s, rf::C2* v, float2* xb,
                                                  int t, int gid) {
    const float2 wt = __ldg(&a.twoy[t]);      // w_2N^t; the other points follow from constants
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<P, P::RA>(t, e);
      const float2 z = n < a.nyp ? s[n] : make_float2(0.f, 0.f);          // rows beyond the film: zero fill
      const float2 zw = rf::cmul_tw1<-1>(z, rf::half_twiddle(wt, e));
      v[e] = {make_float2(z.x, zw.x), make_float2(z.y, zw.y)};
    }
    rf::fft<P, -1, NT, PLANES>(v, xb, t, gid, a.twy);
  }
  // inverse transforms -> first N samples: even part + conj(w)^n odd part -> column (in place)
  template <bool PLANES>
  static __device__ __forceinline__ void inv_store(const Fast2DArgs& a, float2* __restrict__ d, rf::C2* v, float2* xb, int t,
                                                   int gid) {
    const float2 wt = __ldg(&a.twoy[t]);      // w_2N^t; the other points follow from constants
    rf::fft<PI, +1, NT, PLANES>(v, xb, t, gid, a.twy_r);
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RLAST>(t, e);
      const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), rf::half_twiddle(wt, e));
      if (n < a.nyp) d[n] = make_float2(v[e].re.x + u.x, v[e].im.x + u.y);
    }
  }
};

template <class P, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) k2_ycol(Fast2DArgs a, int nxy) {
  if (a.st->skip) return;
  using C = K2Col<P, NT>;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T;
  extern __shared__ float4 smem4[];
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  __builtin_assume(t >= 0 && t < T);          // lets the mirror tests of k2_kidx fold per register slot
  char* mine = reinterpret_cast<char*>(smem4) + (size_t)gid * K2YShape<P>::GROUP_BYTES;
  float4* stash = reinterpret_cast<float4*>(mine);
  float2* xb = reinterpret_cast<float2*>(mine + (size_t)N * 16);
  const bool xy = (int)blockIdx.x < nxy;
  const int kx = xy ? (int)blockIdx.x * G + gid : ((int)blockIdx.x - nxy) * G + gid;
  if (kx >= a.Cx) return;                      // the whole group leaves together
  float2* __restrict__ col = a.spec + (size_t)kx * a.Ny;
  const float* __restrict__ Kc = a.Kt + (size_t)kx * (N + 1);
  // start the kernel-spectrum rows of this column on their way from DRAM to L2
  for (int i = t * 32; i < N + 1; i += T * 32) {
    if (xy) { k2_prefetch_l2(Kc + i); k2_prefetch_l2(Kc + a.kstride + i); k2_prefetch_l2(Kc + 3 * a.kstride + i); }
    else k2_prefetch_l2(Kc + 2 * a.kstride + i);
  }
  {
    // columns that will be wanted soon, on their way from DRAM to L2: this job's second component and
    // the first component of the job that follows on this SM (CTAs are dispatched in order, 512 / NT per SM)
    const int ahead = kx + (512 / NT) * a.nsm * G;
    const float2* nxt = a.spec + (size_t)(xy ? 0 : 2) * a.cstride + (size_t)ahead * a.Ny;
    for (int i = t * 16; i < N; i += T * 16) {
      if (xy) k2_prefetch_l2(col + a.cstride + i);
      if (ahead < a.Cx) k2_prefetch_l2(nxt + i);
    }
  }
  rf::C2 v[E];
  if (xy) {
    C::template load_fwd<true>(a, col, v, xb, t, gid);
#pragma unroll
    for (int e = 0; e < E; ++e) stash[e * T + t] = rf::pack(v[e]);     // own slots: no barrier
    // the kernel rows are needed right after this transform: pull them from L2 into L1 now
    for (int i = t * 32; i < N + 1; i += T * 32) {
      k2_prefetch_l1(Kc + i); k2_prefetch_l1(Kc + a.kstride + i); k2_prefetch_l1(Kc + 3 * a.kstride + i);
    }
    C::template load_fwd<true>(a, col + a.cstride, v, xb, t, gid);
    // B~_x = K_xx M~_x + K_xy M~_y,  B~_y = K_xy M~_x + K_yy M~_y   (Eq. 3; K real, L145)
    const float* __restrict__ Ky = Kc + a.kstride;
    const float* __restrict__ Ko = Kc + (size_t)3 * a.kstride;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      int i0, i1; float s0, s1;
      k2_kidx<N>(rf::slot_index<P, P::RLAST>(t, e), i0, i1, s0, s1);
      const float2 kxx = make_float2(__ldg(&Kc[i0]), __ldg(&Kc[i1]));
      const float2 kyy = make_float2(__ldg(&Ky[i0]), __ldg(&Ky[i1]));
      const float2 kxy = make_float2(s0 * __ldg(&Ko[i0]), s1 * __ldg(&Ko[i1]));
      const rf::C2 X = rf::unpack(stash[e * T + t]), Y = v[e];
      rf::C2 bx;
      bx.re = __ffma2_rn(kxy, Y.re, __fmul2_rn(kxx, X.re));
      bx.im = __ffma2_rn(kxy, Y.im, __fmul2_rn(kxx, X.im));
      stash[e * T + t] = rf::pack(bx);
      v[e].re = __ffma2_rn(kxy, X.re, __fmul2_rn(kyy, Y.re));
      v[e].im = __ffma2_rn(kxy, X.im, __fmul2_rn(kyy, Y.im));
    }
    C::template inv_store<true>(a, col + a.cstride, v, xb, t, gid);
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = rf::unpack(stash[e * T + t]);
    C::template inv_store<true>(a, col, v, xb, t, gid);
  } else {
    float2* __restrict__ cz = col + 2 * a.cstride;
    float2* xz = reinterpret_cast<float2*>(mine);      // no stash needed: 16-byte units, half the barriers
    C::template load_fwd<false>(a, cz, v, xz, t, gid);
    const float* __restrict__ Kz = Kc + (size_t)2 * a.kstride;
#pragma unroll
    for (int e = 0; e < E; ++e) {
      int i0, i1; float s0, s1;
      k2_kidx<N>(rf::slot_index<P, P::RLAST>(t, e), i0, i1, s0, s1);
      const float2 kz = make_float2(__ldg(&Kz[i0]), __ldg(&Kz[i1]));
      v[e].re = __fmul2_rn(kz, v[e].re);
      v[e].im = __fmul2_rn(kz, v[e].im);
    }
    C::template inv_store<false>(a, cz, v, xz, t, gid);
  }
}

// ---------------------------------------------------------------------------------- K_C with TMA
// Same computation as k2_xinv, but the transposed 16G-byte pieces of the CTA's 2G rows arrive as
// TMA boxes {2G rows, KB bins} of a 3-D tensor map over spec (y innermost, then kx, then component):
// a ring of NBUF boxes is in flight while the threads turn the previous box into Z = A + iB and
// its mirror, so the gather costs no LSU global-load wavefronts and no registers.
constexpr int K2_KB = 256;      // kx bins per box
template <int G> struct K2Ring { static constexpr int NBUF = G >= 4 ? 2 : 8 / G; };   // boxes in flight (32-64 KB)

template <class P, int NT>
constexpr size_t k2_tma_smem() {
  return k2_smem<P, NT>() + (size_t)K2Ring<K2Shape<P, NT>::G>::NBUF * K2_KB * K2Shape<P, NT>::G * sizeof(float4) + 128;
}

template <class P, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) k2_xinv_tma(Fast2DArgs a, int dst_role, const __grid_constant__ CUtensorMap map) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T, GP = K2Shape<P, NT>::GP;
  constexpr int NB = (N + 1 + K2_KB - 1) / K2_KB;            // boxes covering kx = 0 .. N
  constexpr int K2_NBUF = K2Ring<G>::NBUF;
  constexpr uint32_t BOX_BYTES = K2_KB * G * sizeof(float4);
  extern __shared__ __align__(128) float4 smem4[];
  __shared__ __align__(8) uint64_t full[K2_NBUF];
  float4* tiles = smem4 + (size_t)G * GP + ((128 - ((size_t)G * GP * 16) % 128) % 128) / 16;   // 128-byte aligned
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float4* xb = smem4 + (size_t)gid * GP;
  const int c = blockIdx.y, r0 = blockIdx.x * 2 * G;
  float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * a.ncell;
  if (tid == 0) {
#pragma unroll
    for (int b = 0; b < K2_NBUF; ++b) tma::mbar_init(&full[b], 1);
    tma::fence_barrier_init();
    tma::fence_proxy_async();
#pragma unroll
    for (int b = 0; b < K2_NBUF && b < NB; ++b) {
      tma::mbar_expect_tx(&full[b], BOX_BYTES);
      tma::load_3d(tiles + (size_t)b * K2_KB * G, &map, 2 * r0, b * K2_KB, c, &full[b]);
    }
  }
  __syncthreads();
#pragma unroll 1
  for (int j = 0; j < NB; ++j) {
    const int b = j % K2_NBUF;
    tma::mbar_wait(&full[b], (j / K2_NBUF) & 1);
    const float4* tile = tiles + (size_t)b * K2_KB * G;
    for (int i = tid; i < K2_KB * G; i += NT) {
      const int p = i % G, kx = j * K2_KB + i / G;
      if (kx > N) continue;
      const float4 e = tile[i];
      float2* st2 = reinterpret_cast<float2*>(smem4 + (size_t)p * GP);
      const int k = kx >> 1, h = kx & 1;
      const float2 z = make_float2(e.x - e.w, e.y + e.z), zm = make_float2(e.x + e.w, e.z - e.y);
      st2[2 * k + h] = z;
      if (h) st2[2 * (N - 1 - k) + 1] = zm;
      else if (k > 0 && k < N / 2) st2[2 * (N - k)] = zm;
    }
    __syncthreads();                       // everyone is done with this box: refill it
    if (tid == 0 && j + K2_NBUF < NB) {
      tma::mbar_expect_tx(&full[b], BOX_BYTES);
      tma::load_3d(tiles + (size_t)b * K2_KB * G, &map, 2 * r0, (j + K2_NBUF) * K2_KB, c, &full[b]);
    }
  }
  {
    rf::C2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = stage_unpack(xb[rf::slot_index<PI, PI::RA>(t, e)]);
    const float2 wt = __ldg(&a.twox[t]);      // w_2N^t; the other points follow from constants
    rf::fft<PI, +1, NT>(v, xb, t, gid, a.twx_r);
    const size_t rowA = (size_t)(r0 + 2 * gid) * a.nxp;      // physical row pitch; n >= nxp is zero fill
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RLAST>(t, e);
      const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), rf::half_twiddle(wt, e));
      if (n < a.nxp) {
        k2_stg(dst + rowA + n, v[e].re.x + u.x);
        k2_stg(dst + rowA + a.nxp + n, v[e].im.x + u.y);
      }
    }
  }
}

// ---------------------------------------------------------------------------------- K_C, direct read
// All bins of the CTA's 2G rows arrive as TMA boxes {2G rows, KB bins} of two tensor maps that walk every second
// column of spec (even kx = 2k, k = 0 .. N/2; odd kx = 2k + 1, k = 0 .. N/2 - 1), every box in flight at once on one
// mbarrier. The landing area IS the FFT exchange buffer: each thread builds its sixteen points of both transforms
// straight from the landed pieces - point n of the even-bin transform is Z[2n], of the odd-bin one Z[2n + 1], with
// Z[b] = A[b] + i B[b] for b <= N and Z[b] = conj(A[2N - b]) + i conj(B[2N - b]) above (A, B: spectra of the two
// real rows of a pair) - then, after one CTA barrier, the buffer is reused for the exchanges. No conversion pass,
// no ring: the whole gather costs 32 shared loads per thread.
template <class P, int NT>
struct K2Inv {
  static constexpr int N = P::N, G = NT / P::T;
  static constexpr int KB = N / 2 < 256 ? N / 2 : 256;                         // bins per box
  static constexpr int NBE = (N / 2 + 1 + KB - 1) / KB, NBO = (N / 2 + KB - 1) / KB;
  static constexpr int LAND4 = (NBE + NBO) * KB * G;                           // float4 units of the landing area
  static constexpr int XB4 = G * K2Shape<P, NT>::GP;                           // float4 units of the exchange buffers
  static constexpr size_t SMEM = sizeof(float4) * (size_t)(LAND4 > XB4 ? LAND4 : XB4) + 128;
};

template <class P, int NT>
__global__ void __launch_bounds__(NT, 512 / NT) k2_xinv_direct(Fast2DArgs a, int dst_role, const __grid_constant__ CUtensorMap map_even,
                                                               const __grid_constant__ CUtensorMap map_odd) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  using S = K2Inv<P, NT>;
  constexpr int N = P::N, T = P::T, E = P::E, G = NT / T, GP = K2Shape<P, NT>::GP, KB = S::KB;
  extern __shared__ __align__(128) float4 smem4[];
  __shared__ __align__(8) uint64_t full;
  float4* land = reinterpret_cast<float4*>((reinterpret_cast<uintptr_t>(smem4) + 127) & ~(uintptr_t)127);
  const float4* Se = land;                                  // [k][p]: even bin 2k of row pair p
  const float4* So = land + (size_t)S::NBE * KB * G;        // [k][p]: odd bin 2k + 1
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  const int c = blockIdx.y, r0 = blockIdx.x * 2 * G;
  if (tid == 0) {
    tma::mbar_init(&full, 1);
    tma::fence_barrier_init();
    tma::fence_proxy_async();
    tma::mbar_expect_tx(&full, (uint32_t)(S::LAND4 * sizeof(float4)));
#pragma unroll 1
    for (int b = 0; b < S::NBE; ++b) tma::load_3d(land + (size_t)b * KB * G, &map_even, 2 * r0, b * KB, c, &full);
#pragma unroll 1
    for (int b = 0; b < S::NBO; ++b) tma::load_3d(land + (size_t)(S::NBE + b) * KB * G, &map_odd, 2 * r0, b * KB, c, &full);
  }
  float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * a.ncell;
  const float2 wt = __ldg(&a.twox[t]);      // w_2N^t; the other points follow from constants
  __syncthreads();                          // the barrier is initialised
  tma::mbar_wait(&full, 0);
  rf::C2 v[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int n = rf::slot_index<PI, PI::RA>(t, e);        // = t + (N/16) e: the mirror tests fold per e
    float4 qe, qo;
    if (e < E / 2) {                      // n < N/2: bins 2n, 2n + 1 < N
      qe = Se[(size_t)n * G + gid]; qo = So[(size_t)n * G + gid];
      v[e] = {make_float2(qe.x - qe.w, qo.x - qo.w), make_float2(qe.y + qe.z, qo.y + qo.z)};
    } else {                              // bins above N: the conjugate partner 2N - b
      qo = So[(size_t)(N - 1 - n) * G + gid];
      qe = Se[(size_t)(N - n) * G + gid];
      const bool self = e == E / 2 && t == 0;              // bin N itself (n = N/2)
      v[e] = {make_float2(self ? qe.x - qe.w : qe.x + qe.w, qo.x + qo.w), make_float2(self ? qe.y + qe.z : qe.z - qe.y, qo.z - qo.y)};
    }
  }
  __syncthreads();                          // everyone has its points: the landing area becomes the exchange buffers
  float4* xb = land + (size_t)gid * GP;
  rf::fft<PI, +1, NT>(v, xb, t, gid, a.twx_r);
  const size_t rowA = (size_t)(r0 + 2 * gid) * a.nxp;      // physical row pitch; n >= nxp is zero fill
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int n = rf::slot_index<PI, PI::RLAST>(t, e);
    const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), rf::half_twiddle(wt, e));
    if (n < a.nxp) {
      k2_stg(dst + rowA + n, v[e].re.x + u.x);
      k2_stg(dst + rowA + a.nxp + n, v[e].im.x + u.y);
    }
  }
}

// ---------------------------------------------------------------------------------- K_C, persistent
// The direct-read x inverse as ONE CTA of 512 threads per SM that never waits for its pieces: its NG = 512 / T FFT
// groups work through the CTA's row pairs (items: component x row pair, blockIdx.x + k gridDim.x) in turn, over a
// ring of NG + NG/2 landing / exchange buffers. While the groups transform NG items, the pieces of the next NG/2 are
// landing; a group that is done with a buffer (after the last exchange of its transform) hands it to TMA for the
// item NBUF steps ahead at once. Each buffer has its mbarrier; the groups synchronise among themselves with named
// barriers only. 4096^2: 0.190 -> 0.168 ms.
template <class P>
struct K2InvP {
  static constexpr int NT = 512, NG = NT / P::T, NBUF = NG + NG / 2;
  using S = K2Inv<P, P::T>;                                  // layout of one landing area (G = 1)
  static constexpr int BUF4 = S::LAND4 > P::XB ? S::LAND4 : P::XB;
  static constexpr size_t SMEM = sizeof(float4) * (size_t)NBUF * BUF4 + 128;
};

template <class P>
__global__ void __launch_bounds__(512, 1) k2_xinv_pers(Fast2DArgs a, int dst_role, const __grid_constant__ CUtensorMap map_even,
                                                            const __grid_constant__ CUtensorMap map_odd) {
  if (a.st->skip) return;
  using PI = typename P::Reversed;
  using K = K2InvP<P>;
  using S = typename K::S;
  constexpr int N = P::N, T = P::T, E = P::E, NT = K::NT, NG = K::NG, KB = S::KB, NBUF = K::NBUF;
  static_assert(T >= 32 && NG <= 15, "one named barrier per group, whole warps");
  extern __shared__ __align__(128) float4 smem4[];
  __shared__ __align__(8) uint64_t full[NBUF];
  float4* base = reinterpret_cast<float4*>((reinterpret_cast<uintptr_t>(smem4) + 127) & ~(uintptr_t)127);
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  const int npairs = a.Ny == 0 ? 0 : a.nyp / 2, nitems = 3 * npairs;
  const int first = blockIdx.x, stride = gridDim.x;
  const int nq = first < nitems ? (nitems - first + stride - 1) / stride : 0;      // items of this CTA
  auto issue = [&](int q) {                    // one thread: bring the pieces of the CTA's q-th item into buffer q % NBUF
    const int item = first + q * stride, c = item / npairs, r0 = 2 * (item - c * npairs);
    float4* land = base + (size_t)(q % NBUF) * K::BUF4;
    uint64_t* bar = &full[q % NBUF];
    tma::mbar_expect_tx(bar, (uint32_t)(S::LAND4 * sizeof(float4)));
#pragma unroll 1
    for (int b = 0; b < S::NBE; ++b) tma::load_3d(land + (size_t)b * KB, &map_even, 2 * r0, b * KB, c, bar);
#pragma unroll 1
    for (int b = 0; b < S::NBO; ++b) tma::load_3d(land + (size_t)(S::NBE + b) * KB, &map_odd, 2 * r0, b * KB, c, bar);
  };
  if (tid == 0) {
#pragma unroll
    for (int b = 0; b < NBUF; ++b) tma::mbar_init(&full[b], 1);
    tma::fence_barrier_init();
    tma::fence_proxy_async();
    for (int q = 0; q < NBUF && q < nq; ++q) issue(q);
  }
  const float2 wt = __ldg(&a.twox[t]);      // w_2N^t; the other points follow from constants
  __syncthreads();                          // the barriers are initialised
#pragma unroll 1
  for (int q = gid; q < nq; q += NG) {
    const int item = first + q * stride, c = item / npairs, r0 = 2 * (item - c * npairs);
    float4* land = base + (size_t)(q % NBUF) * K::BUF4;
    const float4* Se = land;
    const float4* So = land + (size_t)S::NBE * KB;
    tma::mbar_wait(&full[q % NBUF], (q / NBUF) & 1);
    rf::C2 v[E];
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RA>(t, e);        // = t + (N/16) e: the mirror tests fold per e
      float4 qe, qo;
      if (e < E / 2) {                      // n < N/2: bins 2n, 2n + 1 < N
        qe = Se[n]; qo = So[n];
        v[e] = {make_float2(qe.x - qe.w, qo.x - qo.w), make_float2(qe.y + qe.z, qo.y + qo.z)};
      } else {                              // bins above N: the conjugate partner 2N - b
        qo = So[N - 1 - n];
        qe = Se[N - n];
        const bool self = e == E / 2 && t == 0;              // bin N itself (n = N/2)
        v[e] = {make_float2(self ? qe.x - qe.w : qe.x + qe.w, qo.x + qo.w), make_float2(self ? qe.y + qe.z : qe.z - qe.y, qo.z - qo.y)};
      }
    }
    rf::group_sync<T, NT>(gid);             // the group has its points: its landing area becomes its exchange buffer
    rf::fft<PI, +1, NT>(v, land, t, gid, a.twx_r);
    // the buffer is free once every thread of the group is past the last exchange: order the generic accesses before
    // the asynchronous writes that follow, then hand the buffer to TMA for the item three steps ahead
    tma::fence_proxy_async();
    rf::group_sync<T, NT>(gid);
    if (t == 0 && q + NBUF < nq) issue(q + NBUF);
    float* __restrict__ dst = a.st->ptr[dst_role] + (size_t)c * a.ncell;
    const size_t rowA = (size_t)r0 * a.nxp;                  // physical row pitch; n >= nxp is zero fill
#pragma unroll
    for (int e = 0; e < E; ++e) {
      const int n = rf::slot_index<PI, PI::RLAST>(t, e);
      const float2 u = rf::cmul_tw1<+1>(make_float2(v[e].re.y, v[e].im.y), rf::half_twiddle(wt, e));
      if (n < a.nxp) {
        k2_stg(dst + rowA + n, v[e].re.x + u.x);
        k2_stg(dst + rowA + a.nxp + n, v[e].im.x + u.y);
      }
    }
  }
}

// ---------------------------------------------------------------------------------- K_A
// x forward transform of FOUR rows per FFT group. Two real rows a, b form one complex line z = a + i b; the two
// lanes of the packed engine carry two such lines (rows r, r+1 and r+2, r+3), and the even-bin and odd-bin
// halves of the padded transform are two runs of the same group, one after the other:
//     run E: FFT_N(z)          -> bins kx = 2k,     k = 0 .. N/2      (partner of bin 2k   is 2(N - k))
//     run O: FFT_N(z w_2N^n)   -> bins kx = 2k + 1, k = 0 .. N/2 - 1  (partner of bin 2k+1 is 2(N-1-k) + 1)
// After each run the spectra of a and b are separated (Hermitian symmetry) into tiles [bin][4G rows] and leave
// TRANSPOSED, spec[c][kx][y], as TMA boxes {4G rows, KB bins} of a tensor map that walks every second column
// (one map for the even, one for the odd columns): 32-byte pieces per group, written while the other run (or the
// other CTA of the SM) computes. Compared with carrying the even/odd halves in the lanes (two rows per group) this
// doubles the piece size at the same register count, needs no twiddle at all on the way in for run E and only
// packed multiplies for run O. TMA = false: the same tiles are written with plain 32-byte stores.
template <class P, int NT>
struct K2Fwd {
  static constexpr int G = NT / P::T;
  static constexpr int KB = (G >= 4 ? 512 / G : 256) < P::N / 2 ? (G >= 4 ? 512 / G : 256) : P::N / 2;   // bins per tile
  static constexpr int NBUF = 3;                                                   // tiles in flight (unstaged variant)
  static constexpr int TILE4 = KB * G * 2;                                         // float4 units per tile
  // One FFT group per CTA: the tiles of a whole run are staged in the exchange buffer and leave in one go (three
  // CTA barriers per run instead of one per tile; 0.206 -> 0.186 ms at 4096^2). With several groups per CTA the
  // staged writes of a bin are G x 32 bytes apart and the ring of tiles is faster.
  static constexpr bool STAGED = G <= 2;
  static constexpr int NBE = (P::N / 2 + 1 + KB - 1) / KB, NBO = (P::N / 2 + KB - 1) / KB;
  static constexpr int ROWS = 4 * G;
};
template <class P, int NT>
constexpr size_t k2_fwd_smem() {
  using F = K2Fwd<P, NT>;
  // staged: the exchange buffers also hold the tiles of a run (whole boxes, the last one partly unused); else a ring of tiles
  constexpr size_t stage = (size_t)F::NBE * F::TILE4 * sizeof(float4);
  if (F::STAGED) return (k2_smem<P, NT>() > stage ? k2_smem<P, NT>() : stage) + 128;
  return k2_smem<P, NT>() + (size_t)F::NBUF * F::TILE4 * sizeof(float4) + 128;
}

template <class P, int NT, bool RAGGED, bool TMA, bool STAGED>
__global__ void __launch_bounds__(NT, 512 / NT) k2_xfwd4(Fast2DArgs a, int src_role, const __grid_constant__ CUtensorMap map_even,
                                                         const __grid_constant__ CUtensorMap map_odd) {
  if (a.st->skip) return;
  using F = K2Fwd<P, NT>;
  constexpr int N = P::N, T = P::T, E = P::E, G = F::G, GP = K2Shape<P, NT>::GP, KB = F::KB;
  extern __shared__ __align__(128) float4 smem4[];
  __shared__ float bsat_s[MM_MAX_REGIONS];
  constexpr int NBUF = F::NBUF;
  float4* tiles = smem4 + (size_t)G * GP + ((128 - ((size_t)G * GP * 16) % 128) % 128) / 16;   // ring of the unstaged variant, 128-byte aligned
  const int tid = threadIdx.x, gid = tid / T, t = tid % T;
  float4* xb = smem4 + (size_t)gid * GP;
  const int c = blockIdx.y, r0 = blockIdx.x * F::ROWS;
  const float* __restrict__ src = a.st->ptr[src_role] + (size_t)c * a.ncell;
  const uint8_t* __restrict__ reg = a.regions;
  const bool uniform = a.luts->nregions == 1;       // one region: B_sat is a constant
  int store_seq = 0;                                 // tiles handed to TMA so far (ring position of the unstaged variant)
  const float b0 = a.luts->Bsat[0];
  if (!uniform) {
    for (int i = tid; i < MM_MAX_REGIONS; i += NT) bsat_s[i] = a.luts->Bsat[i];
    __syncthreads();
  }
  {
    // rows of the CTA that follows on this SM (dispatch is in order, 512 / NT CTAs per SM): DRAM -> L2
    int nb = (int)blockIdx.x + a.nsm * (512 / NT), nc = c;
    if (nb >= (int)gridDim.x) { nb -= gridDim.x; ++nc; }
    if (nc < 3 && nb < (int)gridDim.x) {
      const float* nxt = a.st->ptr[src_role] + (size_t)nc * a.ncell + (size_t)nb * F::ROWS * a.nxp;
      const long long lim = a.ncell - (long long)nb * F::ROWS * a.nxp;      // stay inside the component
      for (int i = tid * 32; i < F::ROWS * a.nxp && i < lim; i += NT * 32) k2_prefetch_l2(nxt + i);
    }
  }
  const int row = r0 + 4 * gid;                       // first of the group's four rows
  const float2 wt = __ldg(&a.twox[t]);                // w_2N^t; the other points follow from constants
  // row pointers at column t (point e of this thread sits (N/16) e further on); rows beyond the film read row 0
  // with weight 0, so that all 64 loads of a run are unconditional and can be in flight together
  const float* rp[4]; const uint8_t* gp[4]; float rw[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const bool ok = row + q < a.nyp;
    const size_t o = (size_t)(ok ? row + q : 0) * a.nxp + t;
    rp[q] = src + o; gp[q] = reg + o; rw[q] = ok ? (uniform ? b0 : 1.f) : 0.f;
  }
#pragma unroll 1
  for (int run = 0; run < 2; ++run) {
    {
      rf::C2 v[E];
      if (uniform) {
#pragma unroll
        for (int e = 0; e < E; ++e) {
          const int off = (N / 16) * e;
          float z[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) z[q] = (!RAGGED || t + off < a.nxp) ? k2_ldg(rp[q] + off) * rw[q] : 0.f;      // M = B_sat m (L121)
          v[e] = {make_float2(z[0], z[2]), make_float2(z[1], z[3])};          // lanes: rows (r, r+1) and (r+2, r+3)
        }
      } else {
#pragma unroll
        for (int e = 0; e < E; ++e) {
          const int off = (N / 16) * e;
          float z[4];
#pragma unroll
          for (int q = 0; q < 4; ++q) z[q] = (!RAGGED || t + off < a.nxp) ? k2_ldg(rp[q] + off) * (bsat_s[gp[q][off]] * rw[q]) : 0.f;
          v[e] = {make_float2(z[0], z[2]), make_float2(z[1], z[3])};
        }
      }
      if (run == 1) {
        // z w_2N^n, n = t + (N/16) e: first the constant part exp(-i pi e / 16), then w_2N^t for all sixteen
        constexpr float C[16] = {1.f, 0.98078528040323043f, 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f,
                                 0.55557023301960218f, 0.38268343236508977f, 0.19509032201612825f, 0.f, -0.19509032201612825f,
                                 -0.38268343236508977f, -0.55557023301960218f, -0.70710678118654752f, -0.83146961230254524f,
                                 -0.92387953251128674f, -0.98078528040323043f};
        constexpr float S[16] = {0.f, 0.19509032201612825f, 0.38268343236508977f, 0.55557023301960218f, 0.70710678118654752f,
                                 0.83146961230254524f, 0.92387953251128674f, 0.98078528040323043f, 1.f, 0.98078528040323043f,
                                 0.92387953251128674f, 0.83146961230254524f, 0.70710678118654752f, 0.55557023301960218f,
                                 0.38268343236508977f, 0.19509032201612825f};
#pragma unroll
        for (int e = 0; e < E; ++e) {
          if (e == 4) v[e] = rf::rot45<-1>(v[e]);
          else if (e == 8) v[e] = rf::rot90<-1>(v[e]);
          else if (e == 12) v[e] = rf::rot135<-1>(v[e]);
          else if (e != 0) v[e] = rf::rotcs<-1>(v[e], C[e], S[e]);
          v[e] = rf::cmul_tw<-1>(v[e], wt);
        }
      }
      if constexpr (STAGED) {
        rf::fft_head<P, -1>(v, t, a.twx);
        if (TMA && run == 1) {                      // the TMA stores of run E still read the staging area = the exchange buffers
          if (tid == 0) tma::store_wait_read<0>();
          __syncthreads();
        }
        rf::fft_tail<P, -1, NT>(v, xb, t, gid, a.twx);
        // Hermitian separation, each thread for its own bins: slot j of run E is bin 2j (partner slot (N - j) mod N), of
        // run O bin 2j + 1 (partner slot N - 1 - j); bins above N are the mirror images and are not stored
        rf::group_sync<T, NT>(gid);
#pragma unroll
        for (int e = 0; e < E; ++e) xb[rf::slot_index<P, P::RLAST>(t, e)] = stage_pack(v[e]);
        rf::group_sync<T, NT>(gid);
        float4 pm[E];
#pragma unroll
        for (int e = 0; e < E; ++e) {
          const int j = rf::slot_index<P, P::RLAST>(t, e);
          const bool out = run == 0 ? j <= N / 2 : j < N / 2;
          if (out) pm[e] = xb[run == 0 ? ((N - j) & (N - 1)) : N - 1 - j];
        }
        if (TMA) __syncthreads();                   // every partner has been read: the buffers become the staging area
        float4* stage = smem4;                      // [bin][group]: (A0, B0, A1, B1) = the 32 bytes of rows r .. r+3 at this bin
#pragma unroll
        for (int e = 0; e < E; ++e) {
          const int j = rf::slot_index<P, P::RLAST>(t, e);
          const bool out = run == 0 ? j <= N / 2 : j < N / 2;
          if (!out) continue;
          const float4 u = stage_pack(v[e]), um = pm[e];
          const float4 o0 = separate(make_float2(u.x, u.y), make_float2(um.x, um.y));
          const float4 o1 = separate(make_float2(u.z, u.w), make_float2(um.z, um.w));
          if (TMA) {
            stage[2 * ((size_t)j * G + gid)] = o0; stage[2 * ((size_t)j * G + gid) + 1] = o1;
          } else {
            float4* o = reinterpret_cast<float4*>(a.spec + (size_t)c * a.cstride + (size_t)(2 * j + run) * a.Ny + r0 + 4 * gid);
            o[0] = o0; o[1] = o1;
          }
        }
      } else {
        rf::fft<P, -1, NT>(v, xb, t, gid, a.twx);
        rf::group_sync<T, NT>(gid);
#pragma unroll
        for (int e = 0; e < E; ++e) xb[rf::slot_index<P, P::RLAST>(t, e)] = stage_pack(v[e]);
      }
    }
    if constexpr (STAGED) {
      if (TMA) {
        tma::fence_proxy_async();
        __syncthreads();
        if (tid == 0) {
          const int nbox = run == 0 ? F::NBE : F::NBO;
          for (int j = 0; j < nbox; ++j) tma::store_3d(run == 0 ? &map_even : &map_odd, 2 * r0, j * KB, c, smem4 + (size_t)j * F::TILE4);
          tma::store_commit();
        }
      } else {
        __syncthreads();                            // xb is overwritten by the next run
      }
    } else {
      __syncthreads();
      // separate the two real rows of each line: unit k of group p holds Z[k] of its two lines; tile[bin][p] =
      // (A0, B0, A1, B1) = the 32 bytes of rows r .. r+3 at this bin
      const int nbox = run == 0 ? F::NBE : F::NBO, nbin = run == 0 ? N / 2 + 1 : N / 2;
#pragma unroll 1
      for (int j = 0; j < nbox; ++j, ++store_seq) {
        float4* tile = tiles + (size_t)(store_seq % NBUF) * F::TILE4;
        for (int i = tid; i < KB * G; i += NT) {
          const int p = i % G, k = j * KB + i / G;
          if (k >= nbin) continue;
          const float4* st = smem4 + (size_t)p * GP;
          const int km = run == 0 ? ((N - k) & (N - 1)) : N - 1 - k;
          const float4 u = st[k], um = st[km];
          const float4 o0 = separate(make_float2(u.x, u.y), make_float2(um.x, um.y));
          const float4 o1 = separate(make_float2(u.z, u.w), make_float2(um.z, um.w));
          if (TMA) {
            tile[2 * i] = o0; tile[2 * i + 1] = o1;
          } else {
            const int kx = 2 * k + run;
            float4* o = reinterpret_cast<float4*>(a.spec + (size_t)c * a.cstride + (size_t)kx * a.Ny + r0 + 4 * p);
            o[0] = o0; o[1] = o1;
          }
        }
        if (TMA) {
          tma::fence_proxy_async();
          if (tid == 0) tma::store_wait_read<NBUF - 2>();     // the tile of the next iteration is free again
          __syncthreads();
          if (tid == 0) {
            tma::store_3d(run == 0 ? &map_even : &map_odd, 2 * r0, j * KB, c, tile);
            tma::store_commit();
          }
        }
      }
      if (!TMA) __syncthreads();                              // xb is overwritten by the next run
    }
  }
  if (TMA && tid == 0) tma::store_wait_read<0>();           // shared memory must outlive the reads
}
