// fast3d.cu - host side of the register-FFT y and z stages of open 3D boxes (fast3d.cuh): plans, tables, launches.
#include "internal.cuh"
#include "fast3d.cuh"
#include "fft_tables.cuh"

namespace {

// radix plans of the strided axes: sixteen points per thread, T = N / 16 threads per line
template <int N> struct Plan3;
template <> struct Plan3<32> { using P = rf::Plan<32, 2, 16, 2, 1>; };
template <> struct Plan3<64> { using P = rf::Plan<64, 4, 16, 4, 1>; };
template <> struct Plan3<128> { using P = rf::Plan<128, 8, 16, 8, 1>; };
template <> struct Plan3<256> { using P = rf::Plan<256, 16, 16, 16, 1>; };
template <> struct Plan3<512> { using P = rf::Plan<512, 32, 16, 2, 16>; };

// lines per CTA: 256 threads in the y stage, 3 x 128 in the fused z stage
// lines per CTA. Several small CTAs per SM overlap their phases better than few large ones (measured at 256^3 and 128^3):
// 128 threads in the y stage (0.254 -> 0.242 ms, 0.041 -> 0.034 ms), in the x inverse (0.161 -> 0.134 ms) and in the
// periodic x forward kernel (0.123 -> 0.110 ms); the open x forward kernel keeps 256 (0.223 ms; 0.254 ms with 128).
template <int N> constexpr int cy() { return 128 / Plan3<N>::P::T; }
// CTA shape of the fused z stage, measured per line length (threads per component, CTAs per SM):
//   512 points: 128 threads (C = 4 lines), one CTA of 384 threads per SM (fewer lines per CTA would mean 16-byte pieces);
//   128, 256 : 64 threads (C = 8 / 4), two CTAs of 192 threads at 167 registers - two independent CTAs overlap their
//              phases where one of 384 threads cannot (128^3: 0.138 -> 0.109 ms, 256^3 with PBC: 0.300 -> 0.254 ms,
//              256^3 open: unchanged);
//   32, 64   : 64 threads, three CTAs at 96 registers (spills, but a short-line CTA is mostly latency: C3 0.048 -> 0.037 ms).
template <int N> constexpr int zthreads() { return N >= 512 ? 128 : 64; }
template <int N> constexpr int cz() { return zthreads<N>() / Plan3<N>::P::T; }
template <int N> constexpr int zminb() { return N <= 64 ? 3 : (N >= 512 ? 1 : 2); }
template <int N> constexpr size_t smem_y() { return sizeof(float4) * (size_t)N * cy<N>(); }
template <int N> constexpr size_t smem_z() { return K3Z<typename Plan3<N>::P, cz<N>()>::SMEM; }

template <int N>
int attrs_y(mm_sim* s) {
  using P = typename Plan3<N>::P;
  CUDA_TRY(s, cudaFuncSetAttribute(k3_y<P, cy<N>(), false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_y<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_y<P, cy<N>(), true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_y<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_yp<P, cy<N>(), false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_y<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_yp<P, cy<N>(), true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_y<N>()));
  return MM_OK;
}
template <int N>
int attrs_z(mm_sim* s) {
  using P = typename Plan3<N>::P;
  CUDA_TRY(s, cudaFuncSetAttribute(k3_z<P, cz<N>(), zminb<N>()>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_z<N>()));
  // the kernel spectrum in the tile order of the z stage
  constexpr int C = cz<N>();
  const Geometry& g = s->g;
  const int ntiles = (g.Cx + C - 1) / C;
  const size_t n3 = (size_t)g.Hy * ntiles * 6 * g.Hz * C;
  float* K3 = (float*)mm_dev_alloc(s, sizeof(float) * n3);
  if (!K3) return mm_fail(s, MM_ENOMEM, "kernel spectrum (z-stage tiles)");
  k3_pack_kernel<<<s->nsm * 8, 256, 0, s->stream>>>(s->K, K3, g.Cx, g.Hy, g.Hz, C, ntiles);
  s->launches++;
  CUDA_TRY(s, cudaGetLastError());
  s->f3.K3 = K3;
  return MM_OK;
}
template <int N>
void launch_y(mm_sim* s, bool inverse) {
  using P = typename Plan3<N>::P;
  constexpr int C = cy<N>();
  if (s->f3.mode[1] == 2) {                                   // periodic: two neighbouring columns per line group
    const dim3 grid(((s->g.Cx + 1) / 2 + C - 1) / C, s->g.Nz, 3);
    if (inverse) k3_yp<P, C, true><<<grid, P::T * C, smem_y<N>(), s->stream>>>(s->f3);
    else k3_yp<P, C, false><<<grid, P::T * C, smem_y<N>(), s->stream>>>(s->f3);
    return;
  }
  const dim3 grid((s->g.Cx + C - 1) / C, s->g.Nz, 3);
  if (inverse) k3_y<P, C, true><<<grid, P::T * C, smem_y<N>(), s->stream>>>(s->f3);
  else k3_y<P, C, false><<<grid, P::T * C, smem_y<N>(), s->stream>>>(s->f3);
}
template <int N>
void launch_z(mm_sim* s) {
  using P = typename Plan3<N>::P;
  constexpr int C = cz<N>();
  const dim3 grid((s->g.Cx + C - 1) / C, s->g.Py);
  k3_z<P, C, zminb<N>()><<<grid, 3 * P::T * C, smem_z<N>(), s->stream>>>(s->f3);
}

template <int N> constexpr int gxf() { return 256 / Plan3<N>::P::T; }      // x forward, open axis
template <int N> constexpr int gx() { return 128 / Plan3<N>::P::T; }       // x inverse, periodic x forward
template <int N> constexpr size_t smem_x() { return sizeof(float4) * (size_t)f3::row_pitch<typename Plan3<N>::P>() * gx<N>(); }
template <int N> constexpr size_t smem_xf() { return sizeof(float4) * (size_t)f3::row_pitch<typename Plan3<N>::P>() * gxf<N>(); }
template <int N>
int attrs_x(mm_sim* s) {
  using P = typename Plan3<N>::P;
  CUDA_TRY(s, cudaFuncSetAttribute(k3_xfwd<P, gxf<N>()>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_xf<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_xinv<P, gx<N>()>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_xfwd_p<P, gx<N>()>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_xinv_p<P, gx<N>()>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x<N>()));
  return MM_OK;
}
template <int N>
void launch_x(mm_sim* s, bool inverse, int role) {
  using P = typename Plan3<N>::P;
  const bool periodic = s->f3.mode[0] == 2;
  const int nlines = s->g.Ny * s->g.Nz / (periodic ? 4 : 2);      // row pairs, or row quadruples on a periodic axis
  constexpr int G = gx<N>(), GF = gxf<N>();
  const dim3 grid((nlines + G - 1) / G, 3), gridf((nlines + GF - 1) / GF, 3);
  if (periodic) {
    if (inverse) k3_xinv_p<P, G><<<grid, P::T * G, smem_x<N>(), s->stream>>>(s->f3, role);
    else k3_xfwd_p<P, G><<<grid, P::T * G, smem_x<N>(), s->stream>>>(s->f3, role);
  } else {
    if (inverse) k3_xinv<P, G><<<grid, P::T * G, smem_x<N>(), s->stream>>>(s->f3, role);
    else k3_xfwd<P, GF><<<gridf, P::T * GF, smem_xf<N>(), s->stream>>>(s->f3, role);
  }
}

bool pow2_in_range(int n) { return n >= 32 && n <= 512 && (n & (n - 1)) == 0; }

}  // namespace

#define F3_SWITCH(N, CALL)              \
  switch (N) {                          \
    case 32: { CALL(32); break; }       \
    case 64: { CALL(64); break; }       \
    case 128: { CALL(128); break; }     \
    case 256: { CALL(256); break; }     \
    case 512: { CALL(512); break; }     \
  }

// Which stages of a 3D box run on the register engine: an axis qualifies if its extent is a power of two from 32 to
// 512 cells and it is either open (its padded length is then exactly twice the extent) or periodic (not padded;
// x and y only - the rows of a periodic x axis are taken four at a time). The other stages keep the generic kernels;
// all of them share the layout spec[c][z][ky][kx].
void mm_fast3d_modes(const Geometry& g, int* mode) {
  const int N[3] = {g.Nx, g.Ny, g.Nz}, P[3] = {g.Px, g.Py, g.Pz};
  for (int a = 0; a < 3; ++a) {
    mode[a] = 0;
    if (!pow2_in_range(N[a])) continue;
    if (!g.pbc[a] && P[a] == 2 * N[a]) mode[a] = 1;
    else if (g.pbc[a] && P[a] == N[a] && a < 2) mode[a] = 2;
  }
  if (mode[0] == 2 && g.Ny % 4 != 0) mode[0] = 0;
  if (g.Ny % 2 != 0) mode[0] = 0;
  if (g.Nz == 1) mode[0] = mode[1] = mode[2] = 0;           // one-layer films: fast2d.cu or the generic kernels
}

int mm_fast3d_init(mm_sim* s) {
  const Geometry& g = s->g;
  Fast3DArgs& a = s->f3;
  a.g = g;
  mm_fast3d_modes(g, a.mode);
  a.spec = s->spec;
  a.cstride = (long long)g.Nz * g.Py * g.pitch;
  a.st = s->dstate;
  a.regions = s->regions; a.luts = s->luts;
  float2 *f, *r, *h;
  int rc = MM_OK;
#define TY(N) rc = mm_plan_tables<Plan3<N>::P>(s, &f, &r, &h)
#define AX(N) rc = attrs_x<N>(s)
#define AY(N) rc = attrs_y<N>(s)
#define AZ(N) rc = attrs_z<N>(s)
  if (a.mode[0]) {
    F3_SWITCH(g.Nx, TY)
    if (rc) return rc;
    a.twx = f; a.twx_r = r; a.twox = h;
    F3_SWITCH(g.Nx, AX)
    if (rc) return rc;
  }
  if (a.mode[1]) {
    F3_SWITCH(g.Ny, TY)
    if (rc) return rc;
    a.twy = f; a.twy_r = r; a.twoy = h;
    F3_SWITCH(g.Ny, AY)
    if (rc) return rc;
  }
  if (a.mode[2]) {
    F3_SWITCH(g.Nz, TY)
    if (rc) return rc;
    a.twz = f; a.twz_r = r; a.twoz = h;
    F3_SWITCH(g.Nz, AZ)
    if (rc) return rc;
  }
#undef TY
#undef AX
#undef AY
#undef AZ
  return MM_OK;
}

void mm_fast3d_x(mm_sim* s, bool inverse, int role) {
#define LX(N) launch_x<N>(s, inverse, role)
  F3_SWITCH(s->g.Nx, LX)
#undef LX
}
void mm_fast3d_y(mm_sim* s, bool inverse) {
#define LY(N) launch_y<N>(s, inverse)
  F3_SWITCH(s->g.Ny, LY)
#undef LY
}
void mm_fast3d_z(mm_sim* s) {
#define LZ(N) launch_z<N>(s)
  F3_SWITCH(s->g.Nz, LZ)
#undef LZ
}
