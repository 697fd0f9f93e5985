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
template <int N> constexpr int cy() { return 256 / Plan3<N>::P::T; }
#ifndef MM_F3_ZTHREADS
#define MM_F3_ZTHREADS 128
#endif
template <int N> constexpr int cz() { return MM_F3_ZTHREADS / Plan3<N>::P::T; }
constexpr int kZMinBlocks = MM_F3_ZTHREADS == 128 ? 1 : 3;
template <int N> constexpr size_t smem_y() { return sizeof(float4) * (size_t)N * cy<N>(); }
template <int N> constexpr size_t smem_z() { return K3Z<typename Plan3<N>::P, cz<N>()>::SMEM; }

template <int N>
int attrs_y(mm_sim* s) {
  using P = typename Plan3<N>::P;
  CUDA_TRY(s, cudaFuncSetAttribute(k3_y<P, cy<N>(), false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_y<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_y<P, cy<N>(), true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_y<N>()));
  return MM_OK;
}
template <int N>
int attrs_z(mm_sim* s) {
  using P = typename Plan3<N>::P;
  CUDA_TRY(s, cudaFuncSetAttribute(k3_z<P, cz<N>(), kZMinBlocks>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_z<N>()));
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
  const dim3 grid((s->g.Cx + C - 1) / C, s->g.Nz, 3);
  if (inverse) k3_y<P, C, true><<<grid, P::T * C, smem_y<N>(), s->stream>>>(s->f3);
  else k3_y<P, C, false><<<grid, P::T * C, smem_y<N>(), s->stream>>>(s->f3);
}
template <int N>
void launch_z(mm_sim* s) {
  using P = typename Plan3<N>::P;
  constexpr int C = cz<N>();
  const dim3 grid((s->g.Cx + C - 1) / C, s->g.Py);
  k3_z<P, C, kZMinBlocks><<<grid, 3 * P::T * C, smem_z<N>(), s->stream>>>(s->f3);
}

template <int N> constexpr int gx() { return 256 / Plan3<N>::P::T; }
template <int N> constexpr size_t smem_x() { return sizeof(float4) * (size_t)f3::row_pitch<typename Plan3<N>::P>() * gx<N>(); }
template <int N>
int attrs_x(mm_sim* s) {
  using P = typename Plan3<N>::P;
  CUDA_TRY(s, cudaFuncSetAttribute(k3_xfwd<P, gx<N>()>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x<N>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k3_xinv<P, gx<N>()>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_x<N>()));
  return MM_OK;
}
template <int N>
void launch_x(mm_sim* s, bool inverse, int role) {
  using P = typename Plan3<N>::P;
  constexpr int G = gx<N>();
  const int npairs = s->g.Ny * s->g.Nz / 2;
  const dim3 grid((npairs + G - 1) / G, 3);
  if (inverse) k3_xinv<P, G><<<grid, P::T * G, smem_x<N>(), s->stream>>>(s->f3, role);
  else k3_xfwd<P, G><<<grid, P::T * G, smem_x<N>(), s->stream>>>(s->f3, role);
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

// open boxes whose y and z extents are powers of two from 32 to 512 cells (the padded length of such an axis is
// exactly twice its extent); the x stage stays with the generic kernels
bool mm_fast3d_supported(int Nx, int Ny, int Nz, const int* pbc) {
  (void)Nx;
  return !pbc[0] && !pbc[1] && !pbc[2] && pow2_in_range(Ny) && pow2_in_range(Nz);
}

int mm_fast3d_init(mm_sim* s) {
  const Geometry& g = s->g;
  if (g.Py != 2 * g.Ny || g.Pz != 2 * g.Nz) { s->fast3d = false; return MM_OK; }
  Fast3DArgs& a = s->f3;
  a.g = g;
  a.spec = s->spec;
  a.cstride = (long long)g.Nz * g.Py * g.pitch;
  a.st = s->dstate;
  a.regions = s->regions; a.luts = s->luts;
  a.Nxt = (pow2_in_range(g.Nx) && g.Px == 2 * g.Nx) ? g.Nx : 0;
  float2 *f, *r, *h;
  int rc = MM_OK;
#define TY(N) rc = mm_plan_tables<Plan3<N>::P>(s, &f, &r, &h)
  if (a.Nxt) {
    F3_SWITCH(a.Nxt, TY)
    if (rc) return rc;
    a.twx = f; a.twx_r = r; a.twox = h;
#define AX(N) rc = attrs_x<N>(s)
    F3_SWITCH(a.Nxt, AX)
#undef AX
    if (rc) return rc;
  }
  F3_SWITCH(g.Ny, TY)
  if (rc) return rc;
  a.twy = f; a.twy_r = r; a.twoy = h;
  F3_SWITCH(g.Nz, TY)
  if (rc) return rc;
  a.twz = f; a.twz_r = r; a.twoz = h;
#undef TY
#define AY(N) rc = attrs_y<N>(s)
#define AZ(N) rc = attrs_z<N>(s)
  F3_SWITCH(g.Ny, AY)
  if (rc) return rc;
  F3_SWITCH(g.Nz, AZ)
#undef AY
#undef AZ
  return rc;
}

bool mm_fast3d_x(mm_sim* s, bool inverse, int role) {      // false: this box keeps the generic x stage
  if (!s->f3.Nxt) return false;
#define LX(N) launch_x<N>(s, inverse, role)
  F3_SWITCH(s->f3.Nxt, LX)
#undef LX
  return true;
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
