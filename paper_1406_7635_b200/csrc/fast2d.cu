// fast2d.cu - host side of the fast 2D demag path: plan tables, kernel-table layout, launches.
#include <cmath>
#include <vector>
#include "internal.cuh"
#include "fast2d.cuh"
#include "fft_tables.cuh"

namespace {

// per length: the radix plan (T threads and 16 points per thread for one pair of transforms) and
// the CTA size NT; a CTA holds G = NT / T FFT groups and therefore 2G rows in the x kernels
template <int N> struct PlanFor;
// (NTF: CTA size of the forward x kernel, four rows per FFT group; NTI: of the inverse one, two rows per group)
template <> struct PlanFor<4096> { using P = rf::Plan<4096, 256, 16, 16, 16>; static constexpr int NT = 256, NTF = 256, NTI = 256; };
template <> struct PlanFor<2048> { using P = rf::Plan<2048, 128, 16, 8, 16>; static constexpr int NT = 256, NTF = 256, NTI = 256; };
template <> struct PlanFor<1024> { using P = rf::Plan<1024, 64, 16, 4, 16>; static constexpr int NT = 256, NTF = 256, NTI = 256; };
template <> struct PlanFor<512> { using P = rf::Plan<512, 32, 16, 2, 16>; static constexpr int NT = 256, NTF = 256, NTI = 256; };
template <> struct PlanFor<256> { using P = rf::Plan<256, 16, 16, 16, 1>; static constexpr int NT = 128, NTF = 128, NTI = 128; };

// 3-D TMA view of spec: floats along y innermost (2 per bin), then kx, then component; one box =
// {rows * 2 floats, kb bins, 1}. The view starts at column kx0 and walks every kstep-th column (nk of them).
// Returns false if the driver entry point is unavailable.
bool make_spec_map(mm_sim* s, int rows, CUtensorMap* out, int kb = K2_KB, int kx0 = 0, int kstep = 1, int nk = -1) {
  typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                               const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                               CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  void* fn = nullptr;
  cudaDriverEntryPointQueryResult qres;
  if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess || !fn ||
      qres != cudaDriverEntryPointSuccess) {
    cudaGetLastError();
    return false;
  }
  const Fast2DArgs& a = s->f2;
  if (nk < 0) nk = a.Cx;
  const cuuint64_t dims[3] = {(cuuint64_t)2 * a.Ny, (cuuint64_t)nk, 3};
  const cuuint64_t strides[2] = {(cuuint64_t)kstep * a.Ny * sizeof(float2), (cuuint64_t)a.cstride * sizeof(float2)};
  const cuuint32_t box[3] = {(cuuint32_t)(2 * rows), (cuuint32_t)kb, 1};
  const cuuint32_t estr[3] = {1, 1, 1};
  return ((EncodeFn)fn)(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void*)(a.spec + (size_t)kx0 * a.Ny), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

template <int N>
int make_axis_tables(mm_sim* s, float2** fwd, float2** rev, float2** half) {
  return mm_plan_tables<typename PlanFor<N>::P>(s, fwd, rev, half);
}

int axis_tables(mm_sim* s, int N, float2** fwd, float2** rev, float2** half) {
  switch (N) {
    case 4096: return make_axis_tables<4096>(s, fwd, rev, half);
    case 2048: return make_axis_tables<2048>(s, fwd, rev, half);
    case 1024: return make_axis_tables<1024>(s, fwd, rev, half);
    case 512: return make_axis_tables<512>(s, fwd, rev, half);
    case 256: return make_axis_tables<256>(s, fwd, rev, half);
  }
  return mm_fail(s, MM_EINVAL, "fast 2D path: unsupported length");
}

// one persistent CTA per SM with two FFT groups and a ring of three landing buffers: plans whose group is 256 threads
// (4096 and 2048 points: 0.190 -> 0.168 ms and 0.059 -> 0.052 ms; the ring of a 1024-point plan does not fit)
template <int N> constexpr bool xinv_persistent() { return PlanFor<N>::P::T >= 128; }
template <int N>
int x_attrs(mm_sim* s) {
  using F = PlanFor<N>;
  const int fb = (int)k2_fwd_smem<typename F::P, F::NTF>();
  CUDA_TRY(s, cudaFuncSetAttribute(k2_xfwd4<typename F::P, F::NTF, false, false, K2Fwd<typename F::P, F::NTF>::STAGED>, cudaFuncAttributeMaxDynamicSharedMemorySize, fb));
  CUDA_TRY(s, cudaFuncSetAttribute(k2_xfwd4<typename F::P, F::NTF, true, false, K2Fwd<typename F::P, F::NTF>::STAGED>, cudaFuncAttributeMaxDynamicSharedMemorySize, fb));
  CUDA_TRY(s, cudaFuncSetAttribute(k2_xfwd4<typename F::P, F::NTF, false, true, K2Fwd<typename F::P, F::NTF>::STAGED>, cudaFuncAttributeMaxDynamicSharedMemorySize, fb));
  CUDA_TRY(s, cudaFuncSetAttribute(k2_xfwd4<typename F::P, F::NTF, true, true, K2Fwd<typename F::P, F::NTF>::STAGED>, cudaFuncAttributeMaxDynamicSharedMemorySize, fb));
  CUDA_TRY(s, cudaFuncSetAttribute(k2_xinv<typename F::P, F::NTI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)k2_smem<typename F::P, F::NTI>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k2_xinv_tma<typename F::P, F::NTI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)k2_tma_smem<typename F::P, F::NTI>()));
  CUDA_TRY(s, cudaFuncSetAttribute(k2_xinv_direct<typename F::P, F::NTI>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)K2Inv<typename F::P, F::NTI>::SMEM));
  if constexpr (xinv_persistent<N>())
    CUDA_TRY(s, cudaFuncSetAttribute(k2_xinv_pers<typename F::P>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                     (int)K2InvP<typename F::P>::SMEM));
  return MM_OK;
}
// the direct-read x inverse wins where one FFT group fills the CTA (its landed pieces are then read without bank
// conflicts); below that the ring version is kept
template <int N> constexpr bool xinv_direct() { return PlanFor<N>::NTI == PlanFor<N>::P::T || N >= 2048; }
template <int N>
int y_attrs(mm_sim* s) {
  using F = PlanFor<N>;
  CUDA_TRY(s, cudaFuncSetAttribute(k2_ycol<typename F::P, F::NT>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   (int)k2_y_smem<typename F::P, F::NT>()));
  return MM_OK;
}

template <int N>
bool launch_xinv_pers(mm_sim* s, int role) {
  if constexpr (xinv_persistent<N>()) {
    using P = typename PlanFor<N>::P;
    if (s->g.Ny % 2 != 0) return false;
    k2_xinv_pers<P><<<s->nsm, K2InvP<P>::NT, K2InvP<P>::SMEM, s->stream>>>(s->f2, role, s->f2_map_invp_even, s->f2_map_invp_odd);
    return true;
  } else {
    (void)s; (void)role;
    return false;
  }
}
template <int N>
void launch_x(mm_sim* s, bool inverse, int role) {
  using F = PlanFor<N>;
  constexpr int GI = F::NTI / F::P::T;
  constexpr int ROWS = K2Fwd<typename F::P, F::NTF>::ROWS;
  const bool ragged = s->f2.nxp < s->f2.Nx;
  const bool tma_on = s->f2_tma && !s->f2_no_tma;
  if (!inverse) {
    const dim3 gf((s->g.Ny + ROWS - 1) / ROWS, 3);
    const size_t b = k2_fwd_smem<typename F::P, F::NTF>();
    if (tma_on) {
      if (ragged) k2_xfwd4<typename F::P, F::NTF, true, true, K2Fwd<typename F::P, F::NTF>::STAGED><<<gf, F::NTF, b, s->stream>>>(s->f2, role, s->f2_map_fwd, s->f2_map_fwd_odd);
      else k2_xfwd4<typename F::P, F::NTF, false, true, K2Fwd<typename F::P, F::NTF>::STAGED><<<gf, F::NTF, b, s->stream>>>(s->f2, role, s->f2_map_fwd, s->f2_map_fwd_odd);
    } else {
      if (ragged) k2_xfwd4<typename F::P, F::NTF, true, false, K2Fwd<typename F::P, F::NTF>::STAGED><<<gf, F::NTF, b, s->stream>>>(s->f2, role, s->f2_map_fwd, s->f2_map_fwd_odd);
      else k2_xfwd4<typename F::P, F::NTF, false, false, K2Fwd<typename F::P, F::NTF>::STAGED><<<gf, F::NTF, b, s->stream>>>(s->f2, role, s->f2_map_fwd, s->f2_map_fwd_odd);
    }
  }
  else if (tma_on && launch_xinv_pers<N>(s, role)) {}
  else if (tma_on && xinv_direct<N>())
    k2_xinv_direct<typename F::P, F::NTI><<<dim3(s->g.Ny / (2 * GI), 3), F::NTI, K2Inv<typename F::P, F::NTI>::SMEM, s->stream>>>(s->f2, role, s->f2_map_inv_even, s->f2_map_inv_odd);
  else if (tma_on)
    k2_xinv_tma<typename F::P, F::NTI><<<dim3(s->g.Ny / (2 * GI), 3), F::NTI, k2_tma_smem<typename F::P, F::NTI>(), s->stream>>>(s->f2, role, s->f2_map_inv);
  else
    k2_xinv<typename F::P, F::NTI><<<dim3(s->g.Ny / (2 * GI), 3), F::NTI, k2_smem<typename F::P, F::NTI>(), s->stream>>>(s->f2, role);
}
// one launch: XY jobs (one column per FFT group) followed by Z jobs (one column per group)
template <int N>
void launch_y(mm_sim* s) {
  using F = PlanFor<N>;
  constexpr int G = F::NT / F::P::T;
  const int nxy = (s->f2.Cx + G - 1) / G, nz = nxy;
  k2_ycol<typename F::P, F::NT><<<nxy + nz, F::NT, k2_y_smem<typename F::P, F::NT>(), s->stream>>>(s->f2, nxy);
}

template <int N> constexpr int rows_inv_of() { return 2 * (PlanFor<N>::NTI / PlanFor<N>::P::T); }
int rows_per_cta(int N) {      // rows of one CTA of the x inverse kernel (the forward kernel pads its last CTA with zero rows)
  switch (N) {
    case 4096: return rows_inv_of<4096>();
    case 2048: return rows_inv_of<2048>();
    case 1024: return rows_inv_of<1024>();
    case 512: return rows_inv_of<512>();
    case 256: return rows_inv_of<256>();
  }
  return 0;
}

template <int N>
bool make_inv_maps(mm_sim* s) {
  using F = PlanFor<N>;
  using I = K2Inv<typename F::P, F::NTI>;
  using IP = K2Inv<typename F::P, F::P::T>;       // one group per landing area (persistent kernel)
  return make_spec_map(s, 2 * I::G, &s->f2_map_inv_even, I::KB, 0, 2, N / 2 + 1) &&
         make_spec_map(s, 2 * I::G, &s->f2_map_inv_odd, I::KB, 1, 2, N / 2) &&
         make_spec_map(s, 2, &s->f2_map_invp_even, IP::KB, 0, 2, N / 2 + 1) &&
         make_spec_map(s, 2, &s->f2_map_invp_odd, IP::KB, 1, 2, N / 2);
}
template <int N>
bool make_fwd_maps(mm_sim* s) {
  using F = K2Fwd<typename PlanFor<N>::P, PlanFor<N>::NTF>;
  return make_spec_map(s, F::ROWS, &s->f2_map_fwd, F::KB, 0, 2, N / 2 + 1) &&
         make_spec_map(s, F::ROWS, &s->f2_map_fwd_odd, F::KB, 1, 2, N / 2);
}

}  // namespace

#define F2_SWITCH(N, CALL)                    \
  switch (N) {                                \
    case 4096: { CALL(4096); break; }         \
    case 2048: { CALL(2048); break; }         \
    case 1024: { CALL(1024); break; }         \
    case 512: { CALL(512); break; }           \
    case 256: { CALL(256); break; }           \
  }

int mm_fast2d_length(int N) {
  int L = 256;
  while (L < N) L *= 2;
  return L;
}

// open one-layer films up to 4096 cells per side; sizes that are not powers of two are zero-filled
// to the next one (any padded length >= 2N - 1 gives the same linear convolution, #4)
bool mm_fast2d_supported(int Nx, int Ny, int Nz, const int* pbc) {
  if (Nz != 1 || pbc[0] || pbc[1] || pbc[2] || Nx > 4096 || Ny > 4096 || Nx < 64 || Ny < 64) return false;
  const int rg = rows_per_cta(mm_fast2d_length(Nx));
  return rg > 0 && Ny % rg == 0 && Nx % 2 == 0;
}

int mm_fast2d_init(mm_sim* s) {
  const Geometry& g = s->g;
  Fast2DArgs& a = s->f2;
  a.Nx = g.Px / 2; a.Ny = g.Py / 2; a.Cx = a.Nx + 1;
  a.nxp = g.Nx; a.nyp = g.Ny;
  {
    int dev = 0, nsm = 148;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
      cudaGetLastError();
      nsm = 148;
    }
    a.nsm = nsm;
  }
  a.ncell = g.N;
  a.spec = s->spec;
  a.cstride = (long long)a.Cx * a.Ny;
  a.Kt = s->Kt;
  a.kstride = (long long)a.Cx * (a.Ny + 1);
  a.regions = s->regions; a.luts = s->luts; a.st = s->dstate;
  float2 *fx, *rx, *hx, *fy, *ry, *hy;
  int rc;
  if ((rc = axis_tables(s, a.Nx, &fx, &rx, &hx))) return rc;
  if ((rc = axis_tables(s, a.Ny, &fy, &ry, &hy))) return rc;
  a.twx = fx; a.twx_r = rx; a.twox = hx; a.twy = fy; a.twy_r = ry; a.twoy = hy;
#define XA(N) if ((rc = x_attrs<N>(s))) return rc
#define YA(N) if ((rc = y_attrs<N>(s))) return rc
  F2_SWITCH(a.Nx, XA)
  F2_SWITCH(a.Ny, YA)
#undef XA
#undef YA
  int rows_inv = 0;
#define RI(N) rows_inv = rows_inv_of<N>()
  F2_SWITCH(a.Nx, RI)
#undef RI
  bool fwd_ok = false;
#define FM(N) fwd_ok = make_fwd_maps<N>(s)
  F2_SWITCH(a.Nx, FM)
#undef FM
  bool inv_ok = false;
#define IM(N) inv_ok = make_inv_maps<N>(s)
  F2_SWITCH(a.Nx, IM)
#undef IM
  s->f2_tma = make_spec_map(s, rows_inv, &s->f2_map_inv) && fwd_ok && inv_ok;
  return MM_OK;
}

// B_demag of the field in role `src` -> role R_B
void mm_fast2d_demag(mm_sim* s, int src_role) {
#define XF(N) launch_x<N>(s, false, src_role)
#define XI(N) launch_x<N>(s, true, R_B)
#define YC(N) launch_y<N>(s)
  { Launch l(s, KK_F2_XFWD); F2_SWITCH(s->f2.Nx, XF) }
  { Launch l(s, KK_F2_YCOL); F2_SWITCH(s->f2.Ny, YC) }
  { Launch l(s, KK_F2_XINV); F2_SWITCH(s->f2.Nx, XI) }
#undef XF
#undef XI
#undef YC
}
