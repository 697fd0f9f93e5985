// mm_api.cu - the C ABI of include/mm.h: handle, host-side planning, launch sequences.
// Every step of the path runs in the kernels of this directory; nothing here computes fields on
// the host and there is no CPU fallback.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "internal.cuh"
#include "demag_conv.cuh"
#include "local_rk.cuh"

namespace {

constexpr int kMaxFft = 8192;
constexpr size_t kSmemMax = 232448;  // 227 KB opt-in limit per CTA on sm_100

// Dormand-Prince 5(4) tableau (PAPER.md L365 names the method; coefficients: DESIGN.md)
const double DP_A[7][6] = {
    {0, 0, 0, 0, 0, 0},
    {1.0 / 5, 0, 0, 0, 0, 0},
    {3.0 / 40, 9.0 / 40, 0, 0, 0, 0},
    {44.0 / 45, -56.0 / 15, 32.0 / 9, 0, 0, 0},
    {19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729, 0, 0},
    {9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656, 0},
    {35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84}};
const double DP_E[7] = {35.0 / 384 - 5179.0 / 57600, 0.0, 500.0 / 1113 - 7571.0 / 16695, 125.0 / 192 - 393.0 / 640,
                        -2187.0 / 6784 + 92097.0 / 339200, 11.0 / 84 - 187.0 / 2100, -1.0 / 40};


// Bogacki-Shampine 3(2) tableau (PAPER.md L366 names the method; textbook coefficients)
const double BS_A[4][6] = {{0, 0, 0, 0, 0, 0}, {1.0 / 2, 0, 0, 0, 0, 0}, {0, 3.0 / 4, 0, 0, 0, 0}, {2.0 / 9, 1.0 / 3, 4.0 / 9, 0, 0, 0}};
const double BS_E[7] = {2.0 / 9 - 7.0 / 24, 1.0 / 3 - 1.0 / 4, 4.0 / 9 - 1.0 / 3, -1.0 / 8, 0, 0, 0};

bool smooth5(int n) {
  for (int f : {2, 3, 5}) while (n % f == 0) n /= f;
  return n == 1;
}

int padded_length(int N, int periodic) {
  if (periodic) return N;
  if (N == 1) return 1;
  int p = 2 * N - 1;
  while (!smooth5(p)) ++p;
  return p;
}

AxisPlan make_plan(int N, int P) {
  AxisPlan pl;
  memset(&pl, 0, sizeof(pl));
  pl.N = N; pl.P = P;
  int r = P;
  for (int f : {8, 4, 2, 3, 5})
    while (r % f == 0 && pl.npass < MM_MAX_PASSES) { pl.radix[pl.npass++] = f; r /= f; }
  return pl;
}

}  // namespace


namespace {

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int copy_in(mm_sim* s, void* dst, const void* src, size_t bytes) {
  CUDA_TRY(s, cudaMemcpyAsync(dst, src, bytes, is_device_ptr(src) ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice,
                              s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));  // host or device source: the caller may reuse or free it on return
  return MM_OK;
}

int copy_out(mm_sim* s, void* dst, const void* src, size_t bytes) {
  CUDA_TRY(s, cudaMemcpyAsync(dst, src, bytes, is_device_ptr(dst) ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost,
                              s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  return MM_OK;
}

int pull_state(mm_sim* s) {
  CUDA_TRY(s, cudaMemcpyAsync(&s->hst, s->dstate, sizeof(DevState), cudaMemcpyDeviceToHost, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  return MM_OK;
}

int push_state(mm_sim* s) {
  CUDA_TRY(s, cudaMemcpyAsync(s->dstate, &s->hst, sizeof(DevState), cudaMemcpyHostToDevice, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  return MM_OK;
}


int upload_twiddles(mm_sim* s, int P, float2** out) {
  std::vector<float2> tw(P);
  for (int k = 0; k < P; ++k) {
    double a = -2.0 * M_PI * (double)k / (double)P;
    tw[k] = make_float2((float)cos(a), (float)sin(a));
  }
  *out = (float2*)mm_dev_alloc(s, sizeof(float2) * P);
  if (!*out) return mm_fail(s, MM_ENOMEM, "twiddle table");
  CUDA_TRY(s, cudaMemcpy(*out, tw.data(), sizeof(float2) * P, cudaMemcpyHostToDevice));
  return MM_OK;
}

template <typename KernelT>
int opt_in_smem(mm_sim* s, KernelT k) {
  CUDA_TRY(s, cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax));
  return MM_OK;
}

int configure_launches(mm_sim* s) {
  const Geometry& g = s->g;
  int rc;
  if ((rc = opt_in_smem(s, k_x_fwd))) return rc;
  if ((rc = opt_in_smem(s, k_x_inv))) return rc;
  if ((rc = opt_in_smem(s, k_y_axis))) return rc;
  if ((rc = opt_in_smem(s, k_last_fused<1>))) return rc;
  if ((rc = opt_in_smem(s, k_last_fused<2>))) return rc;
  if ((rc = opt_in_smem(s, k_last_fused<3>))) return rc;
  auto pick = [](int P, int nbuf, int want_points, int cmax) {
    size_t per = (size_t)nbuf * P * sizeof(float2);
    int c = want_points / P;
    if (c < 1) c = 1;
    if (c > cmax) c = cmax;
    while (c > 1 && per * c > 98304) --c;       // prefer >= 2 CTAs per SM
    return c;
  };
  s->xL = pick(g.Px, 2, 4096, 64);
  s->xSmem = (size_t)2 * s->xL * g.Px * sizeof(float2);
  s->yC = pick(g.Py, 2, 4096, 32);
  s->ySmem = (size_t)2 * s->yC * g.Py * sizeof(float2);
  s->last_along_z = g.Pz > 1;
  const int Pl = s->last_along_z ? g.Pz : g.Py;
  const int ncs[3] = {2, 1, 3};  // coupled components of modes 0, 1, 2
  for (int mode = 0; mode < 3; ++mode) {
    s->lastC[mode] = pick(Pl, ncs[mode] + 1, 4096, 32);
    s->lastSmem[mode] = (size_t)(ncs[mode] + 1) * s->lastC[mode] * Pl * sizeof(float2);
    const bool used = s->last_along_z ? (mode == 2) : (mode != 2);
    if (used && s->lastSmem[mode] > kSmemMax) return mm_fail(s, MM_EINVAL, "FFT length too large for shared memory");
  }
  if (s->xSmem > kSmemMax || s->ySmem > kSmemMax) return mm_fail(s, MM_EINVAL, "FFT length too large for shared memory");
  return MM_OK;
}

// B_demag of the field in role `src` -> role R_B
void launch_demag(mm_sim* s, int src_role) {
  if (s->fast2d && !s->force_generic) { mm_fast2d_demag(s, src_role); return; }
  const Geometry& g = s->g;
  const int rows = g.Ny * g.Nz, pairs = (rows + 1) / 2;
  const int T = 256;
  dim3 gx((pairs + s->xL - 1) / s->xL, 3);
  const bool f3 = s->fast3d && !s->force_generic;
  const bool f3x = f3 && s->f3.mode[0], f3y = f3 && s->f3.mode[1], f3z = f3 && s->f3.mode[2];      // stage by stage
  if (f3x) { Launch l(s, KK_F3_XFWD); mm_fast3d_x(s, false, src_role); }
  else { Launch l(s, KK_XFWD); k_x_fwd<<<gx, T, s->xSmem, s->stream>>>(s->conv, src_role, s->xL); }
  if (s->last_along_z) {
    dim3 gy((g.Cx + s->yC - 1) / s->yC, g.Nz, 3);
    if (f3y) { Launch l(s, KK_F3_Y); mm_fast3d_y(s, false); }
    else if (g.Py > 1) { Launch l(s, KK_YFWD); k_y_axis<<<gy, T, s->ySmem, s->stream>>>(s->conv, 0, s->yC); }
    dim3 gl((g.Cx + s->lastC[2] - 1) / s->lastC[2], g.Py);
    if (f3z) { Launch l(s, KK_F3_Z); mm_fast3d_z(s); }
    else { Launch l(s, KK_LAST_3D); k_last_fused<3><<<gl, T, s->lastSmem[2], s->stream>>>(s->conv, 2, s->lastC[2]); }
    if (f3y) { Launch l(s, KK_F3_Y); mm_fast3d_y(s, true); }
    else if (g.Py > 1) { Launch l(s, KK_YINV); k_y_axis<<<gy, T, s->ySmem, s->stream>>>(s->conv, 1, s->yC); }
  } else {
    dim3 g0((g.Cx + s->lastC[0] - 1) / s->lastC[0]);
    { Launch l(s, KK_LAST_XY); k_last_fused<2><<<g0, T, s->lastSmem[0], s->stream>>>(s->conv, 0, s->lastC[0]); }
    dim3 g1((g.Cx + s->lastC[1] - 1) / s->lastC[1]);
    { Launch l(s, KK_LAST_Z); k_last_fused<1><<<g1, T, s->lastSmem[1], s->stream>>>(s->conv, 1, s->lastC[1]); }
  }
  if (f3x) { Launch l(s, KK_F3_XINV); mm_fast3d_x(s, true, R_B); }
  else { Launch l(s, KK_XINV); k_x_inv<<<gx, T, s->xSmem, s->stream>>>(s->conv, R_B, s->xL); }
}

// can the four-cells-per-thread local kernel (and with it the fused stage / error variants) run on this box?
bool local4_ok(const mm_sim* s) { return s->g.Nx % 4 == 0 && s->g.Ny <= 65535 && s->g.Nz <= 65535; }

// field (out_torque = 0) or torque over gamma (out_torque = 1, 2) of role `src` into role `dst`.
// fuse = 1: also form the next stage input (tableau row sc) into role ynext; fuse = 2: also reduce the
// error norm with weights ec (both need local4_ok and a torque evaluation).
void launch_local(mm_sim* s, int src_role, int dst_role, unsigned mask, int out_torque, int fuse, const StageCoef* scp,
                  const ErrCoef* ecp, int ynext);

void launch_eval(mm_sim* s, int src_role, int dst_role, unsigned mask, int out_torque, int fuse = 0,
                 const StageCoef* scp = nullptr, const ErrCoef* ecp = nullptr, int ynext = R_Y) {
  if (mask & MM_DEMAG) launch_demag(s, src_role);
  launch_local(s, src_role, dst_role, mask, out_torque, fuse, scp, ecp, ynext);
  if (out_torque && s->stt_on) {      // Slonczewski torque on top (Eq. 28); only reached with fuse == 0
    SttArgs p;
    p.pref = s->stt[0]; p.pol = s->stt[1]; p.lam2 = s->stt[2]; p.eps_prime = s->stt[3];
    p.mp[0] = s->stt[4]; p.mp[1] = s->stt[5]; p.mp[2] = s->stt[6];
    Launch l(s, KK_OTHER);
    k_add_stt<<<blocks_for(s->g.N, 256), 256, 0, s->stream>>>(s->g.N, s->regions, s->luts, s->dstate, src_role, dst_role, p);
  }
  if (out_torque && s->zl_on) {       // Zhang-Li torque on top (Eq. 26)
    ZlArgs p;
    const double muB = 9.2740100783e-24, e = 1.602176634e-19, mu0 = 4e-7 * M_PI, xi = s->zl_xi;
    const double c = muB * mu0 / (2.0 * e * s->hst.gamma * (1.0 + xi * xi));           // u = c j / Bsat  [T m]
    for (int a = 0; a < 3; ++a) p.c[a] = (float)(c * s->zl_j[a] / (2.0 * s->cell[a]));
    p.xi = (float)xi;
    Launch l(s, KK_OTHER);
    k_add_zl<<<blocks_for(s->g.N, 256), 256, 0, s->stream>>>(s->g, s->regions, s->luts, s->dstate, src_role, dst_role, p);
  }
}

void launch_local(mm_sim* s, int src_role, int dst_role, unsigned mask, int out_torque, int fuse, const StageCoef* scp,
                  const ErrCoef* ecp, int ynext) {
  Launch l(s, KK_LOCAL);
  const Geometry& g = s->g;
  StageCoef sc = {};
  ErrCoef ec = {};
  if (scp) sc = *scp;
  if (ecp) ec = *ecp;
  if (s->dmi_on) mask |= MM_DMI_ON;
  if (local4_ok(s)) {
    const int q = g.Nx / 4, bt = q >= 128 ? 128 : (q >= 64 ? 64 : 32);
    const dim3 grid((q + bt - 1) / bt, g.Ny, g.Nz);
    const bool th = (mask & MM_THERMAL) != 0;
#define MM_LOCAL4(U, T, F, D) k_local4<U, T, F, D><<<grid, bt, 0, s->stream>>>(g, s->regions, s->luts, s->dstate, src_role, R_B, dst_role, mask, out_torque, sc, ec, ynext)
#define MM_LOCAL4_PICK(U, D)                                                                                            \
    do {                                                                                                                \
      if (th) MM_LOCAL4(U, true, 0, D); else if (fuse == 1) MM_LOCAL4(U, false, 1, D);                                   \
      else if (fuse == 2) MM_LOCAL4(U, false, 2, D); else MM_LOCAL4(U, false, 0, D);                                    \
    } while (0)
    if (s->nregions == 1 && !s->geom) { if (s->dmi_on) MM_LOCAL4_PICK(true, true); else MM_LOCAL4_PICK(true, false); }
    else { if (s->dmi_on) MM_LOCAL4_PICK(false, true); else MM_LOCAL4_PICK(false, false); }
#undef MM_LOCAL4_PICK
#undef MM_LOCAL4
    return;
  }
  k_local<<<blocks_for(g.N, 256), 256, 0, s->stream>>>(g, s->regions, s->luts, s->dstate, src_role, R_B, dst_role, mask,
                                                       out_torque);
}

// stage input / new state from m0 and the slopes (k_stage; four cells per thread where the components stay 16-byte aligned)
void launch_stage(mm_sim* s, const StageCoef& sc, int dst_role) {
  const long long N = s->g.N;
  if (N % 4 == 0) k_stage4<<<blocks_for(N / 4, 256), 256, 0, s->stream>>>(N, s->dstate, sc, dst_role);
  else k_stage<<<blocks_for(N, 256), 256, 0, s->stream>>>(N, s->dstate, sc, dst_role);
}

void enqueue_step(mm_sim* s) {
  const long long N = s->g.N;
  const int tq = s->precession ? 1 : 2;                       // torque with / without the precession term
  if (s->solver == MM_RK12) {
    // Heun (L367): y = m + h k1, k2 = tau(y), result m + h (k1 + k2) / 2; no FSAL. With a temperature the
    // thermal field of Eq. 24 is part of both evaluations and changes with the step counter, so k1 is
    // evaluated after k_ctrl_begin has fixed h (the field's amplitude depends on it).
    const unsigned mask = s->terms | (s->temperature > 0 ? MM_THERMAL : 0u);
    { Launch l(s, KK_CTRL); k_ctrl_begin<<<1, 1, 0, s->stream>>>(s->dstate); }
    launch_eval(s, R_M, R_K0, mask, tq);
    StageCoef sc;
    for (int j = 0; j < 6; ++j) sc.a[j] = 0.f;
    sc.n = 1; sc.a[0] = 1.f;
    { Launch l(s, KK_STAGE); launch_stage(s, sc, R_Y); }
    launch_eval(s, R_Y, R_K1, mask, tq);
    sc.n = 2; sc.a[0] = 0.5f; sc.a[1] = 0.5f;
    { Launch l(s, KK_STAGE); launch_stage(s, sc, R_MNEW); }
    ErrCoef ec;
    for (int j = 0; j < 7; ++j) ec.e[j] = 0.f;
    ec.e[0] = -0.5f; ec.e[1] = 0.5f;                          // 2nd-order minus Euler weights
    { Launch l(s, KK_ERROR); k_error<<<s->nsm * 8, 256, 0, s->stream>>>(N, s->dstate, ec); }
    { Launch l(s, KK_CTRL); k_ctrl_end<<<1, 1, 0, s->stream>>>(s->dstate); }
    s->have_k1 = false;
    return;
  }
  const bool bs = s->solver == MM_RK23;
  const int ns = bs ? 4 : 7;                                  // stages; the last one is the FSAL evaluation
  if (!s->have_k1) {
    launch_eval(s, R_M, R_K0, s->terms, tq);
    s->have_k1 = true;
    s->extra_evals++;
  }
  { Launch l(s, KK_CTRL); k_ctrl_begin<<<1, 1, 0, s->stream>>>(s->dstate); }
  auto row = [&](int i) {
    StageCoef sc;
    sc.n = i;
    for (int j = 0; j < 6; ++j) sc.a[j] = (float)(bs ? BS_A[i][j] : DP_A[i][j]);
    return sc;
  };
  ErrCoef ec;
  for (int j = 0; j < 7; ++j) ec.e[j] = (float)(bs ? BS_E[j] : DP_E[j]);
  if (local4_ok(s) && !s->stt_on && !s->zl_on) {
    // fused sequence: y_2 by the stage kernel, then every evaluation also forms the next stage input
    // (alternating between two buffers: the exchange stencil is still reading the current one) and the
    // last one reduces the error norm: ns + 1 fewer launches, no slope is read back right after it is written
    const StageCoef s1 = row(1);
    int cur = (ns == 2) ? R_MNEW : R_Y;
    { Launch l(s, KK_STAGE); launch_stage(s, s1, cur); }
    for (int i = 1; i < ns; ++i) {
      if (i < ns - 1) {
        const StageCoef sn = row(i + 1);
        const int next = (i + 1 == ns - 1) ? R_MNEW : (cur == R_Y ? R_Y2 : R_Y);
        launch_eval(s, cur, R_K0 + i, s->terms, tq, 1, &sn, nullptr, next);
        cur = next;
      } else {
        launch_eval(s, cur, R_K0 + i, s->terms, tq, 2, nullptr, &ec);
      }
    }
  } else {
    for (int i = 1; i < ns; ++i) {
      const StageCoef sc = row(i);
      const int yrole = (i == ns - 1) ? R_MNEW : R_Y;
      { Launch l(s, KK_STAGE); launch_stage(s, sc, yrole); }
      launch_eval(s, yrole, R_K0 + i, s->terms, tq);
    }
    { Launch l(s, KK_ERROR); k_error<<<s->nsm * 8, 256, 0, s->stream>>>(N, s->dstate, ec); }
  }
  { Launch l(s, KK_CTRL); k_ctrl_end<<<1, 1, 0, s->stream>>>(s->dstate); }
}

// One attempted step through a CUDA graph of the launch sequence: all control is on the device (DevState), so the
// sequence of a step is the same every time once the FSAL slope exists; small boxes are launch-bound
// (PAPER.md L503 finds the same below 256 000 cells) and the replay removes the per-kernel launch cost.
// Falls back to plain launches while profiling (events bracket every kernel) or if capture is unavailable.
void drop_graph(mm_sim* s) {
  if (s->graph_exec) { cudaGraphExecDestroy(s->graph_exec); s->graph_exec = nullptr; }
  s->graph_dirty = false;
}

void step_once(mm_sim* s) {
  const bool steady = s->have_k1 || s->solver == MM_RK12;      // Heun evaluates k1 inside every step
  if (s->prof_on || s->no_graph || !steady) { enqueue_step(s); return; }
  if (s->graph_dirty) drop_graph(s);
  if (!s->graph_exec) {
    const long before = s->launches;
    if (cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
      cudaGetLastError(); s->no_graph = true; enqueue_step(s); return;
    }
    enqueue_step(s);
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(s->stream, &g);
    s->graph_launches = s->launches - before;
    s->launches = before;                                      // captured, not executed
    if (e == cudaSuccess) e = cudaGraphInstantiate(&s->graph_exec, g, 0);
    if (g) cudaGraphDestroy(g);
    if (e != cudaSuccess) { cudaGetLastError(); s->graph_exec = nullptr; s->no_graph = true; enqueue_step(s); return; }
  }
  if (cudaGraphLaunch(s->graph_exec, s->stream) != cudaSuccess) { cudaGetLastError(); s->no_graph = true; drop_graph(s); enqueue_step(s); return; }
  s->launches += s->graph_launches;
}

// thermal field: Heun and a fixed step only (L310)
int check_thermal(mm_sim* s) {
  if (s->temperature > 0 && (s->solver != MM_RK12 || !(s->hst.fix_dt > 0)))
    return mm_fail(s, MM_ESTATE, "a temperature needs the Heun solver (MM_RK12) and a fixed step (PAPER.md L310)");
  return MM_OK;
}

void clear_skip(mm_sim* s) {
  Launch l(s, KK_OTHER);
  k_clear_skip<<<1, 1, 0, s->stream>>>(s->dstate);
}

int check_ready(mm_sim* s) {
  if (!s) return MM_EINVAL;
  if (!s->have_params) return mm_fail(s, MM_ESTATE, "mm_set_params has not been called");
  if (!s->have_m) return mm_fail(s, MM_ESTATE, "mm_set_m has not been called");
  return MM_OK;
}

int status_to_error(mm_sim* s) {
  if (s->hst.status == MM_ENAN) return mm_fail(s, MM_ENAN, "non-finite error estimate");
  if (s->hst.status == MM_EDT) return mm_fail(s, MM_EDT, "step size fell below dt_min");
  return MM_OK;
}

}  // namespace


static thread_local std::string g_create_error;   // text of the last failed mm_create on this thread

void* mm_default_alloc(size_t bytes, void*) {
  void* p = nullptr;
  if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return p;
}
void mm_default_free(void* p, void*) { cudaFree(p); }

int mm_fail(mm_sim* s, int code, const std::string& msg) {
  if (s) s->err = msg;
  return code;
}

void* mm_dev_alloc(mm_sim* s, size_t bytes) {
  void* p = s->alloc(bytes ? bytes : 16, s->alloc_ctx);
  if (!p) return nullptr;
  s->owned.emplace_back(p, bytes);
  s->cur_bytes += bytes;
  if (s->cur_bytes > s->peak_bytes) s->peak_bytes = s->cur_bytes;
  return p;
}

void mm_dev_free(mm_sim* s, void* p) {
  if (!p) return;
  for (size_t i = 0; i < s->owned.size(); ++i)
    if (s->owned[i].first == p) {
      s->cur_bytes -= s->owned[i].second;
      s->owned.erase(s->owned.begin() + i);
      break;
    }
  s->dealloc(p, s->alloc_ctx);
}

extern "C" {

int mm_create(mm_sim** out, int Nx, int Ny, int Nz, double dx, double dy, double dz, int pbc_x, int pbc_y, int pbc_z) {
  return mm_create_ex(out, Nx, Ny, Nz, dx, dy, dz, pbc_x, pbc_y, pbc_z, nullptr, nullptr, nullptr, nullptr);
}

int mm_create_ex(mm_sim** out, int Nx, int Ny, int Nz, double dx, double dy, double dz, int pbc_x, int pbc_y, int pbc_z,
                 void* (*dev_alloc_cb)(size_t, void*), void (*dev_free_cb)(void*, void*), void* alloc_ctx,
                 void* cuda_stream) {
  if (!out) return MM_EINVAL;
  *out = nullptr;
  g_create_error.clear();
  if (Nx < 1 || Ny < 1 || Nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || pbc_x < 0 || pbc_y < 0 || pbc_z < 0 ||
      !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz) || (dev_alloc_cb == nullptr) != (dev_free_cb == nullptr))
  { g_create_error = "bad grid size, cell size, PBC repeats or allocator pair"; return MM_EINVAL; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); g_create_error = "no CUDA device"; return MM_ECUDA; }
  mm_sim* s = new (std::nothrow) mm_sim();
  if (!s) return MM_ENOMEM;
  if (dev_alloc_cb) { s->alloc = dev_alloc_cb; s->dealloc = dev_free_cb; s->alloc_ctx = alloc_ctx; }
  s->stream = (cudaStream_t)cuda_stream;
  if (!s->stream) {
    // No stream given: a stream of the handle's own. It is a blocking stream, so it stays ordered with work the
    // caller issues on the legacy default stream (PyTorch's default), and unlike that one it can be captured
    // into a CUDA graph (the step replay of mm_steps / mm_run).
    if (cudaStreamCreate(&s->stream) != cudaSuccess) { cudaGetLastError(); delete s; g_create_error = "cudaStreamCreate"; return MM_ECUDA; }
    s->own_stream = true;
  }
  {
    int dev = 0, nsm = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && nsm > 0)
      s->nsm = nsm;
    else
      cudaGetLastError();
  }
  s->cell[0] = dx; s->cell[1] = dy; s->cell[2] = dz;
  s->rep[0] = pbc_x; s->rep[1] = pbc_y; s->rep[2] = pbc_z;
  Geometry& g = s->g;
  g.Nx = Nx; g.Ny = Ny; g.Nz = Nz;
  g.N = (long long)Nx * Ny * Nz;
  g.Px = padded_length(Nx, pbc_x); g.Py = padded_length(Ny, pbc_y); g.Pz = padded_length(Nz, pbc_z);
  s->fast2d = mm_fast2d_supported(Nx, Ny, Nz, s->rep);
  if (s->fast2d) {   // fast 2D path: transform length = next power of two, padded length exactly twice that
    g.Px = 2 * mm_fast2d_length(Nx);
    g.Py = 2 * mm_fast2d_length(Ny);
  }
  g.pbc[0] = pbc_x > 0; g.pbc[1] = pbc_y > 0; g.pbc[2] = pbc_z > 0;
  g.dx = (float)dx; g.dy = (float)dy;
  g.inv_dx2 = (float)(1.0 / (dx * dx)); g.inv_dy2 = (float)(1.0 / (dy * dy)); g.inv_dz2 = (float)(1.0 / (dz * dz));
  auto bail = [&](int code, const char* msg) {
    g_create_error = msg;
    mm_destroy(s);
    return code;
  };
  if (g.Px > kMaxFft || g.Py > kMaxFft || g.Pz > kMaxFft) return bail(MM_EINVAL, "padded FFT length above 8192");
  if (!smooth5(g.Px) || !smooth5(g.Py) || !smooth5(g.Pz)) return bail(MM_EINVAL, "periodic axis length must be 2^a 3^b 5^c");
  g.Cx = g.Px / 2 + 1;
  {
    int mode[3];
    mm_fast3d_modes(g, mode);
    s->fast3d = !s->fast2d && (mode[0] || mode[1] || mode[2]);
  }
  // rows of the spectrum start on 128-byte lines when the strided stages read pieces of neighbouring kx
  g.pitch = s->fast3d ? (g.Cx + 15) / 16 * 16 : g.Cx;
  g.Hy = g.Py / 2 + 1; g.Hz = g.Pz / 2 + 1;
  s->px = make_plan(Nx, g.Px); s->py = make_plan(Ny, g.Py); s->pz = make_plan(Nz, g.Pz);
  int rc;
  if ((rc = configure_launches(s))) { std::string m = s->err; return bail(rc, m.c_str()); }
  // device memory
  const size_t fbytes = sizeof(float) * 3 * (size_t)g.N;
  s->regions = (uint8_t*)mm_dev_alloc(s, (size_t)g.N);
  s->luts = (Luts*)mm_dev_alloc(s, sizeof(Luts));
  s->dstate = (DevState*)mm_dev_alloc(s, sizeof(DevState));
  s->scratch3 = (double*)mm_dev_alloc(s, 3 * sizeof(double));
  s->red_part = (double*)mm_dev_alloc(s, (size_t)(3 * 8 * s->nsm + 1) * sizeof(double));   // per-block partials + ticket
  const int rowsS = (g.Pz == 1) ? g.Ny : g.Nz * g.Py;
  const size_t spec_rows = s->fast2d ? (size_t)g.Py / 2 : (size_t)rowsS;      // fast layout: [Cx][Py / 2]
  s->spec = (float2*)mm_dev_alloc(s, sizeof(float2) * 3 * spec_rows * g.pitch);
  if (!s->regions || !s->luts || !s->dstate || !s->spec || !s->scratch3 || !s->red_part) return bail(MM_ENOMEM, "device buffers");
  s->red_ticket = reinterpret_cast<unsigned*>(s->red_part + 3 * 8 * s->nsm);
  if (cudaMemsetAsync(s->red_ticket, 0, sizeof(double), s->stream) != cudaSuccess) return bail(MM_ECUDA, "memset");
  if (cudaMemsetAsync(s->regions, 0, (size_t)g.N, s->stream) != cudaSuccess) return bail(MM_ECUDA, "memset");
  if ((rc = upload_twiddles(s, g.Px, &s->twx)) || (rc = upload_twiddles(s, g.Py, &s->twy)) ||
      (rc = upload_twiddles(s, g.Pz, &s->twz)))
    return bail(rc, "twiddles");
  if ((rc = mm_build_kernel_spectrum(s, 3))) { std::string m = s->err; return bail(rc, m.c_str()); }
  // convolution arguments
  ConvArgs& c = s->conv;
  c.g = g; c.px = s->px; c.py = s->py; c.pz = s->pz;
  c.twx = s->twx; c.twy = s->twy; c.twz = s->twz;
  c.spec = s->spec; c.rowsS = rowsS; c.cstride = (long long)rowsS * g.pitch;
  c.K = s->K; c.kstride = (long long)g.Cx * g.Hy * g.Hz;
  c.regions = s->regions; c.luts = s->luts; c.st = s->dstate;
  if (s->fast2d && (rc = mm_fast2d_init(s))) { std::string m = s->err; return bail(rc, m.c_str()); }
  if (s->fast3d && (rc = mm_fast3d_init(s))) { std::string m = s->err; return bail(rc, m.c_str()); }
  // a box whose convolution runs entirely on a fast layout (Kt of the 2D path, the z-stage tiles of the 3D path)
  // does not keep the generic layout of the kernel spectrum; MM_OPT_GENERIC_FFT builds it again when asked for
  if (s->fast2d || (s->fast3d && s->f3.mode[2])) {
    if (cudaStreamSynchronize(s->stream) != cudaSuccess) return bail(MM_ECUDA, "kernel set-up");
    mm_dev_free(s, s->K);
    s->K = nullptr; s->conv.K = nullptr;
  }
  // the twelve vector fields come last: the fp64 scratch of the kernel set-up is gone by now, so the peak of the
  // handle's device memory is what it keeps, not set-up scratch on top of it (the paper's B/cell context, L533)
  for (int r = 0; r < R_COUNT; ++r) {
    s->field[r] = (float*)mm_dev_alloc(s, fbytes);
    if (!s->field[r]) return bail(MM_ENOMEM, "field arrays");
    if (cudaMemsetAsync(s->field[r], 0, fbytes, s->stream) != cudaSuccess) return bail(MM_ECUDA, "memset");
  }
  // controller state
  DevState& h = s->hst;
  memset(&h, 0, sizeof(h));
  for (int r = 0; r < R_COUNT; ++r) h.ptr[r] = s->field[r];
  h.max_err = 1e-5; h.headroom = 0.8; h.fix_dt = 0.0; h.dt = 1e-14; h.dt_min = 1e-18; h.dt_max = 1e-9;
  h.gamma = 1.7595e11;
  h.nstage = 7; h.nevals = 6; h.expo = 0.2;
  h.status = MM_OK;
  if ((rc = push_state(s))) { std::string m = s->err; return bail(rc, m.c_str()); }
  *out = s;
  return MM_OK;
}

int mm_destroy(mm_sim* s) {
  if (!s) return MM_OK;
  cudaStreamSynchronize(s->stream);
  drop_graph(s);
  for (auto& e : s->prof) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  for (auto& e : s->ev_pool) cudaEventDestroy(e);
  while (!s->owned.empty()) mm_dev_free(s, s->owned.back().first);
  if (s->own_stream) cudaStreamDestroy(s->stream);
  delete s;
  return MM_OK;
}

// largest region id of a map that lives on the device (4 bytes come back, not the map)
static int max_region_on_device(mm_sim* s, const uint8_t* dev_regions, unsigned* out) {
  unsigned* bits = reinterpret_cast<unsigned*>(s->scratch3);
  CUDA_TRY(s, cudaMemsetAsync(bits, 0, sizeof(unsigned), s->stream));
  { Launch l(s, KK_OTHER); k_max_region<<<s->nsm * 4, 256, 0, s->stream>>>(s->g.N, dev_regions, bits); }
  CUDA_TRY(s, cudaGetLastError());
  CUDA_TRY(s, cudaMemcpyAsync(out, bits, sizeof(unsigned), cudaMemcpyDeviceToHost, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  return MM_OK;
}

static int apply_geometry(mm_sim* s);

int mm_set_regions(mm_sim* s, const uint8_t* regions) {
  if (!s || !regions) return mm_fail(s, MM_EINVAL, "null argument");
  // validate the ids against the current table size before the handle's map is touched
  if (s->have_params) {
    unsigned top = 0;
    if (is_device_ptr(regions)) {
      int rc = max_region_on_device(s, regions, &top);
      if (rc) return rc;
    } else {
      for (long long i = 0; i < s->g.N; ++i) top = regions[i] > top ? regions[i] : top;
    }
    if ((int)top >= s->nregions) return mm_fail(s, MM_EINVAL, "region id >= nregions");
  }
  int rc = copy_in(s, s->geom ? s->regions_user : s->regions, regions, (size_t)s->g.N);
  if (!rc && s->geom) rc = apply_geometry(s);
  s->have_k1 = false; s->graph_dirty = true;
  return rc;
}

// regions = inside the shape ? the caller's index : the reserved vacuum index
static int apply_geometry(mm_sim* s) {
  { Launch l(s, KK_OTHER); k_apply_geometry<<<s->nsm * 8, 256, 0, s->stream>>>(s->g.N, s->regions_user, s->geom, s->regions); }
  CUDA_TRY(s, cudaGetLastError());
  return MM_OK;
}

int mm_set_geometry(mm_sim* s, const uint8_t* inside) {
  if (!s) return MM_EINVAL;
  const size_t N = (size_t)s->g.N;
  int rc;
  if (!inside) {                                    // remove the shape: the caller's map becomes the effective one again
    if (!s->geom) return MM_OK;
    CUDA_TRY(s, cudaMemcpyAsync(s->regions, s->regions_user, N, cudaMemcpyDeviceToDevice, s->stream));
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    mm_dev_free(s, s->geom); mm_dev_free(s, s->regions_user);
    s->geom = s->regions_user = nullptr;
  } else {
    if (s->have_params && s->nregions > MM_MAX_REGIONS - 1)
      return mm_fail(s, MM_EINVAL, "a geometry reserves region index 255: at most 255 regions");
    if (!s->geom) {
      unsigned top = 0;
      if ((rc = max_region_on_device(s, s->regions, &top))) return rc;
      if (top >= MM_MAX_REGIONS - 1) return mm_fail(s, MM_EINVAL, "a geometry reserves region index 255: the region map uses it");
      s->geom = (uint8_t*)mm_dev_alloc(s, N);
      s->regions_user = (uint8_t*)mm_dev_alloc(s, N);
      if (!s->geom || !s->regions_user) {
        mm_dev_free(s, s->geom); mm_dev_free(s, s->regions_user);
        s->geom = s->regions_user = nullptr;
        return mm_fail(s, MM_ENOMEM, "geometry");
      }
      CUDA_TRY(s, cudaMemcpyAsync(s->regions_user, s->regions, N, cudaMemcpyDeviceToDevice, s->stream));
    }
    if ((rc = copy_in(s, s->geom, inside, N))) return rc;
    if ((rc = apply_geometry(s))) return rc;
  }
  // the kernels take their one-region shortcuts from the table size: a box with a shape has two kinds of cells
  const int nreg_dev = s->geom ? MM_MAX_REGIONS : s->nregions;
  CUDA_TRY(s, cudaMemcpyAsync(&s->luts->nregions, &nreg_dev, sizeof(int), cudaMemcpyHostToDevice, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  if (s->have_m) {                                  // cells outside the shape carry no magnetisation
    if ((rc = pull_state(s))) return rc;
    { Launch l(s, KK_OTHER); k_normalise<<<blocks_for(s->g.N, 256), 256, 0, s->stream>>>(s->g.N, s->hst.ptr[R_M], s->regions, s->luts); }
    CUDA_TRY(s, cudaGetLastError());
  }
  s->have_k1 = false; s->graph_dirty = true;
  return MM_OK;
}

int mm_set_params(mm_sim* s, const mm_params* p) {
  if (!s || !p) return mm_fail(s, MM_EINVAL, "null argument");
  const int n = p->nregions;
  if (n < 1 || n > MM_MAX_REGIONS) return mm_fail(s, MM_EINVAL, "nregions out of range");
  if (s->geom && n > MM_MAX_REGIONS - 1) return mm_fail(s, MM_EINVAL, "a geometry reserves region index 255: at most 255 regions");
  if (s->dmi_n > 1 && s->dmi_n != n) return mm_fail(s, MM_EINVAL, "the DM table of mm_set_dmi has another number of regions");
  for (int r = 0; r < n; ++r) {
    if (!(p->Msat[r] >= 0) || !(p->Aex[r] >= 0) || !std::isfinite(p->Msat[r]) || !std::isfinite(p->Aex[r]) ||
        !std::isfinite(p->alpha[r]) || !std::isfinite(p->Ku1[r]) || !std::isfinite(p->Ku2[r]) ||
        !std::isfinite(p->Kc1[r]) || !std::isfinite(p->Kc2[r]) || !std::isfinite(p->Kc3[r]))
      return mm_fail(s, MM_EINVAL, "non-finite or negative material parameter");
  }
  {
    unsigned top = 0;
    int rc = max_region_on_device(s, s->geom ? s->regions_user : s->regions, &top);
    if (rc) return rc;
    if ((int)top >= n) return mm_fail(s, MM_EINVAL, "region map holds an id >= nregions");
  }
  Luts* L = new (std::nothrow) Luts();
  if (!L) return mm_fail(s, MM_ENOMEM, "host LUT");
  memset(L, 0, sizeof(Luts));
  const double mu0 = 4e-7 * M_PI;
  auto unit = [](const double* v, double* o) {
    double nn = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    for (int c = 0; c < 3; ++c) o[c] = nn > 0 ? v[c] / nn : 0.0;
  };
  L->nregions = s->geom ? MM_MAX_REGIONS : n;      // (entries beyond n stay zero: index 255 is the vacuum of a geometry)
  std::vector<double> q(n);
  for (int r = 0; r < n; ++r) {
    const double Ms = p->Msat[r], iMs = Ms > 0 ? 1.0 / Ms : 0.0;
    q[r] = Ms > 0 ? p->Aex[r] / Ms : 0.0;
    L->Bsat[r] = (float)(mu0 * Ms);
    s->hMsat[r] = Ms; s->hAex[r] = p->Aex[r];
    {   // Dzyaloshinskii-Moriya tables (Eq. 10, Eq. 11-13), from the strength last given to mm_set_dmi
      const double D = s->dmi_n == 0 ? 0.0 : s->hD[s->dmi_n == 1 ? 0 : r];
      L->dmi[r] = Ms > 0 ? (float)(2.0 * D / Ms) : 0.f;
      L->dmi_bc[r] = (Ms > 0 && p->Aex[r] > 0) ? (float)(D / (2.0 * p->Aex[r])) : 0.f;
    }
    L->alpha[r] = (float)p->alpha[r];
    L->live[r] = Ms > 0 ? 1.f : 0.f;
    {   // Eq. 24 without T and dt: sqrt(2 mu0 alpha kB / (Bsat gamma dV))
      const double gam = p->gamma_LL > 0 ? p->gamma_LL : 1.7595e11, dV = s->cell[0] * s->cell[1] * s->cell[2];
      L->therm[r] = Ms > 0 && p->alpha[r] > 0 ? (float)std::sqrt(2.0 * mu0 * p->alpha[r] * 1.380649e-23 / (mu0 * Ms * gam * dV)) : 0.f;
    }
    L->ku1[r] = (float)(2.0 * p->Ku1[r] * iMs);
    L->ku2[r] = (float)(4.0 * p->Ku2[r] * iMs);
    L->kc1[r] = (float)(-2.0 * p->Kc1[r] * iMs);
    L->kc2[r] = (float)(-2.0 * p->Kc2[r] * iMs);
    L->kc3[r] = (float)(-4.0 * p->Kc3[r] * iMs);
    double u[3], c1[3], c2[3], c3[3];
    unit(p->anisU[r], u); unit(p->anisC1[r], c1); unit(p->anisC2[r], c2);
    c3[0] = c1[1] * c2[2] - c1[2] * c2[1]; c3[1] = c1[2] * c2[0] - c1[0] * c2[2]; c3[2] = c1[0] * c2[1] - c1[1] * c2[0];
    for (int c = 0; c < 3; ++c) {
      L->u[c][r] = (float)u[c]; L->c1[c][r] = (float)c1[c]; L->c2[c][r] = (float)c2[c]; L->c3[c][r] = (float)c3[c];
    }
    if (p->Ku1[r] != 0 || p->Ku2[r] != 0) L->has_uniaxial = 1;
    if (p->Kc1[r] != 0 || p->Kc2[r] != 0 || p->Kc3[r] != 0) L->has_cubic = 1;
  }
  for (int i = 0; i < n; ++i)
    for (int j = 0; j <= i; ++j) {
      const double sum = q[i] + q[j];
      const double hm = sum > 0 ? 2.0 * q[i] * q[j] / sum : 0.0;                 // Eq. 9
      const double S = p->exch_scale ? p->exch_scale[i * (i + 1) / 2 + j] : 1.0;
      L->exch[i * (i + 1) / 2 + j] = (float)(2.0 * S * hm);                       // the "2" of Eq. 6
    }
  for (int c = 0; c < 3; ++c) L->bext[c] = (float)p->B_ext[c];
  cudaError_t e = cudaMemcpyAsync(s->luts, L, sizeof(Luts), cudaMemcpyHostToDevice, s->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
  delete L;
  CUDA_TRY(s, e);
  int rc;
  if ((rc = pull_state(s))) return rc;
  s->hst.gamma = p->gamma_LL > 0 ? p->gamma_LL : 1.7595e11;
  if ((rc = push_state(s))) return rc;
  s->nregions = n;
  s->have_params = true;
  s->have_k1 = false; s->graph_dirty = true;
  return MM_OK;
}

int mm_set_terms(mm_sim* s, unsigned mask) {
  if (!s) return MM_EINVAL;
  s->terms = mask & MM_ALL;
  s->have_k1 = false; s->graph_dirty = true;
  return MM_OK;
}

int mm_set_solver_kind(mm_sim* s, int kind) {
  if (!s) return MM_EINVAL;
  if (kind != MM_RK45 && kind != MM_RK23 && kind != MM_RK12) return mm_fail(s, MM_EINVAL, "unknown solver");
  int rc;
  if ((rc = pull_state(s))) return rc;
  s->solver = kind;
  s->hst.nstage = kind == MM_RK23 ? 4 : (kind == MM_RK12 ? 2 : 7);
  s->hst.nevals = kind == MM_RK23 ? 3 : (kind == MM_RK12 ? 2 : 6);
  s->hst.expo = kind == MM_RK23 ? 1.0 / 3.0 : (kind == MM_RK12 ? 0.5 : 0.2);
  s->have_k1 = false; s->graph_dirty = true;
  return push_state(s);
}

int mm_set_temperature(mm_sim* s, double kelvin, unsigned long long seed) {
  if (!s) return MM_EINVAL;
  if (!(kelvin >= 0) || !std::isfinite(kelvin)) return mm_fail(s, MM_EINVAL, "bad temperature");
  int rc;
  if ((rc = pull_state(s))) return rc;
  s->temperature = kelvin;
  s->hst.temperature = kelvin;
  s->hst.seed = seed;
  s->have_k1 = false; s->graph_dirty = true;
  return push_state(s);
}

int mm_set_slonczewski(mm_sim* s, double jz, double pol, double lambda, double eps_prime, const double mp[3]) {
  if (!s) return MM_EINVAL;
  if (jz == 0) { s->stt_on = false; s->have_k1 = false; s->graph_dirty = true; return MM_OK; }
  if (!mp || !std::isfinite(jz) || !std::isfinite(pol) || !(lambda > 0) || !std::isfinite(eps_prime))
    return mm_fail(s, MM_EINVAL, "bad spin-torque parameter");
  const double n = std::sqrt(mp[0] * mp[0] + mp[1] * mp[1] + mp[2] * mp[2]);
  if (!(n > 0)) return mm_fail(s, MM_EINVAL, "fixed-layer direction is zero");
  const double hbar = 1.054571817e-34, e = 1.602176634e-19, mu0 = 4e-7 * M_PI, d = s->g.Nz * s->cell[2];
  s->stt[0] = (float)(jz * hbar * mu0 / (e * d));       // beta = this / Bsat
  s->stt[1] = (float)pol; s->stt[2] = (float)(lambda * lambda); s->stt[3] = (float)eps_prime;
  for (int c = 0; c < 3; ++c) s->stt[4 + c] = (float)(mp[c] / n);
  s->stt_on = true;
  s->have_k1 = false; s->graph_dirty = true;
  return MM_OK;
}

int mm_set_zhang_li(mm_sim* s, const double j[3], double xi) {
  if (!s || !j) return mm_fail(s, MM_EINVAL, "null argument");
  if (!std::isfinite(j[0]) || !std::isfinite(j[1]) || !std::isfinite(j[2]) || !std::isfinite(xi))
    return mm_fail(s, MM_EINVAL, "bad spin-torque parameter");
  s->have_k1 = false; s->graph_dirty = true;
  if (j[0] == 0 && j[1] == 0 && j[2] == 0) { s->zl_on = false; return MM_OK; }
  for (int a = 0; a < 3; ++a) s->zl_j[a] = j[a];
  s->zl_xi = xi;
  s->zl_on = true;
  return MM_OK;
}

int mm_set_dmi(mm_sim* s, const double* D, int n) {
  if (!s) return MM_EINVAL;
  if (!s->have_params) return mm_fail(s, MM_ESTATE, "mm_set_params must precede mm_set_dmi");
  if (n < 0 || (n > 1 && n != s->nregions) || (n > 0 && !D)) return mm_fail(s, MM_EINVAL, "DM table: one value or one per region");
  bool any = false;
  for (int r = 0; r < n; ++r) {
    if (!std::isfinite(D[r])) return mm_fail(s, MM_EINVAL, "non-finite DM strength");
    s->hD[r] = D[r];
    any = any || D[r] != 0.0;
  }
  s->dmi_n = any ? n : 0;
  s->dmi_on = any;
  std::vector<float> c(MM_MAX_REGIONS, 0.f), bc(MM_MAX_REGIONS, 0.f);
  for (int r = 0; r < s->nregions && any; ++r) {
    const double Dr = s->hD[n == 1 ? 0 : r], Ms = s->hMsat[r], A = s->hAex[r];
    c[r] = Ms > 0 ? (float)(2.0 * Dr / Ms) : 0.f;
    bc[r] = (Ms > 0 && A > 0) ? (float)(Dr / (2.0 * A)) : 0.f;
  }
  char* base = reinterpret_cast<char*>(s->luts);
  CUDA_TRY(s, cudaMemcpyAsync(base + offsetof(Luts, dmi), c.data(), sizeof(float) * MM_MAX_REGIONS, cudaMemcpyHostToDevice, s->stream));
  CUDA_TRY(s, cudaMemcpyAsync(base + offsetof(Luts, dmi_bc), bc.data(), sizeof(float) * MM_MAX_REGIONS, cudaMemcpyHostToDevice, s->stream));
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  s->have_k1 = false; s->graph_dirty = true;
  return MM_OK;
}

int mm_set_precession(mm_sim* s, int on) {
  if (!s) return MM_EINVAL;
  s->precession = on != 0;
  s->have_k1 = false; s->graph_dirty = true;
  return MM_OK;
}

int mm_step(mm_sim* s, mm_step_info* info) { return mm_step_rk45(s, info); }

int mm_set_option(mm_sim* s, int option, int value) {
  if (!s) return MM_EINVAL;
  switch (option) {
    case MM_OPT_GENERIC_FFT:
      if (value && !s->K) {                    // the generic layout was dropped after the set-up: build it again
        int rc = mm_build_kernel_spectrum(s, 1);
        if (rc) return rc;
        s->conv.K = s->K;
      }
      s->force_generic = value != 0; s->have_k1 = false; s->graph_dirty = true;
      return MM_OK;
    case MM_OPT_NO_TMA: s->f2_no_tma = value != 0; s->have_k1 = false; s->graph_dirty = true; return MM_OK;
    case MM_OPT_NO_GRAPH: s->no_graph = value != 0; return MM_OK;
    default: return mm_fail(s, MM_EINVAL, "unknown option");
  }
}

int mm_set_solver(mm_sim* s, double max_err, double headroom, double fix_dt, double dt_init, double dt_min, double dt_max) {
  if (!s) return MM_EINVAL;
  if (max_err < 0 || headroom < 0 || fix_dt < 0 || dt_init < 0 || dt_min < 0 || dt_max < 0)
    return mm_fail(s, MM_EINVAL, "negative solver setting");
  int rc;
  if ((rc = pull_state(s))) return rc;
  DevState& h = s->hst;
  h.max_err = max_err > 0 ? max_err : 1e-5;
  h.headroom = headroom > 0 ? headroom : 0.8;
  h.fix_dt = fix_dt;
  h.dt_min = dt_min > 0 ? dt_min : 1e-18;
  h.dt_max = dt_max > 0 ? dt_max : 1e-9;
  h.dt = fix_dt > 0 ? fix_dt : (dt_init > 0 ? dt_init : 1e-14);
  h.status = MM_OK;     // a failed step (MM_ENAN / MM_EDT) is cleared here or by mm_set_m; its FSAL slope is not trusted
  h.skip = 0;
  s->have_k1 = false;
  return push_state(s);
}

int mm_set_m(mm_sim* s, const float* m) {
  if (!s || !m) return mm_fail(s, MM_EINVAL, "null argument");
  if (!s->have_params) return mm_fail(s, MM_ESTATE, "mm_set_params must precede mm_set_m");
  int rc;
  if ((rc = pull_state(s))) return rc;
  if ((rc = copy_in(s, s->hst.ptr[R_M], m, sizeof(float) * 3 * (size_t)s->g.N))) return rc;
  { Launch l(s, KK_OTHER); k_normalise<<<blocks_for(s->g.N, 256), 256, 0, s->stream>>>(s->g.N, s->hst.ptr[R_M], s->regions, s->luts); }
  CUDA_TRY(s, cudaGetLastError());
  s->hst.status = MM_OK;
  s->hst.skip = 0;
  if ((rc = push_state(s))) return rc;
  s->have_m = true;
  s->have_k1 = false;
  return MM_OK;
}

int mm_get_m(mm_sim* s, float* m_out) {
  if (!s || !m_out) return mm_fail(s, MM_EINVAL, "null argument");
  int rc;
  if ((rc = pull_state(s))) return rc;
  return copy_out(s, m_out, s->hst.ptr[R_M], sizeof(float) * 3 * (size_t)s->g.N);
}

int mm_b_eff(mm_sim* s, unsigned mask, float* B_out) {
  int rc;
  if ((rc = check_ready(s))) return rc;
  if (!B_out) return mm_fail(s, MM_EINVAL, "null argument");
  clear_skip(s);
  launch_eval(s, R_M, R_B, mask & MM_ALL, 0);
  CUDA_TRY(s, cudaGetLastError());
  if ((rc = pull_state(s))) return rc;
  return copy_out(s, B_out, s->hst.ptr[R_B], sizeof(float) * 3 * (size_t)s->g.N);
}

int mm_torque(mm_sim* s, float* out) {
  int rc;
  if ((rc = check_ready(s))) return rc;
  if (!out) return mm_fail(s, MM_EINVAL, "null argument");
  clear_skip(s);
  launch_eval(s, R_M, R_Y, s->terms, s->precession ? 1 : 2);
  CUDA_TRY(s, cudaGetLastError());
  if ((rc = pull_state(s))) return rc;
  return copy_out(s, out, s->hst.ptr[R_Y], sizeof(float) * 3 * (size_t)s->g.N);
}

int mm_step_rk45(mm_sim* s, mm_step_info* info) {
  int rc;
  if ((rc = check_ready(s)) || (rc = check_thermal(s))) return rc;
  step_once(s);
  CUDA_TRY(s, cudaGetLastError());
  if (!info) return MM_OK;
  if ((rc = pull_state(s))) return rc;
  const DevState& h = s->hst;
  info->t = h.t; info->dt_taken = h.h; info->dt_next = h.fix_dt > 0 ? h.fix_dt : h.dt; info->err = h.last_err;
  info->accepted = h.last_accepted; info->n_eval = (long)h.evals + s->extra_evals;
  return status_to_error(s);
}

int mm_steps(mm_sim* s, int n) {
  int rc;
  if ((rc = check_ready(s)) || (rc = check_thermal(s))) return rc;
  if (n < 0) return mm_fail(s, MM_EINVAL, "negative step count");
  for (int i = 0; i < n; ++i) step_once(s);
  CUDA_TRY(s, cudaGetLastError());
  if ((rc = pull_state(s))) return rc;
  return status_to_error(s);
}

int mm_run(mm_sim* s, double duration) {
  int rc;
  if ((rc = check_ready(s)) || (rc = check_thermal(s))) return rc;
  if (!(duration >= 0) || !std::isfinite(duration)) return mm_fail(s, MM_EINVAL, "bad duration");
  if (duration == 0) return MM_OK;
  if ((rc = pull_state(s))) return rc;
  s->hst.run_mode = 1;
  s->hst.t_end = s->hst.t + duration;
  s->hst.run_duration = duration;
  s->hst.skip = 0;
  if ((rc = push_state(s))) return rc;
  // Steps are enqueued in batches sized from the remaining time and the controller's current suggestion, so that
  // few (if any) attempts are enqueued past t_end (those return at once on the device, but small boxes are
  // launch-bound); the host polls the device time once per batch.
  for (;;) {
    const double dt = s->hst.fix_dt > 0 ? s->hst.fix_dt : s->hst.dt;
    const double est = (s->hst.t_end - s->hst.t) / (dt > 0 ? dt : 1e-18);
    int batch;
    if (s->hst.fix_dt > 0) batch = est > 64 ? 64 : (int)std::ceil(est - 1e-9);
    else batch = est > 86 ? 64 : (int)std::floor(0.75 * est);       // the step may grow (fewer attempts) or be rejected
    if (batch < 1) batch = 1;
    for (int i = 0; i < batch; ++i) step_once(s);
    CUDA_TRY(s, cudaGetLastError());
    if ((rc = pull_state(s))) return rc;
    if (s->hst.skip || s->hst.status != MM_OK) break;
    if (!(s->hst.t_end - s->hst.t > 1e-12 * std::max(duration, 1e-30))) break;      // landed on t_end
  }
  const int st = s->hst.status;
  s->hst.run_mode = 0;
  s->hst.skip = 0;
  if ((rc = push_state(s))) return rc;
  s->hst.status = st;
  return status_to_error(s);
}

int mm_get_time(mm_sim* s, double* t) {
  if (!s || !t) return MM_EINVAL;
  int rc;
  if ((rc = pull_state(s))) return rc;
  *t = s->hst.t;
  return MM_OK;
}

int mm_set_time(mm_sim* s, double t) {
  if (!s) return MM_EINVAL;
  int rc;
  if ((rc = pull_state(s))) return rc;
  s->hst.t = t;
  return push_state(s);
}

int mm_get_avg_m(mm_sim* s, double avg[3]) {
  if (!s || !avg) return MM_EINVAL;
  int rc;
  if ((rc = pull_state(s))) return rc;
  { Launch l(s, KK_OTHER); k_sum3<<<s->nsm * 4, 256, 0, s->stream>>>(s->g.N, s->hst.ptr[R_M], s->red_part, s->red_ticket, s->scratch3); }
  CUDA_TRY(s, cudaGetLastError());
  if ((rc = copy_out(s, avg, s->scratch3, 3 * sizeof(double)))) return rc;
  for (int c = 0; c < 3; ++c) avg[c] /= (double)s->g.N;
  return MM_OK;
}

// energy and maximum torque in two halves - enqueue the reduction, then fetch the scalar - so that the batched
// drivers below can enqueue on every handle before they wait for any of them
static void energy_enqueue(mm_sim* s, unsigned mask) {
  clear_skip(s);
  if (mask & MM_DEMAG) launch_demag(s, R_M);
  { Launch l(s, KK_OTHER); k_energy<<<s->nsm * 8, 256, 0, s->stream>>>(s->g, s->regions, s->luts, s->dstate, R_M, R_B, mask | (s->dmi_on ? MM_DMI_ON : 0u), s->red_part, s->red_ticket, s->scratch3); }
}
static int energy_collect(mm_sim* s, double* joules) {
  CUDA_TRY(s, cudaGetLastError());
  double e = 0.0;
  int rc;
  if ((rc = copy_out(s, &e, s->scratch3, sizeof(double)))) return rc;
  *joules = e / (4e-7 * M_PI) * s->cell[0] * s->cell[1] * s->cell[2];
  return MM_OK;
}
static void max_torque_enqueue(mm_sim* s) {
  clear_skip(s);
  launch_eval(s, R_M, R_Y, s->terms, s->precession ? 1 : 2);       // role R_Y never changes hands: field[R_Y]
  unsigned* bits = reinterpret_cast<unsigned*>(s->scratch3);
  cudaMemsetAsync(bits, 0, sizeof(unsigned), s->stream);
  { Launch l(s, KK_OTHER); k_maxnorm<<<s->nsm * 8, 256, 0, s->stream>>>(s->g.N, s->field[R_Y], bits); }
}
static int max_torque_collect(mm_sim* s, double* tesla) {
  CUDA_TRY(s, cudaGetLastError());
  unsigned b = 0;
  int rc;
  if ((rc = copy_out(s, &b, s->scratch3, sizeof(unsigned)))) return rc;
  float f;
  memcpy(&f, &b, sizeof(f));
  *tesla = (double)f;
  return f == f ? MM_OK : mm_fail(s, MM_ENAN, "non-finite torque");
}

int mm_energy(mm_sim* s, unsigned mask, double* joules) {
  int rc;
  if ((rc = check_ready(s))) return rc;
  if (!joules) return mm_fail(s, MM_EINVAL, "null argument");
  energy_enqueue(s, mask & MM_ALL);
  return energy_collect(s, joules);
}

int mm_max_torque(mm_sim* s, double* tesla) {
  int rc;
  if ((rc = check_ready(s))) return rc;
  if (!tesla) return mm_fail(s, MM_EINVAL, "null argument");
  max_torque_enqueue(s);
  return max_torque_collect(s, tesla);
}

// relax() (L388-L392, #15) as a state machine: every round enqueues 3 steps (or none) and one reduction,
// then fetches one scalar. mm_relax drives one handle; mm_batch_relax drives many, enqueueing a round on every
// handle (each on its own stream, so small boxes overlap on the device) before it waits for any scalar.
namespace {
struct RelaxJob {
  mm_sim* s;
  int solver0; bool prec0; double err0, fix0;
  int phase = 0;            // 0, 1: first two energy samples; 2: energy phase; 3: first torque sample; 4: torque phase
  bool wants_energy = true; // what the pending round has enqueued
  bool done = false;
  int rc = MM_OK;
  long batches = 0;
  double e0 = 0, e1 = 0, t0 = 0, max_err = 0;
};
const long kRelaxMaxBatches = 200000;

int relax_set_err(mm_sim* s, double max_err, double fix_dt) {
  int r = pull_state(s);
  if (r) return r;
  s->hst.max_err = max_err; s->hst.fix_dt = fix_dt;
  return push_state(s);
}
int relax_begin(RelaxJob& j) {
  mm_sim* s = j.s;
  int rc;
  if ((rc = check_ready(s))) return rc;
  if ((rc = pull_state(s))) return rc;
  j.solver0 = s->solver; j.prec0 = s->precession; j.err0 = s->hst.max_err; j.fix0 = s->hst.fix_dt;
  j.max_err = j.err0;
  if ((rc = mm_set_solver_kind(s, MM_RK23))) return rc;
  s->precession = false;
  s->have_k1 = false; s->graph_dirty = true;
  return relax_set_err(s, j.err0, 0.0);
}
int relax_end(RelaxJob& j, int code) {
  mm_sim* s = j.s;
  s->precession = j.prec0;
  int r = mm_set_solver_kind(s, j.solver0);
  if (!r) r = relax_set_err(s, j.err0, j.fix0);
  s->have_k1 = false; s->graph_dirty = true;
  return code ? code : r;
}
// decide what the next round is and enqueue it; sets done when the procedure is over
void relax_enqueue(RelaxJob& j) {
  mm_sim* s = j.s;
  auto advance = [&]() { for (int i = 0; i < 3; ++i) step_once(s); };     // sampled every 3 steps (#15)
  if (j.phase == 2 && !(j.e1 < j.e0 && j.batches++ < kRelaxMaxBatches)) j.phase = 3;   // energy stopped falling
  if (j.phase == 4 && !(j.batches++ < kRelaxMaxBatches)) { j.done = true; return; }
  if (j.phase <= 2) { advance(); energy_enqueue(s, s->terms & MM_ALL); j.wants_energy = true; }
  else { if (j.phase == 4) advance(); max_torque_enqueue(s); j.wants_energy = false; }
}
void relax_collect(RelaxJob& j) {
  mm_sim* s = j.s;
  double v = 0.0;
  if ((j.rc = j.wants_energy ? energy_collect(s, &v) : max_torque_collect(s, &v))) { j.done = true; return; }
  switch (j.phase) {
    case 0: j.e0 = v; j.phase = 1; break;
    case 1: j.e1 = v; j.phase = 2; break;
    case 2: j.e0 = j.e1; j.e1 = v; break;
    case 3: j.t0 = v; j.phase = 4; break;
    default:
      if (v < j.t0) { j.t0 = v; break; }
      if (j.max_err <= 1e-9) { j.done = true; break; }
      j.max_err = std::max(j.max_err / std::sqrt(2.0), 1e-9);       // the torque stopped falling: tighten MaxErr
      if ((j.rc = relax_set_err(s, j.max_err, 0.0))) { j.done = true; break; }
      j.t0 = v;
  }
}
int relax_many(mm_sim* const* sims, int count) {
  std::vector<RelaxJob> jobs((size_t)count);
  int rc = MM_OK;
  for (int i = 0; i < count; ++i) {
    jobs[i].s = sims[i];
    if ((jobs[i].rc = relax_begin(jobs[i]))) { jobs[i].done = true; jobs[i].phase = -1; }
  }
  for (;;) {
    bool any = false;
    for (auto& j : jobs) if (!j.done) relax_enqueue(j);
    for (auto& j : jobs) if (!j.done) { relax_collect(j); any = true; }
    if (!any) break;
  }
  for (auto& j : jobs) {
    int r = j.rc;
    if (j.phase >= 0) {
      if (!r) r = pull_state(j.s);
      r = relax_end(j, r ? r : status_to_error(j.s));
    }
    if (r && !rc) rc = r;
  }
  return rc;
}
}  // namespace

int mm_relax(mm_sim* s) {
  if (!s) return MM_EINVAL;
  return relax_many(&s, 1);
}

// ---- batched independent simulations (the paper's parameter sweeps and its 3000-start search, L426, L800-L803):
// the handles step concurrently, each on its own stream, and the host waits once per round for all of them
static int batch_check(mm_sim* const* sims, int count) {
  if (!sims || count < 0) return MM_EINVAL;
  for (int i = 0; i < count; ++i) if (!sims[i]) return MM_EINVAL;
  return MM_OK;
}

int mm_batch_relax(mm_sim* const* sims, int count) {
  int rc;
  if ((rc = batch_check(sims, count))) return rc;
  return relax_many(sims, count);
}

int mm_batch_steps(mm_sim* const* sims, int count, int n) {
  int rc;
  if ((rc = batch_check(sims, count))) return rc;
  if (n < 0) return MM_EINVAL;
  for (int i = 0; i < count; ++i)
    if ((rc = check_ready(sims[i])) || (rc = check_thermal(sims[i]))) return rc;
  for (int k = 0; k < n; ++k)
    for (int i = 0; i < count; ++i) step_once(sims[i]);
  int first = MM_OK;
  for (int i = 0; i < count; ++i) {
    mm_sim* s = sims[i];
    rc = (cudaGetLastError() == cudaSuccess) ? pull_state(s) : mm_fail(s, MM_ECUDA, "launch failed");
    if (!rc) rc = status_to_error(s);
    if (rc && !first) first = rc;
  }
  return first;
}

int mm_batch_run(mm_sim* const* sims, int count, double duration) {
  int rc;
  if ((rc = batch_check(sims, count))) return rc;
  if (!(duration >= 0) || !std::isfinite(duration)) return MM_EINVAL;
  if (duration == 0 || count == 0) return MM_OK;
  std::vector<char> active((size_t)count, 1);
  for (int i = 0; i < count; ++i) {
    mm_sim* s = sims[i];
    if ((rc = check_ready(s)) || (rc = check_thermal(s)) || (rc = pull_state(s))) return rc;
    s->hst.run_mode = 1; s->hst.t_end = s->hst.t + duration; s->hst.run_duration = duration; s->hst.skip = 0;
    if ((rc = push_state(s))) return rc;
  }
  int first = MM_OK;
  for (bool any = true; any;) {
    for (int i = 0; i < count; ++i) {
      if (!active[i]) continue;
      mm_sim* s = sims[i];
      const double dt = s->hst.fix_dt > 0 ? s->hst.fix_dt : s->hst.dt;
      const double est = (s->hst.t_end - s->hst.t) / (dt > 0 ? dt : 1e-18);
      int batch = s->hst.fix_dt > 0 ? (est > 64 ? 64 : (int)std::ceil(est - 1e-9)) : (est > 86 ? 64 : (int)std::floor(0.75 * est));
      if (batch < 1) batch = 1;
      for (int k = 0; k < batch; ++k) step_once(s);
    }
    any = false;
    for (int i = 0; i < count; ++i) {
      if (!active[i]) continue;
      mm_sim* s = sims[i];
      rc = pull_state(s);
      const bool over = rc || s->hst.skip || s->hst.status != MM_OK ||
                        !(s->hst.t_end - s->hst.t > 1e-12 * std::max(duration, 1e-30));
      if (!over) { any = true; continue; }
      active[i] = 0;
      const int st = s->hst.status;
      s->hst.run_mode = 0; s->hst.skip = 0;
      if (!rc) rc = push_state(s);
      s->hst.status = st;
      if (!rc) rc = status_to_error(s);
      if (rc && !first) first = rc;
    }
  }
  return first;
}

int mm_get_stats(mm_sim* s, long* steps, long* rejected, long* evals, size_t* peak) {
  if (!s) return MM_EINVAL;
  int rc;
  if ((rc = pull_state(s))) return rc;
  if (steps) *steps = (long)s->hst.steps;
  if (rejected) *rejected = (long)s->hst.rejected;
  if (evals) *evals = (long)s->hst.evals + s->extra_evals;
  if (peak) *peak = s->peak_bytes;
  return MM_OK;
}

int mm_get_memory(mm_sim* s, size_t* resident, size_t* peak) {
  if (!s) return MM_EINVAL;
  if (resident) *resident = s->cur_bytes;
  if (peak) *peak = s->peak_bytes;
  return MM_OK;
}

int mm_get_stream(mm_sim* s, void** cuda_stream) {
  if (!s || !cuda_stream) return MM_EINVAL;
  *cuda_stream = (void*)s->stream;
  return MM_OK;
}

int mm_get_fft_size(mm_sim* s, int P[3]) {
  if (!s || !P) return MM_EINVAL;
  P[0] = s->g.Px; P[1] = s->g.Py; P[2] = s->g.Pz;
  return MM_OK;
}

int mm_get_launch_count(mm_sim* s, long* launches) {
  if (!s || !launches) return MM_EINVAL;
  *launches = s->launches;
  return MM_OK;
}

int mm_profile(mm_sim* s, int enable) {
  if (!s) return MM_EINVAL;
  CUDA_TRY(s, cudaStreamSynchronize(s->stream));
  for (auto& e : s->prof) { s->ev_pool.push_back(e.a); s->ev_pool.push_back(e.b); }
  s->prof.clear();
  for (int k = 0; k < KK_COUNT; ++k) { s->prof_ms[k] = 0; s->prof_n[k] = 0; }
  s->prof_on = enable != 0;
  return MM_OK;
}

int mm_profile_read(mm_sim* s, int kind, const char** name, double* total_ms, long* launches) {
  static const char* names[KK_COUNT] = {"x_fwd", "y_fwd", "y_inv", "last_xy", "last_z", "last_3d", "x_inv", "local",
                                        "rk_stage", "rk_error", "rk_ctrl", "other", "f2_xfwd", "f2_ycol", "f2_xinv", "f3_y", "f3_z", "f3_xfwd", "f3_xinv"};
  if (!s || kind < 0 || kind >= KK_COUNT) return MM_EINVAL;
  if (!s->prof.empty()) {
    CUDA_TRY(s, cudaStreamSynchronize(s->stream));
    for (auto& e : s->prof) {
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e.a, e.b);
      s->prof_ms[e.kind] += ms; s->prof_n[e.kind] += 1;
      s->ev_pool.push_back(e.a); s->ev_pool.push_back(e.b);
    }
    s->prof.clear();
  }
  if (name) *name = names[kind];
  if (total_ms) *total_ms = s->prof_ms[kind];
  if (launches) *launches = s->prof_n[kind];
  return MM_OK;
}

const char* mm_last_error(const mm_sim* s) { return s ? s->err.c_str() : g_create_error.c_str(); }

const char* mm_strerror(int code) {
  switch (code) {
    case MM_OK: return "ok";
    case MM_EINVAL: return "invalid argument";
    case MM_ENOMEM: return "out of device memory";
    case MM_ECUDA: return "CUDA error (or no CUDA device)";
    case MM_ESTATE: return "call sequence error";
    case MM_ENAN: return "non-finite error estimate";
    case MM_EDT: return "step size below dt_min";
    default: return "unknown error";
  }
}

const char* mm_version(void) { return "mm_b200 0.2 (sm_100a)"; }

}  // extern "C"
