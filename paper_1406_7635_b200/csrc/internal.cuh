// internal.cuh - handle layout and host helpers shared by the translation units of libmm_b200.so
#pragma once
#include <cuda.h>
#include <string>
#include <utility>
#include <vector>
#include "common.cuh"
#include "demag_conv_args.cuh"

void* mm_default_alloc(size_t bytes, void*);
void mm_default_free(void* p, void*);

// kernel classes for launch counting and per-kernel CUDA-event timing (mm_profile)
enum KernelKind { KK_XFWD = 0, KK_YFWD, KK_YINV, KK_LAST_XY, KK_LAST_Z, KK_LAST_3D, KK_XINV, KK_LOCAL, KK_STAGE,
                  KK_ERROR, KK_CTRL, KK_OTHER, KK_F2_XFWD, KK_F2_YCOL, KK_F2_XINV, KK_F3_Y, KK_F3_Z, KK_F3_XFWD, KK_F3_XINV,
                  KK_COUNT };
struct ProfEntry { int kind; cudaEvent_t a, b; };

struct mm_sim {
  Geometry g;
  AxisPlan px, py, pz;
  double cell[3];
  int rep[3];
  cudaStream_t stream = nullptr;
  bool own_stream = false;     // created by mm_create (no stream was passed): destroyed with the handle
  int nsm = 148;               // SMs of the device (grid sizing of the reductions and persistent kernels)
  void* (*alloc)(size_t, void*) = mm_default_alloc;
  void (*dealloc)(void*, void*) = mm_default_free;
  void* alloc_ctx = nullptr;
  std::vector<std::pair<void*, size_t>> owned;
  size_t cur_bytes = 0, peak_bytes = 0;
  // device memory
  float* field[R_COUNT] = {};
  uint8_t* regions = nullptr;      // effective region index of every cell (what the kernels read)
  uint8_t* regions_user = nullptr; // with a geometry: the caller's region map (regions = inside ? regions_user : 255)
  uint8_t* geom = nullptr;         // with a geometry: the shape, one byte per cell (mm_set_geometry)
  Luts* luts = nullptr;
  DevState* dstate = nullptr;
  float2* spec = nullptr;
  float* K = nullptr;
  float2 *twx = nullptr, *twy = nullptr, *twz = nullptr;
  double* scratch3 = nullptr;
  double* red_part = nullptr;       // per-block partials of the ordered fp64 reductions (k_energy, k_sum3)
  unsigned* red_ticket = nullptr;   // their ticket counter (zero between launches)
  ConvArgs conv;
  float* Kt = nullptr;         // kernel spectrum in the fast 2D layout
  Fast2DArgs f2;
  CUtensorMap f2_map_invp_even, f2_map_invp_odd;        // boxes {2 rows, KB bins}: one row pair per FFT group (persistent x inverse)
  CUtensorMap f2_map_inv_even, f2_map_inv_odd;          // boxes {2G rows, KB bins} over the even / odd columns (direct-read x inverse)
  CUtensorMap f2_map_inv, f2_map_fwd, f2_map_fwd_odd;   // TMA views of spec for the x kernels (inverse: boxes of 2G rows x 256
                                                        // bins; forward: 4G rows x KB bins of the even resp. odd columns)
  bool f2_no_tma = false;      // mm_set_option(MM_OPT_NO_TMA)
  bool f2_tma = false;         // tensor maps valid: the x kernels move their transposed pieces with TMA
  bool fast2d = false;         // fast 2D path available for this box
  Fast3DArgs f3;
  bool fast3d = false;         // some stage of this 3D box runs on the register engine (fast3d.cu, f3.mode)
  bool force_generic = false;  // mm_set_option(MM_OPT_GENERIC_FFT)
  // host state
  DevState hst;
  bool have_params = false, have_m = false, have_k1 = false;
  cudaGraphExec_t graph_exec = nullptr;   // one attempted step of the current configuration (mm_api.cu: step_once)
  long graph_launches = 0;                // kernel launches inside it
  bool graph_dirty = false;               // configuration changed: capture again
  bool no_graph = false;                  // mm_set_option(MM_OPT_NO_GRAPH), or capture failed once
  unsigned terms = MM_ALL;
  int solver = MM_RK45;
  bool precession = true;
  double temperature = 0.0;
  bool zl_on = false;          // Zhang-Li torque enabled (mm_set_zhang_li)
  double zl_j[3] = {};         // current density [A/m^2] and non-adiabaticity as passed; the kernel arguments are
  double zl_xi = 0.0;          // formed at launch time from the gamma_LL in force (mm_set_params may change it)
  bool dmi_on = false;         // a Dzyaloshinskii-Moriya strength is set (mm_set_dmi): exchange takes the boundary-condition path
  int dmi_n = 0;               // entries of hD in use: 0 (off), 1 (uniform) or nregions
  double hD[MM_MAX_REGIONS] = {}, hMsat[MM_MAX_REGIONS] = {}, hAex[MM_MAX_REGIONS] = {};   // host copies for the DM tables
  bool stt_on = false;         // Slonczewski torque enabled (mm_set_slonczewski)
  float stt[7] = {};           // pref, pol, lam2, eps_prime, mp[3]  (SttArgs of local_rk.cuh)
  int nregions = 1;
  long launches = 0;
  long extra_evals = 0;
  bool prof_on = false;
  std::vector<ProfEntry> prof;
  std::vector<cudaEvent_t> ev_pool;
  double prof_ms[KK_COUNT] = {};
  long prof_n[KK_COUNT] = {};
  std::string err;
  // launch configuration
  int xL = 1, yC = 1, lastC[3] = {1, 1, 1};
  size_t xSmem = 0, ySmem = 0, lastSmem[3] = {0, 0, 0};
  bool last_along_z = false;
};

int mm_fail(mm_sim* s, int code, const std::string& msg);
void* mm_dev_alloc(mm_sim* s, size_t bytes);
void mm_dev_free(mm_sim* s, void* p);
int mm_build_kernel_spectrum(mm_sim* s, int layouts);   // setup.cu: bit 0 generic K, bit 1 fast 2D layout Kt
bool mm_fast2d_supported(int Nx, int Ny, int Nz, const int* pbc);   // fast2d.cu
int mm_fast2d_length(int N);      // transform length of the fast path for N physical cells (power of two)
int mm_fast2d_init(mm_sim* s);
void mm_fast2d_demag(mm_sim* s, int src_role);
void mm_fast3d_modes(const Geometry& g, int* mode);   // fast3d.cu: per axis 0 generic, 1 open, 2 periodic
int mm_fast3d_init(mm_sim* s);
void mm_fast3d_x(mm_sim* s, bool inverse, int role);
void mm_fast3d_y(mm_sim* s, bool inverse);
void mm_fast3d_z(mm_sim* s);

#define CUDA_TRY(s, expr)                                                                       \
  do {                                                                                          \
    cudaError_t e_ = (expr);                                                                    \
    if (e_ != cudaSuccess) {                                                                    \
      cudaGetLastError();                                                                       \
      return mm_fail((s), MM_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));       \
    }                                                                                           \
  } while (0)

inline unsigned blocks_for(long long n, int threads) { return (unsigned)((n + threads - 1) / threads); }

// RAII bracket around one kernel launch: counts it and, while profiling, records a CUDA event
// on the launching stream before and after it.
struct Launch {
  mm_sim* s; int kind; cudaEvent_t a = nullptr, b = nullptr;
  static cudaEvent_t get(mm_sim* s) {
    if (!s->ev_pool.empty()) { cudaEvent_t e = s->ev_pool.back(); s->ev_pool.pop_back(); return e; }
    cudaEvent_t e; cudaEventCreate(&e); return e;
  }
  Launch(mm_sim* s_, int kind_) : s(s_), kind(kind_) {
    s->launches++;
    if (s->prof_on) { a = get(s); b = get(s); cudaEventRecord(a, s->stream); }
  }
  ~Launch() {
    if (a) { cudaEventRecord(b, s->stream); s->prof.push_back({kind, a, b}); }
  }
};
