// internal.cuh - handle layout and host helpers shared by the translation units of libmm_b200.so
#pragma once
#include <string>
#include <utility>
#include <vector>
#include "common.cuh"
#include "demag_conv_args.cuh"

void* mm_default_alloc(size_t bytes, void*);
void mm_default_free(void* p, void*);

struct mm_sim {
  Geometry g;
  AxisPlan px, py, pz;
  double cell[3];
  int rep[3];
  cudaStream_t stream = nullptr;
  void* (*alloc)(size_t, void*) = mm_default_alloc;
  void (*dealloc)(void*, void*) = mm_default_free;
  void* alloc_ctx = nullptr;
  std::vector<std::pair<void*, size_t>> owned;
  size_t cur_bytes = 0, peak_bytes = 0;
  // device memory
  float* field[R_COUNT] = {};
  uint8_t* regions = nullptr;
  Luts* luts = nullptr;
  DevState* dstate = nullptr;
  float2* spec = nullptr;
  float* K = nullptr;
  float2 *twx = nullptr, *twy = nullptr, *twz = nullptr;
  double* scratch3 = nullptr;
  ConvArgs conv;
  // host state
  DevState hst;
  bool have_params = false, have_m = false, have_k1 = false;
  unsigned terms = MM_ALL;
  int nregions = 1;
  long launches = 0;
  std::string err;
  // launch configuration
  int xL = 1, yC = 1, lastC[3] = {1, 1, 1};
  size_t xSmem = 0, ySmem = 0, lastSmem[3] = {0, 0, 0};
  bool last_along_z = false;
};

int mm_fail(mm_sim* s, int code, const std::string& msg);
void* mm_dev_alloc(mm_sim* s, size_t bytes);
void mm_dev_free(mm_sim* s, void* p);
int mm_build_kernel_spectrum(mm_sim* s);   // setup.cu

#define CUDA_TRY(s, expr)                                                                       \
  do {                                                                                          \
    cudaError_t e_ = (expr);                                                                    \
    if (e_ != cudaSuccess) {                                                                    \
      cudaGetLastError();                                                                       \
      return mm_fail((s), MM_ECUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));       \
    }                                                                                           \
  } while (0)

inline unsigned blocks_for(long long n, int threads) { return (unsigned)((n + threads - 1) / threads); }
