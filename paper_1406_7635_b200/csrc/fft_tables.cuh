// fft_tables.cuh - host side of the register-FFT plans (fft_reg.cuh): twiddle tables in fp64 -> fp32, uploaded once
// per handle. Shared by the fast 2D (fast2d.cu) and fast 3D (fast3d.cu) paths.
#pragma once
#include <cmath>
#include <vector>
#include "internal.cuh"
#include "fft_reg.cuh"

// forward twiddles of a plan, laid out as fft_reg.cuh reads them
template <class P>
inline std::vector<float2> plan_table() {
  std::vector<float2> tw(P::TW);
  const int N = P::N;
  auto put = [&](size_t i, double turns) {
    const double ang = -2.0 * M_PI * turns;
    tw[i] = make_float2((float)cos(ang), (float)sin(ang));
  };
  for (int s = 1; s < P::RA; ++s)
    for (int bf = 0; bf < N / P::RA; ++bf) put((size_t)(s - 1) * (N / P::RA) + bf, (double)((long long)s * bf % N) / N);
  if (P::NPASS == 3)
    for (int s = 1; s < P::RB; ++s)
      for (int bf = 0; bf < N / P::RB; ++bf)
        put((size_t)P::TW1 + (size_t)(s - 1) * (N / P::RB) + bf, (double)((long long)s * P::RA * (bf % P::M2) % N) / N);
  return tw;
}

inline int mm_upload_table(mm_sim* s, const std::vector<float2>& h, float2** out) {
  *out = (float2*)mm_dev_alloc(s, sizeof(float2) * h.size());
  if (!*out) return mm_fail(s, MM_ENOMEM, "register-FFT twiddles");
  CUDA_TRY(s, cudaMemcpy(*out, h.data(), sizeof(float2) * h.size(), cudaMemcpyHostToDevice));
  return MM_OK;
}

// tables of one axis of length P::N: forward plan, reversed plan (inverse transforms), half-bin twiddles
// exp(-2 pi i n / (2N)) of the zero-padded (2N-point) transform
template <class P>
int mm_plan_tables(mm_sim* s, float2** fwd, float2** rev, float2** half) {
  int rc;
  if ((rc = mm_upload_table(s, plan_table<P>(), fwd))) return rc;
  if ((rc = mm_upload_table(s, plan_table<typename P::Reversed>(), rev))) return rc;
  const int N = P::N;
  std::vector<float2> w(N);
  for (int n = 0; n < N; ++n) {
    const double ang = -M_PI * (double)n / (double)N;
    w[n] = make_float2((float)cos(ang), (float)sin(ang));
  }
  return mm_upload_table(s, w, half);
}
