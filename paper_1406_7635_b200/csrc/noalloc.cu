// noalloc.cu - mm_avg_m_noalloc: the mean of a magnetisation field (the paper's m.average()) for
// callers that cannot allocate device memory (code under CUDA-graph capture, tight serving loops, harnesses that
// forbid cudaMalloc). A variant of k_sum3 / grid_sum_ordered (local_rk.cuh): the per-block partial sums and the
// ticket counter, which mm_get_avg_m keeps in buffers the handle allocated, live here in ONE file-scope device array
// of fixed size that every GPU loading the library holds until the process exits. The entry point calls no
// cudaMalloc, cudaFree or allocating library routine.
//
// The array is shared by every call and keeps the last call's contents: the ticket is cleared on the caller's
// stream before each launch, the partials are overwritten before they are read. Calls that overlap on the GPU
// (different streams, or graph branches that run concurrently) race on it.
#include <cuda_runtime.h>
#include <stdio.h>
#include <mutex>
#include "../../include/mm.h"

namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_CHUNK = 8192;                                        // cells per block: one partial (3 doubles) each
constexpr long long NA_MAX_CHUNKS = MM_NOALLOC_MAX_CELLS / NA_CHUNK;  // 8192
constexpr size_t NA_TICKET_OFF = (size_t)NA_MAX_CHUNKS * 3 * sizeof(double);     // 196 608
constexpr size_t NA_SCRATCH_BYTES = NA_TICKET_OFF + 256;                         // 196 864 bytes per GPU

// In host code this name is a host-side stand-in, not a device address: the host asks for the address with
// cudaGetSymbolAddress (once per device, below) and passes it to the kernel.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NA_SCRATCH_BYTES];

// Block b sums the cells [b * NA_CHUNK, (b + 1) * NA_CHUNK) of the three components in fp64: per thread in index
// order with stride NA_THREADS, lanes by shuffles, warps in index order. The block that draws the last ticket adds
// the partials in block order (256 contiguous segments, then the segments in order) and writes the mean. The
// summation order is fixed by N alone, not by the device or the schedule: the same field gives the same bits.
__global__ void __launch_bounds__(NA_THREADS) k_avg_m_noalloc(long long N, const float* __restrict__ m, double* __restrict__ part,
                                                              unsigned* __restrict__ ticket, double* __restrict__ out) {
  __shared__ double wsum[NA_THREADS / 32][3];
  __shared__ double seg[NA_THREADS][3];
  __shared__ bool last;
  const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
  const long long i0 = (long long)blockIdx.x * NA_CHUNK;
  const long long i1 = i0 + NA_CHUNK < N ? i0 + NA_CHUNK : N;
  double s[3] = {0.0, 0.0, 0.0};
  for (long long i = i0 + tid; i < i1; i += NA_THREADS) {
    s[0] += (double)m[i]; s[1] += (double)m[N + i]; s[2] += (double)m[2 * N + i];
  }
#pragma unroll
  for (int c = 0; c < 3; ++c) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s[c] += __shfl_xor_sync(0xffffffffu, s[c], o);
    if (lane == 0) wsum[w][c] = s[c];
  }
  __syncthreads();
  if (tid == 0) {
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      double a = 0.0;
      for (int i = 0; i < NA_THREADS / 32; ++i) a += wsum[i][c];
      part[(size_t)blockIdx.x * 3 + c] = a;
    }
    __threadfence();
    last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  const unsigned nb = gridDim.x, per = (nb + NA_THREADS - 1) / NA_THREADS;
  const unsigned b0 = tid * per, b1 = b0 + per < nb ? b0 + per : nb;
  double a[3] = {0.0, 0.0, 0.0};
  for (unsigned b = b0; b < b1; ++b) {
    a[0] += __ldcg(&part[(size_t)b * 3]); a[1] += __ldcg(&part[(size_t)b * 3 + 1]); a[2] += __ldcg(&part[(size_t)b * 3 + 2]);
  }
  seg[tid][0] = a[0]; seg[tid][1] = a[1]; seg[tid][2] = a[2];
  __syncthreads();
  if (tid < 3) {
    double t = 0.0;
    for (int i = 0; i < NA_THREADS; ++i) t += seg[i][tid];
    out[tid] = t / (double)N;
  }
  if (tid == 0) *ticket = 0u;
}

constexpr int NA_MAX_DEVICES = 64;
std::mutex g_mu;
unsigned char* g_scratch_ptr[NA_MAX_DEVICES];      // device address of g_noalloc_scratch on each device (nullptr: not asked yet)

int fail(char* errbuf, size_t errlen, int code, const char* what, const char* detail = nullptr) {
  if (errbuf && errlen > 0) {
    if (detail) snprintf(errbuf, errlen, "mm_avg_m_noalloc: %s (%s)", what, detail);
    else snprintf(errbuf, errlen, "mm_avg_m_noalloc: %s", what);
  }
  return code;
}

bool on_device(const void* p, int dev) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return (at.type == cudaMemoryTypeDevice && at.device == dev) || at.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int mm_avg_m_noalloc(const float* m_dev, long long ncells, double* avg_dev, void* cuda_stream, char* errbuf,
                                size_t errlen) {
  if (errbuf && errlen > 0) errbuf[0] = 0;
  if (!m_dev || !avg_dev) return fail(errbuf, errlen, MM_EINVAL, "null pointer");
  if (ncells < 1) return fail(errbuf, errlen, MM_EINVAL, "ncells must be positive");
  if (ncells > MM_NOALLOC_MAX_CELLS) {
    char d[96];
    snprintf(d, sizeof d, "%lld cells > MM_NOALLOC_MAX_CELLS = %lld", ncells, (long long)MM_NOALLOC_MAX_CELLS);
    return fail(errbuf, errlen, MM_EINVAL, "field too large for the fixed scratch array", d);
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(errbuf, errlen, MM_ECUDA, "no CUDA device", cudaGetErrorString(e)); }
  if (dev < 0 || dev >= NA_MAX_DEVICES) return fail(errbuf, errlen, MM_EINVAL, "device ordinal beyond 63");
  if (!on_device(m_dev, dev) || !on_device(avg_dev, dev))
    return fail(errbuf, errlen, MM_EINVAL, "m_dev and avg_dev must be device memory of the current device");
  unsigned char* scratch;
  {
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_scratch_ptr[dev]) {      // once per device, with that device current
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
      if (e != cudaSuccess || !p) {
        cudaGetLastError();
        return fail(errbuf, errlen, MM_ECUDA, "cudaGetSymbolAddress", cudaGetErrorString(e));
      }
      g_scratch_ptr[dev] = static_cast<unsigned char*>(p);
    }
    scratch = g_scratch_ptr[dev];
  }
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double* part = reinterpret_cast<double*>(scratch);
  unsigned* ticket = reinterpret_cast<unsigned*>(scratch + NA_TICKET_OFF);
  // the ticket must start at zero whatever an earlier (possibly failed) call left behind
  e = cudaMemsetAsync(ticket, 0, sizeof(unsigned), st);
  if (e != cudaSuccess) { cudaGetLastError(); return fail(errbuf, errlen, MM_ECUDA, "cudaMemsetAsync", cudaGetErrorString(e)); }
  const unsigned nblocks = (unsigned)((ncells + NA_CHUNK - 1) / NA_CHUNK);
  k_avg_m_noalloc<<<nblocks, NA_THREADS, 0, st>>>(ncells, m_dev, part, ticket, avg_dev);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(errbuf, errlen, MM_ECUDA, "kernel launch", cudaGetErrorString(e));
  return MM_OK;
}
