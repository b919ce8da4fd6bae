// selftest_l2.cu — tpcst_selftest_random_access (include/tpcst.h): what this GPU sustains for the access pattern that bounds the
// selection kernels (select_claim, select_collect, write_ids: PAPER.md L46): 4-byte accesses at
// random positions of an array that fits the L2 cache.  Two plain kernels, nothing of the tracker in them: a gather
// (ld.global.nc) and an atomic maximum whose result is not used (red.global.max).  Every thread keeps kBatch independent
// accesses in flight, indices come from an integer hash of the access number (uniform over the array).  The rates are a
// measured device limit to hold the tracker's kernels against; they are not part of the path.
#include <cstdint>

#include "tpcst_internal.h"

namespace tpcst {
int cuda_status(cudaError_t e, const char* what);   // api.cu
}

namespace {

constexpr int kBatch = 4;

__device__ __forceinline__ uint32_t hash32(uint32_t x) {          // bijective mixer
  x ^= x >> 16; x *= 0x7feb352du; x ^= x >> 15; x *= 0x846ca68bu; x ^= x >> 16;
  return x;
}
__device__ __forceinline__ uint32_t index_of(unsigned long long i, uint32_t n_words) {
  return (uint32_t)(((unsigned long long)hash32((uint32_t)i ^ (uint32_t)(i >> 32) * 0x9e3779b9u) * n_words) >> 32);
}

__global__ void __launch_bounds__(256) l2_red_max(uint32_t* a, uint32_t n_words, unsigned long long n_access) {
  const unsigned long long nth = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n_access; i += nth * kBatch) {
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const unsigned long long j = i + u * nth;
      if (j < n_access) atomicMax(a + index_of(j, n_words), (uint32_t)j);
    }
  }
}

__global__ void __launch_bounds__(256) l2_gather(const uint32_t* __restrict__ a, uint32_t n_words, unsigned long long n_access,
                                                 uint32_t* sink) {
  const unsigned long long nth = (unsigned long long)gridDim.x * blockDim.x;
  uint32_t acc = 0;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n_access; i += nth * kBatch) {
    uint32_t v[kBatch];
#pragma unroll
    for (int u = 0; u < kBatch; ++u) {
      const unsigned long long j = i + u * nth;
      v[u] = j < n_access ? __ldg(a + index_of(j, n_words)) : 0u;
    }
#pragma unroll
    for (int u = 0; u < kBatch; ++u) acc ^= v[u];
  }
  if (acc == 0x9e3779b9u) *sink = acc;                  // keeps the loads alive; practically never taken
}

}  // namespace

extern "C" int tpcst_selftest_random_access(void* cuda_stream, uint32_t n_words, uint64_t n_access, int reps, float* ms_gather,
                                 float* ms_red_max) {
  if (!ms_gather || !ms_red_max || n_words < 1u || n_access < 1u || reps < 1 || reps > 1000) return TPCST_ERR_ARG;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint32_t* a = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  int sms = 0, dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess) e = cudaMalloc((void**)&a, ((size_t)n_words + 1u) * 4u);
  if (e == cudaSuccess) e = cudaEventCreate(&e0);
  if (e == cudaSuccess) e = cudaEventCreate(&e1);
  if (e == cudaSuccess) e = cudaMemsetAsync(a, 0, ((size_t)n_words + 1u) * 4u, st);
  const unsigned grid = (unsigned)(sms > 0 ? sms : 148) * 8u;
  float best[2] = {0.f, 0.f};
  for (int which = 0; which < 2 && e == cudaSuccess; ++which) {
    for (int r = -2; r < reps && e == cudaSuccess; ++r) {           // two untimed warm-up launches
      e = cudaEventRecord(e0, st);
      if (which == 0) l2_gather<<<grid, 256, 0, st>>>(a, n_words, n_access, a + n_words);
      else l2_red_max<<<grid, 256, 0, st>>>(a, n_words, n_access);
      if (e == cudaSuccess) e = cudaGetLastError();
      if (e == cudaSuccess) e = cudaEventRecord(e1, st);
      if (e == cudaSuccess) e = cudaEventSynchronize(e1);
      float ms = 0.f;
      if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
      if (e == cudaSuccess && r >= 0 && (best[which] == 0.f || ms < best[which])) best[which] = ms;
    }
  }
  if (e0) (void)cudaEventDestroy(e0);
  if (e1) (void)cudaEventDestroy(e1);
  if (a) (void)cudaFree(a);
  if (e != cudaSuccess) return tpcst::cuda_status(e, "tpcst_selftest_random_access");
  *ms_gather = best[0];
  *ms_red_max = best[1];
  return TPCST_OK;
}
