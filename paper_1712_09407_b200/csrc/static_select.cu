// static_select.cu — tpcst_select_owners_static (include/tpcst.h): the longest-wins tracklet selection
// (G26, select_mode 0) for callers that may not allocate device memory.
//
// The selection needs one word of scratch per cluster: the best claim key seen so far, raised with atomicMax
// by every tracklet that wants the cluster.  tpcst_track_event keeps those words in the caller's workspace
// (Params::owner).  Here they live in a fixed array that is part of this library's device image, so that a
// caller who only owns its input and output buffers (a trigger loop that must not hit cudaMalloc's device-wide
// synchronisation, a plug-in of a framework that owns all device memory, a process with a frozen memory budget)
// can still run the step.  Nothing in this file calls cudaMalloc, cudaFree, cudaHostAlloc or creates a stream or
// an event; the kernels are variants of select_claim / select_collect (kernels_select.cu) that read the plain
// [tracklet][row] table of cluster indices instead of the tracker's internal sorted-space hit tables.
//
// The array's name means two different things.  In device code `g_static_keys` is the array.  In host code the
// same name is only the host-side shadow the runtime uses to identify the symbol: its address is a HOST address,
// and a kernel handed `g_static_keys` from the host would fault (or, where the GPU can reach host memory, scribble
// over unrelated host data).  The device address is obtained once per device with cudaGetSymbolAddress, with that
// device current, and that pointer is what the kernels and the memset get.
#include <mutex>

#include "tpcst_internal.h"

namespace tpcst {
int cuda_status(cudaError_t e, const char* what);   // api.cu: keeps the error text for tpcst_error_string
}

namespace {

using namespace tpcst;

// One claim key per cluster; 4 MiB on every GPU that loads this file's device code, until the process exits.
// Contents survive from call to call: every call clears the [0, n_clusters) part it is about to use.
static __device__ __align__(256) uint32_t g_static_keys[TPCST_STATIC_MAX_CLUSTERS];

constexpr int kMaxDevices = 64;
struct PerDevice {
  uint32_t* keys = nullptr;    // device address of g_static_keys on this device (cudaGetSymbolAddress)
  uint32_t grid_cap = 0;       // CTAs of a full wave: SMs x 8 CTAs of 256 threads
};
std::mutex g_setup_lock;
PerDevice g_dev[kMaxDevices];

// Once per device, with that device current.
int setup_current_device(int device, PerDevice* out) {
  std::lock_guard<std::mutex> hold(g_setup_lock);
  PerDevice& d = g_dev[device];
  if (!d.keys) {
    void* ptr = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_keys);
    if (e != cudaSuccess) return cuda_status(e, "cudaGetSymbolAddress(g_static_keys)");
    if (!ptr) return cuda_status(cudaErrorInvalidSymbol, "cudaGetSymbolAddress(g_static_keys) gave a null address");
    int sms = 0;
    e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return cuda_status(e, "cudaDeviceGetAttribute(multiprocessor count)");
    d.grid_cap = (uint32_t)(sms > 0 ? sms : 148) * 8u;
    d.keys = static_cast<uint32_t*>(ptr);
  }
  *out = d;
  return TPCST_OK;
}

// Device a pointer belongs to; -1 if it is not device (or managed) memory.
int device_of(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return -1; }
  if (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged) return -1;
  return a.device;
}

struct CurrentDevice {            // make `device` current for the scope, then put the caller's back
  int prev = -1;
  cudaError_t err;
  explicit CurrentDevice(int device) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
    else prev = -1;
  }
  ~CurrentDevice() { if (prev >= 0) (void)cudaSetDevice(prev); }
  CurrentDevice(const CurrentDevice&) = delete;
  CurrentDevice& operator=(const CurrentDevice&) = delete;
};

// G26, select_mode 0: more hits win; among equally long tracklets the lower index wins.  Never 0 (nh >= 1).
__device__ __forceinline__ uint32_t claim_key_static(uint32_t nh, uint32_t t) { return (nh << 24) | (0xFFFFFFu - t); }

// Hits of one tracklet = entries of its row that name a cluster.  Called by all 32 lanes of a warp.
__device__ __forceinline__ uint32_t count_hits(const int32_t* row, uint32_t R, uint32_t N, uint32_t lane) {
  uint32_t nh = 0;
  for (uint32_t k0 = 0; k0 < R; k0 += 32u) {
    const uint32_t k = k0 + lane;
    const bool hit = k < R && (uint32_t)row[k] < N;          // -1 and anything else out of range: no hit
    nh += (uint32_t)__popc(__ballot_sync(0xffffffffu, hit));
  }
  return nh;
}

// One warp per tracklet: count its hits, and if it is long enough raise the key of every cluster it uses.
__global__ void __launch_bounds__(256) select_claim_static(const int32_t* __restrict__ row_hits, uint32_t T, uint32_t R,
                                                           uint32_t N, uint32_t min_clusters, uint32_t* keys) {
  const uint32_t lane = threadIdx.x & 31u, n_warps = gridDim.x * (blockDim.x >> 5);
  for (uint32_t t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); t < T; t += n_warps) {
    const int32_t* row = row_hits + (size_t)t * R;
    const uint32_t nh = count_hits(row, R, N, lane);
    if (nh < min_clusters) continue;                          // warp-uniform
    const uint32_t key = claim_key_static(nh, t);
    for (uint32_t k = lane; k < R; k += 32u) {
      const uint32_t c = (uint32_t)row[k];
      if (c < N) atomicMax(keys + c, key);
    }
  }
}

// After every claim has landed: per tracklet, the hits whose key is still its own; per cluster, the index the
// winning key carries.  Both only read `keys`.
__global__ void __launch_bounds__(256) select_collect_static(const int32_t* __restrict__ row_hits, uint32_t T, uint32_t R,
                                                             uint32_t N, uint32_t min_clusters,
                                                             const uint32_t* __restrict__ keys, uint32_t* __restrict__ owner,
                                                             uint32_t* __restrict__ kept) {
  const uint32_t lane = threadIdx.x & 31u, n_warps = gridDim.x * (blockDim.x >> 5);
  for (uint32_t t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); t < T; t += n_warps) {
    const int32_t* row = row_hits + (size_t)t * R;
    const uint32_t nh = count_hits(row, R, N, lane);
    uint32_t mine = 0;
    if (nh >= min_clusters) {                                 // warp-uniform
      const uint32_t key = claim_key_static(nh, t);
      for (uint32_t k0 = 0; k0 < R; k0 += 32u) {
        const uint32_t k = k0 + lane;
        const uint32_t c = k < R ? (uint32_t)row[k] : 0xffffffffu;
        const bool own = c < N && keys[c] == key;
        mine += (uint32_t)__popc(__ballot_sync(0xffffffffu, own));
      }
    }
    if (lane == 0u) kept[t] = mine;
  }
  const uint32_t n_threads = gridDim.x * blockDim.x;
  for (uint32_t c = blockIdx.x * blockDim.x + threadIdx.x; c < N; c += n_threads) {
    const uint32_t k = keys[c];
    owner[c] = k ? 0xFFFFFFu - (k & 0xFFFFFFu) : 0xffffffffu;
  }
}

}  // namespace

extern "C" int tpcst_select_owners_static(const int32_t* row_hits, uint32_t n_tracklets, uint32_t n_rows, uint32_t n_clusters,
                                          uint32_t min_clusters, uint32_t* owner, uint32_t* kept, void* cuda_stream) {
  // sizes first: these answers need no GPU
  if (n_clusters > TPCST_STATIC_MAX_CLUSTERS) return TPCST_ERR_STATIC_LIMIT;
  if (n_rows < 1u || n_rows > 255u || min_clusters < 1u || min_clusters > 255u || n_tracklets > (1u << 24)) return TPCST_ERR_ARG;
  if ((n_tracklets && (!row_hits || !kept)) || (n_clusters && !owner)) return TPCST_ERR_ARG;
  if (!n_tracklets && !n_clusters) return TPCST_OK;
  // one device for all buffers
  int device = -1;
  const void* bufs[3] = {n_tracklets ? (const void*)row_hits : nullptr, n_tracklets ? (const void*)kept : nullptr,
                         n_clusters ? (const void*)owner : nullptr};
  for (const void* b : bufs) {
    if (!b) continue;
    const int d = device_of(b);
    if (d < 0 || d >= kMaxDevices || (device >= 0 && d != device)) return TPCST_ERR_ARG;
    device = d;
  }
  CurrentDevice cur(device);
  if (cur.err != cudaSuccess) return cuda_status(cur.err, "select the buffers' device");
  PerDevice dev;
  const int rc = setup_current_device(device, &dev);
  if (rc != TPCST_OK) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  uint32_t* const keys = dev.keys;                            // the DEVICE address, never the host-side name g_static_keys
  cudaError_t e = cudaSuccess;
  if (n_clusters) {
    e = cudaMemsetAsync(keys, 0, (size_t)n_clusters * 4u, st);  // the last call's keys are still there
    if (e != cudaSuccess) return cuda_status(e, "clear the static claim keys");
  }
  const uint32_t warps_per_cta = 256u / 32u;
  if (n_tracklets && n_clusters) {
    const uint32_t need = (n_tracklets + warps_per_cta - 1u) / warps_per_cta;
    select_claim_static<<<need < dev.grid_cap ? need : dev.grid_cap, 256, 0, st>>>(row_hits, n_tracklets, n_rows, n_clusters,
                                                                                   min_clusters, keys);
    if ((e = cudaGetLastError()) != cudaSuccess) return cuda_status(e, "select_claim_static");
  }
  {
    const uint32_t need_t = (n_tracklets + warps_per_cta - 1u) / warps_per_cta, need_c = (n_clusters + 255u) / 256u;
    uint32_t grid = need_t > need_c ? need_t : need_c;
    if (grid > dev.grid_cap) grid = dev.grid_cap;
    select_collect_static<<<grid, 256, 0, st>>>(row_hits, n_tracklets, n_rows, n_clusters, min_clusters, keys, owner, kept);
    if ((e = cudaGetLastError()) != cudaSuccess) return cuda_status(e, "select_collect_static");
  }
  return TPCST_OK;
}
