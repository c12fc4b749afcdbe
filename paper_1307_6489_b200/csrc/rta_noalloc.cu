// rta_noalloc.cu — rta_extract_image_noalloc (include/rta.h): extraction + image
// cleaning + moments for callers that cannot allocate device memory.
//
// Who that is. (1) A reconstruction thread in the middle of data taking: cudaMalloc
// and cudaFree synchronise the whole device, so one allocation on the analysis side
// would stall the copy stream that is feeding the next events in. (2) A process whose
// device memory is already handed out in full — a framework's caching allocator set
// to take everything, or a memory-partitioned GPU sized to the job — where an
// allocation made behind the owner's back fails or pushes the owner over its limit.
// rta_extract_image's route for unspecialised shapes asks the driver for scratch
// (16 bytes per trace, stream-ordered pool) and the staged kernels' tile scheduler
// lives in a cudaMalloc'ed pool; neither is acceptable to those callers.
//
// What this file does instead: the scratch is a file-scope device array of fixed size,
// part of the library image. Every device that loads librta.so holds its
// kNoAllocBytes (16 MiB + 256 bytes) from module load until the process exits,
// whether or not this entry point is ever called. Layout:
//
//   [0, 256)                      tile-scheduler words of the extraction kernel
//                                 {next tile, CTAs done}; must be zero when it starts
//   [256, 256 + 16 * n_traces)    out_sum | out_start | out_charge | out_time of this
//                                 call, n_traces entries each (the two float arrays
//                                 are what the moments kernel reads)
//
// The array keeps whatever the previous call left. The per-trace part needs no
// clearing (the extraction kernel writes every element the moments kernel reads);
// the scheduler words are zeroed on the caller's stream before every launch, so a
// call that was aborted half way cannot poison the next one.
//
// All calls on a device share the one array: two calls whose kernels can overlap on
// the GPU (different streams without an ordering between them, or two host threads
// on different streams) race on it and give garbage. Calls on one stream, or on
// streams the caller orders with events, are fine.
#include <cuda_runtime.h>

#include <atomic>
#include <mutex>

#include "../../include/rta.h"
#include "rta_internal.h"

static constexpr size_t kSchedBytes = 256;
static constexpr size_t kNoAllocBytes = kSchedBytes + 16u * (size_t)RTA_NOALLOC_MAX_TRACES;

// In host code this name is only a handle for cudaGetSymbolAddress: it is not a device
// address and must never be passed to a kernel or to cudaMemsetAsync as it stands.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

namespace {

constexpr int kMaxDev = 64;
std::mutex g_setup_mu;
std::atomic<int> g_ready[kMaxDev];
unsigned char* g_scratch_ptr[kMaxDev];  // device address of g_noalloc_scratch on device d

// Device address of the scratch array on the current device. The first call on a
// device asks the runtime for it (cudaGetSymbolAddress loads the module if it has not
// been loaded yet; it allocates nothing of ours); later calls read the cached pointer.
cudaError_t scratch_on_current_device(unsigned char** ptr) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
  if (!g_ready[dev].load(std::memory_order_acquire)) {
    std::lock_guard<std::mutex> lock(g_setup_mu);
    if (!g_ready[dev].load(std::memory_order_relaxed)) {
      void* p = nullptr;
      e = cudaGetSymbolAddress(&p, g_noalloc_scratch);  // `dev` is current
      if (e != cudaSuccess) return e;
      if (p == nullptr || ((uintptr_t)p % 256) != 0) return cudaErrorInvalidSymbol;
      g_scratch_ptr[dev] = static_cast<unsigned char*>(p);
      g_ready[dev].store(1, std::memory_order_release);
    }
  }
  *ptr = g_scratch_ptr[dev];
  return cudaSuccess;
}

}  // namespace

cudaError_t rta_launch_extract_image_noalloc(const void* wf, int64_t n_events, int32_t n_pixels,
                                             int32_t S, const int32_t* pedestal,
                                             const float* gain, int32_t W, const RtaCamera& cam,
                                             const RtaImageOut& out, cudaStream_t stream) {
  if (n_events <= 0) return cudaSuccess;
  const int64_t n_traces = n_events * (int64_t)n_pixels;
  if (n_traces > (int64_t)RTA_NOALLOC_MAX_TRACES) return cudaErrorInvalidValue;  // caller checks first
  if (((uintptr_t)wf % 16) != 0 || !rta_dyn_eligible(S, W)) return cudaErrorNotSupported;
  unsigned char* base = nullptr;
  cudaError_t e = scratch_on_current_device(&base);
  if (e != cudaSuccess) return e;
  uint32_t* sched = reinterpret_cast<uint32_t*>(base);
  int32_t* o_sum = reinterpret_cast<int32_t*>(base + kSchedBytes);
  int32_t* o_start = o_sum + n_traces;
  float* o_charge = reinterpret_cast<float*>(o_start + n_traces);
  float* o_time = o_charge + n_traces;
  // the scheduler words start every launch at zero, whatever the last call left
  if ((e = cudaMemsetAsync(sched, 0, kSchedBytes, stream)) != cudaSuccess) return e;
  e = rta_launch_extract_dyn_sched(wf, n_traces, n_pixels, S, pedestal, gain, W, o_sum, o_start,
                                   o_charge, o_time, stream, sched);
  if (e != cudaSuccess) return e;
  return rta_launch_image_moments(o_charge, o_time, n_events, n_pixels, cam, out, stream);
}
