// rta_api.cu — the C ABI of include/rta.h: validation, error reporting, and the
// host-fed double-buffered stream path (the
// page-locked transfer experiment of PAPER.md:133/139 §5 is its ancestor).
// No CPU fallback exists here: every compute call ends in a kernel launch or
// in an error code.
// The library is built with -fvisibility=hidden: what it exports is what
// include/rta.h declares (plus the test hooks below in librta_testing.so).
#pragma GCC visibility push(default)
#include "../../include/rta.h"
#ifdef RTA_TESTING
extern "C" {
int rta_extract_generic(const uint16_t* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
                        const int32_t* pedestal, const float* gain, int32_t W, int32_t* out_sum,
                        int32_t* out_start, float* out_charge, float* out_time, void* stream);
int rta_extract_image_generic(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                              int32_t n_samples, const int32_t* pedestal, const float* gain,
                              int32_t W, const float* pix_x, const float* pix_y,
                              const int32_t* neighbors, float thr_picture, float thr_boundary,
                              int32_t* out_n_pix, float* out_params, uint8_t* out_mask,
                              void* stream);
void rta_debug_serial_ragged(int on);
void rta_debug_force_generic(int on);
void rta_debug_static_schedule(int on);
void rta_debug_general_cleaning(int on);
void rta_debug_jit(int on);
void rta_debug_lanes_per_trace(int lpt);
void rta_debug_seg_tuning(int L, int TR, int NT, int stages);
}
#endif
#pragma GCC visibility pop

#include <cuda_runtime.h>

#include <algorithm>
#include <atomic>
#include <cstring>
#include <map>
#include <mutex>
#include <new>
#include <thread>
#include <utility>
#include <vector>

#include "rta_internal.h"

namespace {

thread_local int t_last_cuda = 0;
std::atomic<bool> g_serial_ragged{false};  // tests: rta_extract_ragged without side streams
std::atomic<bool> g_force_generic{false};  // tests: route the family entry points to the generic kernel
std::atomic<uint64_t> g_launches{0};

int fail_cuda(cudaError_t e) {
  t_last_cuda = (int)e;
  if (e == cudaErrorMemoryAllocation) return RTA_ERR_NOMEM;
  return RTA_ERR_CUDA;
}

int validate(const void* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
             const void* pedestal, const void* gain, int32_t W, const void* o0, const void* o1,
             const void* o2, const void* o3, int wf_align = 2) {
  if (n_events < 0 || n_pixels < 1 || n_samples < 1 || W < 1 || W > n_samples)
    return RTA_ERR_SHAPE;
  if (n_events * (int64_t)n_pixels >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
  if ((int64_t)n_samples * (int64_t)W * 65535ll >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
  if (n_events == 0) return RTA_OK;
  if (!wf || !pedestal || !gain || !o0 || !o1 || !o2 || !o3) return RTA_ERR_NULL;
  if ((uintptr_t)wf % (uintptr_t)wf_align != 0) return RTA_ERR_ALIGN;
  if (((uintptr_t)o0 | (uintptr_t)o1 | (uintptr_t)o2 | (uintptr_t)o3 | (uintptr_t)pedestal |
       (uintptr_t)gain) % 4 != 0)
    return RTA_ERR_ALIGN;
  return RTA_OK;
}

// ---- workspace of the stream path -----------------------------------------
struct Workspace {
  std::mutex mu;
  int device = -1;
  cudaStream_t copy_stream = nullptr;   // H2D
  cudaStream_t back_stream = nullptr;   // D2H of outputs (rta_extract_host)
  void* dev_buf[2] = {nullptr, nullptr};
  size_t dev_cap = 0;
  void* pin_buf[2] = {nullptr, nullptr};
  size_t pin_cap = 0;
  cudaEvent_t copied[2] = {nullptr, nullptr};    // H2D of buffer b finished
  cudaEvent_t consumed[2] = {nullptr, nullptr};  // kernel reading buffer b finished
  bool consumed_valid[2] = {false, false};
  // rta_extract_host only
  void* out_buf[2] = {nullptr, nullptr};   // 4 arrays x chunk traces
  size_t out_cap = 0;
  void* calib_buf = nullptr;
  size_t calib_cap = 0;
  cudaEvent_t done[2] = {nullptr, nullptr};      // kernel of slot b finished
  cudaEvent_t returned[2] = {nullptr, nullptr};  // D2H of slot b finished
  bool returned_valid[2] = {false, false};
  cudaStream_t host_stream = nullptr;            // compute stream of rta_extract_host
};
// One workspace per device, each behind its own mutex: host threads that feed different
// GPUs of one process neither wait for one another nor tear down each other's buffers
// (until round 3 there was one workspace per process, rebuilt whenever the current device
// changed). A workspace is created by the first host-fed call on its device.
constexpr int kMaxWsDevices = 32;
Workspace g_ws_tab[kMaxWsDevices];

// Which workspace serves `dev`; nullptr = a device index outside the table.
Workspace* ws_for_device(int dev) {
  return (dev >= 0 && dev < kMaxWsDevices) ? &g_ws_tab[dev] : nullptr;
}

// The workspace of the current device (not yet locked or prepared).
Workspace* ws_current(cudaError_t* err) {
  int dev = 0;
  *err = cudaGetDevice(&dev);
  if (*err != cudaSuccess) return nullptr;
  Workspace* w = ws_for_device(dev);
  if (w == nullptr) *err = cudaErrorInvalidDevice;
  return w;
}

void ws_release(Workspace& w) {
  for (int b = 0; b < 2; ++b) {
    if (w.dev_buf[b]) cudaFree(w.dev_buf[b]);
    if (w.pin_buf[b]) cudaFreeHost(w.pin_buf[b]);
    if (w.out_buf[b]) cudaFree(w.out_buf[b]);
    if (w.copied[b]) cudaEventDestroy(w.copied[b]);
    if (w.consumed[b]) cudaEventDestroy(w.consumed[b]);
    if (w.done[b]) cudaEventDestroy(w.done[b]);
    if (w.returned[b]) cudaEventDestroy(w.returned[b]);
    w.dev_buf[b] = w.pin_buf[b] = w.out_buf[b] = nullptr;
    w.copied[b] = w.consumed[b] = w.done[b] = w.returned[b] = nullptr;
    w.consumed_valid[b] = w.returned_valid[b] = false;
  }
  if (w.calib_buf) cudaFree(w.calib_buf);
  w.calib_buf = nullptr;
  if (w.copy_stream) cudaStreamDestroy(w.copy_stream);
  if (w.back_stream) cudaStreamDestroy(w.back_stream);
  if (w.host_stream) cudaStreamDestroy(w.host_stream);
  w.copy_stream = w.back_stream = w.host_stream = nullptr;
  w.dev_cap = w.pin_cap = w.out_cap = w.calib_cap = 0;
  w.device = -1;
}

cudaError_t ws_prepare(Workspace& w) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (w.device != dev) {
    if (w.device >= 0) {
      int cur = dev;
      cudaSetDevice(w.device);
      cudaDeviceSynchronize();
      ws_release(w);
      cudaSetDevice(cur);
    }
    if ((e = cudaStreamCreateWithFlags(&w.copy_stream, cudaStreamNonBlocking)) != cudaSuccess)
      return e;
    if ((e = cudaStreamCreateWithFlags(&w.back_stream, cudaStreamNonBlocking)) != cudaSuccess)
      return e;
    if ((e = cudaStreamCreateWithFlags(&w.host_stream, cudaStreamNonBlocking)) != cudaSuccess)
      return e;
    for (int b = 0; b < 2; ++b) {
      if ((e = cudaEventCreateWithFlags(&w.copied[b], cudaEventDisableTiming)) != cudaSuccess)
        return e;
      if ((e = cudaEventCreateWithFlags(&w.consumed[b], cudaEventDisableTiming)) != cudaSuccess)
        return e;
      if ((e = cudaEventCreateWithFlags(&w.done[b], cudaEventDisableTiming)) != cudaSuccess)
        return e;
      if ((e = cudaEventCreateWithFlags(&w.returned[b], cudaEventDisableTiming)) != cudaSuccess)
        return e;
    }
    w.device = dev;
  }
  return cudaSuccess;
}

// grow a pair of buffers; waits for outstanding users before freeing
template <class Alloc, class Free>
cudaError_t grow_pair(void* buf[2], size_t* cap, size_t need, Alloc alloc, Free release) {
  if (*cap >= need) return cudaSuccess;
  cudaError_t e = cudaDeviceSynchronize();
  if (e != cudaSuccess) return e;
  for (int b = 0; b < 2; ++b) {
    if (buf[b]) release(buf[b]);
    buf[b] = nullptr;
  }
  *cap = 0;
  for (int b = 0; b < 2; ++b) {
    if ((e = alloc(&buf[b], need)) != cudaSuccess) return e;
  }
  *cap = need;
  return cudaSuccess;
}

bool is_pageable(const void* p) {
  cudaPointerAttributes a;
  cudaError_t e = cudaPointerGetAttributes(&a, p);
  if (e != cudaSuccess) {
    cudaGetLastError();  // clear
    return true;
  }
  return a.type == cudaMemoryTypeUnregistered;
}

// Pageable source -> pinned staging slot. One memcpy thread moves about 10 GB/s,
// a fifth of a PCIe Gen5 x16 link; up to 8 threads (at least 8 MiB each, slices on
// page boundaries) keep the staging ahead of the H2D copy of the previous chunk.
void staging_copy(void* dst, const void* src, size_t bytes) {
  const unsigned hw = std::thread::hardware_concurrency();
  size_t n = std::min<size_t>(bytes / ((size_t)8 << 20), std::min<size_t>(8, hw > 1 ? hw / 2 : 1));
  if (n <= 1) {
    std::memcpy(dst, src, bytes);
    return;
  }
  const size_t slice = ((bytes / n) + 4095u) & ~(size_t)4095u;
  std::vector<std::thread> workers;
  workers.reserve(n - 1);
  for (size_t i = 1; i < n; ++i) {
    const size_t lo = i * slice;
    if (lo >= bytes) break;
    const size_t len = std::min(slice, bytes - lo);
    try {
      workers.emplace_back([=] {
        std::memcpy(static_cast<uint8_t*>(dst) + lo, static_cast<const uint8_t*>(src) + lo, len);
      });
    } catch (...) {  // no thread to be had: this one does the slice
      std::memcpy(static_cast<uint8_t*>(dst) + lo, static_cast<const uint8_t*>(src) + lo, len);
    }
  }
  std::memcpy(dst, src, std::min(slice, bytes));
  for (std::thread& t : workers) t.join();
}

struct ChunkPlan {
  int64_t chunk_events;
  int64_t n_chunks;
  size_t event_bits;   // bits of one event in the source format
};
int64_t gcd64(int64_t a, int64_t b) {
  while (b) {
    const int64_t t = a % b;
    a = b;
    b = t;
  }
  return a;
}
// Chunks of whole events of at most chunk_bytes (rounded down, at least one
// event). A P12 chunk must also start on a 16-byte boundary of the stream
// (whole bytes for the copy, 16 bytes for the staged kernels): its event count
// is a multiple of m, the smallest count with m * n_pixels * n_samples % 32 == 0.
ChunkPlan plan_chunks(int64_t n_events, int32_t n_pixels, int32_t n_samples, size_t chunk_bytes,
                      int bits) {
  ChunkPlan p;
  const int64_t ev_samples = (int64_t)n_pixels * (int64_t)n_samples;
  p.event_bits = (size_t)ev_samples * (size_t)bits;
  if (chunk_bytes == 0) chunk_bytes = (size_t)1 << 30;
  if (chunk_bytes > ((size_t)1 << 48)) chunk_bytes = (size_t)1 << 48;  // the products below stay far from 2^64
  const int64_t m = bits == 12 ? 32 / gcd64(ev_samples, 32) : 1;
  int64_t ce = (int64_t)((chunk_bytes / p.event_bits) * 8u +
                         ((chunk_bytes % p.event_bits) * 8u) / p.event_bits);  // whole events
  ce -= ce % m;
  if (ce < m) ce = m;
  if (ce > n_events) ce = n_events > 0 ? n_events : 1;
  p.chunk_events = ce;
  p.n_chunks = (n_events + ce - 1) / ce;
  return p;
}

// Core of the host-fed path: chunks of whole events go through the device
// double buffer; `launch(dev_chunk, ev0, nev, slot)` enqueues the kernel(s) of
// one chunk on `stream`. With out_slot_bytes != 0 the kernels write to one of
// two library-owned device slots (`slot`, else nullptr) and
// `back(ev0, nev, slot, back_stream)` enqueues the D2H copies of that chunk.
template <class Launch, class Back>
int stream_core(Workspace& w, const void* wf_host, int64_t n_events, int32_t n_pixels,
                int32_t n_samples, size_t chunk_bytes, cudaStream_t stream, int bits,
                size_t out_slot_bytes, Launch launch, Back back) {
  cudaError_t e;
  const ChunkPlan plan = plan_chunks(n_events, n_pixels, n_samples, chunk_bytes, bits);
  const size_t buf_bytes = ((size_t)plan.chunk_events * plan.event_bits + 7u) / 8u;
  e = grow_pair(
      w.dev_buf, &w.dev_cap, buf_bytes, [](void** p, size_t n) { return cudaMalloc(p, n); },
      [](void* p) { cudaFree(p); });
  if (e != cudaSuccess) return fail_cuda(e);
  const bool pageable = is_pageable(wf_host);
  if (pageable) {
    e = grow_pair(
        w.pin_buf, &w.pin_cap, buf_bytes,
        [](void** p, size_t n) { return cudaHostAlloc(p, n, cudaHostAllocDefault); },
        [](void* p) { cudaFreeHost(p); });
    if (e != cudaSuccess) return fail_cuda(e);
  }
  const bool to_host = out_slot_bytes != 0;
  if (to_host) {
    e = grow_pair(
        w.out_buf, &w.out_cap, out_slot_bytes,
        [](void** p, size_t n) { return cudaMalloc(p, n); }, [](void* p) { cudaFree(p); });
    if (e != cudaSuccess) return fail_cuda(e);
  }

  for (int64_t k = 0; k < plan.n_chunks; ++k) {
    const int b = (int)(k & 1);
    const int64_t ev0 = k * plan.chunk_events;
    const int64_t nev = (ev0 + plan.chunk_events <= n_events) ? plan.chunk_events : n_events - ev0;
    // ev0 * event_bits is a multiple of 128 (plan_chunks); only the last chunk
    // of a P12 stream can end inside a byte
    const size_t bytes = ((size_t)nev * plan.event_bits + 7u) / 8u;
    const uint8_t* src =
        reinterpret_cast<const uint8_t*>(wf_host) + ((size_t)ev0 * plan.event_bits) / 8u;

    // the device buffer is free once the kernel of chunk k-2 (or of an
    // earlier call) has finished with it
    if (w.consumed_valid[b]) {
      if ((e = cudaStreamWaitEvent(w.copy_stream, w.consumed[b], 0)) != cudaSuccess)
        return fail_cuda(e);
    }
    if (pageable) {
      // pinned staging slot b is free once its previous H2D copy has finished
      // (an event never recorded counts as complete)
      if ((e = cudaEventSynchronize(w.copied[b])) != cudaSuccess) return fail_cuda(e);
      staging_copy(w.pin_buf[b], src, bytes);
      src = reinterpret_cast<const uint8_t*>(w.pin_buf[b]);
    }
    if ((e = cudaMemcpyAsync(w.dev_buf[b], src, bytes, cudaMemcpyHostToDevice, w.copy_stream)) !=
        cudaSuccess)
      return fail_cuda(e);
    if ((e = cudaEventRecord(w.copied[b], w.copy_stream)) != cudaSuccess) return fail_cuda(e);
    if ((e = cudaStreamWaitEvent(stream, w.copied[b], 0)) != cudaSuccess) return fail_cuda(e);

    // output slot b is free once its previous D2H has finished
    if (to_host && w.returned_valid[b]) {
      if ((e = cudaStreamWaitEvent(stream, w.returned[b], 0)) != cudaSuccess) return fail_cuda(e);
    }
    uint8_t* slot = to_host ? reinterpret_cast<uint8_t*>(w.out_buf[b]) : nullptr;
    if ((e = launch(w.dev_buf[b], ev0, nev, slot)) != cudaSuccess) return fail_cuda(e);
    if ((e = cudaEventRecord(w.consumed[b], stream)) != cudaSuccess) return fail_cuda(e);
    w.consumed_valid[b] = true;

    if (to_host) {
      if ((e = cudaStreamWaitEvent(w.back_stream, w.consumed[b], 0)) != cudaSuccess)
        return fail_cuda(e);
      if ((e = back(ev0, nev, slot, w.back_stream)) != cudaSuccess) return fail_cuda(e);
      if ((e = cudaEventRecord(w.returned[b], w.back_stream)) != cudaSuccess) return fail_cuda(e);
      w.returned_valid[b] = true;
    }
  }
  return RTA_OK;
}

// Per-trace extraction through stream_core. When `host_out` is set, per-chunk
// results are written to the device slots and copied back to the host arrays.
struct HostOut {
  int32_t* sum;
  int32_t* start;
  float* charge;
  float* time;
};

int stream_impl(Workspace& w, const void* wf_host, int64_t n_events, int32_t n_pixels,
                int32_t n_samples, const int32_t* pedestal, const float* gain, int32_t W,
                int32_t* out_sum, int32_t* out_start, float* out_charge, float* out_time,
                size_t chunk_bytes, cudaStream_t stream, const HostOut* host_out, int bits = 16) {
  const ChunkPlan plan = plan_chunks(n_events, n_pixels, n_samples, chunk_bytes, bits);
  const size_t chunk_traces = (size_t)plan.chunk_events * (size_t)n_pixels;
  auto launch = [&](const void* dev_chunk, int64_t ev0, int64_t nev, uint8_t* slot) {
    const size_t t0 = (size_t)ev0 * (size_t)n_pixels;
    int32_t *o_sum = out_sum + t0, *o_start = out_start + t0;
    float *o_charge = out_charge + t0, *o_time = out_time + t0;
    if (slot) {
      o_sum = reinterpret_cast<int32_t*>(slot);
      o_start = reinterpret_cast<int32_t*>(slot + chunk_traces * 4u);
      o_charge = reinterpret_cast<float*>(slot + chunk_traces * 8u);
      o_time = reinterpret_cast<float*>(slot + chunk_traces * 12u);
    }
    return rta_launch_extract(dev_chunk, nev * (int64_t)n_pixels, n_pixels, n_samples, pedestal,
                              gain, W, o_sum, o_start, o_charge, o_time, stream, false, nullptr,
                              bits);
  };
  auto back = [&](int64_t ev0, int64_t nev, uint8_t* slot, cudaStream_t bs) {
    const size_t t0 = (size_t)ev0 * (size_t)n_pixels;
    const size_t nb = (size_t)nev * (size_t)n_pixels * 4u;
    void* dst[4] = {host_out->sum + t0, host_out->start + t0, host_out->charge + t0,
                    host_out->time + t0};
    for (int i = 0; i < 4; ++i) {
      const cudaError_t e = cudaMemcpyAsync(dst[i], slot + chunk_traces * 4u * (size_t)i, nb,
                                            cudaMemcpyDeviceToHost, bs);
      if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
  };
  return stream_core(w, wf_host, n_events, n_pixels, n_samples, chunk_bytes, stream, bits,
                     host_out ? chunk_traces * 16u : 0u, launch, back);
}

// Host-to-host path (rta_extract_host, rta_extract_host_packed12): calibration
// up, chunks through stream_impl, results back; synchronous.
int host_impl(const void* wf_host, int64_t n_events, int32_t n_pixels, int32_t n_samples,
              const int32_t* pedestal_host, const float* gain_host, int32_t W,
              int32_t* out_sum_host, int32_t* out_start_host, float* out_charge_host,
              float* out_time_host, size_t chunk_bytes, int bits) {
  const int v = validate(wf_host, n_events, n_pixels, n_samples, pedestal_host, gain_host, W,
                         out_sum_host, out_start_host, out_charge_host, out_time_host,
                         bits == 12 ? 1 : 2);
  if (v != RTA_OK || n_events == 0) return v;
  cudaError_t e0 = cudaSuccess;
  Workspace* wsp = ws_current(&e0);
  if (wsp == nullptr) return fail_cuda(e0);
  Workspace& w = *wsp;
  std::lock_guard<std::mutex> lock(w.mu);
  cudaError_t e = ws_prepare(w);
  if (e != cudaSuccess) return fail_cuda(e);
  const size_t calib_bytes = (size_t)n_pixels * 8u;
  if (w.calib_cap < calib_bytes) {
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return fail_cuda(e);
    if (w.calib_buf) cudaFree(w.calib_buf);
    w.calib_buf = nullptr;
    w.calib_cap = 0;
    if ((e = cudaMalloc(&w.calib_buf, calib_bytes)) != cudaSuccess) return fail_cuda(e);
    w.calib_cap = calib_bytes;
  }
  int32_t* d_ped = reinterpret_cast<int32_t*>(w.calib_buf);
  float* d_gain = reinterpret_cast<float*>(reinterpret_cast<uint8_t*>(w.calib_buf) +
                                           (size_t)n_pixels * 4u);
  // calibration constants may still be read by kernels of an earlier call
  if ((e = cudaStreamSynchronize(w.host_stream)) != cudaSuccess) return fail_cuda(e);
  if ((e = cudaMemcpyAsync(d_ped, pedestal_host, (size_t)n_pixels * 4u, cudaMemcpyHostToDevice,
                           w.host_stream)) != cudaSuccess)
    return fail_cuda(e);
  if ((e = cudaMemcpyAsync(d_gain, gain_host, (size_t)n_pixels * 4u, cudaMemcpyHostToDevice,
                           w.host_stream)) != cudaSuccess)
    return fail_cuda(e);
  const HostOut ho{out_sum_host, out_start_host, out_charge_host, out_time_host};
  const int rc = stream_impl(w, wf_host, n_events, n_pixels, n_samples, d_ped, d_gain, W, nullptr,
                             nullptr, nullptr, nullptr, chunk_bytes, w.host_stream, &ho, bits);
  // synchronous by contract, also on the error path (nothing may outlive the call)
  cudaError_t e1 = cudaStreamSynchronize(w.host_stream);
  cudaError_t e2 = cudaStreamSynchronize(w.back_stream);
  cudaError_t e3 = cudaStreamSynchronize(w.copy_stream);
  if (rc != RTA_OK) return rc;
  if (e1 != cudaSuccess) return fail_cuda(e1);
  if (e2 != cudaSuccess) return fail_cuda(e2);
  if (e3 != cudaSuccess) return fail_cuda(e3);
  return RTA_OK;
}

// ---- image cleaning + moments (NEXT-4; readings R31-R35) ----------
int validate_image(int64_t n_events, int32_t n_pixels, const void* pix_x, const void* pix_y,
                   const void* neighbors, const void* out_n_pix, const void* out_params,
                   const void* out_mask) {
  (void)out_mask;  // optional, bytes: no alignment requirement
  if (n_events < 0 || n_pixels < 1) return RTA_ERR_SHAPE;
  if (n_events * (int64_t)n_pixels >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
  if (n_pixels > rta_image_pixel_limit()) return RTA_ERR_UNSUPPORTED;
  if (n_events == 0) return RTA_OK;
  if (!pix_x || !pix_y || !neighbors || !out_n_pix || !out_params) return RTA_ERR_NULL;
  if (((uintptr_t)pix_x | (uintptr_t)pix_y | (uintptr_t)neighbors | (uintptr_t)out_n_pix |
       (uintptr_t)out_params) % 4 != 0)
    return RTA_ERR_ALIGN;
  return RTA_OK;
}

// extraction-side checks of the fused calls (no per-trace outputs to check)
int validate_fused(const void* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
                   const void* pedestal, const void* gain, int32_t W) {
  if (n_events < 0 || n_pixels < 1 || n_samples < 1 || W < 1 || W > n_samples)
    return RTA_ERR_SHAPE;
  if (n_events * (int64_t)n_pixels >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
  if ((int64_t)n_samples * (int64_t)W * 65535ll >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
  if (n_events == 0) return RTA_OK;
  if (!wf || !pedestal || !gain) return RTA_ERR_NULL;
  if ((uintptr_t)wf % 2 != 0) return RTA_ERR_ALIGN;
  if (((uintptr_t)pedestal | (uintptr_t)gain) % 4 != 0) return RTA_ERR_ALIGN;
  return RTA_OK;
}

// Host-fed fused path: waveform chunks in, event parameters out. `host_out`
// set: results go through the device slots back to host arrays.
struct ImageHostOut {
  int32_t* n_pix;
  float* params;
  uint8_t* mask;
};

int image_stream_impl(Workspace& w, const void* wf_host, int64_t n_events, int32_t n_pixels,
                      int32_t n_samples, const int32_t* pedestal, const float* gain, int32_t W,
                      const RtaCamera& cam, const RtaImageOut& out, size_t chunk_bytes,
                      cudaStream_t stream, const ImageHostOut* host_out) {
  const ChunkPlan plan = plan_chunks(n_events, n_pixels, n_samples, chunk_bytes, 16);
  const size_t ce = (size_t)plan.chunk_events;
  const bool want_mask = host_out ? host_out->mask != nullptr : out.mask != nullptr;
  // slot layout: params [ce][8] float, n_pix [ce] int32, mask [ce][P] bytes
  const size_t slot_bytes = ce * 36u + (want_mask ? ce * (size_t)n_pixels : 0u);
  auto launch = [&](const void* dev_chunk, int64_t ev0, int64_t nev, uint8_t* slot) {
    RtaImageOut o;
    if (slot) {
      o.params = reinterpret_cast<float*>(slot);
      o.n_pix = reinterpret_cast<int32_t*>(slot + ce * 32u);
      o.mask = want_mask ? slot + ce * 36u : nullptr;
    } else {
      o.n_pix = out.n_pix + ev0;
      o.params = out.params + (size_t)ev0 * 8u;
      o.mask = out.mask ? out.mask + (size_t)ev0 * (size_t)n_pixels : nullptr;
    }
    return rta_launch_extract_image(dev_chunk, nev, n_pixels, n_samples, pedestal, gain, W, cam,
                                    o, stream, false);
  };
  auto back = [&](int64_t ev0, int64_t nev, uint8_t* slot, cudaStream_t bs) {
    cudaError_t e = cudaMemcpyAsync(host_out->params + (size_t)ev0 * 8u, slot,
                                    (size_t)nev * 32u, cudaMemcpyDeviceToHost, bs);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(host_out->n_pix + ev0, slot + ce * 32u, (size_t)nev * 4u,
                        cudaMemcpyDeviceToHost, bs);
    if (e != cudaSuccess) return e;
    if (want_mask)
      e = cudaMemcpyAsync(host_out->mask + (size_t)ev0 * (size_t)n_pixels, slot + ce * 36u,
                          (size_t)nev * (size_t)n_pixels, cudaMemcpyDeviceToHost, bs);
    return e;
  };
  return stream_core(w, wf_host, n_events, n_pixels, n_samples, chunk_bytes, stream, 16,
                     host_out ? slot_bytes : 0u, launch, back);
}

}  // namespace

void rta_count_launch() { g_launches.fetch_add(1, std::memory_order_relaxed); }

extern "C" {

int rta_extract(const uint16_t* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
                const int32_t* pedestal, const float* gain, int32_t W, int32_t* out_sum,
                int32_t* out_start, float* out_charge, float* out_time, void* stream) {
  const int v = validate(wf, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum, out_start,
                         out_charge, out_time);
  if (v != RTA_OK || n_events == 0) return v;
  const cudaError_t e =
      rta_launch_extract(wf, n_events * (int64_t)n_pixels, n_pixels, n_samples, pedestal, gain, W,
                         out_sum, out_start, out_charge, out_time, (cudaStream_t)stream, false);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

#ifdef RTA_TESTING
// Same as rta_extract but always through the generic kernel. Only in
// librta_testing.so (built with -DRTA_TESTING; two independent device paths
// must agree); the shipped librta.so exports include/rta.h and nothing else.
int rta_extract_generic(const uint16_t* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
                        const int32_t* pedestal, const float* gain, int32_t W, int32_t* out_sum,
                        int32_t* out_start, float* out_charge, float* out_time, void* stream) {
  const int v = validate(wf, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum, out_start,
                         out_charge, out_time);
  if (v != RTA_OK || n_events == 0) return v;
  const cudaError_t e =
      rta_launch_extract(wf, n_events * (int64_t)n_pixels, n_pixels, n_samples, pedestal, gain, W,
                         out_sum, out_start, out_charge, out_time, (cudaStream_t)stream, true);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}
#endif  // RTA_TESTING

// ---- the other members of the extractor family (NEXT-1; readings R22-R24) ----
int rta_extract_fixed(const uint16_t* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
                      const int32_t* pedestal, const float* gain, int32_t W,
                      const int32_t* window_start, int32_t* out_sum, int32_t* out_start,
                      float* out_charge, float* out_time, void* stream) {
  const int v = validate(wf, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum, out_start,
                         out_charge, out_time);
  if (v != RTA_OK || n_events == 0) return v;
  if (!window_start) return RTA_ERR_NULL;
  if ((uintptr_t)window_start % 4 != 0) return RTA_ERR_ALIGN;
  RtaMode m = {};
  m.kind = RTA_MODE_FIXED;
  m.window_start = window_start;
  const cudaError_t e = rta_launch_extract(wf, n_events * (int64_t)n_pixels, n_pixels, n_samples,
                                           pedestal, gain, W, out_sum, out_start, out_charge,
                                           out_time, (cudaStream_t)stream, g_force_generic, &m);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

int rta_extract_local_peak(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                           int32_t n_samples, const int32_t* pedestal, const float* gain,
                           int32_t W, int32_t shift, int32_t* out_sum, int32_t* out_start,
                           float* out_charge, float* out_time, void* stream) {
  const int v = validate(wf, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum, out_start,
                         out_charge, out_time);
  if (v != RTA_OK || n_events == 0) return v;
  RtaMode m = {};
  m.kind = RTA_MODE_LOCAL_PEAK;
  // |shift| >= n_samples already pins the window to one end of the trace
  m.shift = shift > n_samples ? n_samples : (shift < -n_samples ? -n_samples : shift);
  const cudaError_t e = rta_launch_extract(wf, n_events * (int64_t)n_pixels, n_pixels, n_samples,
                                           pedestal, gain, W, out_sum, out_start, out_charge,
                                           out_time, (cudaStream_t)stream, g_force_generic, &m);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

int rta_extract_fir(const uint16_t* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
                    const int32_t* pedestal, const float* gain, const int32_t* taps,
                    int32_t n_taps, int32_t* out_sum, int32_t* out_start, float* out_charge,
                    float* out_time, void* stream) {
  if (n_events < 0 || n_pixels < 1 || n_samples < 1 || n_taps < 1 || n_taps > n_samples)
    return RTA_ERR_SHAPE;
  if (n_taps > RTA_MAX_TAPS) return RTA_ERR_UNSUPPORTED;
  if (!taps) return RTA_ERR_NULL;
  int64_t abs_sum = 0;
  for (int k = 0; k < n_taps; ++k) abs_sum += taps[k] < 0 ? -(int64_t)taps[k] : (int64_t)taps[k];
  if (abs_sum < 1) abs_sum = 1;
  if ((int64_t)n_samples * 65535ll >= (1ll << 31) / abs_sum) return RTA_ERR_UNSUPPORTED;
  if (n_events * (int64_t)n_pixels >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
  // the remaining checks are those of the plain window with W = 1 (pointers, alignment)
  const int v = validate(wf, n_events, n_pixels, n_samples, pedestal, gain, 1, out_sum, out_start,
                         out_charge, out_time);
  if (v != RTA_OK || n_events == 0) return v;
  RtaMode m = {};
  m.kind = RTA_MODE_FIR;
  m.n_taps = n_taps;
  for (int k = 0; k < n_taps; ++k) m.taps[k] = taps[k];
  const cudaError_t e = rta_launch_extract(wf, n_events * (int64_t)n_pixels, n_pixels, n_samples,
                                           pedestal, gain, n_taps, out_sum, out_start, out_charge,
                                           out_time, (cudaStream_t)stream, g_force_generic, &m);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

int rta_extract_stream(const uint16_t* wf_host, int64_t n_events, int32_t n_pixels,
                       int32_t n_samples, const int32_t* pedestal, const float* gain, int32_t W,
                       int32_t* out_sum, int32_t* out_start, float* out_charge, float* out_time,
                       size_t chunk_bytes, void* stream) {
  const int v = validate(wf_host, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum,
                         out_start, out_charge, out_time);
  if (v != RTA_OK || n_events == 0) return v;
  cudaError_t e = cudaSuccess;
  Workspace* wsp = ws_current(&e);
  if (wsp == nullptr) return fail_cuda(e);
  Workspace& ws = *wsp;
  std::lock_guard<std::mutex> lock(ws.mu);
  e = ws_prepare(ws);
  if (e != cudaSuccess) return fail_cuda(e);
  return stream_impl(ws, wf_host, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum,
                     out_start, out_charge, out_time, chunk_bytes, (cudaStream_t)stream, nullptr);
}

int rta_extract_host(const uint16_t* wf_host, int64_t n_events, int32_t n_pixels,
                     int32_t n_samples, const int32_t* pedestal_host, const float* gain_host,
                     int32_t W, int32_t* out_sum_host, int32_t* out_start_host,
                     float* out_charge_host, float* out_time_host, size_t chunk_bytes) {
  return host_impl(wf_host, n_events, n_pixels, n_samples, pedestal_host, gain_host, W,
                   out_sum_host, out_start_host, out_charge_host, out_time_host, chunk_bytes, 16);
}

// ---- packed 12-bit ingest (NEXT-2; readings R25-R27) -----------------
int rta_extract_packed12(const uint8_t* packed, int64_t n_events, int32_t n_pixels,
                         int32_t n_samples, const int32_t* pedestal, const float* gain,
                         int32_t W, int32_t* out_sum, int32_t* out_start, float* out_charge,
                         float* out_time, void* stream) {
  const int v = validate(packed, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum,
                         out_start, out_charge, out_time, 1);
  if (v != RTA_OK || n_events == 0) return v;
  const cudaError_t e = rta_launch_extract(packed, n_events * (int64_t)n_pixels, n_pixels,
                                           n_samples, pedestal, gain, W, out_sum, out_start,
                                           out_charge, out_time, (cudaStream_t)stream,
                                           g_force_generic, nullptr, 12);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

int rta_extract_stream_packed12(const uint8_t* packed_host, int64_t n_events, int32_t n_pixels,
                                int32_t n_samples, const int32_t* pedestal, const float* gain,
                                int32_t W, int32_t* out_sum, int32_t* out_start,
                                float* out_charge, float* out_time, size_t chunk_bytes,
                                void* stream) {
  const int v = validate(packed_host, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum,
                         out_start, out_charge, out_time, 1);
  if (v != RTA_OK || n_events == 0) return v;
  cudaError_t e = cudaSuccess;
  Workspace* wsp = ws_current(&e);
  if (wsp == nullptr) return fail_cuda(e);
  Workspace& ws = *wsp;
  std::lock_guard<std::mutex> lock(ws.mu);
  e = ws_prepare(ws);
  if (e != cudaSuccess) return fail_cuda(e);
  return stream_impl(ws, packed_host, n_events, n_pixels, n_samples, pedestal, gain, W, out_sum,
                     out_start, out_charge, out_time, chunk_bytes, (cudaStream_t)stream, nullptr,
                     12);
}

int rta_extract_host_packed12(const uint8_t* packed_host, int64_t n_events, int32_t n_pixels,
                              int32_t n_samples, const int32_t* pedestal_host,
                              const float* gain_host, int32_t W, int32_t* out_sum_host,
                              int32_t* out_start_host, float* out_charge_host,
                              float* out_time_host, size_t chunk_bytes) {
  return host_impl(packed_host, n_events, n_pixels, n_samples, pedestal_host, gain_host, W,
                   out_sum_host, out_start_host, out_charge_host, out_time_host, chunk_bytes, 12);
}

// ---- mixed-camera batches (NEXT-3; readings R28-R30) ----------------
struct rta_ragged_plan {
  int device = -1;
  RtaRaggedTile* tiles_dev = nullptr;  // all classes, one after the other
  struct Class {
    int32_t S, W;
    int32_t tile_traces;    // what the class's tiles were cut for (rta_ragged_tile_traces at plan time)
    uint32_t first, count;  // range in tiles_dev
  };
  std::vector<Class> classes;
  int64_t n_blocks = 0, n_traces = 0, n_tiles = 0, wf_bytes = 0, wf_end = 0, out_end = 0;
};

int rta_ragged_plan_create(int32_t n_tel, const int32_t* tel_n_pixels,
                           const int32_t* tel_n_samples, const int32_t* tel_W,
                           const int64_t* tel_calib_offset, int64_t n_blocks,
                           const int32_t* blk_tel, const int64_t* blk_wf_offset,
                           const int64_t* blk_out_offset, rta_ragged_plan** plan) {
  if (!plan) return RTA_ERR_NULL;
  *plan = nullptr;
  if (n_tel < 0 || n_blocks < 0) return RTA_ERR_SHAPE;
  if (n_tel > 0 && (!tel_n_pixels || !tel_n_samples || !tel_W || !tel_calib_offset))
    return RTA_ERR_NULL;
  if (n_blocks > 0 && (!blk_tel || !blk_wf_offset || !blk_out_offset)) return RTA_ERR_NULL;
  for (int32_t k = 0; k < n_tel; ++k) {
    const int64_t P = tel_n_pixels[k], S = tel_n_samples[k], W = tel_W[k];
    if (P < 1 || S < 1 || W < 1 || W > S || tel_calib_offset[k] < 0) return RTA_ERR_SHAPE;
    if (S * W * 65535ll >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
    if (tel_calib_offset[k] + P >= (1ll << 32)) return RTA_ERR_UNSUPPORTED;
  }
  rta_ragged_plan* pl = new (std::nothrow) rta_ragged_plan;
  if (!pl) return RTA_ERR_NOMEM;
  // tiles grouped by shape class, blocks in table order inside a class
  std::map<std::pair<int32_t, int32_t>, std::vector<RtaRaggedTile>> by_shape;
  std::map<std::pair<int32_t, int32_t>, int> tile_of;  // tile size per shape class, asked once
  for (int64_t b = 0; b < n_blocks; ++b) {
    const int32_t k = blk_tel[b];
    if (k < 0 || k >= n_tel || blk_wf_offset[b] < 0 || blk_out_offset[b] < 0) {
      delete pl;
      return RTA_ERR_SHAPE;
    }
    const int64_t P = tel_n_pixels[k], S = tel_n_samples[k];
    // range checks before any arithmetic on the offsets: an offset near 2^62
    // would wrap (P * S < 2^46 by the telescope checks above)
    if (blk_wf_offset[b] >= (1ll << 47) || blk_out_offset[b] >= (1ll << 31)) {
      delete pl;
      return RTA_ERR_UNSUPPORTED;
    }
    const int64_t end_bytes = (blk_wf_offset[b] + P * S) * 2;
    if (blk_out_offset[b] + P >= (1ll << 31) || end_bytes >= (1ll << 48)) {
      delete pl;
      return RTA_ERR_UNSUPPORTED;
    }
    const auto shape = std::make_pair((int32_t)S, tel_W[k]);
    auto tile_it = tile_of.find(shape);
    if (tile_it == tile_of.end())
      tile_it = tile_of.emplace(shape, rta_ragged_tile_traces((int32_t)S, tel_W[k])).first;
    const int64_t tt = tile_it->second;
    std::vector<RtaRaggedTile>& v = by_shape[shape];
    for (int64_t t0 = 0; t0 < P; t0 += tt) {
      const int64_t n = (P - t0 < tt) ? P - t0 : tt;
      RtaRaggedTile t;
      t.src = (unsigned long long)((blk_wf_offset[b] + t0 * S) * 2) | ((unsigned long long)n << 48);
      t.out_base = (uint32_t)(blk_out_offset[b] + t0);
      t.cal0 = (uint32_t)(tel_calib_offset[k] + t0);
      v.push_back(t);
    }
    pl->n_traces += P;
    pl->wf_bytes += P * S * 2;
    if (end_bytes > pl->wf_end) pl->wf_end = end_bytes;
    if (blk_out_offset[b] + P > pl->out_end) pl->out_end = blk_out_offset[b] + P;
  }
  pl->n_blocks = n_blocks;
  std::vector<RtaRaggedTile> all;
  for (auto& kv : by_shape) {
    if (kv.second.size() >= (1ull << 32) || all.size() + kv.second.size() >= (1ull << 32)) {
      delete pl;
      return RTA_ERR_UNSUPPORTED;
    }
    rta_ragged_plan::Class c;
    c.S = kv.first.first;
    c.W = kv.first.second;
    c.tile_traces = tile_of[kv.first];
    c.first = (uint32_t)all.size();
    c.count = (uint32_t)kv.second.size();
    pl->classes.push_back(c);
    all.insert(all.end(), kv.second.begin(), kv.second.end());
  }
  pl->n_tiles = (int64_t)all.size();
  if (!all.empty()) {
    cudaError_t e = cudaGetDevice(&pl->device);
    if (e == cudaSuccess) e = cudaMalloc((void**)&pl->tiles_dev, all.size() * sizeof(RtaRaggedTile));
    if (e == cudaSuccess)
      e = cudaMemcpy(pl->tiles_dev, all.data(), all.size() * sizeof(RtaRaggedTile),
                     cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
      if (pl->tiles_dev) cudaFree(pl->tiles_dev);
      delete pl;
      return fail_cuda(e);
    }
  }
  *plan = pl;
  return RTA_OK;
}

// Side streams for rta_extract_ragged: the launches of one call (one per camera
// shape) are independent, so all but the first run on library-owned streams
// forked from and joined back into the caller's stream. Every launch is a
// persistent grid sized for the whole GPU: the CTAs of the next shape become
// resident as those of the previous one drain, which hides the launch tails.
namespace {
constexpr int kSideStreams = 2;
constexpr int kMaxDev = 32;
struct SideStreams {
  std::mutex mu;
  bool ready[kMaxDev] = {};
  bool failed[kMaxDev] = {};
  cudaStream_t s[kMaxDev][kSideStreams] = {};
  cudaEvent_t fork[kMaxDev] = {};
  cudaEvent_t join[kMaxDev][kSideStreams] = {};
};
SideStreams g_side;

// caller holds g_side.mu
bool side_streams_ready(int dev) {
  if (dev < 0 || dev >= kMaxDev || g_side.failed[dev]) return false;
  if (g_side.ready[dev]) return true;
  bool ok = cudaEventCreateWithFlags(&g_side.fork[dev], cudaEventDisableTiming) == cudaSuccess;
  for (int i = 0; i < kSideStreams && ok; ++i)
    ok = cudaStreamCreateWithFlags(&g_side.s[dev][i], cudaStreamNonBlocking) == cudaSuccess &&
         cudaEventCreateWithFlags(&g_side.join[dev][i], cudaEventDisableTiming) == cudaSuccess;
  if (!ok) {
    cudaGetLastError();
    g_side.failed[dev] = true;  // stay on the caller's stream (what is half-built is leaked once)
    return false;
  }
  g_side.ready[dev] = true;
  return true;
}

// rta_shutdown: the caller has synchronised the devices in use
void side_streams_release() {
  std::lock_guard<std::mutex> lock(g_side.mu);
  int cur = 0;
  const bool have_cur = cudaGetDevice(&cur) == cudaSuccess;
  for (int d = 0; d < kMaxDev; ++d) {
    if (g_side.ready[d] && cudaSetDevice(d) == cudaSuccess) {
      for (int i = 0; i < kSideStreams; ++i) {
        cudaStreamSynchronize(g_side.s[d][i]);
        cudaStreamDestroy(g_side.s[d][i]);
        cudaEventDestroy(g_side.join[d][i]);
      }
      cudaEventDestroy(g_side.fork[d]);
    }
    g_side.ready[d] = false;
    g_side.failed[d] = false;
  }
  if (have_cur) cudaSetDevice(cur);
  cudaGetLastError();
}
}  // namespace

int rta_extract_ragged(const rta_ragged_plan* plan, const uint16_t* wf, const int32_t* pedestal,
                       const float* gain, int32_t* out_sum, int32_t* out_start,
                       float* out_charge, float* out_time, void* stream) {
  if (!plan) return RTA_ERR_NULL;
  if (plan->n_tiles == 0) return RTA_OK;
  if (!wf || !pedestal || !gain || !out_sum || !out_start || !out_charge || !out_time)
    return RTA_ERR_NULL;
  if ((uintptr_t)wf % 2 != 0) return RTA_ERR_ALIGN;
  if (((uintptr_t)out_sum | (uintptr_t)out_start | (uintptr_t)out_charge | (uintptr_t)out_time |
       (uintptr_t)pedestal | (uintptr_t)gain) % 4 != 0)
    return RTA_ERR_ALIGN;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return fail_cuda(e);
  if (dev != plan->device) return fail_cuda(cudaErrorInvalidDevice);
  const cudaStream_t user = (cudaStream_t)stream;
  const size_t n_classes = plan->classes.size();
  std::unique_lock<std::mutex> lock(g_side.mu, std::defer_lock);
  bool forked = false;
  if (n_classes > 1 && !g_serial_ragged.load()) {
    lock.lock();
    forked = side_streams_ready(dev) &&
             cudaEventRecord(g_side.fork[dev], user) == cudaSuccess;
    if (!forked) {
      cudaGetLastError();
      lock.unlock();
    }
  }
  int used = 0;  // side streams that got work
  cudaError_t first_err = cudaSuccess;
  for (size_t i = 0; i < n_classes; ++i) {
    const rta_ragged_plan::Class& c = plan->classes[i];
    cudaStream_t st = user;
    if (forked && i > 0) {
      const int k = (int)((i - 1) % kSideStreams);
      st = g_side.s[dev][k];
      if (k >= used) {  // first work on this side stream: order it after the caller's stream
        e = cudaStreamWaitEvent(st, g_side.fork[dev], 0);
        if (e != cudaSuccess && first_err == cudaSuccess) first_err = e;
        used = k + 1;
      }
    }
    e = rta_launch_ragged(wf, plan->tiles_dev + c.first, c.count, c.S, c.W, c.tile_traces, pedestal, gain,
                          out_sum, out_start, out_charge, out_time, st);
    if (e != cudaSuccess && first_err == cudaSuccess) first_err = e;
  }
  // join, also after an error: the caller's stream must not run ahead of what was enqueued
  for (int k = 0; k < used; ++k) {
    e = cudaEventRecord(g_side.join[dev][k], g_side.s[dev][k]);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(user, g_side.join[dev][k], 0);
    if (e != cudaSuccess && first_err == cudaSuccess) first_err = e;
  }
  if (first_err != cudaSuccess) return fail_cuda(first_err);
  return RTA_OK;
}

int64_t rta_ragged_plan_info(const rta_ragged_plan* plan, int32_t what) {
  if (!plan) return -1;
  switch (what) {
    case RTA_RAGGED_N_LAUNCHES: return (int64_t)plan->classes.size();
    case RTA_RAGGED_N_TILES: return plan->n_tiles;
    case RTA_RAGGED_N_TRACES: return plan->n_traces;
    case RTA_RAGGED_WF_BYTES: return plan->wf_bytes;
    case RTA_RAGGED_WF_END_BYTES: return plan->wf_end;
    case RTA_RAGGED_OUT_END: return plan->out_end;
    default: return -1;
  }
}

void rta_ragged_plan_destroy(rta_ragged_plan* plan) {
  if (!plan) return;
  if (plan->tiles_dev) {
    int cur = 0;
    if (cudaGetDevice(&cur) == cudaSuccess) {
      cudaSetDevice(plan->device);
      cudaDeviceSynchronize();  // kernels of earlier calls may still read the table
      cudaFree(plan->tiles_dev);
      cudaSetDevice(cur);
    }
    cudaGetLastError();
  }
  delete plan;
}

// ---- image cleaning + moments (NEXT-4) ----------------------------------------
int rta_image_moments(const float* charge, const float* time, int64_t n_events,
                      int32_t n_pixels, const float* pix_x, const float* pix_y,
                      const int32_t* neighbors, float thr_picture, float thr_boundary,
                      int32_t* out_n_pix, float* out_params, uint8_t* out_mask, void* stream) {
  const int v = validate_image(n_events, n_pixels, pix_x, pix_y, neighbors, out_n_pix, out_params,
                               out_mask);
  if (v != RTA_OK || n_events == 0) return v;
  if (!charge || !time) return RTA_ERR_NULL;
  if (((uintptr_t)charge | (uintptr_t)time) % 4 != 0) return RTA_ERR_ALIGN;
  const RtaCamera cam{pix_x, pix_y, neighbors, thr_picture, thr_boundary};
  const RtaImageOut out{out_n_pix, out_params, out_mask};
  const cudaError_t e = rta_launch_image_moments(charge, time, n_events, n_pixels, cam, out,
                                                 (cudaStream_t)stream);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

static int extract_image_common(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                                int32_t n_samples, const int32_t* pedestal, const float* gain,
                                int32_t W, const float* pix_x, const float* pix_y,
                                const int32_t* neighbors, float thr_picture, float thr_boundary,
                                int32_t* out_n_pix, float* out_params, uint8_t* out_mask,
                                void* stream, bool force_generic) {
  int v = validate_fused(wf, n_events, n_pixels, n_samples, pedestal, gain, W);
  if (v != RTA_OK) return v;
  v = validate_image(n_events, n_pixels, pix_x, pix_y, neighbors, out_n_pix, out_params, out_mask);
  if (v != RTA_OK || n_events == 0) return v;
  const RtaCamera cam{pix_x, pix_y, neighbors, thr_picture, thr_boundary};
  const RtaImageOut out{out_n_pix, out_params, out_mask};
  const cudaError_t e = rta_launch_extract_image(wf, n_events, n_pixels, n_samples, pedestal, gain,
                                                 W, cam, out, (cudaStream_t)stream, force_generic);
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

int rta_extract_image(const uint16_t* wf, int64_t n_events, int32_t n_pixels, int32_t n_samples,
                      const int32_t* pedestal, const float* gain, int32_t W, const float* pix_x,
                      const float* pix_y, const int32_t* neighbors, float thr_picture,
                      float thr_boundary, int32_t* out_n_pix, float* out_params,
                      uint8_t* out_mask, void* stream) {
  return extract_image_common(wf, n_events, n_pixels, n_samples, pedestal, gain, W, pix_x, pix_y,
                              neighbors, thr_picture, thr_boundary, out_n_pix, out_params,
                              out_mask, stream, false);
}

// The same for callers that cannot allocate device memory (include/rta.h): fixed
// scratch inside the library image, see rta_noalloc.cu. Validation happens here,
// before the first CUDA call.
int rta_extract_image_noalloc(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                              int32_t n_samples, const int32_t* pedestal, const float* gain,
                              int32_t W, const float* pix_x, const float* pix_y,
                              const int32_t* neighbors, float thr_picture, float thr_boundary,
                              int32_t* out_n_pix, float* out_params, uint8_t* out_mask,
                              void* stream) {
  int v = validate_fused(wf, n_events, n_pixels, n_samples, pedestal, gain, W);
  if (v != RTA_OK) return v;
  v = validate_image(n_events, n_pixels, pix_x, pix_y, neighbors, out_n_pix, out_params, out_mask);
  if (v != RTA_OK || n_events == 0) return v;
  if (n_events * (int64_t)n_pixels > (int64_t)RTA_NOALLOC_MAX_TRACES) return RTA_ERR_TOO_LARGE;
  if ((uintptr_t)wf % 16 != 0) return RTA_ERR_ALIGN;
  if (!rta_dyn_eligible(n_samples, W)) return RTA_ERR_UNSUPPORTED;
  const RtaCamera cam{pix_x, pix_y, neighbors, thr_picture, thr_boundary};
  const RtaImageOut out{out_n_pix, out_params, out_mask};
  const cudaError_t e = rta_launch_extract_image_noalloc(wf, n_events, n_pixels, n_samples, pedestal,
                                                         gain, W, cam, out, (cudaStream_t)stream);
  if (e == cudaErrorNotSupported) return RTA_ERR_UNSUPPORTED;
  return e == cudaSuccess ? RTA_OK : fail_cuda(e);
}

#ifdef RTA_TESTING
// Same through the generic fused kernel (librta_testing.so only).
int rta_extract_image_generic(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                              int32_t n_samples, const int32_t* pedestal, const float* gain,
                              int32_t W, const float* pix_x, const float* pix_y,
                              const int32_t* neighbors, float thr_picture, float thr_boundary,
                              int32_t* out_n_pix, float* out_params, uint8_t* out_mask,
                              void* stream) {
  return extract_image_common(wf, n_events, n_pixels, n_samples, pedestal, gain, W, pix_x, pix_y,
                              neighbors, thr_picture, thr_boundary, out_n_pix, out_params,
                              out_mask, stream, true);
}
#endif  // RTA_TESTING

int rta_extract_image_stream(const uint16_t* wf_host, int64_t n_events, int32_t n_pixels,
                             int32_t n_samples, const int32_t* pedestal, const float* gain,
                             int32_t W, const float* pix_x, const float* pix_y,
                             const int32_t* neighbors, float thr_picture, float thr_boundary,
                             int32_t* out_n_pix, float* out_params, uint8_t* out_mask,
                             size_t chunk_bytes, void* stream) {
  int v = validate_fused(wf_host, n_events, n_pixels, n_samples, pedestal, gain, W);
  if (v != RTA_OK) return v;
  v = validate_image(n_events, n_pixels, pix_x, pix_y, neighbors, out_n_pix, out_params, out_mask);
  if (v != RTA_OK || n_events == 0) return v;
  cudaError_t e = cudaSuccess;
  Workspace* wsp = ws_current(&e);
  if (wsp == nullptr) return fail_cuda(e);
  Workspace& ws = *wsp;
  std::lock_guard<std::mutex> lock(ws.mu);
  e = ws_prepare(ws);
  if (e != cudaSuccess) return fail_cuda(e);
  const RtaCamera cam{pix_x, pix_y, neighbors, thr_picture, thr_boundary};
  const RtaImageOut out{out_n_pix, out_params, out_mask};
  return image_stream_impl(ws, wf_host, n_events, n_pixels, n_samples, pedestal, gain, W, cam,
                           out, chunk_bytes, (cudaStream_t)stream, nullptr);
}

int rta_extract_image_host(const uint16_t* wf_host, int64_t n_events, int32_t n_pixels,
                           int32_t n_samples, const int32_t* pedestal_host,
                           const float* gain_host, int32_t W, const float* pix_x_host,
                           const float* pix_y_host, const int32_t* neighbors_host,
                           float thr_picture, float thr_boundary, int32_t* out_n_pix_host,
                           float* out_params_host, uint8_t* out_mask_host, size_t chunk_bytes) {
  int v = validate_fused(wf_host, n_events, n_pixels, n_samples, pedestal_host, gain_host, W);
  if (v != RTA_OK) return v;
  v = validate_image(n_events, n_pixels, pix_x_host, pix_y_host, neighbors_host, out_n_pix_host,
                     out_params_host, out_mask_host);
  if (v != RTA_OK || n_events == 0) return v;
  cudaError_t e0 = cudaSuccess;
  Workspace* wsp = ws_current(&e0);
  if (wsp == nullptr) return fail_cuda(e0);
  Workspace& w = *wsp;
  std::lock_guard<std::mutex> lock(w.mu);
  cudaError_t e = ws_prepare(w);
  if (e != cudaSuccess) return fail_cuda(e);
  // pedestal, gain, pix_x, pix_y: 4 bytes per pixel each; neighbours: 24
  const size_t P = (size_t)n_pixels, calib_bytes = P * 40u;
  if (w.calib_cap < calib_bytes) {
    if ((e = cudaDeviceSynchronize()) != cudaSuccess) return fail_cuda(e);
    if (w.calib_buf) cudaFree(w.calib_buf);
    w.calib_buf = nullptr;
    w.calib_cap = 0;
    if ((e = cudaMalloc(&w.calib_buf, calib_bytes)) != cudaSuccess) return fail_cuda(e);
    w.calib_cap = calib_bytes;
  }
  uint8_t* cb = reinterpret_cast<uint8_t*>(w.calib_buf);
  const void* src[5] = {pedestal_host, gain_host, pix_x_host, pix_y_host, neighbors_host};
  const size_t off[5] = {0, P * 4u, P * 8u, P * 12u, P * 16u};
  const size_t len[5] = {P * 4u, P * 4u, P * 4u, P * 4u, P * 24u};
  // the tables may still be read by kernels of an earlier call
  if ((e = cudaStreamSynchronize(w.host_stream)) != cudaSuccess) return fail_cuda(e);
  for (int i = 0; i < 5; ++i) {
    if ((e = cudaMemcpyAsync(cb + off[i], src[i], len[i], cudaMemcpyHostToDevice,
                             w.host_stream)) != cudaSuccess)
      return fail_cuda(e);
  }
  const RtaCamera cam{reinterpret_cast<const float*>(cb + off[2]),
                      reinterpret_cast<const float*>(cb + off[3]),
                      reinterpret_cast<const int32_t*>(cb + off[4]), thr_picture, thr_boundary};
  const RtaImageOut none{nullptr, nullptr, nullptr};
  const ImageHostOut ho{out_n_pix_host, out_params_host, out_mask_host};
  const int rc = image_stream_impl(w, wf_host, n_events, n_pixels, n_samples,
                                   reinterpret_cast<const int32_t*>(cb + off[0]),
                                   reinterpret_cast<const float*>(cb + off[1]), W, cam, none,
                                   chunk_bytes, w.host_stream, &ho);
  // synchronous by contract, also on the error path (nothing may outlive the call)
  cudaError_t e1 = cudaStreamSynchronize(w.host_stream);
  cudaError_t e2 = cudaStreamSynchronize(w.back_stream);
  cudaError_t e3 = cudaStreamSynchronize(w.copy_stream);
  if (rc != RTA_OK) return rc;
  if (e1 != cudaSuccess) return fail_cuda(e1);
  if (e2 != cudaSuccess) return fail_cuda(e2);
  if (e3 != cudaSuccess) return fail_cuda(e3);
  return RTA_OK;
}

int32_t rta_image_max_pixels(void) { return rta_image_pixel_limit(); }

const char* rta_image_kernel_name(int32_t n_pixels, int32_t n_samples, int32_t W, int aligned16) {
  return rta_pick_image_kernel_name(n_pixels, n_samples, W, aligned16 != 0);
}

const char* rta_strerror(int status) {
  switch (status) {
    case RTA_OK: return "ok";
    case RTA_ERR_NULL: return "null pointer with work to do";
    case RTA_ERR_SHAPE: return "bad shape: need n_events >= 0, n_pixels >= 1, 1 <= W <= n_samples";
    case RTA_ERR_UNSUPPORTED:
      return "unsupported size: n_events*n_pixels >= 2^31 or n_samples*W*65535 >= 2^31";
    case RTA_ERR_ALIGN: return "misaligned pointer (wf: 2 bytes; calibration and outputs: 4 bytes)";
    case RTA_ERR_CUDA: return "CUDA runtime error (see rta_last_cuda_error)";
    case RTA_ERR_NOMEM: return "out of device or pinned host memory";
    case RTA_ERR_TOO_LARGE:
      return "too many traces for the fixed scratch of rta_extract_image_noalloc "
             "(n_events*n_pixels > RTA_NOALLOC_MAX_TRACES): split the batch";
    default: return "unknown status";
  }
}

int rta_last_cuda_error(void) { return t_last_cuda; }

const char* rta_kernel_name(int32_t n_samples, int32_t W, int aligned16) {
  return rta_pick_kernel_name(n_samples, W, aligned16 != 0);
}

int rta_prepare(int32_t n_samples, int32_t W, int32_t extractor, int32_t sample_bits) {
  static_assert((int)RTA_EXTRACTOR_SLIDING == (int)RTA_MODE_SLIDING &&
                    (int)RTA_EXTRACTOR_FIXED == (int)RTA_MODE_FIXED &&
                    (int)RTA_EXTRACTOR_LOCAL_PEAK == (int)RTA_MODE_LOCAL_PEAK &&
                    (int)RTA_EXTRACTOR_FIR == (int)RTA_MODE_FIR,
                "the public extractor numbers are the internal modes");
  if (n_samples < 1 || W < 1 || W > n_samples) return RTA_ERR_SHAPE;
  if (extractor < RTA_EXTRACTOR_SLIDING || extractor > RTA_EXTRACTOR_FIR) return RTA_ERR_SHAPE;
  if (sample_bits != 16 && sample_bits != 12) return RTA_ERR_SHAPE;
  if ((int64_t)n_samples * (int64_t)W * 65535ll >= (1ll << 31)) return RTA_ERR_UNSUPPORTED;
  if (sample_bits == 12 && extractor != RTA_EXTRACTOR_SLIDING) return RTA_ERR_UNSUPPORTED;
  if (extractor == RTA_EXTRACTOR_FIR && W > RTA_MAX_TAPS) return RTA_ERR_UNSUPPORTED;
  // the four BASELINE shapes were compiled with the library
  if (std::strncmp(rta_pick_kernel_name(n_samples, W, true, sample_bits), "tile", 4) == 0) return RTA_OK;
  const cudaError_t e = rta_jit_prepare(n_samples, W, extractor, sample_bits);
  if (e == cudaSuccess) return RTA_OK;
  if (e == cudaErrorNotSupported) return RTA_ERR_UNSUPPORTED;
  return fail_cuda(e);
}

const char* rta_kernel_name_packed12(int32_t n_samples, int32_t W, int aligned16) {
  return rta_pick_kernel_name(n_samples, W, aligned16 != 0, 12);
}

int64_t rta_chunk_events(int64_t n_events, int32_t n_pixels, int32_t n_samples,
                         size_t chunk_bytes, int32_t sample_bits) {
  if (n_events < 0 || n_pixels < 1 || n_samples < 1 || (sample_bits != 16 && sample_bits != 12))
    return -1;
  if ((int64_t)n_pixels * (int64_t)n_samples >= (1ll << 46)) return -1;  // event_bits must fit
  return plan_chunks(n_events, n_pixels, n_samples, chunk_bytes, sample_bits).chunk_events;
}

uint64_t rta_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

void rta_shutdown(void) {
  int cur = 0;
  const bool have_cur = cudaGetDevice(&cur) == cudaSuccess;
  for (int d = 0; d < kMaxWsDevices; ++d) {
    Workspace& w = g_ws_tab[d];
    std::lock_guard<std::mutex> lock(w.mu);
    if (w.device < 0) continue;
    if (cudaSetDevice(w.device) == cudaSuccess) {
      cudaDeviceSynchronize();
      ws_release(w);
    }
  }
  if (have_cur) cudaSetDevice(cur);
  cudaGetLastError();
  side_streams_release();
  rta_image_release();
  rta_jit_release();
  rta_sched_release();
}

#ifdef RTA_TESTING
// Test hooks: process-global switches that exist in librta_testing.so only, so
// that no program linked against the shipped library can flip the dispatch of
// another thread's calls.
// 1 = rta_extract_ragged issues every launch on the caller's stream, one after the other.
void rta_debug_serial_ragged(int on) { g_serial_ragged.store(on != 0); }

// 1 = rta_extract_fixed / _local_peak / _fir /
// _packed12 take the generic kernel whatever the shape (two device paths must agree).
void rta_debug_force_generic(int on) { g_force_generic.store(on != 0); }

// 1 = static round-robin tile schedule,
// 0 = dynamic (default). Results are identical; only the tile->CTA map changes.
void rta_debug_static_schedule(int on) { rta_set_static_schedule(on != 0); }

// 1 = the image cleaning runs the two
// steps of its definition even when the neighbour table is symmetric.
void rta_debug_general_cleaning(int on) { rta_set_general_cleaning(on != 0); }

// 0 = no run-time specialisations: unspecialised shapes take the runtime-shape kernel
// (staged<any>), as they do when libnvrtc is not available. 1 = back on.
void rta_debug_jit(int on) { rta_jit_enable(on != 0); }

// 4 / 8 / 16 / 32 = rta_extract runs the several-lanes-per-trace kernel with that many lanes
// per trace wherever it can (measurements of DESIGN.md section 5g); 0 = normal dispatch.
void rta_debug_lanes_per_trace(int lpt) { rta_set_lanes_per_trace(lpt); }

// Segment kernel: window starts per segment (2 * odd), traces per tile, threads per CTA, stages; 0 =
// chosen per shape. A non-zero L sends every sliding call on an aligned base to that kernel.
void rta_debug_seg_tuning(int L, int TR, int NT, int stages) { rta_set_seg_tuning(L, TR, NT, stages); }
#endif  // RTA_TESTING

}  // extern "C"
