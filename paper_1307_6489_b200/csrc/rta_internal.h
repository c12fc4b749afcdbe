// rta_internal.h — declarations shared by the translation units of librta.so.
// Not part of the public ABI (that is include/rta.h) and never seen by oracle/.
#ifndef RTA_INTERNAL_H
#define RTA_INTERNAL_H

// The extractor family (readings R22-R24): how the window is chosen.
#define RTA_MAX_TAPS 32

#ifdef __CUDACC_RTC__
// Run-time compilation of a specialised tile kernel (rta_jit.cu): device code
// only, no host headers. NVRTC predefines size_t and the CUDA built-ins.
typedef unsigned char uint8_t;
typedef unsigned short uint16_t;
typedef unsigned int uint32_t;
typedef int int32_t;
typedef unsigned long long uint64_t;
typedef long long int64_t;
typedef unsigned long long uintptr_t;
#else
#include <cuda_runtime.h>
#include <stdint.h>
#endif
// Mixed-camera batches: one entry per tile (at most rta_ragged_tile_traces(S, W) traces of one block).
struct alignas(16) RtaRaggedTile {
  unsigned long long src;  // byte offset of the tile's first trace in wf | n_traces << 48
  uint32_t out_base;       // flat output index of the first trace
  uint32_t cal0;           // calibration index of the first trace
};
enum { RTA_MODE_SLIDING = 0, RTA_MODE_FIXED = 1, RTA_MODE_LOCAL_PEAK = 2, RTA_MODE_FIR = 3 };
struct RtaMode {
  int kind;
  const int32_t* window_start;  // RTA_MODE_FIXED: DEVICE [n_pixels]
  int32_t shift;                // RTA_MODE_LOCAL_PEAK
  int32_t n_taps;               // RTA_MODE_FIR (== W passed to rta_launch_extract)
  int32_t taps[RTA_MAX_TAPS];   // RTA_MODE_FIR
};

#ifndef __CUDACC_RTC__
// Enqueue the extraction of `n_traces` traces starting at global trace index 0
// of `wf` on `stream`. Arguments are already validated. Returns a cudaError_t.
// `force_generic` routes every shape to the generic kernel (tests use it to
// compare the two paths). `mode` == nullptr is the sliding-window extractor.
// `sample_bits` is 16 (uint16 samples) or 12 (P12 stream, sliding extractor only).
cudaError_t rta_launch_extract(const void* wf, int64_t n_traces, int32_t n_pixels,
                               int32_t n_samples, const int32_t* pedestal,
                               const float* gain, int32_t W, int32_t* out_sum,
                               int32_t* out_start, float* out_charge, float* out_time,
                               cudaStream_t stream, bool force_generic,
                               const RtaMode* mode = nullptr, int sample_bits = 16);

// Whether an unspecialised (S, W) takes the staged kernel with runtime shape
// (extract_dyn_kernel) when the input is 16-byte aligned.
bool rta_dyn_eligible(int32_t n_samples, int32_t W);

// The sliding extractor through the runtime-shape staged kernel, with the tile
// scheduler's two words supplied by the caller (zero when the kernel starts) instead
// of the library's cudaMalloc'ed per-stream pool. cudaErrorNotSupported unless
// rta_dyn_eligible(n_samples, W) and wf is 16-byte aligned.
cudaError_t rta_launch_extract_dyn_sched(const void* wf, int64_t n_traces, int32_t n_pixels,
                                         int32_t n_samples, const int32_t* pedestal,
                                         const float* gain, int32_t W, int32_t* out_sum,
                                         int32_t* out_start, float* out_charge, float* out_time,
                                         cudaStream_t stream, uint32_t* sched);
// Name of the kernel the dispatcher picks (static string).
const char* rta_pick_kernel_name(int32_t n_samples, int32_t W, bool aligned16, int bits = 16);

// Mixed-camera batches (include/rta.h rta_ragged_plan_*): how many traces of one block a
// tile of shape (S, W) holds at most, decided when the plan is made: the tile of the
// ahead-of-time kernel, else of the run-time specialisation (when the compiler is there),
// else of the runtime-shape kernel.
int rta_ragged_tile_traces(int32_t n_samples, int32_t W);
// One launch over a device-resident tile table whose tiles all have shape (S, W).
// `tile_traces` is what rta_ragged_tile_traces gave when the table was cut.
cudaError_t rta_launch_ragged(const void* wf, const RtaRaggedTile* tiles_dev, uint32_t n_tiles,
                              int32_t n_samples, int32_t W, int32_t tile_traces, const int32_t* pedestal,
                              const float* gain, int32_t* out_sum, int32_t* out_start,
                              float* out_charge, float* out_time, cudaStream_t stream);

void rta_count_launch();

// Tile scheduling of the staged kernels: dynamic (default) or the static
// round-robin (tests compare the two). rta_sched_release frees the per-stream
// scheduler words (rta_shutdown).
// (the three setters below exist in librta_testing.so only: rta_kernels.cu -DRTA_TESTING)
void rta_set_static_schedule(bool on);
// Measurements / tests: 4, 8, 16 or 32 = the sliding extractor runs the several-lanes-per-trace
// kernel with that many lanes wherever it can (n_samples a multiple of 8, aligned base); 0 = normal.
void rta_set_lanes_per_trace(int lpt);
// Measurements / tests: segment length (2 * odd), traces per tile and threads per CTA of the
// segment kernel; 0 = chosen per shape. A non-zero L sends every sliding call on an aligned
// base to that kernel.
void rta_set_seg_tuning(int L, int TR, int NT, int stages);
bool rta_seg_eligible(int32_t n_samples, int32_t W);
void rta_sched_release();
cudaError_t rta_device_sms(int dev, int* sms);
// Allow `func` up to 227 KB of dynamic shared memory on `dev` (set once per kernel and device).
cudaError_t rta_func_allow_max_smem(const void* func, int dev);

// Image cleaning + moments (include/rta.h rta_image_moments, rta_extract_image;
// DESIGN.md readings R31-R35). Device pointers, already validated.
struct RtaCamera {
  const float* pix_x;        // [n_pixels]
  const float* pix_y;        // [n_pixels]
  const int32_t* neighbors;  // [n_pixels][6], -1 (or any index outside [0, n_pixels)) = none
  float thr_picture, thr_boundary;
};
struct RtaImageOut {
  int32_t* n_pix;   // [n_events]
  float* params;    // [n_events][8]
  uint8_t* mask;    // [n_events][n_pixels] or nullptr
};
cudaError_t rta_launch_image_moments(const float* charge, const float* time, int64_t n_events,
                                     int32_t n_pixels, const RtaCamera& cam,
                                     const RtaImageOut& out, cudaStream_t stream);
// Extraction fused with cleaning + moments: per-trace results stay in shared memory.
cudaError_t rta_launch_extract_image(const void* wf, int64_t n_events, int32_t n_pixels,
                                     int32_t n_samples, const int32_t* pedestal,
                                     const float* gain, int32_t W, const RtaCamera& cam,
                                     const RtaImageOut& out, cudaStream_t stream,
                                     bool force_generic);
// rta_noalloc.cu: rta_extract_image_noalloc behind its validation (include/rta.h).
// cudaErrorNotSupported: shape or alignment outside what that call takes.
cudaError_t rta_launch_extract_image_noalloc(const void* wf, int64_t n_events, int32_t n_pixels,
                                             int32_t n_samples, const int32_t* pedestal,
                                             const float* gain, int32_t W,
                                             const RtaCamera& cam,
                                             const RtaImageOut& out, cudaStream_t stream);
// Tests: never take the symmetric-neighbour-table shortcut of the cleaning (both
// ways give the same mask on a symmetric table).
void rta_set_general_cleaning(bool on);
void rta_image_release();  // frees the scratch memory pools (rta_shutdown)
int32_t rta_image_pixel_limit();  // charge, time and flags of one event must fit one CTA
const char* rta_pick_image_kernel_name(int32_t n_pixels, int32_t n_samples, int32_t W,
                                       bool aligned16);

// Run-time specialisation (rta_jit.cu): the staged tile kernel compiled by NVRTC
// for one (n_samples, W, extractor) the first time that shape is seen, cached
// per process. rta_jit_launch returns cudaErrorNotSupported when the shape is
// not eligible or the compiler is not available (the caller then takes the
// runtime-shape kernel); any other error is a launch error.
struct RtaJitArgs {
  const void* wf;
  uint32_t n_traces, n_pixels, pix_inv;
  const int32_t* pedestal;
  const float* gain;
  int32_t *out_sum, *out_start;
  float *out_charge, *out_time;
  uint32_t* sched;
};
bool rta_jit_eligible(int32_t n_samples, int32_t W, int bits = 16);   // shape fits a register copy, JIT enabled
bool rta_jit_available();                              // ... and libnvrtc could be loaded
cudaError_t rta_jit_launch(int32_t n_samples, int32_t W, int mode, const RtaJitArgs& a,
                           const void* mode_args, size_t mode_args_bytes, cudaStream_t stream,
                           int bits = 16);
// Compile / load / set up the specialisation of a shape on the current device now
// (rta_prepare); cudaErrorNotSupported when the shape has none.
cudaError_t rta_jit_prepare(int32_t n_samples, int32_t W, int mode, int bits);
// The same for a tile table of a mixed-camera batch (sliding extractor). rta_jit_tile_traces:
// traces per tile of the specialisation of (S, W), 0 when there is none (not eligible, no compiler).
struct RtaJitRaggedArgs {
  const void* wf;
  const RtaRaggedTile* tiles;
  uint32_t n_tiles;
  const int32_t* pedestal;
  const float* gain;
  int32_t *out_sum, *out_start;
  float *out_charge, *out_time;
  uint32_t* sched;
};
int rta_jit_tile_traces(int32_t n_samples, int32_t W);
cudaError_t rta_jit_launch_ragged(int32_t n_samples, int32_t W, const RtaJitRaggedArgs& a,
                                  cudaStream_t stream);
void rta_jit_enable(bool on);   // tests: switch the run-time specialisations off / on
void rta_jit_release();         // rta_shutdown
#endif  // __CUDACC_RTC__

#endif
