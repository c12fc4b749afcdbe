/* rta.h — C ABI of the B200 sliding-window signal-extraction library (librta.so).
 *
 * The operation (BASELINE.json:north_star sentence 2; the paper names the step
 * only as "signal extraction algorithms [13] ... ported to CUDA"
 * §5, at the front of RT-RECO's calibration, §4): for every
 * trace wf[e][p][0..S-1] of digitised camera samples,
 *
 *     x[s]      = wf[e][p][s] - pedestal[p]
 *     Sum(t)    = x[t] + ... + x[t+W-1],   t = 0 .. S-W      (windows inside the trace)
 *     t*        = smallest t with Sum(t) = max_t Sum(t)       (earliest on ties)
 *     out_sum   = Sum(t*)                      int32, exact
 *     out_start = t*                           int32, exact, 0-based
 *     out_charge= RN32(Sum(t*) * gain[p])      float32
 *     out_time  = RN32(sum_{s=t*}^{t*+W-1} s*x[s] / Sum(t*))  float32, absolute 0-based
 *                 sample index; t* + (W-1)/2 when Sum(t*) <= 0
 *
 * (DESIGN.md "Readings" R1-R18 lists every point the sources leave open.)
 *
 * Conventions for every entry point
 *  - All functions return an int status (RTA_OK or RTA_ERR_*); they never
 *    throw, print or exit. Arguments are validated before anything is enqueued.
 *  - The caller owns every pointer it passes; the library never frees or
 *    retains them. The library owns only rta_extract_stream's workspace (two
 *    device chunk buffers, two pinned staging buffers when the source is
 *    pageable, one copy stream, events), one per device, created lazily by the
 *    first host-fed call on that device, reused, and released by
 *    rta_shutdown(). Host-fed calls on one device serialise on that device's
 *    workspace; calls on different devices do not wait for one another.
 *  - There is no CPU fallback: without a CUDA device every compute call
 *    returns RTA_ERR_CUDA.
 *  - The library links the CUDA runtime only (no libtorch).
 */
#ifndef RTA_H
#define RTA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  RTA_OK = 0,
  RTA_ERR_NULL = 1,        /* a required pointer is NULL while there is work to do */
  RTA_ERR_SHAPE = 2,       /* n_events < 0, n_pixels < 1, n_samples < 1, W < 1 or W > n_samples */
  RTA_ERR_UNSUPPORTED = 3, /* n_events*n_pixels >= 2^31, or n_samples*W*65535 >= 2^31 (int32 guard) */
  RTA_ERR_ALIGN = 4,       /* wf is not 2-byte aligned / an output is not 4-byte aligned (P12: any byte) */
  RTA_ERR_CUDA = 5,        /* CUDA runtime failure; see rta_last_cuda_error() */
  RTA_ERR_NOMEM = 6,       /* workspace allocation failed (device or pinned host) */
  RTA_ERR_TOO_LARGE = 7    /* more work than the fixed scratch of rta_extract_image_noalloc holds */
};

/* Kernel-only path.
 *
 *   wf        DEVICE  uint16 [n_events][n_pixels][n_samples], dense, sample fastest.
 *                     Any uint16 value is accepted (12-bit data is a property of the
 *                     configs, not of the ABI). A 16-byte-aligned base pointer takes
 *                     the staged (TMA / cp.async) kernels — ahead-of-time
 *                     specialisations for the shapes (30,7), (40,7), (25,4), (128,8);
 *                     for any other trace (pair of traces when n_samples is odd) of at
 *                     most 320 bytes the same kernel compiled for the shape at first use
 *                     (NVRTC through dlopen("libnvrtc.so"): 0.3-0.6 s once per shape and
 *                     process; never inside a stream capture; RTA_JIT=0 turns it off);
 *                     without the compiler, and up to 1152 bytes, a kernel with runtime
 *                     (n_samples, W); longer traces a kernel that gives a thread a run of
 *                     window starts ("segments"), or a warp per trace ("lanes<32>":
 *                     n_samples a multiple of 8 with a window much wider than a
 *                     segment, or a trace too long for a segment stage) — these two
 *                     for rta_extract only; the other extractors, P12 input, mixed
 *                     batches and the image calls run the generic kernel on traces
 *                     above 1152 bytes. Any other 2-byte-aligned pointer takes the
 *                     runtime-shape kernel too, unless the trace (pair) is a multiple of
 *                     32 bytes; those take the generic kernel (strided global loads:
 *                     several times slower). Same
 *                     results either way (rta_kernel_name says which). With an
 *                     unaligned base the first bulk copy starts at the 16-byte
 *                     boundary below wf (inside the 16-byte line holding wf[0]);
 *                     nothing past the last sample is read.
 *   pedestal  DEVICE  int32  [n_pixels]; may exceed the samples (x can be negative).
 *   gain      DEVICE  float  [n_pixels]; NaN/Inf propagate into out_charge untouched.
 *   W         window width in samples, 1 <= W <= n_samples.
 *   out_*     DEVICE  flat [n_events*n_pixels], index e*n_pixels + p, 4-byte aligned.
 *   stream    cudaStream_t (NULL = the default stream).
 *
 * Asynchronous: validates, enqueues on `stream`, returns without synchronising.
 * Outputs are valid once `stream` has been synchronised. n_events == 0 is
 * RTA_OK with nothing enqueued and the outputs untouched. Thread-safe across
 * streams. Capturable into a CUDA graph: a captured launch hands its tiles out
 * in a fixed round-robin and touches no library state, so replays may run on
 * any stream, next to one another and next to eager calls. (Eager calls use
 * 128 KB of per-stream tile-scheduler words, allocated by the first eager call
 * on a device, owned by the library and released by rta_shutdown.) */
int rta_extract(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                int32_t n_samples, const int32_t* pedestal, const float* gain,
                int32_t W, int32_t* out_sum, int32_t* out_start,
                float* out_charge, float* out_time, void* stream);

/* ---- Other members of the extractor family ----------
 * The paper says "several signal extraction algorithms [13]" were being ported
 * (§5) and names none; ref [13] is unavailable, so
 * the three below are defined here (readings R22-R24). They share
 * every argument, layout, output and error rule of rta_extract and differ only
 * in how the window is chosen. With x[s] = wf[e][p][s] - pedestal[p]:
 *
 *   rta_extract_fixed       t* = clamp(window_start[p], 0, S-W)
 *                           window_start: DEVICE int32 [n_pixels], 4-byte aligned.
 *   rta_extract_local_peak  t* = clamp(peak - shift, 0, S-W), peak = smallest s
 *                           with x[s] maximal; shift may be negative.
 *   both:                   out_sum = sum_{k<W} x[t*+k], time numerator
 *                           sum_{k<W} (t*+k) x[t*+k]
 *   rta_extract_fir         y(t) = sum_{k<K} taps[k] x[t+k], t = 0..S-K;
 *                           t* = smallest t with y(t) maximal; out_sum = y(t*);
 *                           time numerator sum_{k<K} (t*+k) taps[k] x[t*+k]; W := K.
 *                           taps: HOST int32 [n_taps], copied before returning;
 *                           1 <= n_taps <= min(n_samples, 32) (more: RTA_ERR_UNSUPPORTED);
 *                           n_samples * sum|taps| * 65535 >= 2^31: RTA_ERR_UNSUPPORTED.
 *                           All-ones taps of length W give exactly rta_extract.
 *   always                  out_start = t*, out_charge = RN32(out_sum * gain[p]),
 *                           out_time = RN32(numerator / out_sum), or t* + (W-1)/2
 *                           when out_sum <= 0.
 *
 * Asynchronous on `stream`, like rta_extract. */
int rta_extract_fixed(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                      int32_t n_samples, const int32_t* pedestal, const float* gain,
                      int32_t W, const int32_t* window_start, int32_t* out_sum,
                      int32_t* out_start, float* out_charge, float* out_time,
                      void* stream);

int rta_extract_local_peak(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                           int32_t n_samples, const int32_t* pedestal,
                           const float* gain, int32_t W, int32_t shift,
                           int32_t* out_sum, int32_t* out_start, float* out_charge,
                           float* out_time, void* stream);

int rta_extract_fir(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                    int32_t n_samples, const int32_t* pedestal, const float* gain,
                    const int32_t* taps, int32_t n_taps, int32_t* out_sum,
                    int32_t* out_start, float* out_charge, float* out_time,
                    void* stream);

/* Host-fed path (step a8; BASELINE.json:configs[4]; page-locked transfer test
 * of PAPER.md:133/139 §5). Same operation, but `wf_host` is HOST memory
 * (pinned, or pageable — then it is staged through library-owned pinned
 * buffers). The waveforms are cut into chunks of whole events of at most
 * `chunk_bytes` (0 = 1 GiB; rounded down to whole events, at least one event),
 * and chunk k+1 is copied host->device on a library-owned copy stream while
 * chunk k is extracted on `stream` (two device buffers).
 *
 *   pedestal, gain, out_*   DEVICE, out_* sized for the whole run.
 *
 * Returns after the last kernel has been enqueued and every H2D copy has been
 * issued; all work is ordered on `stream`, so synchronising `stream` makes the
 * outputs valid and `wf_host` reusable. Calls are serialised by a library
 * mutex (single workspace). */
int rta_extract_stream(const uint16_t* wf_host, int64_t n_events,
                       int32_t n_pixels, int32_t n_samples,
                       const int32_t* pedestal, const float* gain, int32_t W,
                       int32_t* out_sum, int32_t* out_start, float* out_charge,
                       float* out_time, size_t chunk_bytes, void* stream);

/* Host-to-host convenience on top of rta_extract_stream, the end-to-end call a
 * user with nothing on the device makes: every pointer is HOST memory
 * (pedestal/gain/outputs pinned or pageable); outputs are copied back
 * device->host chunk by chunk on a third stream, overlapping the next chunk.
 * Synchronous: returns when the outputs are complete in host memory. */
int rta_extract_host(const uint16_t* wf_host, int64_t n_events, int32_t n_pixels,
                     int32_t n_samples, const int32_t* pedestal_host,
                     const float* gain_host, int32_t W, int32_t* out_sum_host,
                     int32_t* out_start_host, float* out_charge_host,
                     float* out_time_host, size_t chunk_bytes);

/* ---- Packed 12-bit ingest -----------------------------
 * The paper's Event-Builder simulator emits DL0 data as "a logical sequence of
 * bits ... according with the definition of the satellite telemetry [12]"
 * (§5); the format itself is not given and refs [11], [12] are
 * unavailable, so the packed format is defined here (readings R25-R27).
 *
 * "P12": the dense sample stream wf[e][p][s] (flat sample index
 * n = (e*n_pixels + p)*n_samples + s; no headers, no padding between traces or
 * events) stored 12 bits per sample, little-endian in bits: sample n occupies
 * bits [12 n, 12 n + 12) of the stream, bit b of the stream being bit (b % 8) of
 * byte (b / 8). For a = sample 2k, b = sample 2k+1:
 *     byte 3k = a & 0xFF;  byte 3k+1 = (a >> 8) | ((b & 0xF) << 4);  byte 3k+2 = b >> 4.
 * The stream holds ceil(12 N / 8) bytes for N samples; with N odd the high
 * nibble of the last byte is padding and is ignored. The library never reads a
 * byte past ceil(12 N / 8).
 *
 * The three calls below decode the stream inside the extraction kernel (no
 * unpacked copy ever exists in device memory) and then compute exactly what
 * rta_extract / rta_extract_stream / rta_extract_host compute on the decoded
 * samples; every other argument, output, error and ordering rule is theirs.
 *
 *   packed   uint8, ceil(12 * n_events*n_pixels*n_samples / 8) bytes, any byte
 *            alignment (DEVICE for rta_extract_packed12, HOST for the other two).
 *            A 16-byte-aligned device pointer takes the staged kernels.
 *   chunk_bytes (host-fed calls): bytes of the PACKED stream per chunk; chunks
 *            hold whole events and start on a 16-byte boundary of the stream, so
 *            the event count per chunk is rounded down to a multiple of
 *            m = 32 / gcd(n_pixels*n_samples, 32) (at least m events); 0 = 1 GiB. */
int rta_extract_packed12(const uint8_t* packed, int64_t n_events, int32_t n_pixels,
                         int32_t n_samples, const int32_t* pedestal, const float* gain,
                         int32_t W, int32_t* out_sum, int32_t* out_start,
                         float* out_charge, float* out_time, void* stream);

int rta_extract_stream_packed12(const uint8_t* packed_host, int64_t n_events,
                                int32_t n_pixels, int32_t n_samples,
                                const int32_t* pedestal, const float* gain, int32_t W,
                                int32_t* out_sum, int32_t* out_start, float* out_charge,
                                float* out_time, size_t chunk_bytes, void* stream);

int rta_extract_host_packed12(const uint8_t* packed_host, int64_t n_events,
                              int32_t n_pixels, int32_t n_samples,
                              const int32_t* pedestal_host, const float* gain_host,
                              int32_t W, int32_t* out_sum_host, int32_t* out_start_host,
                              float* out_charge_host, float* out_time_host,
                              size_t chunk_bytes);

/* ---- Mixed-camera (ragged) batches ---------------------
 * The array has three telescope sizes (§1), runs as "multiple
 * sub-array" configurations (§2.2), and the Central Event Builder
 * merges the telescopes triggered by one event (§4.1). The paper
 * gives no layout for a merged event; this one is defined here (DESIGN.md
 * readings R28-R30):
 *
 *   telescope k = 0..n_tel-1:  camera of tel_n_pixels[k] pixels, tel_n_samples[k]
 *       samples per trace, window tel_W[k]; calibration pedestal[c + p], gain[c + p]
 *       with c = tel_calib_offset[k], p = 0..tel_n_pixels[k]-1 (flat DEVICE arrays
 *       shared by all telescopes).
 *   block b = 0..n_blocks-1:  one event of telescope blk_tel[b]: a dense uint16
 *       [n_pixels][n_samples] array at SAMPLE index blk_wf_offset[b] of `wf`; its
 *       results go to flat output index blk_out_offset[b] + p. Any order; gaps
 *       allowed; output ranges of different blocks must not overlap.
 *
 * Every trace gets exactly rta_extract's result for its telescope's (S, W) and
 * calibration. The tables are HOST arrays, read only by rta_ragged_plan_create,
 * which validates them, cuts each block into tiles, uploads the tile tables to
 * the current device (synchronously) and returns an opaque plan. A plan depends
 * on the tables only — not on wf, calibration or outputs — and can be reused for
 * any number of rta_extract_ragged calls, from any stream, until destroyed.
 *
 * rta_extract_ragged is asynchronous on `stream`: one launch per distinct
 * (n_samples, W) among the blocks (rta_ragged_plan_info(RTA_RAGGED_N_LAUNCHES)).
 * The launches are independent; all but the first run on library-owned side
 * streams that are forked from `stream` and joined back into it before the call
 * returns, so the caller sees ordinary stream order: everything is complete when
 * `stream` reaches the end of the call's work.
 * Shapes (30,7), (40,7), (25,4), (128,8) take the specialised staged kernels,
 * other traces of at most 1152 bytes a staged kernel with runtime shape, longer
 * ones a generic kernel. Blocks starting on a 16-byte boundary of `wf` are fastest
 * (TMA bulk copies); 4-byte-aligned ones use 4-byte cp.async; others plain loads.
 *
 * Errors (plan_create, before any CUDA call): NULL table with entries, or
 * plan == NULL -> RTA_ERR_NULL; a telescope with n_pixels < 1, n_samples < 1,
 * W < 1, W > n_samples or a negative offset, or a block with a telescope index
 * out of range or a negative offset -> RTA_ERR_SHAPE; n_samples*W*65535 >= 2^31,
 * an output index >= 2^31, a calibration index >= 2^32 or a byte offset >= 2^48
 * -> RTA_ERR_UNSUPPORTED. n_blocks == 0 gives a valid empty plan (no device
 * needed) whose extraction is RTA_OK with nothing enqueued. */
typedef struct rta_ragged_plan rta_ragged_plan;

int rta_ragged_plan_create(int32_t n_tel, const int32_t* tel_n_pixels,
                           const int32_t* tel_n_samples, const int32_t* tel_W,
                           const int64_t* tel_calib_offset, int64_t n_blocks,
                           const int32_t* blk_tel, const int64_t* blk_wf_offset,
                           const int64_t* blk_out_offset, rta_ragged_plan** plan);

/* wf, pedestal, gain, out_*: DEVICE. The caller guarantees that the buffers
 * cover every offset in the plan (RTA_RAGGED_WF_END_BYTES, RTA_RAGGED_OUT_END). */
int rta_extract_ragged(const rta_ragged_plan* plan, const uint16_t* wf,
                       const int32_t* pedestal, const float* gain, int32_t* out_sum,
                       int32_t* out_start, float* out_charge, float* out_time,
                       void* stream);

enum {
  RTA_RAGGED_N_LAUNCHES = 0,   /* kernels per rta_extract_ragged call */
  RTA_RAGGED_N_TILES = 1,
  RTA_RAGGED_N_TRACES = 2,     /* sum of n_pixels over the blocks */
  RTA_RAGGED_WF_BYTES = 3,     /* waveform bytes the blocks hold (gaps excluded) */
  RTA_RAGGED_WF_END_BYTES = 4, /* one past the last waveform byte any block reads */
  RTA_RAGGED_OUT_END = 5       /* one past the last output index any block writes */
};
int64_t rta_ragged_plan_info(const rta_ragged_plan* plan, int32_t what);  /* -1: bad argument */

/* Synchronises the plan's device (kernels may still be reading the tables),
 * frees the tables and the plan. NULL is ignored. */
void rta_ragged_plan_destroy(rta_ragged_plan* plan);

/* ---- Image cleaning + image moments ---------------------
 * The first step downstream of the extraction, so that "event-level
 * reconstruction parameters (but not the raw data)" (§2.2) are what
 * leaves the GPU. The paper names the chain only ("calibration, the
 * gamma/hadron separation, and the energy and direction reconstruction",
 * PAPER.md:101 §4.1; RT-RECO is a reduced, fast version, §4.2) and
 * defines none of it; the operation is defined here (readings R31-R35).
 * Per event, with q[p] the pixel charges, t[p] the peak times, (x[p], y[p]) the
 * pixel centres and up to six neighbours per pixel:
 *
 *   core[p] = q[p] >= thr_picture                      (fp32 compare; NaN fails)
 *   keep[p] = core[p] and some neighbour n of p has core[n]
 *   edge[p] = q[p] >= thr_boundary and some neighbour n of p has keep[n]
 *   mask[p] = keep[p] or edge[p]
 *   n_pix   = pixels in the mask;   size = sum q over the mask
 *   cog_x   = sum q x / size,  cog_y = sum q y / size
 *   sxx     = sum q (x - cog_x)^2 / size,  syy likewise,  sxy = sum q (x - cog_x)(y - cog_y) / size
 *   z       = sqrt((sxx - syy)^2 + 4 sxy^2)
 *   length  = sqrt((sxx + syy + z) / 2),   width = sqrt(max(0, (sxx + syy - z) / 2))
 *   psi     = atan2(2 sxy, sxx - syy) / 2            (major-axis angle, (-pi/2, pi/2])
 *   t_mean  = sum q t / size;   q_max = largest q in the mask
 *   out_params[e][0..7] = size, cog_x, cog_y, length, width, psi, t_mean, q_max
 *   n_pix == 0, or size <= 0 or NaN  ->  all eight parameters are 0 (n_pix is still the count).
 *
 * Sums are accumulated in fp64 and rounded once to fp32; n_pix, the mask and
 * q_max are exact. Results do not depend on the launch (no atomics).
 *
 *   pix_x, pix_y  DEVICE float [n_pixels]      pixel centres, any unit
 *   neighbors     DEVICE int32 [n_pixels][6]   neighbour pixel indices; any value outside
 *                                              [0, n_pixels) means "no neighbour". The table is
 *                                              used as given (it need not be symmetric).
 *   out_n_pix     DEVICE int32 [n_events]
 *   out_params    DEVICE float [n_events][8]
 *   out_mask      DEVICE uint8 [n_events][n_pixels] (0/1), or NULL when not wanted
 *
 * rta_image_moments: cleaning + moments of charge / time arrays already on the
 * device (float [n_events][n_pixels], e.g. rta_extract's out_charge / out_time).
 * rta_extract_image: rta_extract's sliding-window extraction and the step above
 * in ONE kernel; charge and peak time stay in shared memory and only the event
 * parameters (36 bytes per event, + the mask if asked for) are written. Shapes
 * (30,7), (40,7), (25,4), (128,8) with a 16-byte-aligned wf and every event
 * starting on a boundary the staged loads accept take the staged kernels; any
 * other 16-byte-aligned shape with traces of at most 1152 bytes runs rta_extract's
 * staged kernel into a stream-ordered scratch buffer (cudaMallocAsync, 16 bytes
 * per trace, freed on the stream) followed by the moments kernel; anything else
 * (or no scratch to be had) a generic fused kernel. Same results either way
 * (rta_image_kernel_name says which). rta_extract_image(...) equals
 * rta_extract(...) followed by rta_image_moments(out_charge, out_time, ...).
 * rta_extract_image_stream / _host: the host-fed variants, chunked and double
 * buffered exactly like rta_extract_stream / rta_extract_host (same chunk rule,
 * same workspace and mutex); _host brings 36 bytes per event (+ mask) back.
 *
 * All asynchronous on `stream` except _host. Errors: the shape/NULL/alignment
 * rules of rta_extract for the waveform side; n_pixels above
 * rta_image_max_pixels() (two events' charges, times and bit masks must fit one
 * CTA's shared memory: 12 288 pixels) -> RTA_ERR_UNSUPPORTED; NULL geometry or
 * output (out_mask excepted) -> RTA_ERR_NULL; 4-byte alignment of every float /
 * int32 array. NaN thresholds give empty masks. n_events == 0 -> RTA_OK. */
int rta_image_moments(const float* charge, const float* time, int64_t n_events,
                      int32_t n_pixels, const float* pix_x, const float* pix_y,
                      const int32_t* neighbors, float thr_picture, float thr_boundary,
                      int32_t* out_n_pix, float* out_params, uint8_t* out_mask, void* stream);

int rta_extract_image(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                      int32_t n_samples, const int32_t* pedestal, const float* gain, int32_t W,
                      const float* pix_x, const float* pix_y, const int32_t* neighbors,
                      float thr_picture, float thr_boundary, int32_t* out_n_pix,
                      float* out_params, uint8_t* out_mask, void* stream);

/* wf_host: HOST (pinned or pageable); everything else DEVICE. */
int rta_extract_image_stream(const uint16_t* wf_host, int64_t n_events, int32_t n_pixels,
                             int32_t n_samples, const int32_t* pedestal, const float* gain,
                             int32_t W, const float* pix_x, const float* pix_y,
                             const int32_t* neighbors, float thr_picture, float thr_boundary,
                             int32_t* out_n_pix, float* out_params, uint8_t* out_mask,
                             size_t chunk_bytes, void* stream);

/* Every pointer HOST; synchronous. */
int rta_extract_image_host(const uint16_t* wf_host, int64_t n_events, int32_t n_pixels,
                           int32_t n_samples, const int32_t* pedestal_host,
                           const float* gain_host, int32_t W, const float* pix_x_host,
                           const float* pix_y_host, const int32_t* neighbors_host,
                           float thr_picture, float thr_boundary, int32_t* out_n_pix_host,
                           float* out_params_host, uint8_t* out_mask_host, size_t chunk_bytes);

/* rta_extract_image for callers that must not allocate device memory.
 *
 * Two kinds of caller are meant. A reconstruction thread during data taking
 * (§4.2, event by event while the telescopes acquire): cudaMalloc and
 * cudaFree synchronise the whole device, so an allocation on the analysis side
 * stalls the copies that bring the next events in. And a process whose device
 * memory is spoken for in full (a framework allocator told to take everything, a
 * GPU partition sized to the job), where an allocation behind the owner's back
 * fails or breaks the owner's budget. rta_extract_image itself is no good to
 * them on a shape without a fused kernel: it takes 16 bytes of scratch per trace
 * from a stream-ordered pool, may compile a kernel at first use, and its tile
 * scheduler lives in a cudaMalloc'ed pool.
 *
 * This call computes the same thing with the same arguments (extraction by the
 * runtime-shape staged kernel into scratch, then the moments kernel) and calls
 * no cudaMalloc, cudaFree, memory pool, run-time compiler or other allocating
 * routine. Its scratch is a static device array inside the library image:
 * 256 bytes of scheduler words + 16 bytes per trace for at most
 * RTA_NOALLOC_MAX_TRACES traces = 16 MiB + 256 bytes, held by every GPU that
 * loads librta.so from module load until the process exits, called or not.
 *
 *  - n_events * n_pixels > RTA_NOALLOC_MAX_TRACES -> RTA_ERR_TOO_LARGE, nothing
 *    enqueued (split the batch: events are independent).
 *  - wf must be 16-byte aligned (else RTA_ERR_ALIGN) and a trace (a pair of
 *    traces when n_samples is odd) at most 1152 bytes, i.e. n_samples <= 576
 *    even / 288 odd (else RTA_ERR_UNSUPPORTED). All four BASELINE shapes qualify.
 *    Every other rule of rta_extract_image applies unchanged.
 *  - The first call on a device looks the array's device address up
 *    (cudaGetSymbolAddress, once per device, with that device current) and sets
 *    kernel attributes; make that first call outside any stream capture.
 *  - The array is shared by every call on the device and keeps the previous
 *    call's bytes. The library zeroes the scheduler words on `stream` before each
 *    launch; the per-trace part is fully rewritten before it is read. Two calls
 *    whose kernels can run at the same time (unordered streams, two host threads)
 *    race on the array and return garbage: keep such calls on one stream or order
 *    them with events. Results equal rta_extract_image's (same integer
 *    extraction, same cleaning and moments code).
 * Asynchronous on `stream`; n_events == 0 -> RTA_OK. */
#define RTA_NOALLOC_MAX_TRACES 1048576
int rta_extract_image_noalloc(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                              int32_t n_samples, const int32_t* pedestal, const float* gain,
                              int32_t W, const float* pix_x, const float* pix_y,
                              const int32_t* neighbors, float thr_picture, float thr_boundary,
                              int32_t* out_n_pix, float* out_params, uint8_t* out_mask,
                              void* stream);

/* "image_tile<S=40,W=7>", ..., "staged<any>+image_moments" or "image_generic". */
const char* rta_image_kernel_name(int32_t n_pixels, int32_t n_samples, int32_t W, int aligned16);
int32_t rta_image_max_pixels(void);

/* Static, never-NULL description of a status code. */
const char* rta_strerror(int status);

/* The cudaError_t behind this thread's most recent RTA_ERR_CUDA / RTA_ERR_NOMEM
 * (0 if none). */
int rta_last_cuda_error(void);

/* Which kernel a shape takes, for tests and profiles: a static string such as
 * "tile<S=40,W=7>", "staged<jit>", "staged<any>", "segments", "lanes<32>" or "generic" for
 * (n_samples, W, 16-byte-aligned?). */
const char* rta_kernel_name(int32_t n_samples, int32_t W, int aligned16);
/* Take the run-time compile off the data path. A shape without an ahead-of-time
 * kernel is compiled for its (n_samples, W, extractor, sample format) the first
 * time a call meets it: 0.3-0.6 s on the host inside that call, and never inside
 * a stream capture (a first call that is being captured records the slower
 * runtime-shape kernel instead). An on-site pipeline that knows its cameras
 * (three telescope types; re-pointing within 90 s)
 * calls this once per shape at configuration time, with the device current that
 * will run the data, before any capture:
 *
 *   extractor    RTA_EXTRACTOR_SLIDING (rta_extract, rta_extract_ragged, the
 *                _stream / _host / _image calls), _FIXED, _LOCAL_PEAK or _FIR
 *                (W = n_taps)
 *   sample_bits  16 (uint16 samples) or 12 (P12 stream; sliding only)
 *
 * RTA_OK: a kernel specialised for the shape is compiled, loaded and set up on
 * the current device (or was built ahead of time); calls of this shape compile
 * nothing from now on. RTA_ERR_UNSUPPORTED: the shape has no specialisation
 * (trace too long for one, libnvrtc not found, RTA_JIT=0) and runs the
 * runtime-shape kernels, which need no preparation either; also P12 with another
 * extractor, and the int32 guard of rta_extract. RTA_ERR_SHAPE: bad n_samples /
 * W / extractor / sample_bits. Thread-safe; compiling one shape does not delay
 * launches of other shapes. rta_shutdown unloads what was compiled. */
enum {
  RTA_EXTRACTOR_SLIDING = 0,
  RTA_EXTRACTOR_FIXED = 1,
  RTA_EXTRACTOR_LOCAL_PEAK = 2,
  RTA_EXTRACTOR_FIR = 3
};
int rta_prepare(int32_t n_samples, int32_t W, int32_t extractor, int32_t sample_bits);

/* Same for a P12 stream: "tile12<S=40,W=7>", "tile12<jit>" (packed units of at most 320
 * bytes, compiled at first use), "generic12". */
const char* rta_kernel_name_packed12(int32_t n_samples, int32_t W, int aligned16);

/* Events per chunk the host-fed calls use for this shape and `chunk_bytes`
 * (sample_bits 16: rta_extract_stream / _host; 12: the _packed12 calls): whole
 * events, rounded down, at least one (P12: a multiple of m, see above), never
 * more than n_events (1 when n_events is 0). Pure host arithmetic; -1 on a bad
 * shape or sample_bits. */
int64_t rta_chunk_events(int64_t n_events, int32_t n_pixels, int32_t n_samples,
                         size_t chunk_bytes, int32_t sample_bits);

/* Number of kernels the library has launched in this process (all threads);
 * bench.py reports the difference over its timed region as gpu_launches. */
uint64_t rta_launch_count(void);

/* Frees the library-owned workspace (device buffers, pinned staging, streams,
 * events). Safe to call at any time no stream call is running; the workspace
 * is rebuilt on demand. */
void rta_shutdown(void);

#ifdef __cplusplus
}
#endif
#endif /* RTA_H */
