// rta_image.cu — image cleaning + image moments on the device, alone and fused
// behind the signal extraction.
//
// What is computed: DESIGN.md readings R31-R35 — the first downstream RT-RECO
// step (the paper names the chain only: "calibration ... direction
// reconstruction" PAPER.md:101 §4.1, a reduced fast version PAPER.md:113 §4.2),
// so that "event-level reconstruction parameters (but not the raw data)"
// (§2.2) are what leaves the GPU: two-threshold neighbour cleaning
// of the per-pixel charges, then the charge-weighted first and second moments
// of the surviving pixels (size, centre of gravity, length, width, psi), the
// charge-weighted mean peak time, the largest charge and the pixel count.
//
// How:
//  * clean_warp: ONE WARP cleans one event. The image is sparse (a few per
//    cent of the pixels pass a threshold), so the work is organised around bit
//    masks of the camera (one bit per pixel: core, low, keep, mask) and
//    compacted pixel lists: only core pixels look at their neighbours' core
//    bits, only pixels above the boundary threshold that are not kept look at
//    their neighbours' keep bits, and the moments run over the list of mask
//    pixels. Sums are fp64 (per-lane partial sums over the list in pixel order,
//    xor butterfly over the lanes: no atomics on floating point, run-to-run
//    deterministic), centred second moments in a second pass like the definition.
//  * extract_image_kernel<C> (fused, staged): a CTA owns one event at a time.
//    NT extraction threads stream the event's traces through the same
//    shared-memory stage ring as extract_tile_kernel (TMA bulk copies, or
//    16-byte cp.async for the padded S = 128 layout; tiles cut per event) and
//    write charge / peak time / threshold bits into one of two per-event
//    buffers in shared memory instead of HBM. One extra warp — the cleaning
//    warp — takes a finished buffer and runs clean_warp on it while the
//    extraction threads are already on the next event (named-barrier hand-off:
//    ready / free per buffer). Events are handed out dynamically (one atomic
//    per event). HBM traffic: the waveform bytes once in, 36 bytes per event
//    out (+ 1 byte per pixel if the mask is asked for).
//  * extract_image_generic_kernel: the same hand-off for any (S, W) and any
//    2-byte alignment; traces are read straight from global memory.
//  * image_moments_kernel: charge / time arrays already in HBM (rta_extract's
//    outputs); one warp per event, the charge row staged in shared memory, peak
//    times gathered from HBM for the mask pixels only.
#include "rta_device.cuh"

namespace {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
  return v;
}
__device__ __forceinline__ void named_sync(const int id, const int n) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory");
}
__device__ __forceinline__ void named_arrive(const int id, const int n) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory");
}

__host__ __device__ constexpr size_t r16(size_t n) { return (n + 15u) & ~(size_t)15u; }
__host__ __device__ constexpr size_t mask_words(int P) { return ((size_t)P + 31u) >> 5; }

// What the producer of an event (extraction threads, or the loading warp
// itself) hands to clean_warp: charges, peak times (shared or global memory)
// and the two threshold bit masks, bit p & 31 of word p >> 5.
struct EventBuf {
  float* q;          // [P]
  float* t;          // [P] (fused kernels only)
  uint32_t* core_w;  // q >= thr_picture
  uint32_t* low_w;   // q >= thr_boundary
  static __host__ __device__ size_t bytes(int P, bool with_t) {
    return (with_t ? 2u : 1u) * r16(4u * (size_t)P) + 2u * r16(4u * mask_words(P));
  }
  __device__ __forceinline__ EventBuf(uint8_t* base, const int P, const bool with_t) {
    q = reinterpret_cast<float*>(base);
    base += r16(4u * (size_t)P);
    t = reinterpret_cast<float*>(base);
    if (with_t) base += r16(4u * (size_t)P);
    core_w = reinterpret_cast<uint32_t*>(base);
    low_w = reinterpret_cast<uint32_t*>(base + r16(4u * mask_words(P)));
  }
};

// Scratch owned by a cleaning warp: keep / mask bit words and one pixel list.
struct CleanScratch {
  uint32_t* keep_w;
  uint32_t* mask_w;
  uint16_t* list;  // [P], pixel indices (< 2^16: rta_image_pixel_limit)
  static __host__ __device__ size_t bytes(int P) {
    return 2u * r16(4u * mask_words(P)) + r16(2u * (size_t)P);
  }
  __device__ __forceinline__ CleanScratch(uint8_t* base, const int P) {
    keep_w = reinterpret_cast<uint32_t*>(base);
    mask_w = reinterpret_cast<uint32_t*>(base + r16(4u * mask_words(P)));
    list = reinterpret_cast<uint16_t*>(base + 2u * r16(4u * mask_words(P)));
  }
};

// Pixel indices of the set bits of word(w), w = 0 .. NW-1, in ascending order
// into list[]; returns their number (same value in every lane). One warp: lane
// l owns the K = ceil(NW / 32) consecutive words l K .. l K + K - 1, so one
// prefix sum over the lanes' bit counts places every lane's run.
template <class F>
__device__ __forceinline__ int compact_bits(const int NW, uint16_t* __restrict__ list, F word) {
  const int lane = threadIdx.x & 31;
  const int K = (NW + 31) >> 5;
  const int w_lo = lane * K, w_hi = min(w_lo + K, NW);
  int c = 0;
  for (int w = w_lo; w < w_hi; ++w) c += __popc(word(w));
  int incl = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
    if (lane >= o) incl += v;
  }
  int off = incl - c;
  for (int w = w_lo; w < w_hi; ++w) {
    uint32_t bits = word(w);
    while (bits) {
      const int b = __ffs((int)bits) - 1;
      bits &= bits - 1u;
      list[off++] = (uint16_t)(32 * w + b);
    }
  }
  const int total = __shfl_sync(0xFFFFFFFFu, incl, 31);
  __syncwarp();
  return total;
}

__device__ __forceinline__ bool test_bit(const uint32_t* w, const int n) {
  return (w[n >> 5] >> (n & 31)) & 1u;
}

// For the n listed pixels: hit = some neighbour's bit is set in in_w; hits set
// the pixel's bit in out_w. Four list entries per lane are in flight at once
// (their neighbour rows are loaded before any is used). Returns "any hit" per
// lane. nb8: the table is 8-byte aligned, so a 24-byte row is three 8-byte loads.
__device__ __forceinline__ int neighbour_pass(const int n, const uint16_t* __restrict__ list,
                                              const int32_t* __restrict__ nbr, const bool nb8,
                                              const int P, const uint32_t* in_w,
                                              uint32_t* out_w) {
  const int lane = threadIdx.x & 31;
  constexpr int U = 2;
  int any = 0;
  for (int i0 = 0; i0 < n; i0 += 32 * U) {
    int p[U], nb[U][6];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = i0 + 32 * u + lane;
      p[u] = i < n ? (int)list[i] : -1;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (p[u] >= 0) {
        const int32_t* row = nbr + 6u * (size_t)p[u];
        if (nb8) {
#pragma unroll
          for (int j = 0; j < 3; ++j) {
            const int2 v = __ldg(reinterpret_cast<const int2*>(row) + j);
            nb[u][2 * j] = v.x, nb[u][2 * j + 1] = v.y;
          }
        } else {
#pragma unroll
          for (int j = 0; j < 6; ++j) nb[u][j] = __ldg(row + j);
        }
      }
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (p[u] >= 0) {
        bool hit = false;
#pragma unroll
        for (int j = 0; j < 6; ++j)
          if ((unsigned)nb[u][j] < (unsigned)P && test_bit(in_w, nb[u][j])) hit = true;
        if (hit) {
          atomicOr(&out_w[p[u] >> 5], 1u << (p[u] & 31));
          any = 1;
        }
      }
    }
  }
  __syncwarp();
  return any;
}

__device__ __forceinline__ double bcast(const double v, const int src) {
  return __shfl_sync(0xFFFFFFFFu, v, src);
}

// Cleaning and moments of event e (readings R31-R35), executed by one whole
// warp. q / core_w / low_w are in shared memory and complete; t points at the
// event's peak times (shared or global memory).
__device__ __forceinline__ void clean_warp(const uint32_t e, const int P, const float* q,
                                           const float* t, const uint32_t* core_w,
                                           const uint32_t* low_w, const CleanScratch& sc,
                                           const RtaCamera& cam, const RtaImageOut& out) {
  const int lane = threadIdx.x & 31;
  const int NW = (int)mask_words(P);
  const bool nb8 = (reinterpret_cast<uintptr_t>(cam.neighbors) & 7u) == 0;
  uint8_t* mrow = out.mask ? out.mask + (size_t)e * (size_t)P : nullptr;

  // keep[p] = core[p] and some neighbour is core (isolated core pixels drop)
  for (int w = lane; w < NW; w += 32) sc.keep_w[w] = 0u;
  const int n_core = compact_bits(NW, sc.list, [&](int w) { return core_w[w]; });
  const int kept = neighbour_pass(n_core, sc.list, cam.neighbors, nb8, P, core_w, sc.keep_w);
  if (!__any_sync(0xFFFFFFFFu, kept)) {  // no surviving core pixel: the mask is empty
    if (mrow)
      for (int p = lane; p < P; p += 32) mrow[p] = 0;
    if (lane == 8) out.n_pix[e] = 0;
    if (lane < 8) out.params[(size_t)e * 8u + lane] = 0.0f;
    return;
  }

  // mask[p] = keep[p] or (q[p] >= thr_boundary and some neighbour is kept)
  for (int w = lane; w < NW; w += 32) sc.mask_w[w] = sc.keep_w[w];
  const int n_cand =
      compact_bits(NW, sc.list, [&](int w) { return low_w[w] & ~sc.keep_w[w]; });
  neighbour_pass(n_cand, sc.list, cam.neighbors, nb8, P, sc.keep_w, sc.mask_w);
  if (mrow)
    for (int p = lane; p < P; p += 32) mrow[p] = test_bit(sc.mask_w, p) ? 1 : 0;

  // pass 1 over the mask pixels in ascending pixel order: lane i takes entries
  // i, i + 32, ...; the first two per lane stay in registers for pass 2
  const int n_pix = compact_bits(NW, sc.list, [&](int w) { return sc.mask_w[w]; });
  double rw[2] = {0.0, 0.0}, rx[2] = {0.0, 0.0}, ry[2] = {0.0, 0.0}, rt[2] = {0.0, 0.0};
  float qm = -INFINITY;
#pragma unroll
  for (int u = 0; u < 2; ++u) {
    const int i = lane + 32 * u;
    if (i < n_pix) {
      const int p = sc.list[i];
      const float qp = q[p];
      rw[u] = (double)qp;
      rx[u] = (double)__ldg(cam.pix_x + p);
      ry[u] = (double)__ldg(cam.pix_y + p);
      rt[u] = (double)t[p];
      qm = fmaxf(qm, qp);
    }
  }
  double s0 = rw[0], sx = rw[0] * rx[0], sy = rw[0] * ry[0], st = rw[0] * rt[0];
  s0 += rw[1], sx += rw[1] * rx[1], sy += rw[1] * ry[1], st += rw[1] * rt[1];
  for (int i = lane + 64; i < n_pix; i += 32) {
    const int p = sc.list[i];
    const float qp = q[p];
    const double w = (double)qp;
    s0 += w;
    sx += w * (double)__ldg(cam.pix_x + p);
    sy += w * (double)__ldg(cam.pix_y + p);
    st += w * (double)t[p];
    qm = fmaxf(qm, qp);
  }
  s0 = warp_sum(s0), sx = warp_sum(sx), sy = warp_sum(sy), st = warp_sum(st);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) qm = fmaxf(qm, __shfl_xor_sync(0xFFFFFFFFu, qm, o));
  if (!(s0 > 0.0)) {  // non-positive (or NaN) total charge: parameters are zero, the count stands
    if (lane == 8) out.n_pix[e] = n_pix;
    if (lane < 8) out.params[(size_t)e * 8u + lane] = 0.0f;
    return;
  }
  // one division for three quotients: lane 0, 1, 2 divide sx, sy, st by s0
  const double r1 = (lane == 0 ? sx : lane == 1 ? sy : st) / s0;
  const double cx = bcast(r1, 0), cy = bcast(r1, 1), tm = bcast(r1, 2);

  // pass 2: centred second moments
  double sxx = 0.0, syy = 0.0, sxy = 0.0;
#pragma unroll
  for (int u = 0; u < 2; ++u) {  // entries past n_pix carry zero weight
    const double dx = rx[u] - cx, dy = ry[u] - cy;
    sxx += rw[u] * dx * dx;
    syy += rw[u] * dy * dy;
    sxy += rw[u] * dx * dy;
  }
  for (int i = lane + 64; i < n_pix; i += 32) {
    const int p = sc.list[i];
    const double w = (double)q[p];
    const double dx = (double)__ldg(cam.pix_x + p) - cx, dy = (double)__ldg(cam.pix_y + p) - cy;
    sxx += w * dx * dx;
    syy += w * dy * dy;
    sxy += w * dx * dy;
  }
  sxx = warp_sum(sxx), syy = warp_sum(syy), sxy = warp_sum(sxy);
  const double r2 = (lane == 0 ? sxx : lane == 1 ? syy : sxy) / s0;
  sxx = bcast(r2, 0), syy = bcast(r2, 1), sxy = bcast(r2, 2);
  const double d = sxx - syy;
  const double z = sqrt(d * d + 4.0 * sxy * sxy);
  // one square root for length (lane 3) and width (lane 4)
  const double r3 = sqrt(lane == 3 ? 0.5 * (sxx + syy + z) : fmax(0.5 * (sxx + syy - z), 0.0));
  const double psi = 0.5 * atan2(2.0 * sxy, d);
  const double v = lane == 0 ? s0 : lane == 1 ? cx : lane == 2 ? cy : lane == 5 ? psi
                 : lane == 6 ? tm : r3;
  if (lane < 7) out.params[(size_t)e * 8u + lane] = (float)v;
  if (lane == 7) out.params[(size_t)e * 8u + 7u] = qm;
  if (lane == 8) out.n_pix[e] = n_pix;
}

// ------------------------------------------------ cleaning on HBM arrays ----
// One warp per event: the charge row comes in by cp.async into one of two
// per-warp buffers (the next event's row is in flight while this one is
// cleaned); peak times stay in HBM and are gathered for the mask pixels only.
__device__ __forceinline__ void row_async(float* dst, const float* src, const int P) {
  const int lane = threadIdx.x & 31;
  int p = 0;
  if ((reinterpret_cast<uintptr_t>(src) & 15u) == 0) {
    const int n4 = P >> 2;
    for (int i = lane; i < n4; i += 32) cp_async16(smem_u32(dst + 4 * i), src + 4 * i);
    p = 4 * n4;
  }
  for (int i = p + lane; i < P; i += 32) cp_async4(smem_u32(dst + i), src + i);
  asm volatile("cp.async.commit_group;" ::: "memory");
}

template <int WARPS>
__global__ void __launch_bounds__(32 * WARPS)
    image_moments_kernel(const float* __restrict__ charge, const float* __restrict__ time,
                         const uint32_t n_events, const int P,
                         const __grid_constant__ RtaCamera cam,
                         const __grid_constant__ RtaImageOut out) {
  extern __shared__ __align__(128) uint8_t smem[];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t row_bytes = r16(4u * (size_t)P);
  const size_t per_warp = row_bytes + EventBuf::bytes(P, false) + CleanScratch::bytes(P);
  uint8_t* mine = smem + (size_t)warp * per_warp;
  float* rows[2] = {reinterpret_cast<float*>(mine), reinterpret_cast<float*>(mine + row_bytes)};
  const EventBuf buf(mine + row_bytes, P, false);  // buf.q == rows[1]; only the bit words are used
  const CleanScratch sc(mine + row_bytes + EventBuf::bytes(P, false), P);
  const float thr_p = cam.thr_picture, thr_b = cam.thr_boundary;
  const uint32_t stride = gridDim.x * WARPS;
  uint32_t e = blockIdx.x * WARPS + warp;
  if (e < n_events) row_async(rows[0], charge + (size_t)e * (size_t)P, P);
  for (int b = 0; e < n_events; e += stride, b ^= 1) {
    if (e + stride < n_events) {
      row_async(rows[b ^ 1], charge + (size_t)(e + stride) * (size_t)P, P);
      asm volatile("cp.async.wait_group 1;" ::: "memory");
    } else {
      asm volatile("cp.async.wait_group 0;" ::: "memory");
    }
    __syncwarp();
    const float* q = rows[b];
#pragma unroll 4
    for (int p0 = 0; p0 < P; p0 += 32) {
      const int p = p0 + lane;
      const bool in = p < P;
      const float v = in ? q[p] : 0.0f;
      const uint32_t c = __ballot_sync(0xFFFFFFFFu, in && v >= thr_p);
      const uint32_t l = __ballot_sync(0xFFFFFFFFu, in && v >= thr_b);
      if (lane == 0) buf.core_w[p0 >> 5] = c, buf.low_w[p0 >> 5] = l;
    }
    __syncwarp();
    clean_warp(e, P, q, time + (size_t)e * (size_t)P, buf.core_w, buf.low_w, sc, cam, out);
    __syncwarp();
  }
}

// ------------------------------------------------- producer / cleaner hand-off ----
// The fused kernels run NT extraction threads and one cleaning warp (threads
// NT .. NT+31). Event number k of the CTA uses buffer k & 1. Named barriers
// (all with NT + 32 participants): READY + b — the extraction threads arrive
// when the buffer is complete, the cleaning warp waits; FREE + b — the
// cleaning warp arrives when it is done with the buffer, the extraction
// threads wait before writing event k + 2 into it. ev_id[b] carries the event
// index (kNoEvent = no more events).
enum : int { BAR_READY = 1, BAR_FREE = 3, BAR_EXTRACT = 5 };
constexpr uint32_t kNoEvent = 0xFFFFFFFFu;

struct FusedShared {
  uint32_t ev_id[2];
};

template <int NT>
__device__ __forceinline__ void cleaner_loop(const int P, uint8_t* ev_base, uint8_t* sc_base,
                                             volatile FusedShared& fs, const RtaCamera& cam,
                                             const RtaImageOut& out) {
  const size_t eb = EventBuf::bytes(P, true);
  const CleanScratch sc(sc_base, P);
  for (uint32_t k = 0;; ++k) {
    const int b = (int)(k & 1u);
    named_sync(BAR_READY + b, NT + 32);
    const uint32_t e = fs.ev_id[b];
    if (e == kNoEvent) break;
    const EventBuf buf(ev_base + (size_t)b * eb, P, true);
    clean_warp(e, P, buf.q, buf.t, buf.core_w, buf.low_w, sc, cam, out);
    __syncwarp();
    named_arrive(BAR_FREE + b, NT + 32);
  }
}

// extraction side: before the first write of the CTA's event number k
template <int NT>
__device__ __forceinline__ void producer_acquire(const uint32_t k) {
  if (k >= 2u) named_sync(BAR_FREE + (int)(k & 1u), NT + 32);
}
// extraction side: every extraction thread, after its last write of event number k
template <int NT>
__device__ __forceinline__ void producer_release(const uint32_t k, const uint32_t e,
                                                 volatile FusedShared& fs, const bool leader) {
  if (leader) fs.ev_id[k & 1u] = e;
  __threadfence_block();
  named_arrive(BAR_READY + (int)(k & 1u), NT + 32);
}

// ----------------------------------------- extraction + cleaning, generic ----
template <int NT>
__global__ void __launch_bounds__(NT + 32)
    extract_image_generic_kernel(const uint8_t* __restrict__ wf, const uint32_t n_events,
                                 const int P, const int S, const int W,
                                 const int* __restrict__ pedestal, const float* __restrict__ gain,
                                 const __grid_constant__ RtaCamera cam,
                                 const __grid_constant__ RtaImageOut out) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ FusedShared fs;
  const int tid = threadIdx.x, lane = tid & 31;
  const size_t eb = EventBuf::bytes(P, true);
  if (tid >= NT) {
    cleaner_loop<NT>(P, smem, smem + 2u * eb, fs, cam, out);
    return;
  }
  const ModeArgs ma = {};
  const float thr_p = cam.thr_picture, thr_b = cam.thr_boundary;
  uint32_t k = 0;
  for (uint32_t e = blockIdx.x; e < n_events; e += gridDim.x, ++k) {
    producer_acquire<NT>(k);
    const EventBuf buf(smem + (size_t)(k & 1u) * eb, P, true);
    const uint8_t* base = wf + (size_t)e * (size_t)P * (size_t)S * 2u;
    for (int p0 = tid - lane; p0 < P; p0 += NT) {  // whole warps: the ballots need every lane
      const int p = p0 + lane;
      float qv = 0.0f;
      const bool in = p < P;
      if (in) {
        const GlobalTrace<16> tr(base, (uint32_t)p, S);
        const Result r = generic_trace<MODE_SLIDING, 16>(tr, S, W, (uint32_t)p, pedestal, gain, ma);
        buf.q[p] = qv = r.charge;
        buf.t[p] = r.time;
      }
      const uint32_t c = __ballot_sync(0xFFFFFFFFu, in && qv >= thr_p);
      const uint32_t l = __ballot_sync(0xFFFFFFFFu, in && qv >= thr_b);
      if (lane == 0) buf.core_w[p0 >> 5] = c, buf.low_w[p0 >> 5] = l;
    }
    producer_release<NT>(k, e, fs, tid == 0);
  }
  producer_acquire<NT>(k);
  producer_release<NT>(k, kNoEvent, fs, tid == 0);
}

// 16 bits -> the even bit positions of 32 bits
__device__ __forceinline__ uint32_t spread16(uint32_t x) {
  x &= 0xFFFFu;
  x = (x | (x << 8)) & 0x00FF00FFu;
  x = (x | (x << 4)) & 0x0F0F0F0Fu;
  x = (x | (x << 2)) & 0x33333333u;
  x = (x | (x << 1)) & 0x55555555u;
  return x;
}

// ------------------------------------------- extraction + cleaning, staged ----
// Work items of a CTA: (event, tile) pairs, tiles 0 .. nt-1 of one event, then
// the next event drawn from the shared counter. The producer side runs STAGES
// items ahead of the consumer through item_q, across event boundaries.
template <class C>
__global__ void __launch_bounds__(C::NT + 32, C::NT >= 256 ? 3 : 1)
    extract_image_kernel(const uint8_t* __restrict__ wf, const uint32_t n_events, const int P,
                         const int* __restrict__ pedestal, const float* __restrict__ gain,
                         const __grid_constant__ RtaCamera cam,
                         const __grid_constant__ RtaImageOut out, uint32_t* __restrict__ sched) {
  static_assert(C::BITS == 16 && C::STAGES >= 2, "uint16 samples, at least two stages");
  static_assert(C::TPT == 1 || C::TPT == 2, "one or two traces per thread");
  // an event may start at any multiple of VEC bytes: the copy starts at the
  // 16-byte boundary below it, so a stage holds up to 16 bytes more than a tile
  constexpr int STG = C::STAGE_BYTES + 16;
  constexpr int NT = C::NT;
  constexpr uint32_t TRACE_BYTES = C::TRACE_BITS / 8;
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[C::STAGES];
  constexpr int QN = C::STAGES + 1;
  __shared__ uint2 item_q[QN];  // {event, tile}
  __shared__ FusedShared fs;
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_u32(full_bar);
  uint8_t* ev_base = smem + C::STAGES * STG;
  const size_t eb = EventBuf::bytes(P, true);
  const ModeArgs ma = {};
  const uint32_t nt = ((uint32_t)P + C::TILE_TRACES - 1u) / C::TILE_TRACES;  // tiles per event
  const unsigned long long EB = (unsigned long long)P * TRACE_BYTES;         // bytes per event
  const unsigned long long total = (unsigned long long)n_events * EB;
  const float thr_p = cam.thr_picture, thr_b = cam.thr_boundary;

  // thread 0: the producer cursor (pev, pt) and one prefetched event index
  uint32_t pev = blockIdx.x, pt = 0, pre_ev = kNoEvent;
  auto fetch_event = [&]() -> uint32_t {
    if (sched == nullptr) return (pev > kNoEvent - gridDim.x) ? kNoEvent : pev + gridDim.x;
    const uint32_t got = pre_ev;
    const uint32_t k = atomicAdd(sched, 1u);
    pre_ev = (k > kNoEvent - gridDim.x) ? kNoEvent : gridDim.x + k;
    return got;
  };
  auto next_item = [&]() -> uint2 {
    const uint2 it = make_uint2(pev, pt);
    if (pev < n_events && ++pt == nt) {
      pt = 0;
      pev = fetch_event();
    }
    return it;
  };

  if (tid == 0) {
    if (sched != nullptr) {
      const uint32_t k = atomicAdd(sched, 1u);
      pre_ev = (k > kNoEvent - gridDim.x) ? kNoEvent : gridDim.x + k;
    }
#pragma unroll
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(bar_base + 8 * s, C::PAD ? NT : 1);
      item_q[s] = next_item();
    }
    fence_mbar_init();
  }
  __syncthreads();
  if (tid >= NT) {  // the cleaning warp
    cleaner_loop<NT>(P, ev_base, ev_base + 2u * eb, fs, cam, out);
    return;
  }

  auto issue = [&](const uint2 it, const int stage) {
    const unsigned long long start = (unsigned long long)it.x * EB +
                                     (unsigned long long)it.y * C::TILE_BYTES;
    const uint32_t left = (uint32_t)P - it.y * C::TILE_TRACES;
    const uint32_t n = left < (uint32_t)C::TILE_TRACES ? left : (uint32_t)C::TILE_TRACES;
    const uint32_t bytes = n * TRACE_BYTES;
    const uint32_t dst = smem_base + stage * STG;
    const uint32_t bar = bar_base + 8 * stage;
    if constexpr (!C::PAD) {
      if (tid == 0) {
        const uint32_t mis = (uint32_t)(start & 15u);
        const unsigned long long lo = start - mis;
        uint32_t len = (mis + bytes + 15u) & ~15u;
        if (lo + len > total) {
          // the last tile of the last event: nothing past the caller's buffer
          // is read; the final < 16 bytes go halfword by halfword
          len = (uint32_t)((total - lo) & ~15ull);
          uint8_t* d = smem + stage * STG;
          for (uint32_t b = len; b < mis + bytes; b += 2u)
            *reinterpret_cast<uint16_t*>(d + b) = *reinterpret_cast<const uint16_t*>(wf + lo + b);
        }
        mbar_expect_tx(bar, len);
        if (len != 0) tma_bulk_g2s(dst, wf + lo, len, bar);
      }
    } else {
      // S = 128: events start on 16-byte boundaries (256-byte traces)
      const uint8_t* src = wf + start;
#pragma unroll 4
      for (uint32_t c = tid; c < bytes / 16u; c += NT) {
        const uint32_t u = c / C::NVEC;  // one extra chunk of padding per unit
        cp_async16(dst + (c + u) * 16u, src + (size_t)c * 16u);
      }
      cp_async_mbar_arrive(bar);
    }
  };

#pragma unroll
  for (int s = 0; s < C::STAGES; ++s) {
    const uint2 it = item_q[s];
    if (it.x < n_events) issue(it, s);
  }

  uint32_t k = 0;  // events of this CTA so far
  for (uint32_t j = 0;; ++j) {
    const uint2 it = item_q[j % QN];
    if (it.x >= n_events) break;  // event indices grow per CTA: nothing later is valid either
    const int stage = (int)(j % C::STAGES);
    const uint32_t parity = (j / C::STAGES) & 1u;
    if (tid == 0) item_q[(j + C::STAGES) % QN] = next_item();
    if (it.y == 0) producer_acquire<NT>(k);
    const EventBuf buf(ev_base + (size_t)(k & 1u) * eb, P, true);
    mbar_wait(bar_base + 8 * stage, parity);
    const uint32_t p0 = it.y * C::TILE_TRACES + (uint32_t)tid * C::TPT;
    float qv[C::TPT];
#pragma unroll
    for (int i = 0; i < C::TPT; ++i) qv[i] = 0.0f;
    if (p0 < (uint32_t)P) {
      uint32_t mis = 0;
      if constexpr (!C::PAD)
        mis = (uint32_t)(((unsigned long long)it.x * EB + (unsigned long long)it.y * C::TILE_BYTES) & 15u);
      const uint8_t* unit = smem + stage * STG + mis + tid * C::UNIT_STRIDE;
      Result res[C::TPT];
      compute_results<C, MODE_SLIDING>(unit, p0, 0u, pedestal, gain, ma, res);
#pragma unroll
      for (int i = 0; i < C::TPT; ++i) {  // P is a multiple of TPT: the unit is whole
        buf.q[p0 + i] = qv[i] = res[i].charge;
        buf.t[p0 + i] = res[i].time;
      }
    }
    // threshold bits of this warp's 32 * TPT pixels (warps past the camera's end write nothing)
    const uint32_t w0 = (it.y * C::TILE_TRACES + (uint32_t)(tid - lane) * C::TPT) >> 5;
    const bool in = p0 < (uint32_t)P;
    if constexpr (C::TPT == 1) {
      const uint32_t c = __ballot_sync(0xFFFFFFFFu, in && qv[0] >= thr_p);
      const uint32_t l = __ballot_sync(0xFFFFFFFFu, in && qv[0] >= thr_b);
      if (lane == 0 && w0 < mask_words(P)) buf.core_w[w0] = c, buf.low_w[w0] = l;
    } else {
      const uint32_t c0 = __ballot_sync(0xFFFFFFFFu, in && qv[0] >= thr_p);
      const uint32_t c1 = __ballot_sync(0xFFFFFFFFu, in && qv[1] >= thr_p);
      const uint32_t l0 = __ballot_sync(0xFFFFFFFFu, in && qv[0] >= thr_b);
      const uint32_t l1 = __ballot_sync(0xFFFFFFFFu, in && qv[1] >= thr_b);
      // lane l holds pixels 2 l and 2 l + 1 of the warp's 64: lanes 0-15 fill word w0, 16-31 word w0 + 1
      if ((lane & 15) == 0) {
        const int sh = lane;  // 0 or 16
        const uint32_t w = w0 + (uint32_t)(lane >> 4);
        if (w < mask_words(P)) {
          buf.core_w[w] = spread16(c0 >> sh) | (spread16(c1 >> sh) << 1);
          buf.low_w[w] = spread16(l0 >> sh) | (spread16(l1 >> sh) << 1);
        }
      }
    }
    named_sync(BAR_EXTRACT, NT);  // the stage is free, the item slot is published
    const uint2 nxt = item_q[(j + C::STAGES) % QN];
    if (nxt.x < n_events) issue(nxt, stage);
    if (it.y + 1u == nt) {
      producer_release<NT>(k, it.x, fs, tid == 0);
      ++k;
    }
  }
  producer_acquire<NT>(k);
  producer_release<NT>(k, kNoEvent, fs, tid == 0);

  if (sched != nullptr && tid == 0) {
    __threadfence();
    if (atomicAdd(sched + 1, 1u) == gridDim.x - 1) {
      sched[0] = 0;
      sched[1] = 0;
      __threadfence();
    }
  }
}

// ------------------------------------------------------------- dispatch ----
constexpr int kGenericNT = 256;
constexpr size_t kSmemLimit = 227u * 1024u;

#ifndef RTA_I30_NT
#define RTA_I30_NT 256
#endif
#ifndef RTA_I30_ST
#define RTA_I30_ST 2
#endif
#ifndef RTA_I40_NT
#define RTA_I40_NT 256
#endif
#ifndef RTA_I40_ST
#define RTA_I40_ST 2
#endif
#ifndef RTA_I25_NT
#define RTA_I25_NT 256
#endif
#ifndef RTA_I25_ST
#define RTA_I25_ST 2
#endif
#ifndef RTA_I128_NT
#define RTA_I128_NT 64
#endif
#ifndef RTA_I128_ST
#define RTA_I128_ST 2
#endif
using ImgS30W7 = TileCfg<30, 7, RTA_I30_NT, RTA_I30_ST>;
using ImgS40W7 = TileCfg<40, 7, RTA_I40_NT, RTA_I40_ST>;
using ImgS25W4 = TileCfg<25, 4, RTA_I25_NT, RTA_I25_ST>;
using ImgS128W8 = TileCfg<128, 8, RTA_I128_NT, RTA_I128_ST>;

// shared memory of one warp of image_moments_kernel: two charge rows, bit words, scratch
size_t moments_warp_bytes(int32_t P) {
  return r16(4u * (size_t)P) + EventBuf::bytes(P, false) + CleanScratch::bytes(P);
}

// shared memory of the fused kernels behind the stage ring: two event buffers
// and the cleaning warp's scratch
size_t fused_image_bytes(int32_t P) {
  return 2u * EventBuf::bytes(P, true) + CleanScratch::bytes(P);
}

// The staged kernel takes a shape when every event starts on a boundary its
// units can be read from (VEC bytes; whole units per event) and the per-event
// buffers fit behind the ring.
template <class C>
bool staged_ok(int32_t P) {
  const size_t eb = (size_t)P * (C::TRACE_BITS / 8);
  if (P % C::TPT != 0 || eb % C::VEC != 0) return false;
  if (C::PAD && eb % 16 != 0) return false;
  return C::STAGES * (size_t)(C::STAGE_BYTES + 16) + fused_image_bytes(P) + 1024u <= kSmemLimit;
}

template <class C>
struct FusedLauncher {
  static cudaError_t launch(const uint8_t* wf, uint32_t n_events, int32_t P,
                            const int32_t* pedestal, const float* gain, const RtaCamera& cam,
                            const RtaImageOut& out, cudaStream_t stream) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if ((e = rta_device_sms(dev, &sms)) != cudaSuccess) return e;
    const size_t smem = C::STAGES * (size_t)(C::STAGE_BYTES + 16) + fused_image_bytes(P);
    // the dynamic shared-memory size depends on n_pixels: set per launch (cheap)
    e = cudaFuncSetAttribute(extract_image_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, extract_image_kernel<C>, C::NT + 32,
                                                      smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    uint32_t grid = (uint32_t)(sms * occ);
    if (grid > n_events) grid = n_events;
    uint32_t* sched = rta_static_schedule() ? nullptr : rta_sched_words(dev, stream);
    extract_image_kernel<C><<<grid, C::NT + 32, smem, stream>>>(wf, n_events, P, pedestal, gain,
                                                                cam, out, sched);
    rta_count_launch();
    return cudaGetLastError();
  }
};

// grid = every CTA the device holds at once (or one per `per_cta` events)
template <class K>
cudaError_t resident_grid(K kernel, int threads, size_t smem, uint32_t n_events, uint32_t per_cta,
                          uint32_t* grid_out) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = rta_device_sms(dev, &sms)) != cudaSuccess) return e;
  if (smem + 1024u > kSmemLimit) return cudaErrorInvalidValue;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  uint32_t grid = (uint32_t)(sms * occ);
  const uint32_t need = (n_events + per_cta - 1u) / per_cta;
  if (grid > need) grid = need;
  *grid_out = grid;
  return cudaSuccess;
}

template <int WARPS>
cudaError_t launch_moments(const float* charge, const float* time, uint32_t n_events, int32_t P,
                           const RtaCamera& cam, const RtaImageOut& out, cudaStream_t stream) {
  const size_t smem = WARPS * moments_warp_bytes(P);
  uint32_t grid = 0;
  cudaError_t e =
      resident_grid(image_moments_kernel<WARPS>, 32 * WARPS, smem, n_events, WARPS, &grid);
  if (e != cudaSuccess) return e;
  image_moments_kernel<WARPS><<<grid, 32 * WARPS, smem, stream>>>(charge, time, n_events, P, cam,
                                                                 out);
  rta_count_launch();
  return cudaGetLastError();
}

}  // namespace

int32_t rta_image_pixel_limit() {
  // two event buffers (charge, time, two bit masks) and the cleaning warp's
  // scratch must fit one CTA's shared memory in the generic fused kernel:
  // about 18.75 bytes per pixel of 227 KB
  return 12288;
}

const char* rta_pick_image_kernel_name(int32_t P, int32_t S, int32_t W, bool aligned16) {
  if (aligned16) {
    if (S == 30 && W == 7 && staged_ok<ImgS30W7>(P)) return "image_tile<S=30,W=7>";
    if (S == 40 && W == 7 && staged_ok<ImgS40W7>(P)) return "image_tile<S=40,W=7>";
    if (S == 25 && W == 4 && staged_ok<ImgS25W4>(P)) return "image_tile<S=25,W=4>";
    if (S == 128 && W == 8 && staged_ok<ImgS128W8>(P)) return "image_tile<S=128,W=8>";
  }
  return "image_generic";
}

cudaError_t rta_launch_image_moments(const float* charge, const float* time, int64_t n_events,
                                     int32_t n_pixels, const RtaCamera& cam,
                                     const RtaImageOut& out, cudaStream_t stream) {
  if (n_events <= 0) return cudaSuccess;
  // as many warps per CTA as keep two CTAs per SM resident
  const size_t per_warp = moments_warp_bytes(n_pixels);
  const size_t half = (kSmemLimit - 2048u) / 2u;
  const uint32_t E = (uint32_t)n_events;
  if (8u * per_warp <= half) return launch_moments<8>(charge, time, E, n_pixels, cam, out, stream);
  if (4u * per_warp <= half) return launch_moments<4>(charge, time, E, n_pixels, cam, out, stream);
  if (2u * per_warp <= half) return launch_moments<2>(charge, time, E, n_pixels, cam, out, stream);
  return launch_moments<1>(charge, time, E, n_pixels, cam, out, stream);
}

cudaError_t rta_launch_extract_image(const void* wf, int64_t n_events, int32_t n_pixels,
                                     int32_t S, const int32_t* pedestal, const float* gain,
                                     int32_t W, const RtaCamera& cam, const RtaImageOut& out,
                                     cudaStream_t stream, bool force_generic) {
  if (n_events <= 0) return cudaSuccess;
  const uint8_t* w = static_cast<const uint8_t*>(wf);
  if (!force_generic && ((uintptr_t)wf % 16) == 0) {
#define RTA_TRY(CFG)                                                                     \
  if (S == CFG::S && W == CFG::W && staged_ok<CFG>(n_pixels))                            \
    return FusedLauncher<CFG>::launch(w, (uint32_t)n_events, n_pixels, pedestal, gain,   \
                                      cam, out, stream);
    RTA_TRY(ImgS30W7)
    RTA_TRY(ImgS40W7)
    RTA_TRY(ImgS25W4)
    RTA_TRY(ImgS128W8)
#undef RTA_TRY
  }
  const size_t smem = fused_image_bytes(n_pixels);
  uint32_t grid = 0;
  cudaError_t e = resident_grid(extract_image_generic_kernel<kGenericNT>, kGenericNT + 32, smem,
                                (uint32_t)n_events, 1u, &grid);
  if (e != cudaSuccess) return e;
  extract_image_generic_kernel<kGenericNT><<<grid, kGenericNT + 32, smem, stream>>>(
      w, (uint32_t)n_events, n_pixels, S, W, pedestal, gain, cam, out);
  rta_count_launch();
  return cudaGetLastError();
}
