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
// How: one CTA owns one event at a time.
//  * extract_image_kernel<C>: the CTA streams the event's traces through the
//    same shared-memory stage ring as extract_tile_kernel (TMA bulk copies, or
//    16-byte cp.async for the padded S = 128 layout), tiles cut per event; each
//    thread's charge and peak time go to two per-event arrays in shared memory
//    instead of HBM. After the event's last tile the CTA cleans the image and
//    reduces the moments from shared memory while the TMA copies of the next
//    event's first tiles are already in flight. Events are handed out
//    dynamically (one atomic per event). HBM traffic: the waveform bytes once
//    in, 36 bytes per event out (+ 1 byte per pixel if the mask is asked for).
//  * extract_image_generic_kernel: any (S, W), any 2-byte alignment; traces are
//    read straight from global memory.
//  * image_moments_kernel: the same cleaning on charge / time arrays already in
//    HBM (rta_extract's outputs).
//  * cleaning is sparse: only pixels above the picture threshold look at their
//    neighbours' charges, only pixels above the boundary threshold look at
//    their neighbours' keep flags, and an event without a surviving core pixel
//    ends after one barrier. Moments are accumulated in fp64 (per-thread
//    partial sums, xor-butterfly per warp, fixed-order sum over the warps: no
//    atomics, run-to-run deterministic), centred second moments in a second
//    pass over the mask like the definition.
#include "rta_device.cuh"

#include <atomic>

namespace {

template <int NT>
struct RedScratch {
  double a[NT / 32][4];  // pass 1: size, sum q x, sum q y, sum q t
  int n[NT / 32];
  float qmax[NT / 32];
  double b[NT / 32][3];  // pass 2: centred sxx, syy, sxy (times size)
};

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
  return v;
}

// bytes of the per-event arrays behind the stage ring: charge, time (fp32) and
// the keep / mask flags (bytes), each rounded to 16 bytes
__host__ __device__ constexpr size_t r16(size_t n) { return (n + 15u) & ~(size_t)15u; }
__host__ __device__ inline size_t image_smem_bytes(int P) {
  return 2u * r16(4u * (size_t)P) + 2u * r16((size_t)P);
}

struct EventArrays {
  float* q;
  float* t;
  uint8_t* keep;
  uint8_t* mask;
  __device__ __forceinline__ EventArrays(uint8_t* base, const int P) {
    q = reinterpret_cast<float*>(base);
    t = reinterpret_cast<float*>(base + r16(4u * (size_t)P));
    keep = base + 2u * r16(4u * (size_t)P);
    mask = keep + r16((size_t)P);
  }
};

__device__ __forceinline__ void store_empty(const uint32_t e, const int n_pix,
                                            const RtaImageOut& out) {
  out.n_pix[e] = n_pix;
  float* o = out.params + (size_t)e * 8u;
#pragma unroll
  for (int i = 0; i < 8; ++i) o[i] = 0.0f;
}

// Cleaning and moments of event e from the charge / time arrays in shared
// memory (readings R31-R35). Called by every thread of the CTA after a barrier
// that published ev.q / ev.t; every read of ev.q / ev.t is followed by a
// barrier inside, so the caller may overwrite them right after it returns.
template <int NT>
__device__ __forceinline__ void clean_event(const uint32_t e, const int P, const EventArrays& ev,
                                            RedScratch<NT>& red, const RtaCamera& cam,
                                            const RtaImageOut& out) {
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const float thr_p = cam.thr_picture, thr_b = cam.thr_boundary;

  // keep[p] = core[p] and some neighbour is core (isolated core pixels drop)
  int any_keep = 0;
  for (int p = tid; p < P; p += NT) {
    bool k = false;
    if (ev.q[p] >= thr_p) {
      const int32_t* nb = cam.neighbors + 6u * (size_t)p;
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        const int n = __ldg(nb + j);
        if ((unsigned)n < (unsigned)P && ev.q[n] >= thr_p) k = true;
      }
    }
    ev.keep[p] = k ? 1 : 0;
    any_keep |= k ? 1 : 0;
  }
  any_keep = __syncthreads_or(any_keep);
  uint8_t* mrow = out.mask ? out.mask + (size_t)e * (size_t)P : nullptr;
  if (!any_keep) {  // no surviving core pixel: the mask is empty
    if (mrow)
      for (int p = tid; p < P; p += NT) mrow[p] = 0;
    if (tid == 0) store_empty(e, 0, out);
    return;
  }

  // mask[p] = keep[p] or (q[p] >= thr_boundary and some neighbour is kept); pass 1 sums
  int n = 0;
  double s0 = 0.0, sx = 0.0, sy = 0.0, st = 0.0;
  float qm = -INFINITY;
  for (int p = tid; p < P; p += NT) {
    const float q = ev.q[p];
    bool m = ev.keep[p] != 0;
    if (!m && q >= thr_b) {
      const int32_t* nb = cam.neighbors + 6u * (size_t)p;
#pragma unroll
      for (int j = 0; j < 6; ++j) {
        const int nn = __ldg(nb + j);
        if ((unsigned)nn < (unsigned)P && ev.keep[nn] != 0) m = true;
      }
    }
    ev.mask[p] = m ? 1 : 0;
    if (mrow) mrow[p] = m ? 1 : 0;
    if (m) {
      const double w = (double)q;
      ++n;
      s0 += w;
      sx += w * (double)__ldg(cam.pix_x + p);
      sy += w * (double)__ldg(cam.pix_y + p);
      st += w * (double)ev.t[p];
      qm = fmaxf(qm, q);
    }
  }
  if (__any_sync(0xFFFFFFFFu, n > 0)) {
    n = __reduce_add_sync(0xFFFFFFFFu, n);
    s0 = warp_sum(s0), sx = warp_sum(sx), sy = warp_sum(sy), st = warp_sum(st);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) qm = fmaxf(qm, __shfl_xor_sync(0xFFFFFFFFu, qm, o));
  }
  if (lane == 0) {
    red.a[warp][0] = s0, red.a[warp][1] = sx, red.a[warp][2] = sy, red.a[warp][3] = st;
    red.n[warp] = n;
    red.qmax[warp] = qm;
  }
  __syncthreads();
  n = 0, s0 = sx = sy = st = 0.0, qm = -INFINITY;
#pragma unroll
  for (int w = 0; w < NT / 32; ++w) {
    n += red.n[w];
    s0 += red.a[w][0], sx += red.a[w][1], sy += red.a[w][2], st += red.a[w][3];
    qm = fmaxf(qm, red.qmax[w]);
  }
  if (!(s0 > 0.0)) {  // non-positive (or NaN) total charge: parameters are zero, the count stands
    if (tid == 0) store_empty(e, n, out);
    return;
  }
  const double cx = sx / s0, cy = sy / s0;

  // pass 2: centred second moments over the mask
  double sxx = 0.0, syy = 0.0, sxy = 0.0;
  bool mine = false;
  for (int p = tid; p < P; p += NT) {
    if (ev.mask[p]) {
      const double w = (double)ev.q[p];
      const double dx = (double)__ldg(cam.pix_x + p) - cx, dy = (double)__ldg(cam.pix_y + p) - cy;
      sxx += w * dx * dx;
      syy += w * dy * dy;
      sxy += w * dx * dy;
      mine = true;
    }
  }
  if (__any_sync(0xFFFFFFFFu, mine)) sxx = warp_sum(sxx), syy = warp_sum(syy), sxy = warp_sum(sxy);
  if (lane == 0) red.b[warp][0] = sxx, red.b[warp][1] = syy, red.b[warp][2] = sxy;
  __syncthreads();
  if (tid == 0) {
    sxx = syy = sxy = 0.0;
#pragma unroll
    for (int w = 0; w < NT / 32; ++w) sxx += red.b[w][0], syy += red.b[w][1], sxy += red.b[w][2];
    sxx /= s0, syy /= s0, sxy /= s0;
    const double d = sxx - syy;
    const double z = sqrt(d * d + 4.0 * sxy * sxy);
    const double l2 = 0.5 * (sxx + syy + z);
    double w2 = 0.5 * (sxx + syy - z);
    if (w2 < 0.0) w2 = 0.0;
    out.n_pix[e] = n;
    float* o = out.params + (size_t)e * 8u;
    o[0] = (float)s0;
    o[1] = (float)cx;
    o[2] = (float)cy;
    o[3] = (float)sqrt(l2);
    o[4] = (float)sqrt(w2);
    o[5] = (float)(0.5 * atan2(2.0 * sxy, d));
    o[6] = (float)(st / s0);
    o[7] = qm;
  }
}

// ------------------------------------------------ cleaning on HBM arrays ----
template <int NT>
__global__ void __launch_bounds__(NT)
    image_moments_kernel(const float* __restrict__ charge, const float* __restrict__ time,
                         const uint32_t n_events, const int P,
                         const __grid_constant__ RtaCamera cam,
                         const __grid_constant__ RtaImageOut out) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ RedScratch<NT> red;
  const EventArrays ev(smem, P);
  const int tid = threadIdx.x;
  for (uint32_t e = blockIdx.x; e < n_events; e += gridDim.x) {
    const float* q = charge + (size_t)e * (size_t)P;
    const float* t = time + (size_t)e * (size_t)P;
    if ((((uintptr_t)q | (uintptr_t)t) & 15u) == 0) {
      const int n4 = P >> 2;
      for (int i = tid; i < n4; i += NT) {
        reinterpret_cast<float4*>(ev.q)[i] = __ldcs(reinterpret_cast<const float4*>(q) + i);
        reinterpret_cast<float4*>(ev.t)[i] = __ldcs(reinterpret_cast<const float4*>(t) + i);
      }
      for (int p = 4 * n4 + tid; p < P; p += NT) ev.q[p] = __ldcs(q + p), ev.t[p] = __ldcs(t + p);
    } else {
      for (int p = tid; p < P; p += NT) ev.q[p] = __ldcs(q + p), ev.t[p] = __ldcs(t + p);
    }
    __syncthreads();
    clean_event<NT>(e, P, ev, red, cam, out);
  }
}

// ----------------------------------------- extraction + cleaning, generic ----
template <int NT>
__global__ void __launch_bounds__(NT)
    extract_image_generic_kernel(const uint8_t* __restrict__ wf, const uint32_t n_events,
                                 const int P, const int S, const int W,
                                 const int* __restrict__ pedestal, const float* __restrict__ gain,
                                 const __grid_constant__ RtaCamera cam,
                                 const __grid_constant__ RtaImageOut out) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ RedScratch<NT> red;
  const EventArrays ev(smem, P);
  const ModeArgs ma = {};
  for (uint32_t e = blockIdx.x; e < n_events; e += gridDim.x) {
    const uint8_t* base = wf + (size_t)e * (size_t)P * (size_t)S * 2u;
    for (int p = threadIdx.x; p < P; p += NT) {
      const GlobalTrace<16> tr(base, (uint32_t)p, S);
      const Result r = generic_trace<MODE_SLIDING, 16>(tr, S, W, (uint32_t)p, pedestal, gain, ma);
      ev.q[p] = r.charge;
      ev.t[p] = r.time;
    }
    __syncthreads();
    clean_event<NT>(e, P, ev, red, cam, out);
  }
}

// ------------------------------------------- extraction + cleaning, staged ----
// Work items of a CTA: (event, tile) pairs, tiles 0 .. nt-1 of one event, then
// the next event drawn from the shared counter. The producer side runs STAGES
// items ahead of the consumer through item_q, across event boundaries.
template <class C>
__global__ void __launch_bounds__(C::NT)
    extract_image_kernel(const uint8_t* __restrict__ wf, const uint32_t n_events, const int P,
                         const int* __restrict__ pedestal, const float* __restrict__ gain,
                         const __grid_constant__ RtaCamera cam,
                         const __grid_constant__ RtaImageOut out, uint32_t* __restrict__ sched) {
  static_assert(C::BITS == 16 && C::STAGES >= 2, "uint16 samples, at least two stages");
  // an event may start at any multiple of VEC bytes: the copy starts at the
  // 16-byte boundary below it, so a stage holds up to 16 bytes more than a tile
  constexpr int STG = C::STAGE_BYTES + 16;
  constexpr uint32_t TRACE_BYTES = C::TRACE_BITS / 8;
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[C::STAGES];
  constexpr int QN = C::STAGES + 1;
  __shared__ uint2 item_q[QN];  // {event, tile}
  __shared__ RedScratch<C::NT> red;
  const int tid = threadIdx.x;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_u32(full_bar);
  const EventArrays ev(smem + C::STAGES * STG, P);
  const ModeArgs ma = {};
  const uint32_t nt = ((uint32_t)P + C::TILE_TRACES - 1u) / C::TILE_TRACES;  // tiles per event
  const unsigned long long EB = (unsigned long long)P * TRACE_BYTES;         // bytes per event
  const unsigned long long total = (unsigned long long)n_events * EB;

  // thread 0: the producer cursor (pev, pt) and one prefetched event index
  uint32_t pev = blockIdx.x, pt = 0, pre_ev = 0xFFFFFFFFu;
  auto fetch_event = [&]() -> uint32_t {
    if (sched == nullptr)
      return (pev > 0xFFFFFFFFu - gridDim.x) ? 0xFFFFFFFFu : pev + gridDim.x;
    const uint32_t got = pre_ev;
    const uint32_t k = atomicAdd(sched, 1u);
    pre_ev = (k > 0xFFFFFFFFu - gridDim.x) ? 0xFFFFFFFFu : gridDim.x + k;
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
      pre_ev = (k > 0xFFFFFFFFu - gridDim.x) ? 0xFFFFFFFFu : gridDim.x + k;
    }
#pragma unroll
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(bar_base + 8 * s, C::PAD ? C::NT : 1);
      item_q[s] = next_item();
    }
    fence_mbar_init();
  }
  __syncthreads();

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
      for (uint32_t c = tid; c < bytes / 16u; c += C::NT) {
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

  for (uint32_t j = 0;; ++j) {
    const uint2 it = item_q[j % QN];
    if (it.x >= n_events) break;  // event indices grow per CTA: nothing later is valid either
    const int stage = (int)(j % C::STAGES);
    const uint32_t parity = (j / C::STAGES) & 1u;
    if (tid == 0) item_q[(j + C::STAGES) % QN] = next_item();
    mbar_wait(bar_base + 8 * stage, parity);
    const uint32_t p0 = it.y * C::TILE_TRACES + (uint32_t)tid * C::TPT;
    if (p0 < (uint32_t)P) {
      uint32_t mis = 0;
      if constexpr (!C::PAD)
        mis = (uint32_t)(((unsigned long long)it.x * EB + (unsigned long long)it.y * C::TILE_BYTES) & 15u);
      const uint8_t* unit = smem + stage * STG + mis + tid * C::UNIT_STRIDE;
      Result res[C::TPT];
      compute_results<C, MODE_SLIDING>(unit, p0, 0u, pedestal, gain, ma, res);
#pragma unroll
      for (int i = 0; i < C::TPT; ++i) {
        if (p0 + i < (uint32_t)P) {
          ev.q[p0 + i] = res[i].charge;
          ev.t[p0 + i] = res[i].time;
        }
      }
    }
    __syncthreads();  // the stage is free, the item slot is published, ev.q / ev.t are visible
    const uint2 nxt = item_q[(j + C::STAGES) % QN];
    if (nxt.x < n_events) issue(nxt, stage);
    if (it.y + 1u == nt) clean_event<C::NT>(it.x, P, ev, red, cam, out);
  }

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

// The staged kernel takes a shape when every event starts on a boundary its
// units can be read from (VEC bytes; whole units per event) and the per-event
// arrays fit behind the ring.
template <class C>
bool staged_ok(int32_t P) {
  const size_t eb = (size_t)P * (C::TRACE_BITS / 8);
  if (P % C::TPT != 0 || eb % C::VEC != 0) return false;
  if (C::PAD && eb % 16 != 0) return false;
  return C::STAGES * (size_t)(C::STAGE_BYTES + 16) + image_smem_bytes(P) <= kSmemLimit;
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
    const size_t smem = C::STAGES * (size_t)(C::STAGE_BYTES + 16) + image_smem_bytes(P);
    // the dynamic shared-memory size depends on n_pixels: set per launch (cheap)
    e = cudaFuncSetAttribute(extract_image_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                             (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, extract_image_kernel<C>, C::NT, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    uint32_t grid = (uint32_t)(sms * occ);
    if (grid > n_events) grid = n_events;
    uint32_t* sched = rta_static_schedule() ? nullptr : rta_sched_words(dev, stream);
    extract_image_kernel<C><<<grid, C::NT, smem, stream>>>(wf, n_events, P, pedestal, gain, cam,
                                                           out, sched);
    rta_count_launch();
    return cudaGetLastError();
  }
};

template <class K>
cudaError_t launch_per_event(K kernel, size_t smem, uint32_t n_events, int* grid_out) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = rta_device_sms(dev, &sms)) != cudaSuccess) return e;
  if (smem > kSmemLimit) return cudaErrorInvalidValue;
  e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, kGenericNT, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  uint32_t grid = (uint32_t)(sms * occ);
  if (grid > n_events) grid = n_events;
  *grid_out = (int)grid;
  return cudaSuccess;
}

}  // namespace

int32_t rta_image_pixel_limit() {
  // charge + time + two flag bytes per pixel must fit one CTA's shared memory,
  // next to 1 KB of static scratch (reduction partials) and the rounding of
  // the four arrays to 16 bytes
  return (int32_t)((kSmemLimit - 1024u - 64u) / 10u);
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
  const size_t smem = image_smem_bytes(n_pixels);
  int grid = 0;
  cudaError_t e = launch_per_event(image_moments_kernel<kGenericNT>, smem, (uint32_t)n_events, &grid);
  if (e != cudaSuccess) return e;
  image_moments_kernel<kGenericNT><<<grid, kGenericNT, smem, stream>>>(
      charge, time, (uint32_t)n_events, n_pixels, cam, out);
  rta_count_launch();
  return cudaGetLastError();
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
  const size_t smem = image_smem_bytes(n_pixels);
  int grid = 0;
  cudaError_t e =
      launch_per_event(extract_image_generic_kernel<kGenericNT>, smem, (uint32_t)n_events, &grid);
  if (e != cudaSuccess) return e;
  extract_image_generic_kernel<kGenericNT><<<grid, kGenericNT, smem, stream>>>(
      w, (uint32_t)n_events, n_pixels, S, W, pedestal, gain, cam, out);
  rta_count_launch();
  return cudaGetLastError();
}
