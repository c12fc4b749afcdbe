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
//  * clean_event: ONE WARP cleans one event. The image is sparse (a few per
//    cent of the pixels pass a threshold), so the work is organised around bit
//    masks of the camera (one bit per pixel) and compacted pixel lists. When
//    the neighbour table is symmetric (checked by every CTA when it starts,
//    6 P look-ups spread over its threads) one pass over the core pixels does
//    both cleaning steps: a core pixel with a core neighbour is kept and marks
//    those of its neighbours that pass the boundary threshold; otherwise the
//    two steps of the definition are run as written (pull, two lists). The
//    moments are ONE pass over the list of mask pixels, about the first mask
//    pixel as origin (fp64, per-lane partial sums in list order, xor butterfly:
//    no floating-point atomics, run-to-run deterministic). The scalar tail
//    (divisions, square roots, atan2) is not run per event: each event's sums
//    are parked in the registers of one lane and 32 events are finished at
//    once, one event per lane.
//  * extract_image_kernel<C, G> (fused, staged): ONE persistent CTA per SM.
//    G groups of NT extraction threads each stream tiles of the CTA's current
//    events through their own TMA / cp.async stage ring and write charge, peak
//    time and threshold bits into one of NB per-event buffers in shared memory
//    instead of HBM; NC cleaning warps take finished buffers (mbarrier
//    hand-off: ready[b] counts one arrival per warp and tile, free[b] one per
//    cleaned event). HBM traffic: the waveform bytes once in, 36 bytes per
//    event out (+ 1 byte per pixel if the mask is asked for).
//  * extract_image_generic_kernel: one cleaning warp beside 256 extraction
//    threads (named barriers) for any (S, W), camera size and 2-byte alignment;
//    traces are read straight from global memory.
//  * image_moments_kernel: charge / time arrays already in HBM (rta_extract's
//    outputs); one warp per event builds the threshold bits from one coalesced
//    sweep over the charge row and gathers charge and peak time of the mask
//    pixels from L2.
#include "rta_device.cuh"

#include <atomic>
#include <mutex>

// most warps per CTA of image_moments_kernel (the launch bound caps the registers
// per thread at 65536 / (32 warps))
#ifndef RTA_MOM_WARPS
#define RTA_MOM_WARPS 24
#endif
// how the fused kernels form the arg-max keys (compute_results KEYMUL): 1 = IMAD
// with a constant-bank multiplier (fma pipe); these kernels are alu-pipe-bound
#ifndef RTA_IMG_KEYMODE
#define RTA_IMG_KEYMODE 1
#endif

namespace {

__device__ __forceinline__ void named_sync(const int id, const int n) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory");
}
__device__ __forceinline__ void named_arrive(const int id, const int n) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}

// wait with back-off: for warps that are idle most of the time (the spin of
// mbar_wait would take issue slots from the extraction warps)
__device__ __forceinline__ void mbar_wait_idle(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  for (;;) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    if (ok) break;
    __nanosleep(256);
  }
}

__host__ __device__ constexpr size_t r16(size_t n) { return (n + 15u) & ~(size_t)15u; }
__host__ __device__ constexpr size_t mask_words(int P) { return ((size_t)P + 31u) >> 5; }

// What the producer of an event hands to clean_event: charges, peak times and
// the two threshold bit masks, bit p & 31 of word p >> 5 (bits past P are 0).
struct EventBuf {
  float* q;          // [P]
  float* t;          // [P]
  uint32_t* core_w;  // q >= thr_picture
  uint32_t* low_w;   // q >= thr_boundary
  static __host__ __device__ size_t bytes(int P) {
    return 2u * r16(4u * (size_t)P) + 2u * r16(4u * mask_words(P));
  }
  __device__ __forceinline__ EventBuf(uint8_t* base, const int P) {
    q = reinterpret_cast<float*>(base);
    base += r16(4u * (size_t)P);
    t = reinterpret_cast<float*>(base);
    base += r16(4u * (size_t)P);
    core_w = reinterpret_cast<uint32_t*>(base);
    low_w = reinterpret_cast<uint32_t*>(base + r16(4u * mask_words(P)));
  }
};

// The same for the staged fused kernel, whose extraction threads hand over the start t* of
// the winning window instead of the peak time (TimeFromWaveform): one byte per pixel
// (n_samples <= 256), so that more event buffers fit behind the stage rings.
struct EventBuf8 {
  float* q;          // [P]
  uint8_t* tstar;    // [P]
  uint32_t* core_w;
  uint32_t* low_w;
  static __host__ __device__ size_t bytes(int P) {
    return r16(4u * (size_t)P) + r16((size_t)P) + 2u * r16(4u * mask_words(P));
  }
  __device__ __forceinline__ EventBuf8(uint8_t* base, const int P) {
    q = reinterpret_cast<float*>(base);
    base += r16(4u * (size_t)P);
    tstar = base;
    base += r16((size_t)P);
    core_w = reinterpret_cast<uint32_t*>(base);
    low_w = reinterpret_cast<uint32_t*>(base + r16(4u * mask_words(P)));
  }
};

// Scratch owned by a cleaning warp: keep / mask bit words and one pixel list of
// `cap` entries (cap >= 384 = 32 lanes x 12 words, the most one lane's run of
// words can hold for P <= 12288). A list longer than cap is produced and
// consumed in rounds (compact_bits); sparse images need one round.
struct CleanScratch {
  uint32_t* keep_w;
  uint32_t* mask_w;
  uint16_t* list;  // [cap], pixel indices (< 2^16: rta_image_pixel_limit)
  int cap;
  static __host__ __device__ size_t bytes(int P, int cap) {
    return 2u * r16(4u * mask_words(P)) + r16(2u * (size_t)cap);
  }
  __device__ __forceinline__ CleanScratch(uint8_t* base, const int P, const int cap_) : cap(cap_) {
    keep_w = reinterpret_cast<uint32_t*>(base);
    mask_w = reinterpret_cast<uint32_t*>(base + r16(4u * mask_words(P)));
    list = reinterpret_cast<uint16_t*>(base + 2u * r16(4u * mask_words(P)));
  }
};
constexpr int kListCapMin = 512;

// Pixel indices of the set bits of word(w), w = w_begin .. NW-1, in ascending
// order into list[], at most `cap` of them; returns their number (same value in
// every lane) and moves w_begin to the first word not covered (NW when done).
// One warp: lane l owns the K = ceil(NW / 32) consecutive words from
// w_begin + l K, so one prefix sum over the lanes' bit counts places every
// lane's run; a round ends before the first lane whose run would pass `cap`
// (cap >= 32 K, so every round covers at least lane 0's words).
template <class F>
__device__ __forceinline__ int compact_bits(const int NW, int& w_begin, uint16_t* __restrict__ list,
                                            const int cap, F word) {
  const int lane = threadIdx.x & 31;
  if (NW <= 64 && w_begin == 0) {
    // cameras of up to 2048 pixels (every BASELINE shape): lane l owns words 2 l and 2 l + 1,
    // read once into registers; one round unless the list is too short for the bits
    const int w0 = 2 * lane;
    uint32_t b0 = w0 < NW ? word(w0) : 0u, b1 = w0 + 1 < NW ? word(w0 + 1) : 0u;
    const int c = __popc(b0) + __popc(b1);
    int incl = c;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
      if (lane >= o) incl += v;
    }
    const int total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    if (total <= cap) {
      int off = incl - c;
      const int base = 64 * lane;
      while (b0) {
        const int b = __ffs((int)b0) - 1;
        b0 &= b0 - 1u;
        list[off++] = (uint16_t)(base + b);
      }
      while (b1) {
        const int b = __ffs((int)b1) - 1;
        b1 &= b1 - 1u;
        list[off++] = (uint16_t)(base + 32 + b);
      }
      w_begin = NW;
      __syncwarp();
      return total;
    }
  }
  const int K = (NW + 31) >> 5;
  const int w_lo = min(w_begin + lane * K, NW), w_hi = min(w_lo + K, NW);
  int c = 0;
  for (int w = w_lo; w < w_hi; ++w) c += __popc(word(w));
  int incl = c;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, o);
    if (lane >= o) incl += v;
  }
  const uint32_t over = __ballot_sync(0xFFFFFFFFu, incl > cap);
  const int n_lanes = over ? __ffs((int)over) - 1 : 32;  // lanes whose runs fit
  if (lane < n_lanes) {
    int off = incl - c;
    for (int w = w_lo; w < w_hi; ++w) {
      uint32_t bits = word(w);
      while (bits) {
        const int b = __ffs((int)bits) - 1;
        bits &= bits - 1u;
        list[off++] = (uint16_t)(32 * w + b);
      }
    }
  }
  const int total = __shfl_sync(0xFFFFFFFFu, incl, max(n_lanes, 1) - 1);
  w_begin = min(w_begin + n_lanes * K, NW);
  __syncwarp();
  return n_lanes ? total : 0;
}

__device__ __forceinline__ bool test_bit(const uint32_t* w, const int n) {
  return (w[n >> 5] >> (n & 31)) & 1u;
}

// The neighbour table as the cleaning code reads it: the caller's int32 [P][6]
// in global memory, or a copy as uint16 [P][6] in shared memory (0xFFFF = none;
// 12 bytes per pixel) that the CTA makes when it starts and there is room.
struct NbrTable {
  const int32_t* g;    // global, as given
  const uint16_t* s;   // shared copy, or nullptr
  bool g8;             // g is 8-byte aligned: a 24-byte row is three 8-byte loads
  __device__ __forceinline__ void row(const int p, int (&nb)[6]) const {
    if (s != nullptr) {
      const uint32_t* r = reinterpret_cast<const uint32_t*>(s + 6 * p);  // 12 p: word aligned
#pragma unroll
      for (int j = 0; j < 3; ++j) {
        const uint32_t v = r[j];
        nb[2 * j] = (int)(v & 0xFFFFu), nb[2 * j + 1] = (int)(v >> 16);
      }
    } else {
      const int32_t* r = g + 6u * (size_t)p;
      if (g8) {
#pragma unroll
        for (int j = 0; j < 3; ++j) {
          const int2 v = __ldg(reinterpret_cast<const int2*>(r) + j);
          nb[2 * j] = v.x, nb[2 * j + 1] = v.y;
        }
      } else {
#pragma unroll
        for (int j = 0; j < 6; ++j) nb[j] = __ldg(r + j);
      }
    }
  }
};

// For the n listed pixels: hit = some neighbour's bit is set in in_w; hits set
// the pixel's bit in out_w. Two list entries per lane are in flight at once
// (their neighbour rows are loaded before any is used). Returns "any hit" per lane.
__device__ __forceinline__ int neighbour_pass(const int n, const uint16_t* __restrict__ list,
                                              const NbrTable& nbr, const int P,
                                              const uint32_t* in_w, uint32_t* out_w) {
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
    for (int u = 0; u < U; ++u)
      if (p[u] >= 0) nbr.row(p[u], nb[u]);
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

// Peak time of pixel p for the moment sums: from an array, or recomputed from the
// waveform for the fused staged kernel, whose extraction threads leave step a7
// out (only the few mask pixels of an event ever need a peak time; the samples
// are still in L2). tstar[p] holds t*; the same finish_trace as in
// the extraction gives the same bits.
struct TimeFromArray {
  const float* t;
  __device__ __forceinline__ float operator()(const int p) const { return t[p]; }
};
struct TimeFromWaveform {
  const uint16_t* wf;  // the event's first sample (global memory)
  const uint8_t* tstar;  // [P], t*
  const int* pedestal;
  const float* gain;
  int S, W;
  __device__ __forceinline__ float operator()(const int p) const {
    const int ts = (int)tstar[p];
    const uint16_t* x = wf + (size_t)p * (size_t)S + ts;
    int rawsum = 0, relnum = 0;
    for (int k = 0; k < W; ++k) {
      const int v = (int)__ldg(x + k);
      rawsum += v;
      relnum += k * v;
    }
    return finish_trace(W, rawsum, ts, relnum, __ldg(pedestal + p), __ldg(gain + p), W,
                        (W * (W - 1)) / 2).time;
  }
};

// "q[n] >= thr_boundary" for the symmetric pass: from the bit mask the producer
// of the event made, or straight from a charge row in shared memory (the
// moments kernel, which then never builds that mask for a symmetric table).
struct LowFromBits {
  const uint32_t* low_w;
  __device__ __forceinline__ bool operator()(const int n) const { return test_bit(low_w, n); }
};
struct LowFromRow {
  const float* row;
  float thr;
  __device__ __forceinline__ bool operator()(const int n) const { return row[n] >= thr; }
};

// Symmetric neighbour table (p in nbr[n] whenever n in nbr[p]): "n has a kept
// neighbour" is the same as "a kept pixel lists n", so one pass over the core
// pixels does both steps of the cleaning. A core pixel with a core neighbour is
// kept: its own bit goes into mask_w, and so does every neighbour that passes
// the boundary threshold. Returns "any pixel kept" per lane.
// Two forms with the same result. One pass (symmetric_pass_one): every core pixel tests its
// neighbours for both thresholds at once: the shorter chain of dependent steps, which is
// what the fused kernels' few cleaning warps are bound by (their table is in global
// memory). Two phases (symmetric_pass): fewer instructions (the boundary tests run for the
// kept pixels only), which is what image_moments_kernel is bound by (measured both ways).
template <class Low>
__device__ __forceinline__ int symmetric_pass_one(const int n, const uint16_t* __restrict__ list,
                                              const NbrTable& nbr, const int P,
                                              const uint32_t* core_w, const Low& low,
                                              uint32_t* mask_w) {
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
    for (int u = 0; u < U; ++u)
      if (p[u] >= 0) nbr.row(p[u], nb[u]);
#pragma unroll
    for (int u = 0; u < U; ++u) {
      if (p[u] >= 0) {
        bool hit = false;
        uint32_t lw[6];
#pragma unroll
        for (int j = 0; j < 6; ++j) {
          const bool ok = (unsigned)nb[u][j] < (unsigned)P;
          const int m = ok ? nb[u][j] : 0;
          const uint32_t bit = ok ? (1u << (m & 31)) : 0u;
          if (core_w[m >> 5] & bit) hit = true;
          lw[j] = (ok && low(m)) ? bit : 0u;
        }
        if (hit) {
          atomicOr(&mask_w[p[u] >> 5], 1u << (p[u] & 31));
#pragma unroll
          for (int j = 0; j < 6; ++j)
            if (lw[j]) atomicOr(&mask_w[nb[u][j] >> 5], lw[j]);
          any = 1;
        }
      }
    }
  }
  __syncwarp();
  return any;
}

template <class Low>
__device__ __forceinline__ int symmetric_pass(const int n, uint16_t* __restrict__ list,
                                              const NbrTable& nbr, const int P,
                                              const uint32_t* core_w, const Low& low,
                                              uint32_t* mask_w) {
  const int lane = threadIdx.x & 31;
  const uint32_t lt = (1u << lane) - 1u;
  constexpr int U = 2;
  // Phase A: which core pixels have a core neighbour? Those are kept: their own mask bit is
  // set and they move to the front of the list (most core pixels of a sparse image are
  // isolated noise, so the boundary tests and mask updates below run for a few entries only).
  int n_kept = 0;
  for (int i0 = 0; i0 < n; i0 += 32 * U) {
    int p[U];
    bool hit[U];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = i0 + 32 * u + lane;
      p[u] = i < n ? (int)list[i] : -1;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      hit[u] = false;
      if (p[u] >= 0) {
        int nb[6];
        nbr.row(p[u], nb);
#pragma unroll
        for (int j = 0; j < 6; ++j) {
          const bool ok = (unsigned)nb[j] < (unsigned)P;
          const int m = ok ? nb[j] : 0;
          if (ok && ((core_w[m >> 5] >> (m & 31)) & 1u)) hit[u] = true;
        }
      }
    }
    __syncwarp();  // every entry of the round has been read: the front of the list may be rewritten
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const uint32_t bal = __ballot_sync(0xFFFFFFFFu, hit[u]);
      if (hit[u]) {
        list[n_kept + __popc(bal & lt)] = (uint16_t)p[u];
        atomicOr(&mask_w[p[u] >> 5], 1u << (p[u] & 31));
      }
      n_kept += __popc(bal);
    }
  }
  __syncwarp();
  // Phase B: every kept pixel marks those of its neighbours that pass the boundary threshold.
  for (int i = lane; i < n_kept; i += 32) {
    const int p = (int)list[i];
    int nb[6];
    nbr.row(p, nb);
#pragma unroll
    for (int j = 0; j < 6; ++j) {
      const bool ok = (unsigned)nb[j] < (unsigned)P;
      const int m = ok ? nb[j] : 0;
      if (ok && low(m)) atomicOr(&mask_w[m >> 5], 1u << (m & 31));
    }
  }
  __syncwarp();
  return n_kept;  // the same in every lane
}

// Every thread of the CTA: is the neighbour table symmetric? One (pixel, slot)
// entry per thread and step, four steps' loads in flight at once; the answer
// is the same in every thread. Contains __syncthreads.
__device__ __forceinline__ int table_is_symmetric(const int32_t* __restrict__ nbr, const int P) {
  int ok = 1;
  const int n_entries = 6 * P;
  constexpr int U = 4;
  for (int i0 = threadIdx.x; i0 < n_entries; i0 += U * blockDim.x) {
    int n[U], r[U][6];
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int i = i0 + u * blockDim.x;
      n[u] = i < n_entries ? __ldg(nbr + i) : -1;
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int32_t* row = nbr + 6u * (size_t)((unsigned)n[u] < (unsigned)P ? n[u] : 0);
#pragma unroll
      for (int j = 0; j < 6; ++j) r[u][j] = __ldg(row + j);
    }
#pragma unroll
    for (int u = 0; u < U; ++u) {
      const int p = (i0 + u * (int)blockDim.x) / 6;
      bool back = false;
#pragma unroll
      for (int j = 0; j < 6; ++j) back |= (r[u][j] == p);
      if ((unsigned)n[u] < (unsigned)P && !back) ok = 0;
    }
  }
  return __syncthreads_and(ok);
}

// The same on a uint16 copy of the table in shared memory (complete and visible
// to the CTA; 0xFFFF = none). Contains __syncthreads.
__device__ __forceinline__ int table_is_symmetric_s16(const uint16_t* nbr, const int P) {
  int ok = 1;
  const int n_entries = 6 * P;
  for (int i = threadIdx.x; i < n_entries; i += blockDim.x) {
    const int n = nbr[i];
    if (n < P) {
      const int p = i / 6;
      const uint16_t* r = nbr + 6 * n;
      bool back = false;
#pragma unroll
      for (int j = 0; j < 6; ++j) back |= ((int)r[j] == p);
      if (!back) ok = 0;
    }
  }
  return __syncthreads_and(ok);
}

// The sums of one event (readings R33 / R34), about the origin (x0, y0).
struct EventSums {
  double s0, sx, sy, st, sxx, syy, sxy;
  float x0, y0, qm;
  int n_pix;
  uint32_t e;
};
using Pending = EventSums;  // parked in one lane until 32 events are finished together

// One lane, one event: the scalar tail of readings R33 / R34.
__device__ __forceinline__ void finish_event(const Pending& pd, const RtaImageOut& out) {
  float o[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) o[i] = 0.0f;
  if (pd.n_pix > 0 && pd.s0 > 0.0) {  // else: non-positive (or NaN) total charge, parameters are zero
    const double mx = __ddiv_rn(pd.sx, pd.s0), my = __ddiv_rn(pd.sy, pd.s0);
    // centred second moments from the ones about the origin: E[d^2] - E[d]^2
    const double sxx = __fma_rn(-mx, mx, __ddiv_rn(pd.sxx, pd.s0));
    const double syy = __fma_rn(-my, my, __ddiv_rn(pd.syy, pd.s0));
    const double sxy = __fma_rn(-mx, my, __ddiv_rn(pd.sxy, pd.s0));
    const double d = __dsub_rn(sxx, syy);
    const double z = sqrt(__fma_rn(d, d, __dmul_rn(4.0, __dmul_rn(sxy, sxy))));
    const double tr = __dadd_rn(sxx, syy);
    o[0] = (float)pd.s0;
    o[1] = (float)__dadd_rn((double)pd.x0, mx);
    o[2] = (float)__dadd_rn((double)pd.y0, my);
    o[3] = (float)sqrt(__dmul_rn(0.5, __dadd_rn(tr, z)));
    o[4] = (float)sqrt(fmax(__dmul_rn(0.5, __dsub_rn(tr, z)), 0.0));
    o[5] = (float)__dmul_rn(0.5, atan2(__dmul_rn(2.0, sxy), d));
    o[6] = (float)__ddiv_rn(pd.st, pd.s0);
    o[7] = pd.qm;
  }
  float* dst = out.params + (size_t)pd.e * 8u;
  if ((reinterpret_cast<uintptr_t>(dst) & 15u) == 0) {
    reinterpret_cast<float4*>(dst)[0] = make_float4(o[0], o[1], o[2], o[3]);
    reinterpret_cast<float4*>(dst)[1] = make_float4(o[4], o[5], o[6], o[7]);
  } else {
#pragma unroll
    for (int i = 0; i < 8; ++i) dst[i] = o[i];
  }
  out.n_pix[pd.e] = pd.n_pix;
}

__device__ __forceinline__ void flush_pending(const Pending& pd, int& n_pend,
                                              const RtaImageOut& out) {
  if ((int)(threadIdx.x & 31) < n_pend) finish_event(pd, out);
  n_pend = 0;
  __syncwarp();
}

__device__ __forceinline__ double shfl_xor_f64(const double v, const int o) {
  return __shfl_xor_sync(0xFFFFFFFFu, v, o);
}

// Cleaning and moment sums of event e (readings R31-R35), executed by one whole
// warp; the sums come back in every lane. core_w (and low_w for the general
// path) are in shared memory and complete; `low(n)` answers q[n] >= thr_boundary
// for the symmetric pass; q points at the event's charges (shared or global
// memory) and t(p) gives pixel p's peak time. `after_pass()` runs once the threshold tests are
// over (the moments kernel hands its row buffer back to the copy engine there).
template <bool TWO_PHASE, class Time, class Low, class AfterPass>
__device__ __forceinline__ void clean_event_sums(const uint32_t e, const int P, const float* q,
                                                 const Time& t, const uint32_t* core_w,
                                                 const uint32_t* low_w, const Low& low,
                                                 const CleanScratch& sc, const NbrTable& nbr,
                                                 const RtaCamera& cam, const RtaImageOut& out,
                                                 const bool symmetric, AfterPass after_pass,
                                                 EventSums& cur) {
  const int lane = threadIdx.x & 31;
  const int NW = (int)mask_words(P);
  uint8_t* mrow = out.mask ? out.mask + (size_t)e * (size_t)P : nullptr;

  cur.s0 = cur.sx = cur.sy = cur.st = cur.sxx = cur.syy = cur.sxy = 0.0;
  cur.x0 = cur.y0 = cur.qm = 0.0f;
  cur.n_pix = 0;
  cur.e = e;

  int kept = 0;
  if (symmetric) {
    for (int w = lane; w < NW; w += 32) sc.mask_w[w] = 0u;
    __syncwarp();
    for (int wb = 0; wb < NW;) {
      const int n_core = compact_bits(NW, wb, sc.list, sc.cap, [&](int w) { return core_w[w]; });
      kept |= TWO_PHASE ? symmetric_pass(n_core, sc.list, nbr, P, core_w, low, sc.mask_w)
                        : symmetric_pass_one(n_core, sc.list, nbr, P, core_w, low, sc.mask_w);
    }
  } else {
    // keep[p] = core[p] and some neighbour is core (isolated core pixels drop)
    for (int w = lane; w < NW; w += 32) sc.keep_w[w] = 0u;
    __syncwarp();
    for (int wb = 0; wb < NW;) {
      const int n_core = compact_bits(NW, wb, sc.list, sc.cap, [&](int w) { return core_w[w]; });
      kept |= neighbour_pass(n_core, sc.list, nbr, P, core_w, sc.keep_w);
    }
  }
  kept = __any_sync(0xFFFFFFFFu, kept);
  if (kept && !symmetric) {
    // mask[p] = keep[p] or (q[p] >= thr_boundary and some neighbour is kept)
    for (int w = lane; w < NW; w += 32) sc.mask_w[w] = sc.keep_w[w];
    __syncwarp();
    for (int wb = 0; wb < NW;) {
      const int n_cand = compact_bits(NW, wb, sc.list, sc.cap,
                                      [&](int w) { return low_w[w] & ~sc.keep_w[w]; });
      neighbour_pass(n_cand, sc.list, nbr, P, sc.keep_w, sc.mask_w);
    }
  }
  after_pass();
  if (kept) {
    if (mrow)
      for (int p = lane; p < P; p += 32) mrow[p] = test_bit(sc.mask_w, p) ? 1 : 0;

    // one pass over the mask pixels in ascending pixel order: in every round lane i
    // takes entries i, i + 32, ...; origin = the first mask pixel
    float qm = -INFINITY, x0 = 0.0f, y0 = 0.0f;
    double X0 = 0.0, Y0 = 0.0;
    double s0 = 0.0, sx = 0.0, sy = 0.0, st = 0.0, sxx = 0.0, syy = 0.0, sxy = 0.0;
    int n_pix = 0;
    for (int wb = 0; wb < NW;) {
      const int n = compact_bits(NW, wb, sc.list, sc.cap, [&](int w) { return sc.mask_w[w]; });
      // lane i's first entry of the round is entry i: its loads go out before anything
      // waits, and lane 0's coordinates become the origin in the first non-empty round
      int p = lane < n ? (int)sc.list[lane] : 0;
      float qp = 0.0f, tp = 0.0f, xp = 0.0f, yp = 0.0f;
      if (lane < n) qp = q[p], tp = t(p), xp = __ldg(cam.pix_x + p), yp = __ldg(cam.pix_y + p);
      if (n_pix == 0 && n > 0) {
        x0 = __shfl_sync(0xFFFFFFFFu, xp, 0), y0 = __shfl_sync(0xFFFFFFFFu, yp, 0);
        X0 = (double)x0, Y0 = (double)y0;
      }
      n_pix += n;
      for (int i = lane; i < n; i += 32) {
        if (i != lane) {
          p = sc.list[i];
          qp = q[p], tp = t(p), xp = __ldg(cam.pix_x + p), yp = __ldg(cam.pix_y + p);
        }
        const double w = (double)qp;
        const double dx = __dsub_rn((double)xp, X0);
        const double dy = __dsub_rn((double)yp, Y0);
        const double wx = __dmul_rn(w, dx), wy = __dmul_rn(w, dy);
        s0 = __dadd_rn(s0, w);
        sx = __dadd_rn(sx, wx);
        sy = __dadd_rn(sy, wy);
        sxx = __fma_rn(wx, dx, sxx);
        syy = __fma_rn(wy, dy, syy);
        sxy = __fma_rn(wx, dy, sxy);
        qm = fmaxf(qm, qp);
        st = __fma_rn(w, (double)tp, st);  // last: the peak time comes from furthest away
      }
      __syncwarp();  // the list is rewritten by the next round
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      s0 = __dadd_rn(s0, shfl_xor_f64(s0, o));
      sx = __dadd_rn(sx, shfl_xor_f64(sx, o));
      sy = __dadd_rn(sy, shfl_xor_f64(sy, o));
      sxx = __dadd_rn(sxx, shfl_xor_f64(sxx, o));
      syy = __dadd_rn(syy, shfl_xor_f64(syy, o));
      sxy = __dadd_rn(sxy, shfl_xor_f64(sxy, o));
      qm = fmaxf(qm, __shfl_xor_sync(0xFFFFFFFFu, qm, o));
      st = __dadd_rn(st, shfl_xor_f64(st, o));
    }
    cur.s0 = s0, cur.sx = sx, cur.sy = sy, cur.st = st;
    cur.sxx = sxx, cur.syy = syy, cur.sxy = sxy;
    cur.x0 = x0, cur.y0 = y0, cur.qm = qm;
    cur.n_pix = n_pix;
  } else if (mrow) {  // no surviving core pixel: the mask is empty
    for (int p = lane; p < P; p += 32) mrow[p] = 0;
  }
}

// The fused kernels' cleaning warps: threshold masks from the producer, the
// neighbour table in global memory, sums parked in lane n_pend's `pd`; after 32
// events the warp finishes them together.
template <class Time>
__device__ __forceinline__ void clean_event(const uint32_t e, const int P, const float* q,
                                            const Time& t, const uint32_t* core_w,
                                            const uint32_t* low_w, const CleanScratch& sc,
                                            const RtaCamera& cam, const RtaImageOut& out,
                                            const bool symmetric, Pending& pd, int& n_pend) {
  const NbrTable nbr{cam.neighbors, nullptr, (reinterpret_cast<uintptr_t>(cam.neighbors) & 7u) == 0};
  EventSums cur;
  clean_event_sums<false>(e, P, q, t, core_w, low_w, LowFromBits{low_w}, sc, nbr, cam, out, symmetric,
                   [] {}, cur);
  if ((int)(threadIdx.x & 31) == n_pend) pd = cur;
  if (++n_pend == 32) flush_pending(pd, n_pend, out);
}

// ------------------------------------------------ cleaning on HBM arrays ----
// One warp per event, one persistent CTA per SM, as many warps as shared memory
// holds (about 20 for an 1800-pixel camera).
//  * Every warp owns a row buffer that ONE bulk copy (TMA, mbarrier complete_tx)
//    fills with the charge row of the warp's next event while the warp is still
//    cleaning the current one: the row loads of all warps are always in flight
//    and no warp spends issue slots or a DRAM latency on them. Rows start at any
//    multiple of 4 bytes: the copy starts at the 16-byte boundary below the row
//    (the row lands `mis` bytes into the buffer) and stops at the last boundary
//    inside the array; the final < 16 bytes of the array are read with plain loads.
//  * The sweep builds ONE bit mask (q >= thr_picture; lane = pixel mod 32, so a
//    ballot is a word). With a symmetric neighbour table the boundary threshold
//    is only ever asked of the neighbours of kept pixels, which the symmetric
//    pass reads straight from the row buffer; the buffer goes back to the copy
//    engine right after that pass.
//  * The CTA copies the neighbour table into shared memory as uint16 (12 bytes
//    per pixel) when there is room: the table look-up is the one dependent load
//    in front of every bit test.
//  * The scalar tail (divisions, square roots, atan2: about 400 dependent
//    instructions) is never run per event: a warp pushes the event's sums into a
//    CTA-wide queue in shared memory, and whichever warp completes a batch of 32
//    records finishes them, one event per lane; the last partial batch is
//    finished after a __syncthreads. No cleaning warp keeps parked sums in
//    registers.
constexpr int kQueueBatches = 4;   // batch slots of 32 records
struct FinishQueue {
  uint32_t head;                     // records claimed so far
  uint32_t written[kQueueBatches];   // records completely written, per slot
  uint32_t freed[kQueueBatches];     // batches read out of the slot so far
  uint32_t pad[7];
  float4 rec[kQueueBatches * 32][5];  // 80 bytes per record
};
static_assert(sizeof(FinishQueue) % 16 == 0, "the per-warp buffers behind it stay 16-byte aligned");

// lanes < n: read record `first + lane` and run the scalar tail for it
__device__ __forceinline__ void queue_finish(FinishQueue& Q, const uint32_t slot, const int n,
                                             const RtaImageOut& out) {
  const int lane = threadIdx.x & 31;
  Pending pd;
  if (lane < n) {
    const float4* r = Q.rec[slot * 32u + (uint32_t)lane];
    const float4 a = r[0], b = r[1], c = r[2], d = r[3], f = r[4];
    pd.s0 = __hiloint2double(__float_as_int(a.y), __float_as_int(a.x));
    pd.sx = __hiloint2double(__float_as_int(a.w), __float_as_int(a.z));
    pd.sy = __hiloint2double(__float_as_int(b.y), __float_as_int(b.x));
    pd.st = __hiloint2double(__float_as_int(b.w), __float_as_int(b.z));
    pd.sxx = __hiloint2double(__float_as_int(c.y), __float_as_int(c.x));
    pd.syy = __hiloint2double(__float_as_int(c.w), __float_as_int(c.z));
    pd.sxy = __hiloint2double(__float_as_int(d.y), __float_as_int(d.x));
    pd.x0 = d.z, pd.y0 = d.w, pd.qm = f.x;
    pd.n_pix = __float_as_int(f.y);
    pd.e = (uint32_t)__float_as_int(f.z);
  }
  __syncwarp();
  if (lane == 0) {  // the slot may be refilled
    __threadfence_block();
    Q.written[slot] = 0u;
    // the reset must be visible before the slot is handed back: a writer of the next
    // batch waits on `freed` and then counts itself into `written`
    __threadfence_block();
    atomicAdd(&Q.freed[slot], 1u);
  }
  if (lane < n) finish_event(pd, out);
  __syncwarp();
}

// whole warp; `cur` holds the same sums in every lane
__device__ __forceinline__ void queue_push(FinishQueue& Q, const EventSums& cur,
                                           const RtaImageOut& out) {
  const int lane = threadIdx.x & 31;
  uint32_t done = 0, slot = 0;
  if (lane == 0) {
    const uint32_t idx = atomicAdd(&Q.head, 1u);
    const uint32_t batch = idx >> 5;
    slot = batch % kQueueBatches;
    // the batch that used this slot before must have been read out (it almost always has)
    while (*reinterpret_cast<volatile uint32_t*>(&Q.freed[slot]) < batch / kQueueBatches) __nanosleep(64);
    __threadfence_block();
    float4* r = Q.rec[slot * 32u + (idx & 31u)];
    const auto lo = [](double v) { return __int_as_float(__double2loint(v)); };
    const auto hi = [](double v) { return __int_as_float(__double2hiint(v)); };
    r[0] = make_float4(lo(cur.s0), hi(cur.s0), lo(cur.sx), hi(cur.sx));
    r[1] = make_float4(lo(cur.sy), hi(cur.sy), lo(cur.st), hi(cur.st));
    r[2] = make_float4(lo(cur.sxx), hi(cur.sxx), lo(cur.syy), hi(cur.syy));
    r[3] = make_float4(lo(cur.sxy), hi(cur.sxy), cur.x0, cur.y0);
    r[4] = make_float4(cur.qm, __int_as_float(cur.n_pix), __int_as_float((int)cur.e), 0.0f);
    __threadfence_block();
    done = atomicAdd(&Q.written[slot], 1u) + 1u;
  }
  done = __shfl_sync(0xFFFFFFFFu, done, 0);
  if (done == 32u) {
    slot = __shfl_sync(0xFFFFFFFFu, slot, 0);
    __threadfence_block();
    queue_finish(Q, slot, 32, out);
  }
}

size_t moments_row_bytes(int32_t P) { return r16(4u * (size_t)P) + 32u; }
size_t moments_warp_bytes(int32_t P) {
  return moments_row_bytes(P) + 2u * r16(4u * mask_words(P)) + CleanScratch::bytes(P, kListCapMin);
}
size_t moments_table_bytes(int32_t P) { return r16(12u * (size_t)P); }

template <int WARPS, bool S16>
__global__ void __launch_bounds__(32 * WARPS, 1)
    image_moments_kernel(const float* __restrict__ charge, const float* __restrict__ time,
                         const uint32_t n_events, const int P,
                         const __grid_constant__ RtaCamera cam,
                         const __grid_constant__ RtaImageOut out, const int force_general) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t row_bar[WARPS];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  FinishQueue& Q = *reinterpret_cast<FinishQueue*>(smem);
  uint16_t* nbr16 = reinterpret_cast<uint16_t*>(smem + sizeof(FinishQueue));
  const size_t wb = r16(4u * mask_words(P));
  const size_t rb = r16(4u * (size_t)P) + 32u;
  const size_t per_warp = rb + 2u * wb + CleanScratch::bytes(P, kListCapMin);
  uint8_t* mine = smem + sizeof(FinishQueue) + (S16 ? r16(12u * (size_t)P) : 0u) + (size_t)warp * per_warp;
  uint32_t* core_w = reinterpret_cast<uint32_t*>(mine + rb);
  uint32_t* low_w = reinterpret_cast<uint32_t*>(mine + rb + wb);
  const CleanScratch sc(mine + rb + 2u * wb, P, kListCapMin);
  const uint32_t bar = smem_u32(&row_bar[warp]);
  const uint32_t row_s = smem_u32(mine);
  if (threadIdx.x < (sizeof(FinishQueue) - sizeof(Q.rec)) / 4u)
    reinterpret_cast<uint32_t*>(smem)[threadIdx.x] = 0u;  // head, written[], freed[]
  if (lane == 0) {
    mbar_init(bar, 1);
    fence_mbar_init();
  }
  __syncwarp();

  const uintptr_t base = reinterpret_cast<uintptr_t>(charge);
  const uintptr_t end_all = base + (uintptr_t)n_events * (uintptr_t)P * 4u;
  const uint32_t row_bytes = 4u * (uint32_t)P;
  // lane 0: start the copy of event e's row into this warp's buffer
  const auto issue = [&](const uint32_t e) {
    const uintptr_t a = base + (uintptr_t)e * row_bytes;
    const uint32_t mis = (uint32_t)(a & 15u);
    const uintptr_t lo = a - mis;
    uint32_t len = (mis + row_bytes + 15u) & ~15u;
    if (lo + len > end_all) {  // the last row of the array: whole 16-byte lines, then words
      len = (uint32_t)((end_all - lo) & ~(uintptr_t)15u);
      for (uint32_t b = len; b < mis + row_bytes; b += 4u)
        *reinterpret_cast<float*>(mine + b) = *reinterpret_cast<const float*>(lo + b);
    }
    mbar_expect_tx(bar, len);
    if (len != 0) tma_bulk_g2s(row_s, reinterpret_cast<const void*>(lo), len, bar);
  };

  // The CTA owns a contiguous range of events; its warps draw them from a shared-memory
  // counter (with a fixed warp -> event map the CTA waits for the warps that have one
  // event more than the others: 7 against 6.1 on C3). Lane 0 draws the next index when
  // it hands the row buffer back, so the copy of that row is issued a whole event ahead.
  __shared__ uint32_t next_event;
  const uint32_t ev_lo = (uint32_t)(((uint64_t)n_events * blockIdx.x) / gridDim.x);
  const uint32_t ev_hi = (uint32_t)(((uint64_t)n_events * (blockIdx.x + 1u)) / gridDim.x);
  if (threadIdx.x == 0) next_event = ev_lo + WARPS;
  uint32_t e = ev_lo + warp, e_next = ev_hi;
  if (lane == 0 && e < ev_hi) issue(e);
  // the table copy and check overlap the first loads
  bool symmetric;
  if constexpr (S16) {
    // eight loads in flight per thread (one at a time this copy was 8 % of the kernel)
    constexpr int step = 32 * WARPS;
    for (int i0 = threadIdx.x; i0 < 6 * P; i0 += 8 * step) {
      int v[8];
#pragma unroll
      for (int u = 0; u < 8; ++u) v[u] = i0 + u * step < 6 * P ? __ldg(cam.neighbors + i0 + u * step) : -1;
#pragma unroll
      for (int u = 0; u < 8; ++u)
        if (i0 + u * step < 6 * P)
          nbr16[i0 + u * step] = (unsigned)v[u] < (unsigned)P ? (uint16_t)v[u] : (uint16_t)0xFFFFu;
    }
    __syncthreads();
    symmetric = table_is_symmetric_s16(nbr16, P) && !force_general;
  } else {
    symmetric = table_is_symmetric(cam.neighbors, P) && !force_general;  // contains __syncthreads
  }
  const NbrTable nbr{cam.neighbors, S16 ? nbr16 : nullptr,
                     (reinterpret_cast<uintptr_t>(cam.neighbors) & 7u) == 0};
  const float thr_p = cam.thr_picture, thr_b = cam.thr_boundary;
  const int NW = (int)mask_words(P), NWF = P >> 5;  // words, full words
  for (uint32_t k = 0; e < ev_hi; e = __shfl_sync(0xFFFFFFFFu, e_next, 0), ++k) {
    const uint32_t mis = (uint32_t)((base + (uintptr_t)e * row_bytes) & 15u);
    const float* row = reinterpret_cast<const float*>(mine + mis);
    mbar_wait(bar, k & 1u);
    // sweep: word w of a mask = ballot over pixels 32 w .. 32 w + 31; four words per
    // step (loads first), lane 0 stores them with one 16-byte store
    const auto sweep = [&](const float thr, uint32_t* words) {
      int w = 0;
#pragma unroll 2
      for (; w + 4 <= NWF; w += 4) {
        float v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = row[32 * (w + u) + lane];
        uint4 m;
        m.x = __ballot_sync(0xFFFFFFFFu, v[0] >= thr);
        m.y = __ballot_sync(0xFFFFFFFFu, v[1] >= thr);
        m.z = __ballot_sync(0xFFFFFFFFu, v[2] >= thr);
        m.w = __ballot_sync(0xFFFFFFFFu, v[3] >= thr);
        if (lane == 0) *reinterpret_cast<uint4*>(words + w) = m;
      }
      for (; w < NW; ++w) {  // the last words; the very last may be partial
        const int p = 32 * w + lane;
        const float v = p < P ? row[p] : 0.0f;
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, p < P && v >= thr);
        if (lane == 0) words[w] = m;
      }
    };
    sweep(thr_p, core_w);
    if (!symmetric) sweep(thr_b, low_w);  // the general path asks for every boundary candidate
    __syncwarp();
    EventSums cur;
    clean_event_sums<true>(
        e, P, charge + (size_t)e * (size_t)P, TimeFromArray{time + (size_t)e * (size_t)P}, core_w, low_w,
        LowFromRow{row, thr_b}, sc, nbr, cam, out, symmetric,
        [&] {  // every lane is done with the row: the buffer goes back to the copy engine
          __syncwarp();
          if (lane == 0) {
            e_next = atomicAdd(&next_event, 1u);
            if (e_next < ev_hi) issue(e_next);
          }
        },
        cur);
    queue_push(Q, cur, out);
  }
  __syncthreads();
  if (warp == 0) {  // the last, partial batch
    const uint32_t total = *reinterpret_cast<volatile uint32_t*>(&Q.head);
    if (total & 31u) queue_finish(Q, (total >> 5) % kQueueBatches, (int)(total & 31u), out);
  }
}

// ------------------------------------------------- producer / cleaner hand-off ----
// The generic fused kernel runs NT extraction threads and one cleaning warp
// (threads NT .. NT+31). Event number k of the CTA uses buffer k & 1. Named
// barriers (all with NT + 32 participants): READY + b — the extraction threads
// arrive when the buffer is complete, the cleaning warp waits; FREE + b — the
// cleaning warp arrives when it is done with the buffer, the extraction
// threads wait before writing event k + 2 into it. ev_id[b] carries the event
// index (kNoEvent = no more events).
enum : int { BAR_READY = 1, BAR_FREE = 3 };
constexpr uint32_t kNoEvent = 0xFFFFFFFFu;

struct FusedShared {
  uint32_t ev_id[2];
};

template <int NT>
__device__ __forceinline__ void cleaner_loop(const int P, uint8_t* ev_base, uint8_t* sc_base,
                                             volatile FusedShared& fs, const RtaCamera& cam,
                                             const RtaImageOut& out, const bool symmetric) {
  const size_t eb = EventBuf::bytes(P);
  const CleanScratch sc(sc_base, P, P);
  Pending pd = {};
  int n_pend = 0;
  for (uint32_t k = 0;; ++k) {
    const int b = (int)(k & 1u);
    named_sync(BAR_READY + b, NT + 32);
    const uint32_t e = fs.ev_id[b];
    if (e == kNoEvent) break;
    const EventBuf buf(ev_base + (size_t)b * eb, P);
    clean_event(e, P, buf.q, TimeFromArray{buf.t}, buf.core_w, buf.low_w, sc, cam, out, symmetric,
                pd, n_pend);
    __syncwarp();
    named_arrive(BAR_FREE + b, NT + 32);
  }
  flush_pending(pd, n_pend, out);
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
                                 const __grid_constant__ RtaImageOut out, const int force_general) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ FusedShared fs;
  const int tid = threadIdx.x, lane = tid & 31;
  const size_t eb = EventBuf::bytes(P);
  const bool symmetric = table_is_symmetric(cam.neighbors, P) && !force_general;
  if (tid >= NT) {
    cleaner_loop<NT>(P, smem, smem + 2u * eb, fs, cam, out, symmetric);
    return;
  }
  const ModeArgs ma = {};
  const float thr_p = cam.thr_picture, thr_b = cam.thr_boundary;
  uint32_t k = 0;
  for (uint32_t e = blockIdx.x; e < n_events; e += gridDim.x, ++k) {
    producer_acquire<NT>(k);
    const EventBuf buf(smem + (size_t)(k & 1u) * eb, P);
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

// ------------------------------------------- extraction + cleaning, staged ----
// One persistent CTA per SM: G extraction groups of NT threads (thread t of
// group g = thread g NT + t) and up to NCMAX cleaning warps behind them. The
// CTA's events are e_k = blockIdx.x + k gridDim.x, k = 0, 1, ...; event k is
// written into buffer k mod NB and cleaned by warp k mod NC. The (event, tile)
// items of the CTA, in order, are dealt round-robin to the groups: group g
// takes items g, g + G, ...; every thread derives its group's item sequence
// arithmetically, so there is no queue. Each group has its own ring of STAGES
// stages filled by TMA bulk copies (16-byte cp.async for the padded S = 128
// layout) and its own named barrier.
//   full[g][s]  the stage's bytes have landed (TMA complete_tx / cp.async arrive)
//   ready[b]    one arrival per extraction warp and tile of the event in buffer b:
//               nt * NT / 32 arrivals per phase; the cleaning warp waits
//   freeb[b]    one arrival by the cleaning warp per cleaned event; the extraction
//               threads wait before the first write of event k >= NB
constexpr int kMaxBuf = 12;
constexpr int kFusedListCap = 512;  // entries of a cleaning warp's pixel list (longer lists go in rounds)

// XREGS / CREGS: registers per thread of the extraction / cleaning warpgroups after the split
template <class C, int G, int NCMAX, int XREGS, int CREGS>
__global__ void __launch_bounds__(G * C::NT + 32 * NCMAX, 1)
    extract_image_kernel(const uint8_t* __restrict__ wf, const uint32_t n_events, const int P,
                         const int* __restrict__ pedestal, const float* __restrict__ gain,
                         const __grid_constant__ RtaCamera cam,
                         const __grid_constant__ RtaImageOut out, const int NB, const int NC,
                         const int force_general, const __grid_constant__ ModeArgs ma) {
  static_assert(C::BITS == 16 && C::STAGES >= 2, "uint16 samples, at least two stages");
  static_assert(C::TPT == 1 || C::TPT == 2, "one or two traces per thread");
  static_assert(G >= 1 && G <= 14, "named barriers 1 .. G");
  static_assert(C::S <= 256, "t* travels as one byte");
  // an event may start at any multiple of VEC bytes: the copy starts at the
  // 16-byte boundary below it, so a stage holds up to 16 bytes more than a tile
  constexpr int STG = C::STAGE_BYTES + 16;
  constexpr int NT = C::NT, NX = G * NT;
  constexpr uint32_t TRACE_BYTES = C::TRACE_BITS / 8;
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[G * C::STAGES];
  __shared__ __align__(8) uint64_t ready_bar[kMaxBuf];
  __shared__ __align__(8) uint64_t free_bar[kMaxBuf];
  const int tid = threadIdx.x, lane = tid & 31;
  const uint32_t nt = ((uint32_t)P + C::TILE_TRACES - 1u) / C::TILE_TRACES;  // tiles per event
  uint8_t* ev_base = smem + (size_t)G * C::STAGES * STG;
  const size_t eb = EventBuf8::bytes(P);
  const uint32_t ready0 = smem_u32(ready_bar), free0 = smem_u32(free_bar);

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < G * C::STAGES; ++s) mbar_init(smem_u32(full_bar) + 8 * s, C::PAD ? NT : 1);
    for (int b = 0; b < NB; ++b) {
      mbar_init(ready0 + 8 * b, nt * (NT / 32));
      mbar_init(free0 + 8 * b, 1);
    }
    fence_mbar_init();
  }
  __syncthreads();
  // event number k of this CTA. n_events < 2^31 and the walks stop a few items
  // past the end, so 32 bits hold every index that is formed
  const auto event_of = [&](const uint32_t k) -> uint32_t { return blockIdx.x + k * gridDim.x; };
  // Register split (whole warpgroups only): the extraction code needs 48-56
  // registers (XREGS, tuned per shape), the cleaning code about 130; the CTA is
  // launched with the same number for everyone and the warpgroups trade them here.
  constexpr bool REGSPLIT = (NX % 128 == 0) && (NCMAX % 4 == 0);

  if (tid >= NX) {  // ------------------------------------------------ cleaning warps
    if constexpr (REGSPLIT) asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CREGS));
    const bool symmetric = table_is_symmetric(cam.neighbors, P) && !force_general;
    const int c = (tid - NX) >> 5;
    if (c >= NC) return;
    const CleanScratch sc(ev_base + (size_t)NB * eb + (size_t)c * CleanScratch::bytes(P, kFusedListCap), P,
                          kFusedListCap);
    Pending pd = {};
    int n_pend = 0;
    for (uint32_t k = (uint32_t)c; event_of(k) < n_events; k += (uint32_t)NC) {
      const uint32_t b = k % (uint32_t)NB, use = k / (uint32_t)NB;
      mbar_wait_idle(ready0 + 8 * b, use & 1u);
      const EventBuf8 buf(ev_base + (size_t)b * eb, P);
      const uint32_t ev = event_of(k);
      const TimeFromWaveform tw{reinterpret_cast<const uint16_t*>(wf) + (size_t)ev * (size_t)P * C::S,
                                buf.tstar, pedestal, gain, C::S, C::W};
      clean_event(ev, P, buf.q, tw, buf.core_w, buf.low_w, sc, cam, out, symmetric, pd, n_pend);
      __syncwarp();
      if (lane == 0) mbar_arrive(free0 + 8 * b);
    }
    flush_pending(pd, n_pend, out);
    return;
  }

  // ---------------------------------------------------------------- extraction groups
  if constexpr (REGSPLIT) asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(XREGS));
  const int g = tid / NT, gt = tid - g * NT;
  const uint32_t ring = smem_u32(smem) + (uint32_t)(g * C::STAGES * STG);
  uint8_t* ringp = smem + (size_t)g * C::STAGES * STG;
  const uint32_t bar_base = smem_u32(full_bar) + 8u * (uint32_t)(g * C::STAGES);
  const unsigned long long EB = (unsigned long long)P * TRACE_BYTES;  // bytes per event
  const unsigned long long total = (unsigned long long)n_events * EB;
  const float thr_p = cam.thr_picture, thr_b = cam.thr_boundary;

  // item cursor: event number k (kept as its event index ev and its buffer
  // b = k mod NB, use = k div NB) and tile; advance by G items
  struct Cursor {
    uint32_t ev, tile, b, use;
  };
  const auto advance = [&](Cursor& c) {
    c.tile += (uint32_t)G;
    while (c.tile >= nt) {
      c.tile -= nt;
      c.ev += gridDim.x;
      if (++c.b == (uint32_t)NB) c.b = 0, ++c.use;
    }
  };
  const auto issue = [&](const uint32_t ev, const uint32_t tile, const int stage) {
    const unsigned long long start = (unsigned long long)ev * EB +
                                     (unsigned long long)tile * C::TILE_BYTES;
    const uint32_t left = (uint32_t)P - tile * C::TILE_TRACES;
    const uint32_t n = left < (uint32_t)C::TILE_TRACES ? left : (uint32_t)C::TILE_TRACES;
    const uint32_t bytes = n * TRACE_BYTES;
    const uint32_t dst = ring + stage * STG;
    const uint32_t bar = bar_base + 8 * stage;
    if constexpr (!C::PAD) {
      if (gt == 0) {
        const uint32_t mis = (uint32_t)(start & 15u);
        const unsigned long long lo = start - mis;
        uint32_t len = (mis + bytes + 15u) & ~15u;
        if (lo + len > total) {
          // the last tile of the last event: nothing past the caller's buffer
          // is read; the final < 16 bytes go halfword by halfword
          len = (uint32_t)((total - lo) & ~15ull);
          uint8_t* d = ringp + stage * STG;
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
      for (uint32_t c = gt; c < bytes / 16u; c += NT) {
        const uint32_t u = c / C::NVEC;  // one extra chunk of padding per unit
        cp_async16(dst + (c + u) * 16u, src + (size_t)c * 16u);
      }
      cp_async_mbar_arrive(bar);
    }
  };

  // consumer cursor = item g; the producer cursor runs STAGES items ahead
  Cursor cc = {blockIdx.x, 0u, 0u, 0u};
  if (g != 0) {  // items 0 .. g-1 belong to the groups before this one
    cc.tile = (uint32_t)g - (uint32_t)G;
    advance(cc);
  }
  Cursor pc = cc;
#pragma unroll
  for (int s = 0; s < C::STAGES; ++s) {
    if (pc.ev < n_events) issue(pc.ev, pc.tile, s);
    advance(pc);
  }
  // the table check overlaps the first loads (its __syncthreads pairs with the cleaning warps')
  table_is_symmetric(cam.neighbors, P);

  uint32_t cur_ev = 0xFFFFFFFFu;
  const uint32_t EB32 = (uint32_t)EB;  // low bits are all that the 16-byte phase needs
  const uint32_t NW = (uint32_t)mask_words(P);
  for (uint32_t j = 0;; ++j) {
    const uint32_t ev = cc.ev, tile = cc.tile, b = cc.b;
    if (ev >= n_events) break;
    const int stage = (int)(j % C::STAGES);
    const uint32_t parity = (j / C::STAGES) & 1u;
    if (ev != cur_ev) {  // first tile of this group in this event: the buffer must be free
      cur_ev = ev;
      if (cc.use != 0) mbar_wait(free0 + 8 * b, (cc.use - 1u) & 1u);
    }
    const EventBuf8 buf(ev_base + (size_t)b * eb, P);
    mbar_wait(bar_base + 8 * stage, parity);
    const uint32_t p0 = tile * C::TILE_TRACES + (uint32_t)gt * C::TPT;
    float qv[C::TPT];
#pragma unroll
    for (int i = 0; i < C::TPT; ++i) qv[i] = 0.0f;
    const bool in = p0 < (uint32_t)P;
    if (in) {
      uint32_t mis = 0;
      if constexpr (!C::PAD) mis = (ev * EB32) & 15u;  // TILE_BYTES is a multiple of 16
      const uint8_t* unit = ringp + stage * STG + mis + gt * C::UNIT_STRIDE;
      Result res[C::TPT];
      // step a7 is left to the cleaning warp (TimeFromWaveform): res[].time = bits of t*
      compute_results<C, MODE_SLIDING, RTA_IMG_KEYMODE, false>(unit, p0, 0u, pedestal, gain, ma, res);
#pragma unroll
      for (int i = 0; i < C::TPT; ++i) {  // P is a multiple of TPT: the unit is whole
        buf.q[p0 + i] = qv[i] = res[i].charge;
        buf.tstar[p0 + i] = (uint8_t)__float_as_int(res[i].time);
      }
    }
    // threshold bits of this warp's 32 * TPT pixels (warps past the camera's end write nothing)
    const uint32_t w0 = (tile * C::TILE_TRACES + (uint32_t)(gt - lane) * C::TPT) >> 5;
    if constexpr (C::TPT == 1) {
      const uint32_t c = __ballot_sync(0xFFFFFFFFu, in && qv[0] >= thr_p);
      const uint32_t l = __ballot_sync(0xFFFFFFFFu, in && qv[0] >= thr_b);
      if (lane == 0 && w0 < NW) buf.core_w[w0] = c, buf.low_w[w0] = l;
    } else {
      // lane l holds pixels 2 l and 2 l + 1 of the warp's 64: each half-warp ORs
      // its lanes' bit pairs into one word (lanes 0-15: word w0, 16-31: w0 + 1)
      const uint32_t sh = 2u * (uint32_t)(lane & 15);
      uint32_t cb = 0, lb = 0;
      if (in) {
        cb = ((qv[0] >= thr_p ? 1u : 0u) | (qv[1] >= thr_p ? 2u : 0u)) << sh;
        lb = ((qv[0] >= thr_b ? 1u : 0u) | (qv[1] >= thr_b ? 2u : 0u)) << sh;
      }
      const bool hi = (lane & 16) != 0;
      const uint32_t c_lo = __reduce_or_sync(0xFFFFFFFFu, hi ? 0u : cb);
      const uint32_t c_hi = __reduce_or_sync(0xFFFFFFFFu, hi ? cb : 0u);
      const uint32_t l_lo = __reduce_or_sync(0xFFFFFFFFu, hi ? 0u : lb);
      const uint32_t l_hi = __reduce_or_sync(0xFFFFFFFFu, hi ? lb : 0u);
      if (lane == 0) {
        if (w0 < NW) buf.core_w[w0] = c_lo, buf.low_w[w0] = l_lo;
        if (w0 + 1u < NW) buf.core_w[w0 + 1u] = c_hi, buf.low_w[w0 + 1u] = l_hi;
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(ready0 + 8 * b);  // release: this warp's share of the tile is in the buffer
    named_sync(1 + g, NT);                       // every thread of the group is done with the stage
    // (an empty-stage mbarrier that only the issuing thread waits on, so that the other
    // warps run ahead, was measured: no gain on C2, 4 % slower on C3)
    if (C::PAD || gt == 0) {  // dense layouts: only the thread that issues the bulk copy keeps the producer cursor
      if (pc.ev < n_events) issue(pc.ev, pc.tile, stage);
      advance(pc);
    }
    advance(cc);
  }
}

// ------------------------------------------------------------- dispatch ----
constexpr int kGenericNT = 256;
constexpr size_t kSmemLimit = 227u * 1024u;
std::atomic<bool> g_general_cleaning{false};  // tests: never take the symmetric-table shortcut

// Staged fused kernels of the four config shapes: threads per group, stages
// per group (TileCfg), groups, cleaning warps (tuned on B200).
#ifndef RTA_I30_NT
#define RTA_I30_NT 128
#endif
#ifndef RTA_I30_G
#define RTA_I30_G 6
#endif
#ifndef RTA_I40_NT
#define RTA_I40_NT 128
#endif
#ifndef RTA_I40_G
#define RTA_I40_G 6
#endif
#ifndef RTA_I25_NT
#define RTA_I25_NT 128
#endif
#ifndef RTA_I25_G
#define RTA_I25_G 5
#endif
#ifndef RTA_I128_NT
#define RTA_I128_NT 64
#endif
#ifndef RTA_I128_G
#define RTA_I128_G 5
#endif
#ifndef RTA_IMG_NC
#define RTA_IMG_NC 4
#endif
#ifndef RTA_I128_NC
#define RTA_I128_NC 2
#endif
template <class C_, int G_, int NCMAX_, int XREGS_ = 56, int CREGS_ = 152>
struct ImgCfg {
  using C = C_;
  static constexpr int G = G_, NCMAX = NCMAX_, XREGS = XREGS_, CREGS = CREGS_;
  static constexpr int THREADS = G * C::NT + 32 * NCMAX;
  static constexpr size_t RING = (size_t)G * C::STAGES * (C::STAGE_BYTES + 16);
  static_assert(THREADS <= 1024, "one CTA");
  // the register split of extract_image_kernel (same condition as there): the
  // warpgroups trade registers inside what the CTA was launched with, which is
  // the launch bound's cap (ptxas allocates it in full when setmaxnreg is used);
  // a split that does not fit would leave setmaxnreg.inc waiting for ever
  static constexpr bool REGSPLIT = ((G * C::NT) % 128 == 0) && (NCMAX % 4 == 0);
  static constexpr int LAUNCH_REGS = ((65536 / THREADS) / 8) * 8;
  static constexpr int SPLIT_REGS = G * C::NT * XREGS + 32 * NCMAX * CREGS;
  static_assert(!REGSPLIT || SPLIT_REGS <= THREADS * LAUNCH_REGS, "register split exceeds the CTA's pool");
};
#ifndef RTA_I30_XREGS
#define RTA_I30_XREGS 56
#endif
#ifndef RTA_I30_CREGS
#define RTA_I30_CREGS 152
#endif
using ImgS30W7 = ImgCfg<TileCfg<30, 7, RTA_I30_NT, 2>, RTA_I30_G, RTA_IMG_NC, RTA_I30_XREGS, RTA_I30_CREGS>;
// 48 registers for the S = 40 extraction code: 0.253 ms on C2 against 0.268 ms at 56 (and 0.290 at 40)
#ifndef RTA_I40_XREGS
#define RTA_I40_XREGS 56
#endif
#ifndef RTA_I40_CREGS
#define RTA_I40_CREGS 152
#endif
using ImgS40W7 = ImgCfg<TileCfg<40, 7, RTA_I40_NT, 2>, RTA_I40_G, RTA_IMG_NC, RTA_I40_XREGS, RTA_I40_CREGS>;
#ifndef RTA_I25_XREGS
#define RTA_I25_XREGS 64
#endif
#ifndef RTA_I25_CREGS
#define RTA_I25_CREGS 152
#endif
using ImgS25W4 = ImgCfg<TileCfg<25, 4, RTA_I25_NT, 2>, RTA_I25_G, RTA_IMG_NC, RTA_I25_XREGS, RTA_I25_CREGS>;
using ImgS128W8 = ImgCfg<TileCfg<128, 8, RTA_I128_NT, 2>, RTA_I128_G, RTA_I128_NC>;

// Cleaning warps NC and event buffers NB = NC + 1 that fit behind the ring
// (0 = not even one warp and two buffers fit).
template <class I>
int fused_cleaners(int32_t P) {
  for (int nc = I::NCMAX; nc >= 1; --nc) {
    const size_t need = I::RING + (size_t)(nc + 1) * EventBuf8::bytes(P) +
                        (size_t)nc * CleanScratch::bytes(P, kFusedListCap) + 1024u;
    if (need <= kSmemLimit) return nc;
  }
  return 0;
}

// The staged kernel takes a shape when every event starts on a boundary its
// units can be read from (VEC bytes; whole units per event) and the per-event
// buffers fit behind the ring.
template <class I>
bool staged_ok(int32_t P) {
  using C = typename I::C;
  const size_t eb = (size_t)P * (C::TRACE_BITS / 8);
  if (P % C::TPT != 0 || eb % C::VEC != 0) return false;
  if (C::PAD && eb % 16 != 0) return false;
  return fused_cleaners<I>(P) >= 1;
}

template <class I>
struct FusedLauncher {
  static cudaError_t launch(const uint8_t* wf, uint32_t n_events, int32_t P,
                            const int32_t* pedestal, const float* gain, const RtaCamera& cam,
                            const RtaImageOut& out, cudaStream_t stream) {
    using C = typename I::C;
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if ((e = rta_device_sms(dev, &sms)) != cudaSuccess) return e;
    const int nc = fused_cleaners<I>(P);
    int nb = nc + 1;
    size_t smem = I::RING + (size_t)nb * EventBuf8::bytes(P) +
                  (size_t)nc * CleanScratch::bytes(P, kFusedListCap);
    // more buffers while there is room: the extraction groups run further ahead
    while (nb + 1 <= kMaxBuf && nb < nc + 3 && smem + EventBuf8::bytes(P) + 1024u <= kSmemLimit) {
      ++nb;
      smem += EventBuf8::bytes(P);
    }
    auto kernel = extract_image_kernel<C, I::G, I::NCMAX, I::XREGS, I::CREGS>;
    if (I::REGSPLIT) {  // never launch a split that the allocated registers cannot serve
      cudaFuncAttributes fa;
      if ((e = cudaFuncGetAttributes(&fa, kernel)) != cudaSuccess) return e;
      if (fa.numRegs * I::THREADS < I::SPLIT_REGS) return cudaErrorLaunchOutOfResources;
    }
    // the dynamic shared-memory size depends on n_pixels
    if ((e = rta_func_allow_max_smem((const void*)kernel, dev)) != cudaSuccess) return e;
    uint32_t grid = (uint32_t)sms;
    if (grid > n_events) grid = n_events;
    ModeArgs ma = {};  // constant-bank operands of compute_results (KEYMUL)
    ma.key_mul = 1u << C::KB;
    ma.one = 1u;
    ma.minus_one = 0xFFFFFFFFu;
    kernel<<<grid, I::THREADS, smem, stream>>>(wf, n_events, P, pedestal, gain, cam, out, nb, nc,
                                               g_general_cleaning.load() ? 1 : 0, ma);
    rta_count_launch();
    return cudaGetLastError();
  }
};

template <int WARPS, bool S16>
cudaError_t launch_moments(const float* charge, const float* time, uint32_t n_events, int32_t P,
                           const RtaCamera& cam, const RtaImageOut& out, cudaStream_t stream) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = rta_device_sms(dev, &sms)) != cudaSuccess) return e;
  const size_t smem = sizeof(FinishQueue) + (S16 ? moments_table_bytes(P) : 0u) +
                      WARPS * moments_warp_bytes(P);
  auto kernel = image_moments_kernel<WARPS, S16>;
  if ((e = rta_func_allow_max_smem((const void*)kernel, dev)) != cudaSuccess) return e;
  uint32_t grid = (uint32_t)sms;  // one CTA per SM (launch bounds)
  const uint32_t need = (n_events + WARPS - 1u) / WARPS;
  if (grid > need) grid = need;
  kernel<<<grid, 32 * WARPS, smem, stream>>>(charge, time, n_events, P, cam, out,
                                             g_general_cleaning.load() ? 1 : 0);
  rta_count_launch();
  return cudaGetLastError();
}

// Library-owned stream-ordered memory pool of the current device for the scratch
// of the two-kernel route of rta_launch_extract_image. Its release threshold is
// unlimited, so the scratch of one call is reused by the next instead of going
// back to the driver at every synchronisation. nullptr = no pool (generic route).
constexpr int kMaxPoolDev = 32;
std::mutex g_pool_mu;
cudaMemPool_t g_pool[kMaxPoolDev] = {};
bool g_pool_failed[kMaxPoolDev] = {};

cudaMemPool_t scratch_pool() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxPoolDev) return nullptr;
  std::lock_guard<std::mutex> lock(g_pool_mu);
  if (g_pool[dev] == nullptr && !g_pool_failed[dev]) {
    cudaMemPoolProps props = {};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = dev;
    cudaMemPool_t pool = nullptr;
    unsigned long long keep = ~0ull;
    if (cudaMemPoolCreate(&pool, &props) == cudaSuccess &&
        cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep) == cudaSuccess) {
      g_pool[dev] = pool;
    } else {
      if (pool) cudaMemPoolDestroy(pool);
      cudaGetLastError();
      g_pool_failed[dev] = true;
    }
  }
  return g_pool[dev];
}

}  // namespace

// rta_shutdown: the caller has synchronised the devices in use
void rta_image_release() {
  std::lock_guard<std::mutex> lock(g_pool_mu);
  for (int d = 0; d < kMaxPoolDev; ++d) {
    if (g_pool[d]) cudaMemPoolDestroy(g_pool[d]);
    g_pool[d] = nullptr;
    g_pool_failed[d] = false;
  }
  cudaGetLastError();
}

void rta_set_general_cleaning(bool on) { g_general_cleaning.store(on); }

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
    if (rta_dyn_eligible(S, W)) return "staged<any>+image_moments";
  }
  return "image_generic";
}

cudaError_t rta_launch_image_moments(const float* charge, const float* time, int64_t n_events,
                                     int32_t n_pixels, const RtaCamera& cam,
                                     const RtaImageOut& out, cudaStream_t stream) {
  if (n_events <= 0) return cudaSuccess;
  // As many warps as one CTA's shared memory holds (row buffer + masks + scratch
  // per warp, behind the finish queue). The uint16 copy of the neighbour table
  // goes in front when at least 12 warps still fit behind it.
  const size_t per_warp = moments_warp_bytes(n_pixels);
  const size_t room = kSmemLimit - 1024u - sizeof(FinishQueue);
  const size_t table = moments_table_bytes(n_pixels);
  const uint32_t E = (uint32_t)n_events;
  if (table + 12u * per_warp <= room) {
#define RTA_TRY(W) \
  if (W <= RTA_MOM_WARPS && table + (size_t)W * per_warp <= room) \
    return launch_moments<W, true>(charge, time, E, n_pixels, cam, out, stream);
    RTA_TRY(24) RTA_TRY(22) RTA_TRY(20) RTA_TRY(18) RTA_TRY(16)
    return launch_moments<12, true>(charge, time, E, n_pixels, cam, out, stream);
#undef RTA_TRY
  }
#define RTA_TRY(W) \
  if (W <= RTA_MOM_WARPS && (size_t)W * per_warp <= room) \
    return launch_moments<W, false>(charge, time, E, n_pixels, cam, out, stream);
  RTA_TRY(24) RTA_TRY(20) RTA_TRY(16) RTA_TRY(12) RTA_TRY(8) RTA_TRY(4) RTA_TRY(2)
#undef RTA_TRY
  return launch_moments<1, false>(charge, time, E, n_pixels, cam, out, stream);
}

cudaError_t rta_launch_extract_image(const void* wf, int64_t n_events, int32_t n_pixels,
                                     int32_t S, const int32_t* pedestal, const float* gain,
                                     int32_t W, const RtaCamera& cam, const RtaImageOut& out,
                                     cudaStream_t stream, bool force_generic) {
  if (n_events <= 0) return cudaSuccess;
  const uint8_t* w = static_cast<const uint8_t*>(wf);
  if (!force_generic && ((uintptr_t)wf % 16) == 0) {
#define RTA_TRY(CFG)                                                                     \
  if (S == CFG::C::S && W == CFG::C::W && staged_ok<CFG>(n_pixels))                      \
    return FusedLauncher<CFG>::launch(w, (uint32_t)n_events, n_pixels, pedestal, gain,   \
                                      cam, out, stream);
    RTA_TRY(ImgS30W7)
    RTA_TRY(ImgS40W7)
    RTA_TRY(ImgS25W4)
    RTA_TRY(ImgS128W8)
#undef RTA_TRY
    // Any other shape the staged runtime-shape kernel takes: extraction into a
    // stream-ordered scratch buffer (16 bytes per trace), then the moments kernel.
    // Same charges and the same cleaning code, so the same bits as the generic
    // fused kernel, 4-6 times faster (that kernel reads its traces with strided
    // global loads). Falls through when the scratch cannot be had.
    if (rta_dyn_eligible(S, W)) {
      const size_t n_traces = (size_t)n_events * (size_t)n_pixels;
      void* scratch = nullptr;
      cudaMemPool_t pool = scratch_pool();
      if (pool != nullptr &&
          cudaMallocFromPoolAsync(&scratch, 16u * n_traces, pool, stream) == cudaSuccess) {
        int32_t* o_sum = static_cast<int32_t*>(scratch);
        int32_t* o_start = o_sum + n_traces;
        float* o_charge = reinterpret_cast<float*>(o_start + n_traces);
        float* o_time = o_charge + n_traces;
        cudaError_t e = rta_launch_extract(wf, (int64_t)n_traces, n_pixels, S, pedestal, gain, W, o_sum,
                                           o_start, o_charge, o_time, stream, false);
        if (e == cudaSuccess)
          e = rta_launch_image_moments(o_charge, o_time, n_events, n_pixels, cam, out, stream);
        const cudaError_t ef = cudaFreeAsync(scratch, stream);
        return e != cudaSuccess ? e : ef;
      }
      cudaGetLastError();
    }
  }
  const size_t smem = 2u * EventBuf::bytes(n_pixels) + CleanScratch::bytes(n_pixels, n_pixels);
  if (smem + 1024u > kSmemLimit) return cudaErrorInvalidValue;
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = rta_device_sms(dev, &sms)) != cudaSuccess) return e;
  auto kernel = extract_image_generic_kernel<kGenericNT>;
  if ((e = rta_func_allow_max_smem((const void*)kernel, dev)) != cudaSuccess) return e;
  int occ = 0;
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, kGenericNT + 32, smem);
  if (e != cudaSuccess) return e;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  uint32_t grid = (uint32_t)(sms * occ);
  if (grid > (uint32_t)n_events) grid = (uint32_t)n_events;
  kernel<<<grid, kGenericNT + 32, smem, stream>>>(w, (uint32_t)n_events, n_pixels, S, W, pedestal,
                                                  gain, cam, out,
                                                  g_general_cleaning.load() ? 1 : 0);
  rta_count_launch();
  return cudaGetLastError();
}
