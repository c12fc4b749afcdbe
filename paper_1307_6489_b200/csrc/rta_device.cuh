// rta_device.cuh — device code shared by the translation units of librta.so
// (rta_kernels.cu: per-trace extraction; rta_image.cu: extraction fused with
// image cleaning and moments). PTX wrappers, the tile configuration, the
// per-trace arithmetic of steps a2-a7 and the generic trace
// walker. Everything is in an anonymous namespace: each TU gets its own copy.
// Never seen by oracle/.
#ifndef RTA_DEVICE_CUH
#define RTA_DEVICE_CUH

#include "rta_internal.h"

namespace {

// ------------------------------------------------------------------ PTX ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!ok);
}
// TMA 1-D bulk copy global -> shared, completion on an mbarrier (bytes % 16 == 0)
__device__ __forceinline__ void tma_bulk_g2s(uint32_t dst, const void* src, uint32_t bytes,
                                             uint32_t bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_mbar_arrive(uint32_t bar) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}

// ------------------------------------------------------------ utilities ----
__host__ __device__ constexpr int ilog2_ceil(int n) {
  int b = 0;
  while ((1 << b) < n) ++b;
  return b;
}

// g mod d with inv = min(floor(2^32 / d), 2^32 - 1): the estimate is short by
// at most one, so one conditional subtract finishes it.
__device__ __forceinline__ uint32_t fastmod(uint32_t g, uint32_t d, uint32_t inv) {
  const uint32_t q = __umulhi(g, inv);
  const uint32_t r = g - q * d;
  return r >= d ? r - d : r;
}

struct Result {
  int sum, start;
  float charge, time;
};

constexpr int kMaxTaps = RTA_MAX_TAPS;

// Steps a5-a7 from the raw (pedestal-deferred) quantities of one trace. With
// window weights c[k] (all ones except for the FIR extractor):
//   rawsum = sum_k c[k] raw[tstar + k],  relnum = sum_k k c[k] raw[tstar + k],
//   c0 = sum_k c[k],  c1 = sum_k k c[k],  W = number of weights.
// The ABI guard n_samples * sum|c| * 65535 < 2^31 keeps tstar*rawsum + relnum
// inside int32; everything touched by the pedestal is int64.
__device__ __forceinline__ Result finish_trace(const int W, const int rawsum, const int tstar,
                                               const int relnum, const int ped, const float gain,
                                               const int c0, const int c1) {
  Result r;
  r.start = tstar;
  constexpr int lim = 1 << 24;
  // every operand below 2^24 in magnitude is an exactly representable integer:
  // one IEEE operation each, bit-identical to rounding the double-precision result
  const auto small_floats = [&](const int sum, const int num) {
    int n = num, d = sum;
    if (d <= 0) {  // degenerate mean -> window centre = (2 t* + W - 1) / 2
      n = 2 * tstar + W - 1;
      d = 2;
    }
    r.charge = __fmul_rn((float)sum, gain);
    r.time = __fdiv_rn((float)n, (float)d);
  };
  const auto in24 = [](const int x) { return (unsigned)(x + (lim - 1)) < (unsigned)(2 * lim - 1); };
  if ((unsigned)ped <= 65535u) {
    // A pedestal inside the sample range (every config): x = raw - ped lies in
    // [-65535, 65535], so Sum and the numerator are bounded by the ABI guard
    // n_samples * sum|c| * 65535 < 2^31 and 32-bit arithmetic (exact modulo 2^32
    // in the intermediate products) gives them exactly.
    const int sum = rawsum - c0 * ped;
    const int num = tstar * rawsum + relnum - ped * (tstar * c0 + c1);
    r.sum = sum;
    if (in24(sum) && in24(num)) {
      small_floats(sum, num);
    } else {
      r.charge = (float)((double)sum * (double)gain);
      r.time = sum > 0 ? (float)((double)num / (double)sum)
                       : (float)((double)tstar + 0.5 * (double)(W - 1));
    }
    return r;
  }
  const long long sum64 = (long long)rawsum - (long long)c0 * (long long)ped;
  const long long num64 = (long long)(tstar * rawsum + relnum) -
                          (long long)ped * ((long long)tstar * (long long)c0 + (long long)c1);
  r.sum = (int)sum64;
  if (sum64 > -lim && sum64 < lim && num64 > -lim && num64 < lim) {
    small_floats((int)sum64, (int)num64);
  } else {
    r.charge = (float)((double)sum64 * (double)gain);
    r.time = sum64 > 0 ? (float)((double)num64 / (double)sum64)
                       : (float)((double)tstar + 0.5 * (double)(W - 1));
  }
  return r;
}

// Steps a5-a6 only (all-ones window): sum and charge as finish_trace forms them;
// `time` carries the bits of t* for a later finish_trace on the same trace.
__device__ __forceinline__ Result finish_charge(const int W, const int rawsum, const int tstar,
                                                const int ped, const float gain) {
  Result r;
  r.start = tstar;
  r.time = __int_as_float(tstar);
  constexpr int lim = 1 << 24;
  if ((unsigned)ped <= 65535u) {
    const int sum = rawsum - W * ped;
    r.sum = sum;
    r.charge = ((unsigned)(sum + (lim - 1)) < (unsigned)(2 * lim - 1))
                   ? __fmul_rn((float)sum, gain)
                   : (float)((double)sum * (double)gain);
    return r;
  }
  const long long sum64 = (long long)rawsum - (long long)W * (long long)ped;
  r.sum = (int)sum64;
  r.charge = (sum64 > -lim && sum64 < lim) ? __fmul_rn((float)(int)sum64, gain)
                                           : (float)((double)sum64 * (double)gain);
  return r;
}

// ---- the extractor family (readings R22-R24): how t* is chosen ----
enum : int { MODE_SLIDING = 0, MODE_FIXED = 1, MODE_LOCAL_PEAK = 2, MODE_FIR = 3 };

struct ModeArgs {
  const int32_t* window_start;  // MODE_FIXED: device, [n_pixels]
  int32_t shift;                // MODE_LOCAL_PEAK
  int32_t c0, c1;               // MODE_FIR: sum c[k], sum k c[k]
  int32_t taps[kMaxTaps];       // MODE_FIR
  // MODE_FIR, every tap in [-128, 127]: tap pair m = (c[2m], c[2m+1]) as two
  // signed bytes in half (m & 1) of word m >> 1 (a missing last tap is 0), for
  // one dp2a per two samples on the packed uint16 pairs; fir_packed = 1 selects it
  uint32_t taps2[kMaxTaps / 4];
  int32_t fir_packed;
  // 2^KB of the launched TileCfg, read from the constant bank: the arg-max key
  // sum * 2^KB + (2^KB - 1 - t) then compiles to one IMAD (fma pipe) instead of
  // one LEA (alu pipe), which is the pipe these kernels fill first
  uint32_t key_mul;
  uint32_t one, minus_one;  // 1 and 2^32 - 1, for the same reason (TileCfg::SLIDEMODE)
};

// d = c + a.u16[0] * b.s8[2 hi] + a.u16[1] * b.s8[2 hi + 1]  (SASS IDP.2A)
template <int HI>
__device__ __forceinline__ int dp2a_u16_s8(const uint32_t a, const uint32_t b, const int c) {
  int d;
  if constexpr (HI)
    asm("dp2a.hi.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  else
    asm("dp2a.lo.u32.s32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(c));
  return d;
}

__device__ __forceinline__ int clamp_start(const int t, const int S, const int W) {
  return min(max(t, 0), S - W);
}

#ifndef RTA_SLIDEMODE_P12
#define RTA_SLIDEMODE_P12 2
#endif
#ifndef RTA_SLIDEMODE_U16
#define RTA_SLIDEMODE_U16 0
#endif
#ifndef RTA_KEYMODE_P12
#define RTA_KEYMODE_P12 1
#endif
#ifndef RTA_KEYMODE_P40
#define RTA_KEYMODE_P40 1
#endif
#ifndef RTA_KEYMODE_U16
#define RTA_KEYMODE_U16 1
#endif
// ------------------------------------------------------- tile kernel cfg ----
// BITS = 16: uint16 samples (include/rta.h rta_extract). BITS = 12: the P12
// stream of rta_extract_packed12 (readings R25-R27): sample n sits at
// bits [12 n, 12 n + 12) of the byte stream, little-endian in bits.
template <int S_, int W_, int NT_, int STAGES_, int BITS_ = 16>
struct TileCfg {
  static constexpr int S = S_, W = W_, NT = NT_, STAGES = STAGES_, BITS = BITS_;
  static_assert(BITS == 16 || BITS == 12, "sample formats: uint16 or P12");
  static constexpr int TRACE_BITS = BITS * S;
  // traces per thread: the smallest count whose bytes a thread can own
  // (uint16: a multiple of 4 bytes; P12: a whole number of bytes)
  static constexpr int TPT = (BITS == 16) ? ((TRACE_BITS % 32 == 0) ? 1 : 2)
                                          : ((TRACE_BITS % 8 == 0) ? 1 : 2);
  static constexpr int UNIT_BYTES = TRACE_BITS * TPT / 8;     // bytes one thread owns
  // P12 units of 45 or 75 bytes do not start on a word: the thread reads the
  // aligned words around its unit and realigns them with one funnel shift each
  static constexpr bool MISALIGNED = (UNIT_BYTES % 4 != 0);
  static constexpr int VEC = MISALIGNED              ? 4
                             : (UNIT_BYTES % 16 == 0) ? 16
                             : (UNIT_BYTES % 8 == 0)  ? 8
                                                      : 4;
  static constexpr int NWORDS = (UNIT_BYTES + 3) / 4;          // words holding one unit
  static constexpr int NVEC = MISALIGNED ? NWORDS + 1 : UNIT_BYTES / VEC;  // loads per thread
  // an even number of 16-byte chunks per unit puts the lanes of a quarter-warp
  // on the same banks: pad each unit by one chunk
  static constexpr bool PAD = (VEC == 16) && (NVEC % 2 == 0);
  static constexpr int UNIT_STRIDE = UNIT_BYTES + (PAD ? 16 : 0);
  static constexpr int TILE_TRACES = NT * TPT;
  static constexpr int TILE_BYTES = NT * UNIT_BYTES;
  // misaligned units read up to 7 bytes past their end: keep the stage's tail inside the stage
  static constexpr int STAGE_BYTES = ((NT * UNIT_STRIDE + (MISALIGNED ? 16 : 0) + 127) / 128) * 128;
  static constexpr int SMEM_BYTES = STAGES * STAGE_BYTES;
  static constexpr int NWIN = S - W + 1;
  static constexpr int KB = ilog2_ceil(NWIN);
  static constexpr uint32_t KM = (1u << KB) - 1u;
  static constexpr int PB = ilog2_ceil(S);  // local-peak key: sample index bits
  // how the arg-max keys are formed (compute_results KEYMUL): tuned per shape on B200
  static constexpr int SLIDEMODE = (BITS == 12) ? RTA_SLIDEMODE_P12 : RTA_SLIDEMODE_U16;
  static constexpr int KEYMODE = (BITS == 12) ? ((S == 40 || S == 30) ? RTA_KEYMODE_P40 : RTA_KEYMODE_P12)
                                              : RTA_KEYMODE_U16;
  static constexpr uint32_t XMAX = (BITS == 16) ? 65535u : 4095u;
  static_assert(16 + PB <= 32, "peak key must fit 32 bits");
  static_assert(W >= 1 && W <= S, "window must fit the trace");
  static_assert(NT % 32 == 0, "whole warps");
  static_assert(TILE_BYTES % 16 == 0, "TMA bulk copies move multiples of 16 bytes");
  static_assert((unsigned long long)W * XMAX * (1ull << KB) + KM < (1ull << 32),
                "arg-max key must fit 32 bits for any sample value");
};

// raw sample h (sample index inside the thread's unit) from the register copy
// w[] of the unit; h is a compile-time constant once the caller's loops are
// unrolled, so every branch below folds away.
template <class C>
__device__ __forceinline__ uint32_t unit_sample(const uint32_t* w, const int h) {
  if constexpr (C::BITS == 16) {
    return (h & 1) ? (w[h >> 1] >> 16) : (w[h >> 1] & 0xFFFFu);
  } else {
    const int bit = 12 * h, i = bit >> 5, sh = bit & 31;
    if (sh == 20) return w[i] >> 20;
    if (sh < 20) return (w[i] >> sh) & 0xFFFu;
    const int i1 = (i + 1 < C::NWORDS) ? i + 1 : i;  // a straddling sample always has a next word
    return __funnelshift_r(w[i], w[i1], sh) & 0xFFFu;
  }
}
#define RTA_X(w, h) unit_sample<C>(w, h)

// Samples n0, n0+1, ... of a unit in shared memory at a data-dependent n0
// (the winning window): read(k) returns sample n0 + k, k a compile-time
// constant. uint16: one 16-bit load. P12: sample n occupies the two bytes at
// floor(3 n / 2), shifted by 4 bits when n is odd; the byte address advances
// by exactly 3 bytes per two samples, so one base per parity is enough.
template <class C>
struct WindowReader {
  const uint8_t* be;   // bytes of sample n0 (even k)
  const uint8_t* bo;   // bytes of sample n0 + 1 (odd k); P12 only
  uint32_t she, sho;   // P12: 0 or 4
  __device__ __forceinline__ WindowReader(const uint8_t* unit, const int n0) {
    if constexpr (C::BITS == 16) {
      be = unit + 2 * n0;
      bo = be;
      she = sho = 0;
    } else {
      be = unit + ((3 * n0) >> 1);
      bo = unit + ((3 * n0 + 3) >> 1);
      she = (uint32_t)(n0 & 1) << 2;
      sho = she ^ 4u;
    }
  }
  __device__ __forceinline__ int read(const int k) const {
    if constexpr (C::BITS == 16) {
      return (int)reinterpret_cast<const uint16_t*>(be)[k];
    } else {
      const uint8_t* b = (k & 1) ? bo + 3 * (k >> 1) : be + 3 * (k >> 1);
      const uint32_t v = (uint32_t)b[0] | ((uint32_t)b[1] << 8);
      return (int)((v >> ((k & 1) ? sho : she)) & 0xFFFu);
    }
  }
};

// Steps a2-a7 for the C::TPT traces of one thread's unit in shared memory.
// p0: calibration index of the first trace; it wraps to 0 after n_pixels - 1
// (a uniform batch runs through the camera again; n_pixels = 0 never wraps).
// KEYMUL != 0: `ma` comes from the launch (constant bank) and carries key_mul /
// one / minus_one, which lets part of the integer work run on the fma pipe.
// WANT_TIME = false (sliding extractor only): step a7 is left out. res[].time then
// holds the BITS of t* (the caller recomputes the peak time where it is needed:
// the fused image kernel, for the few pixels that survive the cleaning).
template <class C, int MODE, int KEYMUL = 0, bool WANT_TIME = true>
__device__ __forceinline__ void compute_results(const uint8_t* __restrict__ unit,
                                                const uint32_t p0, const uint32_t n_pixels,
                                                const int* __restrict__ pedestal,
                                                const float* __restrict__ gain,
                                                const ModeArgs& ma, Result (&res)[C::TPT]) {
  constexpr int S = C::S, W = C::W;
  // the fixed window touches W samples only: no register copy of the trace
  constexpr bool NEED_W = (MODE != MODE_FIXED);
  uint32_t w[NEED_W ? C::NWORDS : 1];
  if constexpr (NEED_W) {
    if constexpr (C::MISALIGNED) {
      // aligned words around the unit, then one funnel shift per word
      const uint32_t ph = (uint32_t)(reinterpret_cast<uintptr_t>(unit) & 3u);
      const uint32_t* src = reinterpret_cast<const uint32_t*>(unit - ph);
      uint32_t raw[C::NWORDS + 1];
#pragma unroll
      for (int i = 0; i <= C::NWORDS; ++i) raw[i] = src[i];
#pragma unroll
      for (int i = 0; i < C::NWORDS; ++i) w[i] = __funnelshift_r(raw[i], raw[i + 1], 8u * ph);
    } else if constexpr (C::VEC == 16) {
#pragma unroll
      for (int i = 0; i < C::NVEC; ++i) {
        const uint4 v = *reinterpret_cast<const uint4*>(unit + 16 * i);
        w[4 * i] = v.x, w[4 * i + 1] = v.y, w[4 * i + 2] = v.z, w[4 * i + 3] = v.w;
      }
    } else if constexpr (C::VEC == 8) {
#pragma unroll
      for (int i = 0; i < C::NVEC; ++i) {
        const uint2 v = *reinterpret_cast<const uint2*>(unit + 8 * i);
        w[2 * i] = v.x, w[2 * i + 1] = v.y;
      }
    } else {
#pragma unroll
      for (int i = 0; i < C::NVEC; ++i) w[i] = *reinterpret_cast<const uint32_t*>(unit + 4 * i);
    }
  }

  uint32_t p = p0;
#pragma unroll
  for (int j = 0; j < C::TPT; ++j) {
    const int h0 = j * S;  // compile-time after unrolling
    int tstar, rawsum, relnum = 0;
    if constexpr (MODE == MODE_SLIDING) {
      // a3 + a4 on raw samples: sliding sum, packed (sum, earliest) key
      uint32_t sum = 0;
#pragma unroll
      for (int k = 0; k < W; ++k) sum += RTA_X(w, h0 + k);
      // KEYMUL 1: every key by IMAD with the constant-bank multiplier; 2: every other one
      const auto make_key = [&](const uint32_t s, const int t) -> uint32_t {
        const uint32_t low = C::KM - (uint32_t)t;
        if (KEYMUL == 1 || (KEYMUL == 2 && (t & 1)))
          return s * ma.key_mul + low;
        else
          return (s << C::KB) + low;
      };
      uint32_t best = make_key(sum, 0);
#pragma unroll
      for (int t = 1; t < C::NWIN; ++t) {
        if (KEYMUL != 0 && (C::SLIDEMODE == 1 || (C::SLIDEMODE == 2 && (t & 1)))) {
          // the same update as two IMADs with constant-bank multipliers 1 and -1 (fma pipe)
          sum = RTA_X(w, h0 + t + W - 1) * ma.one + sum;
          sum = RTA_X(w, h0 + t - 1) * ma.minus_one + sum;
        } else {
          sum = sum + RTA_X(w, h0 + t + W - 1) - RTA_X(w, h0 + t - 1);
        }
        best = max(best, make_key(sum, t));
      }
      tstar = (int)(C::KM - (best & C::KM));
      rawsum = (int)(best >> C::KB);
      if constexpr (WANT_TIME) {
        // a7 numerator: re-read the winning window (dynamic index -> shared memory)
        const WindowReader<C> tr(unit, h0 + tstar);
#pragma unroll
        for (int k = 1; k < W; ++k) relnum += k * tr.read(k);
      }
    } else if constexpr (MODE == MODE_FIR) {
      // response on raw samples (the pedestal shifts every y(t) by the same
      // c0*ped); signed compare, strict '>' scanning upwards = earliest on ties
      int best = 0;
      tstar = 0;
      bool done = false;
      if constexpr (C::BITS == 16) {
        if (ma.fir_packed) {
          // small taps: the register copy already holds sample pairs (x[2i], x[2i+1]);
          // windows at odd samples use the pairs (x[2i+1], x[2i+2]); one IDP.2A per pair
          constexpr int KP = (W + 1) / 2, NWD = C::NWORDS;
          uint32_t wo[NWD];
#pragma unroll
          for (int i = 0; i < NWD; ++i)
            wo[i] = __funnelshift_r(w[i], i + 1 < NWD ? w[i + 1] : 0u, 16);
#pragma unroll
          for (int t = 0; t < C::NWIN; ++t) {
            int y = 0;
#pragma unroll
            for (int m = 0; m < KP; ++m) {
              const int n = h0 + t + 2 * m;  // first sample of the pair (compile time)
              const int i = n >> 1;
              const uint32_t a = i < NWD ? ((n & 1) ? wo[i] : w[i]) : 0u;
              y = (m & 1) ? dp2a_u16_s8<1>(a, ma.taps2[m >> 1], y)
                          : dp2a_u16_s8<0>(a, ma.taps2[m >> 1], y);
            }
            if (t == 0 || y > best) {
              best = y;
              tstar = t;
            }
          }
          done = true;
        }
      }
      if (!done) {
#pragma unroll
        for (int k = 0; k < W; ++k) best += ma.taps[k] * (int)RTA_X(w, h0 + k);
#pragma unroll
        for (int t = 1; t < C::NWIN; ++t) {
          int y = 0;
#pragma unroll
          for (int k = 0; k < W; ++k) y += ma.taps[k] * (int)RTA_X(w, h0 + t + k);
          if (y > best) {
            best = y;
            tstar = t;
          }
        }
      }
      rawsum = best;
      const WindowReader<C> tr(unit, h0 + tstar);
#pragma unroll
      for (int k = 1; k < W; ++k) relnum += k * ma.taps[k] * tr.read(k);
    } else {
      if constexpr (MODE == MODE_FIXED) {
        tstar = clamp_start(__ldg(ma.window_start + p), S, W);
      } else {  // MODE_LOCAL_PEAK: largest sample, earliest on ties, one max per sample
        constexpr int PB = C::PB;
        constexpr uint32_t PM = (1u << PB) - 1u;
        uint32_t best = (RTA_X(w, h0) << PB) | PM;
#pragma unroll
        for (int k = 1; k < S; ++k)
          best = max(best, (RTA_X(w, h0 + k) << PB) + (PM - (uint32_t)k));
        tstar = clamp_start((int)(PM - (best & PM)) - ma.shift, S, W);
      }
      const WindowReader<C> tr(unit, h0 + tstar);
      rawsum = tr.read(0);
#pragma unroll
      for (int k = 1; k < W; ++k) {
        const int x = tr.read(k);
        rawsum += x;
        relnum += k * x;
      }
    }
    const int ped = __ldg(pedestal + p);
    const float gn = __ldg(gain + p);
    if constexpr (!WANT_TIME) {
      static_assert(WANT_TIME || MODE == MODE_SLIDING, "only the sliding extractor defers a7");
      res[j] = finish_charge(W, rawsum, tstar, ped, gn);
    } else if constexpr (MODE == MODE_FIR)
      res[j] = finish_trace(W, rawsum, tstar, relnum, ped, gn, ma.c0, ma.c1);
    else
      res[j] = finish_trace(W, rawsum, tstar, relnum, ped, gn, W, (W * (W - 1)) / 2);
    p = (p + 1 == n_pixels) ? 0u : p + 1;
  }
}

// Step a5 and the float stores: results of the unit's first n_valid traces to
// flat output index g0, g0 + 1.
template <class C>
__device__ __forceinline__ void store_results(const Result (&res)[C::TPT], const uint32_t g0,
                                              const uint32_t n_valid, int* __restrict__ out_sum,
                                              int* __restrict__ out_start,
                                              float* __restrict__ out_charge,
                                              float* __restrict__ out_time,
                                              const bool vec_store) {
  if constexpr (C::TPT == 1) {
    if (n_valid >= 1) {
      __stcs(out_sum + g0, res[0].sum);
      __stcs(out_start + g0, res[0].start);
      __stcs(out_charge + g0, res[0].charge);
      __stcs(out_time + g0, res[0].time);
    }
  } else {
    if (n_valid >= 2 && vec_store) {  // g0 is even: 8-byte stores
      __stcs(reinterpret_cast<int2*>(out_sum + g0), make_int2(res[0].sum, res[1].sum));
      __stcs(reinterpret_cast<int2*>(out_start + g0), make_int2(res[0].start, res[1].start));
      __stcs(reinterpret_cast<float2*>(out_charge + g0),
             make_float2(res[0].charge, res[1].charge));
      __stcs(reinterpret_cast<float2*>(out_time + g0), make_float2(res[0].time, res[1].time));
    } else {
#pragma unroll
      for (int j = 0; j < C::TPT; ++j) {
        if ((uint32_t)j < n_valid) {
          __stcs(out_sum + g0 + j, res[j].sum);
          __stcs(out_start + g0 + j, res[j].start);
          __stcs(out_charge + g0 + j, res[j].charge);
          __stcs(out_time + g0 + j, res[j].time);
        }
      }
    }
  }
}

template <class C, int MODE, int KEYMUL = 0>
__device__ __forceinline__ void compute_unit(const uint8_t* __restrict__ unit, const uint32_t g0,
                                             const uint32_t n_valid, const uint32_t p0,
                                             const uint32_t n_pixels,
                                             const int* __restrict__ pedestal,
                                             const float* __restrict__ gain,
                                             int* __restrict__ out_sum, int* __restrict__ out_start,
                                             float* __restrict__ out_charge,
                                             float* __restrict__ out_time, const bool vec_store,
                                             const ModeArgs& ma) {
  Result res[C::TPT];
  compute_results<C, MODE, KEYMUL>(unit, p0, n_pixels, pedestal, gain, ma, res);
  store_results<C>(res, g0, n_valid, out_sum, out_start, out_charge, out_time, vec_store);
}

// -------------------------------------------------------- generic kernel ----
// Any (S, W) inside the ABI guards, any alignment the format allows (uint16: 2
// bytes; P12: 1 byte): one thread per trace, samples read straight from global
// memory (L1/L2 absorb the re-reads).
template <int BITS>
struct GlobalTrace {
  const uint8_t* base;  // uint16: first byte of the trace; P12: first byte of the stream
  size_t n0;            // P12: flat index of the trace's first sample
  __device__ __forceinline__ GlobalTrace(const uint8_t* wf, const uint32_t g, const int S) {
    if constexpr (BITS == 16) {
      base = wf + (size_t)g * (size_t)S * 2u;
      n0 = 0;
    } else {
      base = wf;
      n0 = (size_t)g * (size_t)S;
    }
  }
  __device__ __forceinline__ uint32_t operator[](const int s) const {
    if constexpr (BITS == 16) {
      return reinterpret_cast<const uint16_t*>(base)[s];
    } else {
      const size_t n = n0 + (size_t)s;
      const uint8_t* b = base + ((3u * n) >> 1);
      const uint32_t v = (uint32_t)b[0] | ((uint32_t)b[1] << 8);
      return (v >> ((uint32_t)(n & 1u) << 2)) & 0xFFFu;
    }
  }
};

// One trace through the definition with runtime (S, W): p = calibration index.
template <int MODE, int BITS>
__device__ __forceinline__ Result generic_trace(const GlobalTrace<BITS>& tr, const int S,
                                                const int W, const uint32_t p,
                                                const int* __restrict__ pedestal,
                                                const float* __restrict__ gain,
                                                const ModeArgs& ma) {
  int tstar = 0, rawsum = 0, relnum = 0;
  if constexpr (MODE == MODE_SLIDING) {
    uint32_t sum = 0;
    for (int k = 0; k < W; ++k) sum += tr[k];
    uint32_t best = sum;
    for (int t = 1; t + W <= S; ++t) {
      sum = sum + tr[t + W - 1] - tr[t - 1];
      if (sum > best) {  // strict: earliest on ties
        best = sum;
        tstar = t;
      }
    }
    rawsum = (int)best;
    for (int k = 1; k < W; ++k) relnum += k * (int)tr[tstar + k];
  } else if constexpr (MODE == MODE_FIR) {
    int best = 0;
    for (int t = 0; t + W <= S; ++t) {
      int y = 0;
      for (int k = 0; k < W; ++k) y += ma.taps[k] * (int)tr[t + k];
      if (t == 0 || y > best) {
        best = y;
        tstar = t;
      }
    }
    rawsum = best;
    for (int k = 1; k < W; ++k) relnum += k * ma.taps[k] * (int)tr[tstar + k];
  } else {
    if constexpr (MODE == MODE_FIXED) {
      tstar = clamp_start(__ldg(ma.window_start + p), S, W);
    } else {
      int peak = 0;
      uint32_t top = tr[0];
      for (int k = 1; k < S; ++k) {
        const uint32_t x = tr[k];
        if (x > top) {
          top = x;
          peak = k;
        }
      }
      tstar = clamp_start(peak - ma.shift, S, W);
    }
    for (int k = 0; k < W; ++k) {
      const int x = (int)tr[tstar + k];
      rawsum += x;
      relnum += k * x;
    }
  }
  const int c0 = (MODE == MODE_FIR) ? ma.c0 : W;
  const int c1 = (MODE == MODE_FIR) ? ma.c1 : (W * (W - 1)) / 2;
  return finish_trace(W, rawsum, tstar, relnum, __ldg(pedestal + p), __ldg(gain + p), c0, c1);
}

// The four shapes of BASELINE.json:configs (NT, STAGES tuned on B200; see
// DESIGN.md "Kernels" for the shared-memory budget of each).
// Compile-time tunables, e.g. -DRTA_S40_NT=256 -DRTA_S40_ST=3 (threads per CTA, stages).
#ifndef RTA_S30_NT
#define RTA_S30_NT 256
#endif
#ifndef RTA_S30_ST
#define RTA_S30_ST 3
#endif
#ifndef RTA_S40_NT
#define RTA_S40_NT 256
#endif
#ifndef RTA_S40_ST
#define RTA_S40_ST 3
#endif
#ifndef RTA_S25_NT
#define RTA_S25_NT 256
#endif
#ifndef RTA_S25_ST
#define RTA_S25_ST 2
#endif
#ifndef RTA_S128_NT
#define RTA_S128_NT 64
#endif
#ifndef RTA_S128_ST
#define RTA_S128_ST 2
#endif
using CfgS30W7 = TileCfg<30, 7, RTA_S30_NT, RTA_S30_ST>;
using CfgS40W7 = TileCfg<40, 7, RTA_S40_NT, RTA_S40_ST>;
using CfgS25W4 = TileCfg<25, 4, RTA_S25_NT, RTA_S25_ST>;
using CfgS128W8 = TileCfg<128, 8, RTA_S128_NT, RTA_S128_ST>;
// The same shapes fed by a P12 stream (rta_extract_packed12).
#ifndef RTA_P30_NT
#define RTA_P30_NT 256
#endif
#ifndef RTA_P30_ST
#define RTA_P30_ST 3
#endif
#ifndef RTA_P40_NT
#define RTA_P40_NT 256
#endif
#ifndef RTA_P40_ST
#define RTA_P40_ST 3
#endif
#ifndef RTA_P25_NT
#define RTA_P25_NT 256
#endif
#ifndef RTA_P25_ST
#define RTA_P25_ST 3
#endif
#ifndef RTA_P128_NT
#define RTA_P128_NT 64
#endif
#ifndef RTA_P128_ST
#define RTA_P128_ST 2
#endif
using CfgP30W7 = TileCfg<30, 7, RTA_P30_NT, RTA_P30_ST, 12>;
using CfgP40W7 = TileCfg<40, 7, RTA_P40_NT, RTA_P40_ST, 12>;
using CfgP25W4 = TileCfg<25, 4, RTA_P25_NT, RTA_P25_ST, 12>;
using CfgP128W8 = TileCfg<128, 8, RTA_P128_NT, RTA_P128_ST, 12>;

}  // namespace

#endif
