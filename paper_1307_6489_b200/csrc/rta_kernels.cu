// rta_kernels.cu — sm_100a kernels for sliding-window signal extraction.
//
// What is computed is BASELINE.json:north_star sentence 2 (steps a1-a7 of
// SURVEY.md §8(a); the paper names the step at PAPER.md:141 §5). How it is
// computed is this file's own design:
//
//  * a1 ingest: persistent CTAs stream contiguous tiles of whole traces from
//    HBM into a ring of shared-memory stages. Dense layouts (S = 30, 40, 25)
//    use one TMA bulk copy per tile (cp.async.bulk + mbarrier complete_tx);
//    the S = 128 layout, whose 256-byte trace stride would put every lane of
//    a quarter-warp on the same banks, is copied with 16-byte cp.async into a
//    layout padded by one 16-byte chunk per trace, completion tracked by the
//    same mbarriers (cp.async.mbarrier.arrive).
//  * a2 pedestal: deferred. The pedestal is constant inside a trace, so the
//    arg-max runs on raw samples and Sum = rawsum - W*ped once per trace.
//  * a3/a4: one thread owns one trace (two when 2*S is not a multiple of 4),
//    reads it from shared memory with the widest conflict-free vector load,
//    slides the window in O(1) per step and keeps the maximum of the key
//    rawsum * 2^KB + (2^KB - 1 - t): one unsigned max per window yields the
//    largest sum and, among equals, the smallest t (earliest on ties).
//  * a5-a7: W-1 re-reads of the winning window from shared memory give the
//    time numerator; integers stay exact (int64 where a pedestal could
//    overflow int32), floats are one IEEE multiply / one IEEE divide on
//    exactly representable operands, with a double-precision path when an
//    operand exceeds 2^24 (bit-identical to rounding the double result).
//  * outputs: four coalesced 4-byte (or 8-byte) stores per thread.
//
// A generic kernel (any S, W, any 2-byte alignment) reads global memory
// directly; it is the path for shapes without a specialisation.
#include "rta_tile_kernel.cuh"

#include <atomic>
#include <mutex>
#include <unordered_map>

namespace {

template <int MODE, int BITS>
__global__ void __launch_bounds__(256)
    extract_generic_kernel(const uint8_t* __restrict__ wf, const uint32_t n_traces, const int S,
                           const int W, const uint32_t n_pixels, const uint32_t pix_inv,
                           const int* __restrict__ pedestal, const float* __restrict__ gain,
                           int* __restrict__ out_sum, int* __restrict__ out_start,
                           float* __restrict__ out_charge, float* __restrict__ out_time,
                           const __grid_constant__ ModeArgs ma) {
  for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < n_traces;
       g += gridDim.x * blockDim.x) {
    const GlobalTrace<BITS> tr(wf, g, S);
    const Result r = generic_trace<MODE, BITS>(tr, S, W, fastmod(g, n_pixels, pix_inv), pedestal,
                                               gain, ma);
    out_sum[g] = r.sum;
    out_start[g] = r.start;
    out_charge[g] = r.charge;
    out_time[g] = r.time;
  }
}

// ------------------------------------------- any shape, staged (runtime S, W) ----
// The sliding-window extractor for shapes without a specialisation (a 60-sample
// NectarCam-like readout, a 96-sample trace, another window width ...): the same
// stage ring, TMA ingest and dynamic tile scheduler as extract_tile_kernel, with
// S and W as kernel arguments. A thread still owns one unit (one trace, or two
// when S is odd), but walks it in shared memory with 16-bit loads instead of a
// register copy (register arrays need compile-time indices). What makes that
// fast for any stride:
//  * lanes l and l' hit the same bank with different words iff (l - l') * s = 0
//    mod 32, s = words per unit; with g = gcd(s, 32) those are the lanes
//    l + (32 / g) b, b = 0 .. g-1. Lane group b runs the sliding loop 2 b samples
//    behind (one word): the loop has 2 (g - 1) more iterations than windows and
//    every access of every iteration is conflict-free;
//  * g is kept <= 4: units of a multiple of 32 bytes (g >= 8) are copied with
//    16-byte cp.async into a layout padded by one chunk (as the S = 128 kernel),
//    everything else arrives by one TMA bulk copy per tile.
struct DynShape {
  int32_t S, W, n_win;
  int32_t tpt;          // traces per unit: 1 (S even) or 2
  int32_t unit_bytes;   // 2 S tpt
  int32_t unit_stride;  // unit_bytes (+ 16 when padded)
  int32_t tile_bytes;   // blockDim.x * unit_bytes
  int32_t stage_bytes;  // blockDim.x * unit_stride + slack, multiple of 128
  int32_t stages;
  int32_t g;            // gcd(unit_stride / 4, 32): 1, 2 or 4
  int32_t kb;           // key bits: 2^kb >= n_win
  uint32_t key_mul;     // 2^kb
  uint32_t peak_mul;    // local peak: 2^ceil(log2 S)
  int32_t cpu_shift;    // padded layout: log2(16-byte chunks per unit) when that is a power of two, else -1
};
constexpr int kDynMaxStages = 4;

// Steps a2-a7 of one unit (its first n_valid traces) at `unit` in shared memory,
// shape and extractor as kernel arguments. p: calibration index of the unit's
// first trace; it wraps to 0 after n_pixels - 1 (n_pixels = 0 never wraps).
template <int G, int MODE>
__device__ __forceinline__ void dyn_compute_unit(
    const DynShape& sh, const ModeArgs& ma, const uint8_t* unit, const uint32_t g0,
    const uint32_t n_valid, uint32_t p, const uint32_t n_pixels, const int* __restrict__ pedestal,
    const float* __restrict__ gain, int* __restrict__ out_sum, int* __restrict__ out_start,
    float* __restrict__ out_charge, float* __restrict__ out_time) {
  const int S = sh.S, W = sh.W, n_win = sh.n_win;
  const uint32_t KM = sh.key_mul - 1u;
  // lane group b = lane * g / 32 runs 2 b samples behind; d_max = 2 (g - 1)
  const int d = 2 * ((((int)threadIdx.x & 31) * G) >> 5);
  constexpr int d_max = 2 * (G - 1);
  for (int j = 0; j < sh.tpt; ++j) {
    const uint16_t* x = reinterpret_cast<const uint16_t*>(unit) + j * S;
    int tstar = 0, rawsum = 0, relnum = 0;
    // a loop of `n` steps in which lane group b handles index i - d at step i:
    // `body(index)` for the lanes whose index lies in [first, first + n)
    const auto skewed = [&](const int first, const int n, auto&& body) {
      int i = first;
      if (n > d_max) {
#pragma unroll
        for (int h = 0; h < d_max; ++h, ++i)  // head: the groups start one after the other
          if ((uint32_t)(i - d - first) < (uint32_t)n) body(i - d);
#pragma unroll 8
        for (; i < first + n; ++i) body(i - d);  // steady state: no predicates
#pragma unroll
        for (int h = 0; h < d_max; ++h, ++i)  // tail: the groups finish one after the other
          if ((uint32_t)(i - d - first) < (uint32_t)n) body(i - d);
      } else {
        for (; i < first + n + d_max; ++i)
          if ((uint32_t)(i - d - first) < (uint32_t)n) body(i - d);
      }
    };
    if constexpr (MODE == MODE_SLIDING) {
      uint32_t sum = 0;
#pragma unroll 4
      for (int k = 0; k < W; ++k) sum += x[k];
      uint32_t best = sum * sh.key_mul + KM;
      // window t enters x[t + W - 1] and leaves x[t - 1]; lanes outside [1, n_win)
      // read neighbouring bytes of the stage and discard them
      const uint32_t mul = sh.key_mul;
      const uint16_t* xe = x + (W - 1);
      const uint16_t* xl = x - 1;
      uint32_t low = KM;  // KM - t: every lane visits t = 1, 2, ... in order
      skewed(1, n_win - 1, [&](const int t) {
        sum = sum + xe[t] - xl[t];
        --low;
        best = max(best, sum * mul + low);
      });
      tstar = (int)(KM - (best & KM));
      rawsum = (int)(best >> sh.kb);
#pragma unroll 4
      for (int k = 1; k < W; ++k) relnum += k * (int)x[tstar + k];
    } else if constexpr (MODE == MODE_FIR) {
      // response on raw samples; strict '>' scanning upwards = earliest on ties
      int best = 0;
      for (int k = 0; k < W; ++k) best += ma.taps[k] * (int)x[k];
      skewed(1, n_win - 1, [&](const int t) {
        int y = 0;
#pragma unroll 4
        for (int k = 0; k < W; ++k) y += ma.taps[k] * (int)x[t + k];
        if (y > best) best = y, tstar = t;
      });
      rawsum = best;
      for (int k = 1; k < W; ++k) relnum += k * ma.taps[k] * (int)x[tstar + k];
    } else {
      if constexpr (MODE == MODE_FIXED) {
        tstar = clamp_start(__ldg(ma.window_start + p), S, W);
      } else {  // MODE_LOCAL_PEAK: largest sample, earliest on ties
        const uint32_t pmul = sh.peak_mul, PM = sh.peak_mul - 1u;
        uint32_t best = (uint32_t)x[0] * pmul + PM;
        skewed(1, S - 1, [&](const int k) {
          best = max(best, (uint32_t)x[k] * pmul + (PM - (uint32_t)k));
        });
        tstar = clamp_start((int)(PM - (best & PM)) - ma.shift, S, W);
      }
      rawsum = (int)x[tstar];
#pragma unroll 4
      for (int k = 1; k < W; ++k) {
        const int v = (int)x[tstar + k];
        rawsum += v;
        relnum += k * v;
      }
    }
    const int c0 = (MODE == MODE_FIR) ? ma.c0 : W;
    const int c1 = (MODE == MODE_FIR) ? ma.c1 : (W * (W - 1)) / 2;
    const Result r = finish_trace(W, rawsum, tstar, relnum, __ldg(pedestal + p), __ldg(gain + p),
                                  c0, c1);
    if ((uint32_t)j < n_valid) {
      __stcs(out_sum + g0 + j, r.sum);
      __stcs(out_start + g0 + j, r.start);
      __stcs(out_charge + g0 + j, r.charge);
      __stcs(out_time + g0 + j, r.time);
    }
    p = (p + 1 == n_pixels) ? 0u : p + 1;
  }
}

template <bool PAD, int G, int MODE>
__global__ void __launch_bounds__(256)
    extract_dyn_kernel(const uint8_t* __restrict__ wf, const uint32_t n_traces,
                       const uint32_t n_pixels, const uint32_t pix_inv,
                       const int* __restrict__ pedestal, const float* __restrict__ gain,
                       int* __restrict__ out_sum, int* __restrict__ out_start,
                       float* __restrict__ out_charge, float* __restrict__ out_time,
                       uint32_t* __restrict__ sched, const __grid_constant__ DynShape sh,
                       const __grid_constant__ ModeArgs ma) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[kDynMaxStages];
  __shared__ uint32_t tile_q[kDynMaxStages + 1];
  const int tid = threadIdx.x, NT = blockDim.x;
  const int STAGES = sh.stages, QN = STAGES + 1;
  const uint32_t tile_traces = (uint32_t)(NT * sh.tpt);
  const uint32_t n_full = n_traces / tile_traces;
  const uint32_t rem = n_traces - n_full * tile_traces;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_u32(full_bar);

  TileFeed feed(sched, n_full, STAGES);  // thread 0 only

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(bar_base + 8 * s, PAD ? NT : 1);
      tile_q[s] = feed.fetch_static();
    }
    fence_mbar_init();
    feed.prime();
  }
  __syncthreads();

  const uint32_t chunks_per_unit = (uint32_t)sh.unit_bytes / 16u;  // PAD only
  // A base pointer that is only 2-byte aligned (dense layouts only): the bulk copy
  // starts at the 16-byte boundary below the tile, so the tile lands `mis` bytes
  // into the stage; the 16-bit walk does not care. The copy of the very last
  // tile stops at the last boundary inside the caller's buffer and the final
  // < 16 bytes go halfword by halfword: nothing past the buffer is read. (The
  // first copy starts up to 14 bytes before `wf`, inside the 16-byte line that
  // holds wf[0].)
  const uint32_t mis = PAD ? 0u : (uint32_t)(reinterpret_cast<uintptr_t>(wf) & 15u);
  auto issue = [&](const uint32_t tile, const int stage) {
    const uint8_t* src = wf + (size_t)tile * (size_t)sh.tile_bytes;
    const uint32_t dst = smem_base + (uint32_t)(stage * sh.stage_bytes);
    const uint32_t bar = bar_base + 8 * stage;
    if constexpr (!PAD) {
      if (tid == 0) {
        uint32_t len = (uint32_t)sh.tile_bytes + (mis ? 16u : 0u);
        if (mis != 0 && (unsigned long long)(tile + 1u) * (unsigned long long)sh.tile_bytes + 16u - mis >
                            (unsigned long long)n_traces * 2ull * (unsigned long long)sh.S) {
          len = (uint32_t)sh.tile_bytes;  // whole 16-byte lines inside the buffer
          uint8_t* d = smem + stage * sh.stage_bytes;
          for (uint32_t b = len; b < mis + (uint32_t)sh.tile_bytes; b += 2u)
            *reinterpret_cast<uint16_t*>(d + b) = *reinterpret_cast<const uint16_t*>(src - mis + b);
        }
        mbar_expect_tx(bar, len);
        tma_bulk_g2s(dst, src - mis, len, bar);
      }
    } else {
      // chunk c of the tile belongs to unit c / chunks_per_unit: one chunk of padding per unit
      const uint32_t n_chunks = (uint32_t)sh.tile_bytes / 16u;
      if (sh.cpu_shift >= 0) {  // a power of two chunks per unit: the unit index is a shift
#pragma unroll 4
        for (uint32_t c = tid; c < n_chunks; c += NT)
          cp_async16(dst + (c + (c >> sh.cpu_shift)) * 16u, src + (size_t)c * 16u);
      } else {
        uint32_t u = (uint32_t)tid / chunks_per_unit, r = (uint32_t)tid - u * chunks_per_unit;
        const uint32_t du = (uint32_t)NT / chunks_per_unit, dr = (uint32_t)NT - du * chunks_per_unit;
        for (uint32_t c = tid; c < n_chunks; c += NT) {
          cp_async16(dst + (c + u) * 16u, src + (size_t)c * 16u);
          u += du;
          r += dr;
          if (r >= chunks_per_unit) r -= chunks_per_unit, ++u;
        }
      }
      cp_async_mbar_arrive(bar);
    }
  };

  for (int s = 0; s < STAGES; ++s) {
    const uint32_t tile = tile_q[s];
    if (tile < n_full) issue(tile, s);
  }
  uint32_t pre = 0;
  if (tid == 0) pre = feed.fetch();

  const int S = sh.S;

  auto compute = [&](const uint8_t* unit, const uint32_t g0, const uint32_t n_valid, const uint32_t p) {
    dyn_compute_unit<G, MODE>(sh, ma, unit, g0, n_valid, p, n_pixels, pedestal, gain, out_sum,
                              out_start, out_charge, out_time);
  };

  uint32_t tile;
  for (uint32_t j = 0;; ++j) {
    tile = tile_q[j % QN];
    if (tile >= n_full) break;
    const int stage = (int)(j % (uint32_t)STAGES);
    const uint32_t parity = (j / (uint32_t)STAGES) & 1u;
    if (tid == 0) {
      tile_q[(j + STAGES) % QN] = pre;
      pre = feed.fetch();
    }
    mbar_wait(bar_base + 8 * stage, parity);
    const uint8_t* unit = smem + stage * sh.stage_bytes + mis + tid * sh.unit_stride;
    const uint32_t g0 = tile * tile_traces + (uint32_t)(tid * sh.tpt);
    compute(unit, g0, (uint32_t)sh.tpt, fastmod(g0, n_pixels, pix_inv));
    __syncthreads();
    const uint32_t next = tile_q[(j + STAGES) % QN];
    if (next < n_full) issue(next, stage);
  }

  // ragged tail (< one tile of traces): plain copies, by the CTA that drew index n_full
  if (rem != 0 && tile == n_full) {
    const uint8_t* src = wf + (size_t)n_full * (size_t)sh.tile_bytes;
    const uint32_t n_hw = rem * (uint32_t)S;  // halfwords
    const uint32_t unit_hw = (uint32_t)sh.unit_bytes / 2u, pad_hw = (uint32_t)(sh.unit_stride - sh.unit_bytes) / 2u;
    for (uint32_t i = tid; i < n_hw; i += NT) {
      const uint32_t dsti = PAD ? i + (i / unit_hw) * pad_hw : i;
      reinterpret_cast<uint16_t*>(smem)[dsti] = reinterpret_cast<const uint16_t*>(src)[i];
    }
    __syncthreads();
    const uint32_t first = (uint32_t)(tid * sh.tpt);
    if (first < rem) {
      const uint8_t* unit = smem + tid * sh.unit_stride;
      const uint32_t g0 = n_full * tile_traces + first;
      compute(unit, g0, rem - first, fastmod(g0, n_pixels, pix_inv));
    }
  }

  if (tid == 0) feed.leave();
}

// ------------------------------------------------- mixed-camera batches ----
// SURVEY.md §8(f) NEXT-3 (readings R28-R30). The host plan cuts every
// block (one telescope, one event) into tiles of at most TILE_TRACES traces of
// one shape; one launch per shape class walks its tile table with the same
// stage ring and dynamic scheduler as the uniform kernel. A tile whose source
// is 16-byte aligned arrives by TMA bulk copy (cp.async 16 for the padded
// S = 128 layout); a 4-byte-aligned one by 4-byte cp.async; anything else by
// plain halfword copies. Every thread arrives on the stage's mbarrier through
// cp.async.mbarrier.arrive, so the three ways share one completion mechanism.
// (RaggedTile, the ingest helpers and the kernel body live in rta_tile_kernel.cuh: the run-time
// specialisations compile the same source)
template <class C>
__global__ void __launch_bounds__(C::NT)
    extract_ragged_kernel(const uint8_t* __restrict__ wf, const RaggedTile* __restrict__ tiles,
                          const uint32_t n_tiles, const int* __restrict__ pedestal,
                          const float* __restrict__ gain, int* __restrict__ out_sum,
                          int* __restrict__ out_start, float* __restrict__ out_charge,
                          float* __restrict__ out_time, const int vec_store,
                          uint32_t* __restrict__ sched) {
  ragged_kernel_body<C>(wf, tiles, n_tiles, pedestal, gain, out_sum, out_start, out_charge, out_time,
                        vec_store, sched);
}

// Mixed-camera blocks of a shape without a specialisation: the tile table and
// ingest of extract_ragged_kernel with the runtime-shape walk of extract_dyn_kernel.
template <bool PAD, int G>
__global__ void __launch_bounds__(256)
    extract_ragged_dyn_kernel(const uint8_t* __restrict__ wf, const RaggedTile* __restrict__ tiles,
                              const uint32_t n_tiles, const int* __restrict__ pedestal,
                              const float* __restrict__ gain, int* __restrict__ out_sum,
                              int* __restrict__ out_start, float* __restrict__ out_charge,
                              float* __restrict__ out_time, uint32_t* __restrict__ sched,
                              const __grid_constant__ DynShape sh) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[kDynMaxStages];
  __shared__ uint32_t tile_q[kDynMaxStages + 1];
  __shared__ RaggedTile desc_q[kDynMaxStages + 1];
  const int tid = threadIdx.x, NT = blockDim.x;
  const int STAGES = sh.stages, QN = STAGES + 1;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_u32(full_bar);
  const ModeArgs ma = {};

  TileFeed feed(sched, n_tiles, STAGES);  // thread 0 only
  const auto entry = [&](const uint32_t ti) -> RaggedTile {
    if (ti < n_tiles) return tiles[ti];
    return RaggedTile{0ull, 0u, 0u};
  };
  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(bar_base + 8 * s, NT);
      tile_q[s] = feed.fetch_static();
      desc_q[s] = entry(tile_q[s]);
    }
    fence_mbar_init();
    feed.prime();
  }
  __syncthreads();

  const uint32_t UB = (uint32_t)sh.unit_bytes, PADB = (uint32_t)(sh.unit_stride - sh.unit_bytes);
  const uint32_t TRACE_BYTES = 2u * (uint32_t)sh.S;
  auto issue = [&](const int slot, const int stage) {
    const RaggedTile t = desc_q[slot];
    const uint8_t* src = wf + (size_t)(t.src & kRaggedOffMask);
    const uint32_t bytes = (uint32_t)(t.src >> 48) * TRACE_BYTES;
    uint8_t* dstp = smem + stage * sh.stage_bytes;
    const uint32_t dst = smem_base + (uint32_t)(stage * sh.stage_bytes);
    const uint32_t bar = bar_base + 8 * stage;
    const uint32_t mis = (uint32_t)(reinterpret_cast<uintptr_t>(src) & 15u);
    uint32_t done;  // bytes moved by the wide path; the rest goes halfword by halfword
    if (mis == 0) {
      if constexpr (!PAD) {
        done = bytes & ~15u;
        if (tid == 0 && done != 0) {
          mbar_expect_tx_only(bar, done);
          tma_bulk_g2s(dst, src, done, bar);
        }
      } else {
        done = bytes & ~15u;  // whole units are whole chunks; a last half unit may not be
        const uint32_t cpu = UB / 16u;  // chunks per unit: one chunk of padding after each
        if (sh.cpu_shift >= 0) {
          for (uint32_t c = tid; c < done / 16u; c += NT)
            cp_async16(dst + (c + (c >> sh.cpu_shift)) * 16u, src + (size_t)c * 16u);
        } else {
          uint32_t u = (uint32_t)tid / cpu, r = (uint32_t)tid - u * cpu;
          const uint32_t du = (uint32_t)NT / cpu, dr = (uint32_t)NT - du * cpu;
          for (uint32_t c = tid; c < done / 16u; c += NT) {
            cp_async16(dst + (c + u) * 16u, src + (size_t)c * 16u);
            u += du;
            r += dr;
            if (r >= cpu) r -= cpu, ++u;
          }
        }
      }
    } else if ((mis & 3u) == 0) {
      done = bytes & ~3u;
      for (uint32_t c = tid; c < done / 4u; c += NT) {
        uint32_t d = c * 4u;
        if constexpr (PAD) d += (d / UB) * PADB;
        cp_async4(dst + d, src + (size_t)c * 4u);
      }
    } else {
      done = 0;
    }
    for (uint32_t b = done + 2u * tid; b < bytes; b += 2u * NT) {
      uint32_t d = b;
      if constexpr (PAD) d += (b / UB) * PADB;
      *reinterpret_cast<uint16_t*>(dstp + d) = *reinterpret_cast<const uint16_t*>(src + b);
    }
    cp_async_mbar_arrive(bar);  // counts once this thread's cp.async copies have landed
  };

  for (int s = 0; s < STAGES; ++s) {
    const uint32_t tile = tile_q[s];
    if (tile < n_tiles) issue(s, s);
  }
  uint32_t pre = 0;
  RaggedTile pre_d = {0ull, 0u, 0u};
  if (tid == 0) {
    pre = feed.fetch();
    pre_d = entry(pre);
  }

  for (uint32_t j = 0;; ++j) {
    const uint32_t tile = tile_q[j % QN];
    if (tile >= n_tiles) break;
    const int stage = (int)(j % (uint32_t)STAGES);
    const uint32_t parity = (j / (uint32_t)STAGES) & 1u;
    if (tid == 0) {
      tile_q[(j + STAGES) % QN] = pre;
      desc_q[(j + STAGES) % QN] = pre_d;
      pre = feed.fetch();
      pre_d = entry(pre);
    }
    const RaggedTile t = desc_q[j % QN];
    const uint32_t n = (uint32_t)(t.src >> 48);
    mbar_wait(bar_base + 8 * stage, parity);
    const uint32_t first = (uint32_t)(tid * sh.tpt);
    if (first < n) {
      const uint8_t* unit = smem + stage * sh.stage_bytes + tid * sh.unit_stride;
      dyn_compute_unit<G, MODE_SLIDING>(sh, ma, unit, t.out_base + first, n - first,
                                        t.cal0 + first, t.cal0 + n, pedestal, gain, out_sum,
                                        out_start, out_charge, out_time);  // wrap: see above
    }
    __syncthreads();
    const uint32_t next = tile_q[(j + STAGES) % QN];
    if (next < n_tiles) issue((int)((j + STAGES) % QN), stage);
  }

  if (tid == 0) feed.leave();
}

// Shapes without a specialisation: one thread per trace, one tile (<= 256 traces) per CTA pass.
__global__ void __launch_bounds__(256)
    extract_ragged_generic_kernel(const uint8_t* __restrict__ wf,
                                  const RaggedTile* __restrict__ tiles, const uint32_t n_tiles,
                                  const int S, const int W, const int* __restrict__ pedestal,
                                  const float* __restrict__ gain, int* __restrict__ out_sum,
                                  int* __restrict__ out_start, float* __restrict__ out_charge,
                                  float* __restrict__ out_time) {
  const ModeArgs ma = {};
  for (uint32_t ti = blockIdx.x; ti < n_tiles; ti += gridDim.x) {
    const RaggedTile t = tiles[ti];
    const uint32_t n = (uint32_t)(t.src >> 48);
    // a tile may hold more traces than the CTA has threads (tables cut for the 512-trace
    // tiles of the staged kernels can end up here when those are not available)
    for (uint32_t i = threadIdx.x; i < n; i += blockDim.x) {
      const GlobalTrace<16> tr(wf + (size_t)(t.src & kRaggedOffMask), i, S);
      const Result r = generic_trace<MODE_SLIDING, 16>(tr, S, W, t.cal0 + i, pedestal, gain, ma);
      const uint32_t g = t.out_base + i;
      out_sum[g] = r.sum;
      out_start[g] = r.start;
      out_charge[g] = r.charge;
      out_time[g] = r.time;
    }
  }
}

// ------------------------------------------ several lanes per trace ----
// LPT lanes own one trace (32 / LPT traces per warp at a time): the formulation
// with warp-shuffle prefix sums that BASELINE.json:north_star (b) names. Lane j
// of a group loads the 16-byte chunks j, j + LPT, ... of the trace straight
// from global memory (coalesced), forms the inclusive prefix sums of its 8
// samples, a shuffle scan over the group's lanes adds the lanes in front and a
// carry the rounds before, and the exclusive prefix array X[i] = x[0] + ... + x[i-1]
// goes to shared memory. Window sums are then X[t + W] - X[t] (a lane takes four
// consecutive t per step with a 16-byte load), the arg-max key is reduced over the group
// by shuffles, and lane 0 of the group finishes the trace. Any n_samples that
// is a multiple of 8 on a 16-byte-aligned base, any W: this is the kernel for
// traces too long for a thread (units above 1152 bytes), where the alternative
// is the strided generic kernel; on S = 128 it was measured against the
// thread-per-trace specialisation.
template <int LPT>
__global__ void __launch_bounds__(256)
    extract_lanes_kernel(const uint8_t* __restrict__ wf, const uint32_t n_traces, const int S,
                         const int W, const int kb, const uint32_t n_pixels,
                         const uint32_t pix_inv, const int* __restrict__ pedestal,
                         const float* __restrict__ gain, int* __restrict__ out_sum,
                         int* __restrict__ out_start, float* __restrict__ out_charge,
                         float* __restrict__ out_time) {
  extern __shared__ __align__(16) uint32_t lanes_smem[];
  const int lane = threadIdx.x & 31, j = lane % LPT;
  const uint32_t gmask = LPT == 32 ? 0xFFFFFFFFu : (((1u << (LPT & 31)) - 1u) << (lane - j));
  const uint32_t groups = blockDim.x / LPT, gi = threadIdx.x / LPT;
  // per group: the EXCLUSIVE prefix sums X[i] = x[0] + ... + x[i-1], i = 0 .. S (X[0] = 0),
  // 16-byte aligned, padded so that the 4-window steps below may read up to X[S + 6]
  const uint32_t pstride = (uint32_t)S + 12u;
  uint32_t* X = lanes_smem + gi * pstride;
  const int n_chunks = S >> 3, n_win = S - W + 1;
  const uint32_t key_mul = 1u << kb, KM = key_mul - 1u;
  constexpr int U = 4;  // chunks in flight per lane: the loads of a step go out before any is used
  for (uint32_t g = blockIdx.x * groups + gi; g < n_traces; g += gridDim.x * groups) {
    const uint4* src = reinterpret_cast<const uint4*>(wf + (size_t)g * (size_t)S * 2u);
    uint32_t carry = 0;
    for (int c0 = 0; c0 < n_chunks; c0 += U * LPT) {
      uint4 v[U];
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int c = c0 + u * LPT + j;
        v[u] = c < n_chunks ? __ldcs(src + c) : make_uint4(0u, 0u, 0u, 0u);
      }
#pragma unroll
      for (int u = 0; u < U; ++u) {
        const int c = c0 + u * LPT + j;
        uint4 lo, hi;  // exclusive prefix sums inside the chunk, then its total
        lo.x = 0u;
        lo.y = v[u].x & 0xFFFFu;
        lo.z = lo.y + (v[u].x >> 16);
        lo.w = lo.z + (v[u].y & 0xFFFFu);
        hi.x = lo.w + (v[u].y >> 16);
        hi.y = hi.x + (v[u].z & 0xFFFFu);
        hi.z = hi.y + (v[u].z >> 16);
        hi.w = hi.z + (v[u].w & 0xFFFFu);
        const uint32_t total = hi.w + (v[u].w >> 16);
        uint32_t incl = total;  // scan of the chunk totals over the group's lanes
#pragma unroll
        for (int o = 1; o < LPT; o <<= 1) {
          const uint32_t up = __shfl_up_sync(gmask, incl, o, LPT);
          if (j >= o) incl += up;
        }
        const uint32_t base = carry + incl - total;
        if (c < n_chunks) {
          uint4* dst = reinterpret_cast<uint4*>(X + 8 * c);
          dst[0] = make_uint4(base, base + lo.y, base + lo.z, base + lo.w);
          dst[1] = make_uint4(base + hi.x, base + hi.y, base + hi.z, base + hi.w);
        }
        carry += __shfl_sync(gmask, incl, LPT - 1, LPT);
      }
    }
    if (j == 0) X[S] = carry;  // the sum of the whole trace
    __syncwarp(gmask);
    // a3 + a4: Sum(t) = X[t + W] - X[t], four consecutive windows per lane and step
    // (16-byte loads; windows past the end are masked), packed (sum, earliest) key
    uint32_t best = 0;  // every key is >= 0 and window 0 exists
    for (int t = 4 * j; t < n_win; t += 4 * LPT) {
      const uint4 a = *reinterpret_cast<const uint4*>(X + t);
      const uint32_t* e = X + t + W;
      const uint32_t k0 = (e[0] - a.x) * key_mul + (KM - (uint32_t)t);
      const uint32_t k1 = (e[1] - a.y) * key_mul + (KM - (uint32_t)t - 1u);
      const uint32_t k2 = (e[2] - a.z) * key_mul + (KM - (uint32_t)t - 2u);
      const uint32_t k3 = (e[3] - a.w) * key_mul + (KM - (uint32_t)t - 3u);
      best = max(best, k0);
      if (t + 1 < n_win) best = max(best, k1);
      if (t + 2 < n_win) best = max(best, k2);
      if (t + 3 < n_win) best = max(best, k3);
    }
#pragma unroll
    for (int o = LPT / 2; o > 0; o >>= 1) best = max(best, __shfl_xor_sync(gmask, best, o, LPT));
    const int tstar = (int)(KM - (best & KM));
    const int rawsum = (int)(best >> kb);
    // a7 numerator: sum_k k raw[t* + k], raw[i] = X[i + 1] - X[i]
    int relnum = 0;
    for (int k = j; k < W; k += LPT) relnum += k * (int)(X[tstar + k + 1] - X[tstar + k]);
#pragma unroll
    for (int o = LPT / 2; o > 0; o >>= 1) relnum += __shfl_xor_sync(gmask, relnum, o, LPT);
    if (j == 0) {
      const uint32_t p = fastmod(g, n_pixels, pix_inv);
      const Result r = finish_trace(W, rawsum, tstar, relnum, __ldg(pedestal + p), __ldg(gain + p),
                                    W, (W * (W - 1)) / 2);
      __stcs(out_sum + g, r.sum);
      __stcs(out_start + g, r.start);
      __stcs(out_charge + g, r.charge);
      __stcs(out_time + g, r.time);
    }
    __syncwarp(gmask);  // the prefix array is rewritten by the next trace
  }
}

// ------------------------------------------ long traces: a thread per segment ----
// Traces too long for one thread (units above 1152 bytes). A tile is TR whole
// traces in a ring of 2-4 stages (mbarrier per stage, dynamic tile scheduler as
// in the other staged kernels). The n_win windows of a trace are cut into
// segments of L consecutive window starts; a thread takes one segment: it sums
// the first window (W loads) and then slides like the runtime-shape kernel (two
// 16-bit shared-memory loads per window; the samples up to W - 1 past its
// segment belong to the same trace), keeping the packed (sum, earliest) key of
// its segment. The keys of a trace meet in one atomicMax on a shared-memory word
// per trace: the packed key orders by sum first and earlier start second across
// segments exactly as inside one. After a barrier thread i finishes trace i of
// the tile (a5-a7).
// Banks: L / 2 is odd, so consecutive segments of a trace start on consecutive
// (odd-stride) banks. When n_samples is a multiple of 8 every trace is copied by
// its own bulk copy to a stride of `trace_stride` bytes chosen so that segment 0
// of the next trace continues that bank sequence (slots per trace nslot = nseg
// rounded up to a multiple of 4, stride = nslot L / 2 words mod 32): 32
// consecutive slots never share a bank. Other n_samples keep the dense layout
// (one bulk copy per tile, TR n_samples a multiple of 8 so tiles start on
// 16-byte boundaries; a last tile whose byte count is not a multiple of 16 gets
// its last bytes halfword by halfword from the issuing thread).
struct SegShape {
  int32_t S, W, n_win;
  int32_t L;             // window starts per segment
  int32_t nseg;          // ceil(n_win / L)
  int32_t nslot;         // thread slots per trace (>= nseg; the extra ones idle)
  uint32_t nslot_inv;    // min(floor(2^32 / nslot), 2^32 - 1)
  int32_t TR;            // traces per tile
  int32_t trace_stride;  // bytes between traces in a stage: 2 S (dense) or padded
  int32_t stage_bytes;   // multiple of 128
  int32_t stages;
  int32_t kb;
  uint32_t key_mul;
};
constexpr int kSegMaxStages = 4;
constexpr int kSegMaxTR = 64;

// The windows 1 .. nw-1 of a segment whose window 0 starts at x (sum = its sum, low = the
// low key bits of window 0): the best packed key of the segment.
// 16-bit loads, any alignment: window i enters x[W-1+i] and leaves x[i-1].
__device__ __forceinline__ uint32_t seg_slide_u16(const uint16_t* x, const int W, const int nw,
                                                  uint32_t sum, const uint32_t mul, uint32_t low) {
  uint32_t best = sum * mul + low;
  const uint16_t* xe = x + (W - 1);
  const uint16_t* xl = x - 1;
  // one add-sub per window, in order: left to the compiler the unrolled sums are
  // re-associated into a tree that costs twice the adds (measured)
#pragma unroll 8
  for (int i = 1; i < nw; ++i) {
    const uint32_t e = xe[i], l = xl[i];
    asm("{ .reg .u32 t; add.u32 t, %0, %1; sub.u32 %0, t, %2; }" : "+r"(sum) : "r"(e), "r"(l));
    --low;
    best = max(best, sum * mul + low);
  }
  return best;
}

// x on a 4-byte boundary: two windows per step from one 32-bit load per stream. The
// leaving pair (x[2m], x[2m+1]) is word m; the entering pair (x[W+2m], x[W+2m+1]) is
// word W/2 + m, or for odd W the funnel shift of two consecutive words (the second is
// kept for the next step). Both window sums come from the sum two windows back by
// dp2a (IDP.2A): + e.lo - l.lo and + e.lo + e.hi - l.lo - l.hi.
template <bool WODD>
__device__ __forceinline__ uint32_t seg_slide_pairs(const uint16_t* x, const int W, const int nw,
                                                    uint32_t sum, const uint32_t mul, uint32_t low) {
  uint32_t best = sum * mul + low;
  const uint32_t* xl = reinterpret_cast<const uint32_t*>(x);
  const uint32_t* xe = xl + (W >> 1);
  constexpr uint32_t kPlus = 0x01010001u;   // bytes (1, 0 | 1, 1): .lo adds a.lo, .hi adds a.lo + a.hi
  constexpr uint32_t kMinus = 0xFFFF00FFu;  // bytes (-1, 0 | -1, -1)
  const int np = (nw - 1) >> 1;
  uint32_t ecur = WODD ? xe[0] : 0u;
  int s = (int)sum;
#pragma unroll 4
  for (int m = 0; m < np; ++m) {
    const uint32_t lw = xl[m];
    uint32_t ew;
    if constexpr (WODD) {
      const uint32_t enext = xe[m + 1];
      ew = __funnelshift_r(ecur, enext, 16);
      ecur = enext;
    } else {
      ew = xe[m];
    }
    const int s1 = dp2a_u16_s8<0>(lw, kMinus, dp2a_u16_s8<0>(ew, kPlus, s));
    s = dp2a_u16_s8<1>(lw, kMinus, dp2a_u16_s8<1>(ew, kPlus, s));
    low -= 2u;
    best = max(best, (uint32_t)s1 * mul + (low + 1u));
    best = max(best, (uint32_t)s * mul + low);
  }
  if ((nw - 1) & 1) {  // the last window of an even-length segment
    const int i = nw - 1;
    s += (int)x[W - 1 + i] - (int)x[i - 1];
    best = max(best, (uint32_t)s * mul + (low - 1u));
  }
  return best;
}

__global__ void __launch_bounds__(256)
    extract_seg_kernel(const uint8_t* __restrict__ wf, const uint32_t n_traces,
                       const uint32_t n_pixels, const uint32_t pix_inv,
                       const int* __restrict__ pedestal, const float* __restrict__ gain,
                       int* __restrict__ out_sum, int* __restrict__ out_start,
                       float* __restrict__ out_charge, float* __restrict__ out_time,
                       uint32_t* __restrict__ sched, const __grid_constant__ SegShape sh) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[kSegMaxStages];
  __shared__ uint32_t tile_q[kSegMaxStages + 1];
  __shared__ uint32_t bestk_all[kSegMaxStages][kSegMaxTR];  // per stage: tile j + 1 collects keys while tile j is finished
  const int tid = threadIdx.x, NT = blockDim.x;
  const int STAGES = sh.stages, QN = STAGES + 1;
  const int S = sh.S, W = sh.W;
  const uint32_t TR = (uint32_t)sh.TR;
  const uint32_t n_tiles = (n_traces + TR - 1u) / TR;
  const uint32_t trace_bytes = 2u * (uint32_t)S;
  const bool dense = (uint32_t)sh.trace_stride == trace_bytes;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_u32(full_bar);

  TileFeed feed(sched, n_tiles, STAGES);  // thread 0 only

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(bar_base + 8 * s, 1);
      tile_q[s] = feed.fetch_static();
    }
    fence_mbar_init();
    feed.prime();
  }
  for (int i = tid; i < kSegMaxStages * kSegMaxTR; i += NT) (&bestk_all[0][0])[i] = 0u;  // every key is >= 0 and window 0 always exists
  __syncthreads();

  auto tile_traces = [&](const uint32_t tile) {
    const uint32_t left = n_traces - tile * TR;
    return left < TR ? left : TR;
  };
  auto issue = [&](const uint32_t tile, const int stage) {  // thread 0
    const uint8_t* src = wf + (size_t)tile * (size_t)TR * (size_t)trace_bytes;
    const uint32_t n_tr = tile_traces(tile);
    const uint32_t bar = bar_base + 8 * stage;
    const uint32_t dst = smem_base + (uint32_t)(stage * sh.stage_bytes);
    if (dense) {
      const uint32_t bytes = n_tr * trace_bytes;
      const uint32_t len = bytes & ~15u;
      uint8_t* d = smem + stage * sh.stage_bytes;
      for (uint32_t b = len; b < bytes; b += 2u)  // the last tile only: nothing past the buffer is read
        *reinterpret_cast<uint16_t*>(d + b) = *reinterpret_cast<const uint16_t*>(src + b);
      mbar_expect_tx(bar, len);
      if (len != 0) tma_bulk_g2s(dst, src, len, bar);
    } else {  // one copy per trace (a multiple of 16 bytes each) to the padded stride
      mbar_expect_tx(bar, n_tr * trace_bytes);
      for (uint32_t i = 0; i < n_tr; ++i)
        tma_bulk_g2s(dst + i * (uint32_t)sh.trace_stride, src + (size_t)i * trace_bytes, trace_bytes, bar);
    }
  };

  if (tid == 0) {
    for (int s = 0; s < STAGES; ++s)
      if (tile_q[s] < n_tiles) issue(tile_q[s], s);
  }
  uint32_t pre = 0;
  if (tid == 0) pre = feed.fetch();

  const uint32_t mul = sh.key_mul, KM = sh.key_mul - 1u;
  const uint32_t stride_hw = (uint32_t)sh.trace_stride / 2u;
  // every segment starts on a 4-byte boundary (L is even) when the traces do
  const bool pairs = (stride_hw & 1u) == 0u;
  for (uint32_t j = 0;; ++j) {
    const uint32_t tile = tile_q[j % QN];
    if (tile >= n_tiles) break;
    const int stage = (int)(j % (uint32_t)STAGES);
    const uint32_t parity = (j / (uint32_t)STAGES) & 1u;
    if (tid == 0) {
      tile_q[(j + STAGES) % QN] = pre;
      pre = feed.fetch();
    }
    const uint32_t n_tr = tile_traces(tile);
    // the thread that will finish trace `tid` of the tile asks for its calibration now
    int ped = 0;
    float gn = 0.0f;
    if ((uint32_t)tid < n_tr) {
      const uint32_t p = fastmod(tile * TR + (uint32_t)tid, n_pixels, pix_inv);
      ped = __ldg(pedestal + p), gn = __ldg(gain + p);
    }
    mbar_wait(bar_base + 8 * stage, parity);
    const uint16_t* base = reinterpret_cast<const uint16_t*>(smem + stage * sh.stage_bytes);
    uint32_t* bestk = bestk_all[stage];
    const uint32_t n_q = n_tr * (uint32_t)sh.nslot;
    const int lane = tid & 31;
    for (uint32_t q0 = (uint32_t)(tid - lane); q0 < n_q; q0 += NT) {  // whole warps: the key reduction needs every lane
      const uint32_t q = q0 + (uint32_t)lane;
      uint32_t tr = __umulhi(q, sh.nslot_inv);
      uint32_t seg = q - tr * (uint32_t)sh.nslot;
      if (seg >= (uint32_t)sh.nslot) seg -= (uint32_t)sh.nslot, ++tr;
      const bool active = q < n_q && seg < (uint32_t)sh.nseg;  // not past the tile, not a padding slot
      uint32_t best = 0u;  // every real key is >= 0
      if (active) {
        const int t0 = (int)seg * sh.L;
        const int nw = min(sh.L, sh.n_win - t0);
        const uint16_t* x = base + tr * stride_hw + t0;
        uint32_t sum = 0;
#pragma unroll 4
        for (int k = 0; k < W; ++k) sum += x[k];
        best = pairs ? ((W & 1) ? seg_slide_pairs<true>(x, W, nw, sum, mul, KM - (uint32_t)t0)
                                : seg_slide_pairs<false>(x, W, nw, sum, mul, KM - (uint32_t)t0))
                     : seg_slide_u16(x, W, nw, sum, mul, KM - (uint32_t)t0);
      }
      // the segments of a trace meet in bestk[tr]: one REDUX + one atomic per warp when the warp's
      // lanes all work on one trace (32 same-address atomics serialise), else one atomic per lane
      const uint32_t act = __ballot_sync(0xFFFFFFFFu, active);
      if (act != 0u) {
        const uint32_t tr_ref = __shfl_sync(0xFFFFFFFFu, tr, __ffs((int)act) - 1);
        if (__all_sync(0xFFFFFFFFu, !active || tr == tr_ref)) {
          const uint32_t m = __reduce_max_sync(0xFFFFFFFFu, best);
          if (lane == 0) atomicMax(&bestk[tr_ref], m);
        } else if (active) {
          atomicMax(&bestk[tr], best);
        }
      }
    }
    __syncthreads();
    if ((uint32_t)tid < n_tr) {
      const uint32_t best = bestk[tid];
      bestk[tid] = 0u;
      const int tstar = (int)(KM - (best & KM));
      const int rawsum = (int)(best >> sh.kb);
      const uint16_t* x = base + (uint32_t)tid * stride_hw + tstar;
      int relnum = 0;
#pragma unroll 4
      for (int k = 1; k < W; ++k) relnum += k * (int)x[k];
      const uint32_t g = tile * TR + (uint32_t)tid;
      const Result r = finish_trace(W, rawsum, tstar, relnum, ped, gn, W, (W * (W - 1)) / 2);
      __stcs(out_sum + g, r.sum);
      __stcs(out_start + g, r.start);
      __stcs(out_charge + g, r.charge);
      __stcs(out_time + g, r.time);
    }
    // The stage may be refilled once the finishing threads are done with it. They all sit in
    // warp 0 when a tile holds at most 32 traces: the other warps go on to the next tile (its
    // own stage and key words) without waiting; the next barrier orders everything else.
    if (TR > 32u) __syncthreads(); else __syncwarp();
    if (tid == 0) {
      const uint32_t next = tile_q[(j + STAGES) % QN];
      if (next < n_tiles) issue(next, stage);
    }
  }
  if (tid == 0) feed.leave();
}

// ------------------------------------------------------------- dispatch ----
constexpr int kMaxDevices = 32;
#ifdef RTA_TESTING
// Process-wide dispatch switches: in librta_testing.so only (this file is compiled a
// second time with -DRTA_TESTING for it).
std::atomic<int> g_force_lanes{0};  // tests / measurements: lanes per trace to use wherever the lanes kernel can run
std::atomic<bool> g_static_schedule{false};  // tests: force the static round-robin
// tests / measurements: segment length, traces per tile and threads per CTA of the segment
// kernel (0 = chosen per shape); a forced L also sends shapes that have a faster kernel there
std::atomic<int> g_seg_L{0}, g_seg_TR{0}, g_seg_NT{0}, g_seg_ST{0};
#else
// The shipped library has no switches: every read below is the constant 0 / false, and
// what only a switch could select (the lanes kernel with fewer than 32 lanes, the
// segment kernel on shapes that have a faster one) is not compiled into it.
struct NoSwitch {
  constexpr int load(std::memory_order = std::memory_order_relaxed) const { return 0; }
  constexpr operator bool() const { return false; }
};
constexpr NoSwitch g_static_schedule{}, g_seg_L{}, g_seg_TR{}, g_seg_NT{}, g_seg_ST{};
#endif

struct DeviceInfo {
  std::atomic<int> ready{0};
  int sms = 0;
};
DeviceInfo g_dev[kMaxDevices];

cudaError_t device_sms(int dev, int* sms) {
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  DeviceInfo& d = g_dev[dev];
  if (!d.ready.load(std::memory_order_acquire)) {
    int n = 0;
    cudaError_t e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return e;
    d.sms = n;
    d.ready.store(1, std::memory_order_release);
  }
  *sms = d.sms;
  return cudaSuccess;
}

// ---- scheduler words: one {next tile, CTAs done} pair per (device, stream) ----
// Eager launches on one stream run one after the other, so a pair owned by a
// stream is never shared by two running kernels; the kernel leaves it zeroed.
// Launches recorded into a CUDA graph get no pair (sched_words).
constexpr int kSchedSlots = 1024;      // distinct streams per device before falling back
constexpr int kSchedSlotWords = 32;    // 128 bytes apart: one L2 line per pair

struct SchedPool {
  std::mutex mu;
  uint32_t* base[kMaxDevices] = {};
  bool failed[kMaxDevices] = {};
  std::unordered_map<uintptr_t, int> slot_of[kMaxDevices];
};
SchedPool g_sched;

// nullptr = no pair available (static round-robin is used instead)
uint32_t* sched_words(int dev, cudaStream_t stream) {
  if (stream == cudaStreamPerThread) return nullptr;  // one handle, many streams
  // A captured launch keeps its kernel arguments for every replay, and replays
  // may run on any stream, next to eager calls on the capture stream or to other
  // graphs captured on it: two running grids would then draw from one counter.
  // Captured launches therefore take the static round-robin (no shared state).
  cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(stream, &cap) != cudaSuccess) {
    cudaGetLastError();
    return nullptr;
  }
  if (cap != cudaStreamCaptureStatusNone) return nullptr;
  std::lock_guard<std::mutex> lock(g_sched.mu);
  if (g_sched.failed[dev]) return nullptr;
  if (g_sched.base[dev] == nullptr) {
    const size_t bytes = (size_t)kSchedSlots * kSchedSlotWords * sizeof(uint32_t);
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess || cudaMemset(p, 0, bytes) != cudaSuccess ||
        cudaDeviceSynchronize() != cudaSuccess) {
      cudaGetLastError();  // e.g. first call inside a stream capture: stay static on this device
      if (p) cudaFree(p);
      g_sched.failed[dev] = true;
      return nullptr;
    }
    g_sched.base[dev] = static_cast<uint32_t*>(p);
  }
  auto& m = g_sched.slot_of[dev];
  const uintptr_t key = (uintptr_t)stream;
  auto it = m.find(key);
  int slot;
  if (it != m.end()) {
    slot = it->second;
  } else {
    if ((int)m.size() >= kSchedSlots) return nullptr;
    slot = (int)m.size();
    m.emplace(key, slot);
  }
  return g_sched.base[dev] + (size_t)slot * kSchedSlotWords;
}

}  // namespace

// cudaFuncAttributeMaxDynamicSharedMemorySize of `func` on `dev`, raised once to
// the most a CTA can have (227 KB with its static part) for kernels whose dynamic shared memory
// depends on the call (shape, camera size): a per-launch set would let one host
// thread lower it between another thread's set and its launch.
cudaError_t rta_func_allow_max_smem(const void* func, int dev) {
  static std::mutex mu;
  static std::unordered_map<uintptr_t, uint32_t> done;  // kernel -> bit per device
  if (dev < 0 || dev >= 32) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  uint32_t& bits = done[(uintptr_t)func];
  if (bits & (1u << dev)) return cudaSuccess;
  // the opt-in limit covers static + dynamic shared memory
  cudaFuncAttributes fa;
  cudaError_t e = cudaFuncGetAttributes(&fa, func);
  if (e != cudaSuccess) return e;
  int optin = 0;
  if ((e = cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev)) != cudaSuccess)
    return e;
  e = cudaFuncSetAttribute(func, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           optin - (int)fa.sharedSizeBytes);
  if (e == cudaSuccess) bits |= 1u << dev;
  return e;
}

namespace {

template <class C, int MODE>
struct TileLauncher {
  static std::atomic<int> ready[kMaxDevices];
  static int ctas_per_sm[kMaxDevices];

  static cudaError_t prepare(int dev) {
    if (ready[dev].load(std::memory_order_acquire)) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(extract_tile_kernel<C, MODE>,
                                         cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, extract_tile_kernel<C, MODE>, C::NT,
                                                      C::SMEM_BYTES);
    if (e != cudaSuccess) return e;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    ctas_per_sm[dev] = occ;
    ready[dev].store(1, std::memory_order_release);
    return cudaSuccess;
  }

  static cudaError_t launch(const uint8_t* wf, uint32_t n_traces, uint32_t n_pixels,
                            uint32_t pix_inv, const int32_t* pedestal, const float* gain,
                            int32_t* out_sum, int32_t* out_start, float* out_charge,
                            float* out_time, cudaStream_t stream, const ModeArgs& ma) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
    if ((e = prepare(dev)) != cudaSuccess) return e;
    const uint32_t n_full = n_traces / C::TILE_TRACES;
    uint32_t grid = (uint32_t)(sms * ctas_per_sm[dev]);
    if (grid > n_full) grid = n_full;
    if (grid < 1) grid = 1;
    const uintptr_t o = (uintptr_t)out_sum | (uintptr_t)out_start | (uintptr_t)out_charge |
                        (uintptr_t)out_time;
    const int vec_store = (o % 8 == 0) ? 1 : 0;
    uint32_t* sched = g_static_schedule ? nullptr : sched_words(dev, stream);
    ModeArgs m = ma;
    m.key_mul = 1u << C::KB;
    m.one = 1u;
    m.minus_one = 0xFFFFFFFFu;
    extract_tile_kernel<C, MODE><<<grid, C::NT, C::SMEM_BYTES, stream>>>(
        wf, n_traces, n_pixels, pix_inv, pedestal, gain, out_sum, out_start, out_charge, out_time,
        vec_store, sched, m);
    rta_count_launch();
    return cudaGetLastError();
  }
};
template <class C, int MODE>
std::atomic<int> TileLauncher<C, MODE>::ready[kMaxDevices];
template <class C, int MODE>
int TileLauncher<C, MODE>::ctas_per_sm[kMaxDevices];


}  // namespace

#ifdef RTA_TESTING
void rta_set_static_schedule(bool on) { g_static_schedule.store(on); }
void rta_set_lanes_per_trace(int lpt) { g_force_lanes.store(lpt); }
void rta_set_seg_tuning(int L, int TR, int NT, int stages) {
  g_seg_L.store(L);
  g_seg_TR.store(TR);
  g_seg_NT.store(NT);
  g_seg_ST.store(stages);
}
#endif
cudaError_t rta_device_sms(int dev, int* sms) { return device_sms(dev, sms); }

// rta_shutdown: the caller has synchronised the device(s)
void rta_sched_release() {
  std::lock_guard<std::mutex> lock(g_sched.mu);
  int cur = 0;
  const bool have_cur = cudaGetDevice(&cur) == cudaSuccess;
  for (int d = 0; d < kMaxDevices; ++d) {
    if (g_sched.base[d]) {
      if (cudaSetDevice(d) == cudaSuccess) {
        cudaDeviceSynchronize();
        cudaFree(g_sched.base[d]);
      }
      g_sched.base[d] = nullptr;
    }
    g_sched.failed[d] = false;
    g_sched.slot_of[d].clear();
  }
  if (have_cur) cudaSetDevice(cur);
  cudaGetLastError();
}

// The segment kernel takes the sliding extractor on a 16-byte-aligned base when two
// stages of at least one tile-aligned group of traces fit a CTA and the window is
// not much wider than the longest segment (the first window of every segment costs
// W loads; the lanes kernel does not care about W).
bool rta_seg_eligible(int32_t S, int32_t W) {
  if (S < 1 || W < 1 || W > S || W - 1 > 2 * 258) return false;
  int step = 1;  // traces per tile in the dense layout: tiles start on 16-byte boundaries
  if (S % 8 != 0)
    while (((long long)step * S) % 8 != 0) step *= 2;
  const long long stage = (((long long)step * (2 * S + 128) + 127) / 128) * 128;
  return 2 * stage <= 200 * 1024;
}

const char* rta_pick_kernel_name(int32_t S, int32_t W, bool aligned16, int bits) {
  if (bits == 12) {
    if (aligned16) {
      if (S == 30 && W == 7) return "tile12<S=30,W=7>";
      if (S == 40 && W == 7) return "tile12<S=40,W=7>";
      if (S == 25 && W == 4) return "tile12<S=25,W=4>";
      if (S == 128 && W == 8) return "tile12<S=128,W=8>";
      if (rta_jit_eligible(S, W, 12) && rta_jit_available()) return "tile12<jit>";  // compiled at first use
    }
    return "generic12";
  }
  if (aligned16) {
    if (S == 30 && W == 7) return "tile<S=30,W=7>";
    if (S == 40 && W == 7) return "tile<S=40,W=7>";
    if (S == 25 && W == 4) return "tile<S=25,W=4>";
    if (S == 128 && W == 8) return "tile<S=128,W=8>";
    if (rta_jit_eligible(S, W) && rta_jit_available()) return "staged<jit>";  // compiled for (S, W) at first use
    if (S >= 1 && S <= ((S & 1) ? 288 : 576)) return "staged<any>";  // dyn_shape: units up to 1152 bytes
  } else if (rta_dyn_eligible(S, W) && (2 * S * ((S & 1) ? 2 : 1)) % 32 != 0) {
    return "staged<any>";  // dense layout: any 2-byte alignment (also for the specialised shapes)
  }
  if (aligned16 && rta_seg_eligible(S, W)) return "segments";  // a thread per segment of a long trace
  if (aligned16 && S >= 8 && S % 8 == 0 && 4u * ((size_t)S + 12u) <= 200u * 1024u)
    return "lanes<32>";  // a warp per trace: very wide windows or very long traces
  return "generic";
}

namespace {

struct LaunchArgs {
  const uint8_t* wf;
  uint32_t n_traces, n_pixels, pix_inv;
  int32_t S, W;
  const int32_t* pedestal;
  const float* gain;
  int32_t *out_sum, *out_start;
  float *out_charge, *out_time;
  cudaStream_t stream;
  bool staged;  // 16-byte aligned input and not forced to the generic kernel
  bool unaligned_staged;  // any other input not forced to the generic kernel
};

template <int MODE, int BITS>
cudaError_t launch_generic(const LaunchArgs& a, const ModeArgs& ma) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
  uint32_t grid = (a.n_traces + 255u) / 256u;
  const uint32_t cap = (uint32_t)sms * 8u;
  if (grid > cap) grid = cap;
  extract_generic_kernel<MODE, BITS><<<grid, 256, 0, a.stream>>>(
      a.wf, a.n_traces, a.S, a.W, a.n_pixels, a.pix_inv, a.pedestal, a.gain, a.out_sum,
      a.out_start, a.out_charge, a.out_time, ma);
  rta_count_launch();
  return cudaGetLastError();
}

// Shape of the any-shape staged kernel for (S, W); false = not eligible (units
// above 1152 bytes: the generic kernel takes them).
bool dyn_shape(int32_t S, int32_t W, DynShape* sh, int* threads, int force_threads = 0) {
  const int tpt = (S & 1) ? 2 : 1;
  const long long ub = 2ll * S * tpt;
  if (ub > 1152) return false;
  const bool pad = (ub % 32 == 0);  // word stride a multiple of 8: one chunk of padding
  const int stride = (int)ub + (pad ? 16 : 0);
  int g = 1;
  while (g < 32 && (stride / 4) % (2 * g) == 0) g *= 2;
  if (g > 4 || (pad && g != 4)) return false;  // cannot happen (see the kernel's header)
  // threads per CTA: the candidate that keeps most warps resident (two stages per
  // CTA in 227 KB of shared memory; about 62 registers per thread: 32 warps at most)
  int nt = 32, best_warps = 0;
  const int candidates[5] = {stride >= 160 ? 64 : 128, 128, 256, 64, 32};  // ties go to the earlier entry (measured: long units prefer small CTAs)
  for (const int cand : candidates) {
    const int stage = ((cand * stride + 64 + 127) / 128) * 128;
    int ctas = (227 * 1024) / (2 * stage + 1024);
    if (ctas > 32) ctas = 32;
    int warps = ctas * (cand / 32);
    if (warps > 32) warps = 32;
    if (warps > best_warps) best_warps = warps, nt = cand;
  }
  if (force_threads != 0) {  // a tile table cut for another tile size (mixed-camera plans)
    if (force_threads % 32 != 0 || force_threads > 256 ||
        2 * (((force_threads * stride + 64 + 127) / 128) * 128) + 1024 > 227 * 1024)
      return false;
    nt = force_threads;
  } else if (best_warps == 0) {
    return false;
  }
  sh->S = S;
  sh->W = W;
  sh->n_win = S - W + 1;
  sh->tpt = tpt;
  sh->unit_bytes = (int)ub;
  sh->unit_stride = stride;
  sh->tile_bytes = nt * (int)ub;
  sh->stage_bytes = ((nt * stride + 64 + 127) / 128) * 128;
  sh->stages = 2;  // more resident CTAs beat a deeper ring (registers allow 32 warps per SM)
  sh->g = g;
  sh->kb = ilog2_ceil(sh->n_win);
  sh->key_mul = 1u << sh->kb;
  sh->peak_mul = 1u << ilog2_ceil(S);
  const int cpu = (int)(ub / 16);
  sh->cpu_shift = (pad && (cpu & (cpu - 1)) == 0) ? ilog2_ceil(cpu) : -1;
  *threads = nt;
  return true;
}

template <int MODE>
cudaError_t launch_dyn(const LaunchArgs& a, const DynShape& sh, int threads, const ModeArgs& ma) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
  const bool pad = sh.unit_stride != sh.unit_bytes;
  using Kernel = void (*)(const uint8_t*, uint32_t, uint32_t, uint32_t, const int*, const float*, int*,
                          int*, float*, float*, uint32_t*, DynShape, ModeArgs);
  // unpadded layouts have g = 1, 2 or 4; the padded one always 4
  const Kernel kernel = pad          ? extract_dyn_kernel<true, 4, MODE>
                        : sh.g == 1 ? extract_dyn_kernel<false, 1, MODE>
                        : sh.g == 2 ? extract_dyn_kernel<false, 2, MODE>
                                    : extract_dyn_kernel<false, 4, MODE>;
  const int smem = sh.stages * sh.stage_bytes;
  // the dynamic shared-memory size depends on the shape
  if ((e = rta_func_allow_max_smem((const void*)kernel, dev)) != cudaSuccess) return e;
  int occ = 0;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem)) != cudaSuccess)
    return e;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  const uint32_t n_full = a.n_traces / (uint32_t)(threads * sh.tpt);
  uint32_t grid = (uint32_t)(sms * occ);
  if (grid > n_full) grid = n_full;
  if (grid < 1) grid = 1;
  uint32_t* sched = g_static_schedule ? nullptr : sched_words(dev, a.stream);
  kernel<<<grid, threads, smem, a.stream>>>(a.wf, a.n_traces, a.n_pixels, a.pix_inv, a.pedestal,
                                            a.gain, a.out_sum, a.out_start, a.out_charge,
                                            a.out_time, sched, sh, ma);
  rta_count_launch();
  return cudaGetLastError();
}

// The lanes kernel takes the sliding extractor on a 16-byte-aligned base when n_samples
// is a multiple of 8 and one group's prefix array fits a CTA.
bool lanes_eligible(const LaunchArgs& a) {
  return a.staged && a.S >= 8 && a.S % 8 == 0 && 4u * ((size_t)a.S + 12u) <= 200u * 1024u;
}

template <int LPT>
cudaError_t launch_lanes(const LaunchArgs& a) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
  const size_t per_group = 4u * ((size_t)a.S + 12u);
  int threads = 256;  // as many groups per CTA as fit about a third of an SM's shared memory
  while (threads > LPT && (size_t)(threads / LPT) * per_group > 72u * 1024u) threads /= 2;
  const size_t smem = (size_t)(threads / LPT) * per_group;
  auto kernel = extract_lanes_kernel<LPT>;
  if ((e = rta_func_allow_max_smem((const void*)kernel, dev)) != cudaSuccess) return e;
  int occ = 0;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem)) != cudaSuccess)
    return e;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  const uint32_t groups = (uint32_t)(threads / LPT);
  uint32_t grid = (uint32_t)(sms * occ);
  const uint32_t need = (a.n_traces + groups - 1u) / groups;
  if (grid > need) grid = need;
  kernel<<<grid, threads, smem, a.stream>>>(a.wf, a.n_traces, a.S, a.W, ilog2_ceil(a.S - a.W + 1),
                                            a.n_pixels, a.pix_inv, a.pedestal, a.gain, a.out_sum,
                                            a.out_start, a.out_charge, a.out_time);
  rta_count_launch();
  return cudaGetLastError();
}

// Shape of the segment kernel for (S, W); false = not eligible. L is 2 * odd (bank
// spread), a tile is at most 64 traces, TR * S is a multiple of 8 when the layout is
// dense (tiles start on 16-byte boundaries).
bool seg_shape_for(int32_t S, int32_t W, int L, int TR, int NT, int stages, SegShape* sh, int* threads) {
  if (S < 1 || W < 1 || W > S || L < 2 || (L / 2) % 2 == 0 || L % 2 != 0) return false;
  if (TR < 1 || TR > kSegMaxTR) return false;
  if (NT < 32 || NT > 256 || NT % 32 != 0 || NT < TR) return false;
  if (stages < 2 || stages > kSegMaxStages) return false;
  const bool per_trace = S % 8 == 0;
  if (!per_trace && ((long long)TR * S) % 8 != 0) return false;
  sh->S = S;
  sh->W = W;
  sh->n_win = S - W + 1;
  sh->L = L;
  sh->nseg = (sh->n_win + L - 1) / L;
  sh->nslot = per_trace ? ((sh->nseg + 3) / 4) * 4 : sh->nseg;
  sh->nslot_inv = sh->nslot == 1 ? 0xFFFFFFFFu : (uint32_t)(0x100000000ull / (unsigned long long)sh->nslot);
  long long stride = 2ll * S;
  if (per_trace) {
    // words between traces = nslot L / 2 (mod 32), at least S / 2, a multiple of 4
    const int want = (int)(((long long)sh->nslot * (L / 2)) % 32);
    long long w = S / 2;
    while (w % 32 != want) w += 4;  // S / 2 and `want` are multiples of 4: at most 7 steps
    stride = 4 * w;
  }
  const long long stage = (((long long)TR * stride + 127) / 128) * 128;
  if (stages * stage > 200 * 1024) return false;
  sh->TR = TR;
  sh->trace_stride = (int32_t)stride;
  sh->stage_bytes = (int32_t)stage;
  sh->stages = stages;
  sh->kb = ilog2_ceil(sh->n_win);
  sh->key_mul = 1u << sh->kb;
  *threads = NT;
  return true;
}

// The shape the dispatch uses: segments of 66 window starts (130 and 258 for wide
// windows), tiles of about 16 KB in two stages (measured: more resident warps beat a
// deeper ring), as many threads as the tile has slots.
bool seg_shape(int32_t S, int32_t W, SegShape* sh, int* threads) {
  const int fL = g_seg_L.load(std::memory_order_relaxed), fTR = g_seg_TR.load(std::memory_order_relaxed);
  const int fNT = g_seg_NT.load(std::memory_order_relaxed), fST = g_seg_ST.load(std::memory_order_relaxed);
  const int L = fL ? fL : (W - 1 <= 66 ? 66 : W - 1 <= 130 ? 130 : 258);
  int step = 1;  // TR must be a multiple of this in the dense layout
  if (S % 8 != 0)
    while (((long long)step * S) % 8 != 0) step *= 2;
  int TR = fTR ? fTR : (int)((16 * 1024) / (2ll * S) / step) * step;
  if (TR < step) TR = step;
  if (TR > kSegMaxTR) TR = (kSegMaxTR / step) * step;
  const int n_win = S - W + 1;
  const int nseg = (n_win + L - 1) / L;
  const int nslot = S % 8 == 0 ? ((nseg + 3) / 4) * 4 : nseg;
  int NT = fNT;
  if (!NT) {
    const long long slots = (long long)TR * nslot;
    NT = slots <= 32 ? 32 : slots <= 64 ? 64 : slots <= 128 ? 128 : 256;
    if (NT < TR) NT = ((TR + 31) / 32) * 32;
  }
  for (int stages = fST ? fST : 2; stages >= 2; --stages)
    if (seg_shape_for(S, W, L, TR, NT, stages, sh, threads)) return true;
  return false;
}

cudaError_t launch_seg(const LaunchArgs& a, const SegShape& sh, int threads) {
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
  const int smem = sh.stages * sh.stage_bytes;
  if ((e = rta_func_allow_max_smem((const void*)extract_seg_kernel, dev)) != cudaSuccess) return e;
  int occ = 0;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, extract_seg_kernel, threads, smem)) !=
      cudaSuccess)
    return e;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  const uint32_t n_tiles = (a.n_traces + (uint32_t)sh.TR - 1u) / (uint32_t)sh.TR;
  uint32_t grid = (uint32_t)(sms * occ);
  if (grid > n_tiles) grid = n_tiles;
  if (grid < 1) grid = 1;
  uint32_t* sched = g_static_schedule ? nullptr : sched_words(dev, a.stream);
  extract_seg_kernel<<<grid, threads, smem, a.stream>>>(a.wf, a.n_traces, a.n_pixels, a.pix_inv,
                                                        a.pedestal, a.gain, a.out_sum, a.out_start,
                                                        a.out_charge, a.out_time, sched, sh);
  rta_count_launch();
  return cudaGetLastError();
}

#define RTA_TRY(CFG)                                                                          \
  if (a.S == CFG::S && a.W == CFG::W)                                                         \
    return TileLauncher<CFG, MODE>::launch(a.wf, a.n_traces, a.n_pixels, a.pix_inv,           \
                                           a.pedestal, a.gain, a.out_sum, a.out_start,        \
                                           a.out_charge, a.out_time, a.stream, ma);
template <int MODE>
cudaError_t launch_mode(const LaunchArgs& a, const ModeArgs& ma) {
  // The fixed window touches W samples of a trace: beyond about three 32-byte
  // sectors per trace, gathering them from global memory (the generic kernel)
  // moves less than streaming whole tiles (S = 128: 0.99 ms against 1.69 ms).
  const bool gather = (MODE == MODE_FIXED) && 2 * a.S > 96;
#ifdef RTA_TESTING
  if (MODE == MODE_SLIDING && a.staged && g_seg_L.load(std::memory_order_relaxed) != 0) {
    SegShape sg;  // measurements / tests only: the segment kernel on any shape
    int threads = 0;
    if (seg_shape(a.S, a.W, &sg, &threads)) return launch_seg(a, sg, threads);
  }
  if (MODE == MODE_SLIDING && lanes_eligible(a)) {
    switch (g_force_lanes.load(std::memory_order_relaxed)) {  // measurements only
      case 4: return launch_lanes<4>(a);
      case 8: return launch_lanes<8>(a);
      case 16: return launch_lanes<16>(a);
      case 32: return launch_lanes<32>(a);
      default: break;
    }
  }
#endif
  if (a.staged && !gather) {
    RTA_TRY(CfgS30W7)
    RTA_TRY(CfgS40W7)
    RTA_TRY(CfgS25W4)
    RTA_TRY(CfgS128W8)
    // any other shape whose unit fits a register copy: the same kernel source compiled
    // for this (S, W) at run time (rta_jit.cu); not available -> the runtime-shape kernel
    if (rta_jit_eligible(a.S, a.W)) {
      int dev = 0;
      cudaError_t e = cudaGetDevice(&dev);
      if (e != cudaSuccess) return e;
      ModeArgs m = ma;
      m.key_mul = 1u << ilog2_ceil(a.S - a.W + 1);
      m.one = 1u;
      m.minus_one = 0xFFFFFFFFu;
      const RtaJitArgs ja{a.wf,      a.n_traces,  a.n_pixels,  a.pix_inv,
                          a.pedestal, a.gain,      a.out_sum,   a.out_start,
                          a.out_charge, a.out_time,
                          g_static_schedule ? nullptr : sched_words(dev, a.stream)};
      e = rta_jit_launch(a.S, a.W, MODE, ja, &m, sizeof m, a.stream);
      if (e != cudaErrorNotSupported) return e;
    }
    DynShape sh;
    int threads = 0;
    if (dyn_shape(a.S, a.W, &sh, &threads)) return launch_dyn<MODE>(a, sh, threads, ma);
  } else if (a.unaligned_staged && !gather) {
    // a base that is only 2-byte aligned: the runtime-shape kernel with a dense
    // layout takes it (the specialisations and the padded layout need 16 bytes)
    DynShape sh;
    int threads = 0;
    if (dyn_shape(a.S, a.W, &sh, &threads) && sh.unit_stride == sh.unit_bytes)
      return launch_dyn<MODE>(a, sh, threads, ma);
  }
  // traces too long for one thread: a thread per segment of a trace; windows much wider
  // than a segment, or traces too long for a stage, a warp per trace (shuffle scan,
  // prefix array in shared memory: its cost does not depend on W)
  if (MODE == MODE_SLIDING && a.staged) {
    SegShape sg;
    int threads = 0;
    if (rta_seg_eligible(a.S, a.W) && seg_shape(a.S, a.W, &sg, &threads)) return launch_seg(a, sg, threads);
  }
  if (MODE == MODE_SLIDING && lanes_eligible(a)) return launch_lanes<32>(a);
  return launch_generic<MODE, 16>(a, ma);
}

// P12 input: the sliding-window extractor only (include/rta.h)
cudaError_t launch_packed12(const LaunchArgs& a, const ModeArgs& ma) {
  constexpr int MODE = MODE_SLIDING;
  if (a.staged) {
    RTA_TRY(CfgP30W7)
    RTA_TRY(CfgP40W7)
    RTA_TRY(CfgP25W4)
    RTA_TRY(CfgP128W8)
    // any other shape whose packed unit fits a register copy: compiled for (S, W) at first use
    if (rta_jit_eligible(a.S, a.W, 12)) {
      int dev = 0;
      cudaError_t e = cudaGetDevice(&dev);
      if (e != cudaSuccess) return e;
      ModeArgs m = ma;
      m.key_mul = 1u << ilog2_ceil(a.S - a.W + 1);
      m.one = 1u;
      m.minus_one = 0xFFFFFFFFu;
      const RtaJitArgs ja{a.wf,      a.n_traces,  a.n_pixels,  a.pix_inv,
                          a.pedestal, a.gain,      a.out_sum,   a.out_start,
                          a.out_charge, a.out_time,
                          g_static_schedule ? nullptr : sched_words(dev, a.stream)};
      e = rta_jit_launch(a.S, a.W, MODE, ja, &m, sizeof m, a.stream, 12);
      if (e != cudaErrorNotSupported) return e;
    }
  }
  return launch_generic<MODE, 12>(a, ma);
}
#undef RTA_TRY

template <class C>
struct RaggedLauncher {
  static std::atomic<int> ready[kMaxDevices];
  static int ctas_per_sm[kMaxDevices];
  static cudaError_t launch(const uint8_t* wf, const RaggedTile* tiles, uint32_t n_tiles,
                            const int32_t* pedestal, const float* gain, int32_t* out_sum,
                            int32_t* out_start, float* out_charge, float* out_time,
                            cudaStream_t stream) {
    int dev = 0, sms = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
    if (!ready[dev].load(std::memory_order_acquire)) {
      e = cudaFuncSetAttribute(extract_ragged_kernel<C>,
                               cudaFuncAttributeMaxDynamicSharedMemorySize, C::SMEM_BYTES);
      if (e != cudaSuccess) return e;
      int occ = 0;
      e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, extract_ragged_kernel<C>, C::NT,
                                                        C::SMEM_BYTES);
      if (e != cudaSuccess) return e;
      if (occ < 1) return cudaErrorLaunchOutOfResources;
      ctas_per_sm[dev] = occ;
      ready[dev].store(1, std::memory_order_release);
    }
    uint32_t grid = (uint32_t)(sms * ctas_per_sm[dev]);
    if (grid > n_tiles) grid = n_tiles;
    const uintptr_t o = (uintptr_t)out_sum | (uintptr_t)out_start | (uintptr_t)out_charge |
                        (uintptr_t)out_time;
    uint32_t* sched = g_static_schedule ? nullptr : sched_words(dev, stream);
    extract_ragged_kernel<C><<<grid, C::NT, C::SMEM_BYTES, stream>>>(
        wf, tiles, n_tiles, pedestal, gain, out_sum, out_start, out_charge, out_time,
        (o % 8 == 0) ? 1 : 0, sched);
    rta_count_launch();
    return cudaGetLastError();
  }
};
template <class C>
std::atomic<int> RaggedLauncher<C>::ready[kMaxDevices];
template <class C>
int RaggedLauncher<C>::ctas_per_sm[kMaxDevices];

}  // namespace

bool rta_dyn_eligible(int32_t S, int32_t W) {
  DynShape sh;
  int threads = 0;
  return S >= 1 && W >= 1 && W <= S && dyn_shape(S, W, &sh, &threads);
}

// The sliding extractor through the runtime-shape staged kernel with scheduler words
// the caller owns (rta_noalloc.cu: words in a static device array, zeroed on the
// stream ahead of this launch). Nothing here allocates device memory: no per-stream
// scheduler pool, no run-time compile. A separate copy of launch_dyn's body so that
// the dispatch above stays as it is. cudaErrorNotSupported: (S, W) is not
// rta_dyn_eligible, or wf is not 16-byte aligned.
cudaError_t rta_launch_extract_dyn_sched(const void* wf, int64_t n_traces64, int32_t n_pixels,
                                         int32_t S, const int32_t* pedestal, const float* gain,
                                         int32_t W, int32_t* out_sum, int32_t* out_start,
                                         float* out_charge, float* out_time, cudaStream_t stream,
                                         uint32_t* sched) {
  if (n_traces64 <= 0) return cudaSuccess;
  DynShape sh;
  int threads = 0;
  if (((uintptr_t)wf % 16) != 0 || S < 1 || W < 1 || W > S || !dyn_shape(S, W, &sh, &threads))
    return cudaErrorNotSupported;
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
  const bool pad = sh.unit_stride != sh.unit_bytes;
  using Kernel = void (*)(const uint8_t*, uint32_t, uint32_t, uint32_t, const int*, const float*, int*,
                          int*, float*, float*, uint32_t*, DynShape, ModeArgs);
  const Kernel kernel = pad          ? extract_dyn_kernel<true, 4, MODE_SLIDING>
                        : sh.g == 1 ? extract_dyn_kernel<false, 1, MODE_SLIDING>
                        : sh.g == 2 ? extract_dyn_kernel<false, 2, MODE_SLIDING>
                                    : extract_dyn_kernel<false, 4, MODE_SLIDING>;
  const int smem = sh.stages * sh.stage_bytes;
  if ((e = rta_func_allow_max_smem((const void*)kernel, dev)) != cudaSuccess) return e;
  int occ = 0;
  if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem)) != cudaSuccess)
    return e;
  if (occ < 1) return cudaErrorLaunchOutOfResources;
  const uint32_t n_traces = (uint32_t)n_traces64, P = (uint32_t)n_pixels;
  const uint32_t n_full = n_traces / (uint32_t)(threads * sh.tpt);
  uint32_t grid = (uint32_t)(sms * occ);
  if (grid > n_full) grid = n_full;
  if (grid < 1) grid = 1;
  const uint64_t inv64 = (1ull << 32) / P;
  const uint32_t pix_inv = inv64 > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)inv64;
  const ModeArgs ma = {};
  kernel<<<grid, threads, smem, stream>>>(static_cast<const uint8_t*>(wf), n_traces, P, pix_inv,
                                          pedestal, gain, out_sum, out_start, out_charge, out_time,
                                          sched, sh, ma);
  rta_count_launch();
  return cudaGetLastError();
}

int rta_ragged_tile_traces(int32_t S, int32_t W) {
  if (S == CfgS30W7::S && W == CfgS30W7::W) return CfgS30W7::TILE_TRACES;
  if (S == CfgS40W7::S && W == CfgS40W7::W) return CfgS40W7::TILE_TRACES;
  if (S == CfgS25W4::S && W == CfgS25W4::W) return CfgS25W4::TILE_TRACES;
  if (S == CfgS128W8::S && W == CfgS128W8::W) return CfgS128W8::TILE_TRACES;
  const int jit = rta_jit_tile_traces(S, W);  // the run-time specialisation of the tile-table kernel
  if (jit > 0) return jit;
  DynShape sh;
  int threads = 0;
  if (dyn_shape(S, W, &sh, &threads)) return threads * sh.tpt;  // extract_ragged_dyn_kernel
  return 256;  // extract_ragged_generic_kernel: one thread per trace, 256 threads
}

cudaError_t rta_launch_ragged(const void* wf, const RtaRaggedTile* tiles_dev, uint32_t n_tiles,
                              int32_t S, int32_t W, int32_t tile_traces, const int32_t* pedestal,
                              const float* gain,
                              int32_t* out_sum, int32_t* out_start, float* out_charge,
                              float* out_time, cudaStream_t stream) {
  if (n_tiles == 0) return cudaSuccess;
  const uint8_t* w = static_cast<const uint8_t*>(wf);
#define RTA_TRY(CFG)                                                                        \
  if (S == CFG::S && W == CFG::W)                                                           \
    return RaggedLauncher<CFG>::launch(w, tiles_dev, n_tiles, pedestal, gain, out_sum,      \
                                       out_start, out_charge, out_time, stream);
  RTA_TRY(CfgS30W7)
  RTA_TRY(CfgS40W7)
  RTA_TRY(CfgS25W4)
  RTA_TRY(CfgS128W8)
#undef RTA_TRY
  int dev = 0, sms = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if ((e = device_sms(dev, &sms)) != cudaSuccess) return e;
  // the run-time specialisation, when the table was cut for its tile
  if (tile_traces == rta_jit_tile_traces(S, W)) {
    const RtaJitRaggedArgs ja{w, tiles_dev, n_tiles, pedestal, gain, out_sum, out_start, out_charge, out_time,
                              g_static_schedule ? nullptr : sched_words(dev, stream)};
    e = rta_jit_launch_ragged(S, W, ja, stream);
    if (e != cudaErrorNotSupported) return e;
  }
  // the runtime-shape kernel with as many threads as a tile has units (the table may have been
  // cut for the specialisation's tile while the compiler has gone away since)
  DynShape sh;
  int threads = 0;
  const int tpt = (S & 1) ? 2 : 1;
  if (tile_traces % tpt == 0 && dyn_shape(S, W, &sh, &threads, tile_traces / tpt)) {
    const bool pad = sh.unit_stride != sh.unit_bytes;
    using Kernel = void (*)(const uint8_t*, const RaggedTile*, uint32_t, const int*, const float*,
                            int*, int*, float*, float*, uint32_t*, DynShape);
    const Kernel kernel = pad          ? extract_ragged_dyn_kernel<true, 4>
                          : sh.g == 1 ? extract_ragged_dyn_kernel<false, 1>
                          : sh.g == 2 ? extract_ragged_dyn_kernel<false, 2>
                                      : extract_ragged_dyn_kernel<false, 4>;
    const int smem = sh.stages * sh.stage_bytes;
    if ((e = rta_func_allow_max_smem((const void*)kernel, dev)) != cudaSuccess) return e;
    int occ = 0;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem)) != cudaSuccess)
      return e;
    if (occ < 1) return cudaErrorLaunchOutOfResources;
    uint32_t grid = (uint32_t)(sms * occ);
    if (grid > n_tiles) grid = n_tiles;
    uint32_t* sched = g_static_schedule ? nullptr : sched_words(dev, stream);
    kernel<<<grid, threads, smem, stream>>>(w, tiles_dev, n_tiles, pedestal, gain, out_sum, out_start,
                                            out_charge, out_time, sched, sh);
    rta_count_launch();
    return cudaGetLastError();
  }
  uint32_t grid = n_tiles;
  const uint32_t cap = (uint32_t)sms * 8u;
  if (grid > cap) grid = cap;
  extract_ragged_generic_kernel<<<grid, 256, 0, stream>>>(w, tiles_dev, n_tiles, S, W, pedestal,
                                                          gain, out_sum, out_start, out_charge,
                                                          out_time);
  rta_count_launch();
  return cudaGetLastError();
}

cudaError_t rta_launch_extract(const void* wf, int64_t n_traces64, int32_t n_pixels,
                               int32_t S, const int32_t* pedestal, const float* gain, int32_t W,
                               int32_t* out_sum, int32_t* out_start, float* out_charge,
                               float* out_time, cudaStream_t stream, bool force_generic,
                               const RtaMode* mode, int sample_bits) {
  if (n_traces64 <= 0) return cudaSuccess;
  const uint32_t P = (uint32_t)n_pixels;
  const uint64_t inv64 = (1ull << 32) / P;
  LaunchArgs a;
  a.wf = static_cast<const uint8_t*>(wf);
  a.n_traces = (uint32_t)n_traces64;
  a.n_pixels = P;
  a.pix_inv = inv64 > 0xFFFFFFFFull ? 0xFFFFFFFFu : (uint32_t)inv64;
  a.S = S;
  a.W = W;
  a.pedestal = pedestal;
  a.gain = gain;
  a.out_sum = out_sum;
  a.out_start = out_start;
  a.out_charge = out_charge;
  a.out_time = out_time;
  a.stream = stream;
  a.staged = !force_generic && ((uintptr_t)wf % 16) == 0;
  a.unaligned_staged = !force_generic && !a.staged && sample_bits == 16;
  ModeArgs ma = {};
  const int kind = mode ? mode->kind : RTA_MODE_SLIDING;
  if (sample_bits == 12)
    return kind == RTA_MODE_SLIDING ? launch_packed12(a, ma) : cudaErrorInvalidValue;
  if (sample_bits != 16) return cudaErrorInvalidValue;
  switch (kind) {
    case RTA_MODE_SLIDING:
      return launch_mode<MODE_SLIDING>(a, ma);
    case RTA_MODE_FIXED:
      ma.window_start = mode->window_start;
      return launch_mode<MODE_FIXED>(a, ma);
    case RTA_MODE_LOCAL_PEAK:
      ma.shift = mode->shift;
      return launch_mode<MODE_LOCAL_PEAK>(a, ma);
    case RTA_MODE_FIR: {
      // W == mode->n_taps (checked by the caller)
      ma.fir_packed = 1;
      for (int k = 0; k < W; ++k) {
        const int32_t c = mode->taps[k];
        ma.taps[k] = c;
        ma.c0 += c;
        ma.c1 += k * c;
        if (c < -128 || c > 127) ma.fir_packed = 0;
        const int m = k >> 1;  // pair m: byte (k & 1) of half (m & 1) of word m >> 1
        ma.taps2[m >> 1] |= ((uint32_t)c & 0xFFu) << (16 * (m & 1) + 8 * (k & 1));
      }
      return launch_mode<MODE_FIR>(a, ma);
    }
    default:
      return cudaErrorInvalidValue;
  }
}
