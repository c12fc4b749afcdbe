// rta_tile_kernel.cuh — the staged tile kernel of the per-trace extractors
// (steps a1-a7 of SURVEY.md section 8(a)): tile scheduler + stage ring + the
// per-trace arithmetic of rta_device.cuh. Included by rta_kernels.cu (ahead-of-
// time instantiations) and embedded as text in librta.so for the run-time
// specialisations of rta_jit.cu (NVRTC). Never seen by oracle/.
#ifndef RTA_TILE_KERNEL_CUH
#define RTA_TILE_KERNEL_CUH

#include "rta_device.cuh"

namespace {

// Tile indices of one CTA (used by its thread 0 only). Tiles are handed out
// dynamically: SMs do not stream at the same rate (near / far L2 die, DRAM
// channel load), and with a static round-robin the launch ends when the slowest
// CTA has finished its fixed share (measured: 4-7 % of SM-time idle). `sched`
// points at {next tile, CTAs done}, both zero on entry; the last CTA to leave
// zeroes them again, so the pair is reusable by the next launch on the same
// stream. sched == nullptr selects the static round-robin (same code path,
// locally generated indices); launches captured into a CUDA graph use it.
// The first `stages` tiles of every CTA are the static round-robin ones (no
// atomic round trip before the first load); the shared counter hands out the
// tiles after those, in runs of up to kMaxRun consecutive tiles per atomic:
// same-address atomics retire at only ~0.3 G/s on B200 (measured), which one
// atomic per 10-20 KB tile would saturate. Runs shrink to single tiles near
// the end so the CTAs still finish together.
struct TileFeed {
  static constexpr uint32_t kMaxRun = 8;
  uint32_t* sched;
  uint32_t n_tiles, dyn_base;
  // static sequence, current run [cur, end), prefetched run [nxt, nxt + n_run)
  uint32_t static_next, cur, end, nxt, n_run;

  __device__ __forceinline__ TileFeed(uint32_t* sched_, const uint32_t n_tiles_, const int stages)
      : sched(sched_), n_tiles(n_tiles_), dyn_base((uint32_t)stages * gridDim.x),
        static_next(blockIdx.x), cur(0), end(0), nxt(0), n_run(0) {}
  __device__ __forceinline__ uint32_t fetch_static() {
    const uint32_t t = static_next;
    // saturate: indices past the end must stay past the end
    static_next = (t > 0xFFFFFFFFu - gridDim.x) ? 0xFFFFFFFFu : t + gridDim.x;
    return t;
  }
  __device__ __forceinline__ uint32_t run_length(const uint32_t seen) const {
    const uint32_t left = n_tiles > seen ? n_tiles - seen : 0u;
    const uint32_t k = left / (8u * gridDim.x);
    return k < 1u ? 1u : (k > kMaxRun ? kMaxRun : k);
  }
  // after the static tiles have been drawn: ask for the first dynamic run
  __device__ __forceinline__ void prime() {
    if (sched != nullptr) {
      n_run = run_length(dyn_base);
      nxt = dyn_base + atomicAdd(sched, n_run);
    }
  }
  __device__ __forceinline__ uint32_t fetch() {
    if (sched == nullptr) return fetch_static();
    if (cur == end) {  // take the prefetched run, ask for the one after it
      cur = nxt;
      end = nxt + n_run;
      n_run = run_length(cur);
      nxt = dyn_base + atomicAdd(sched, n_run);
    }
    return cur++;
  }
  // hand the scheduler words back zeroed (all of this CTA's fetches precede this)
  __device__ __forceinline__ void leave() const {
    if (sched == nullptr) return;
    __threadfence();
    if (atomicAdd(sched + 1, 1u) == gridDim.x - 1) {
      sched[0] = 0;
      sched[1] = 0;
      __threadfence();
    }
  }
};

// The body of the staged tile kernel: instantiated ahead of time for the four
// BASELINE shapes (extract_tile_kernel below) and at run time, through NVRTC,
// for any other shape whose unit fits the register copy (rta_jit.cu).
template <class C, int MODE>
__device__ __forceinline__ void tile_kernel_body(
    const uint8_t* __restrict__ wf, const uint32_t n_traces, const uint32_t n_pixels,
    const uint32_t pix_inv, const int* __restrict__ pedestal, const float* __restrict__ gain,
    int* __restrict__ out_sum, int* __restrict__ out_start, float* __restrict__ out_charge,
    float* __restrict__ out_time, const int vec_store, uint32_t* __restrict__ sched,
    const ModeArgs& ma) {
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[C::STAGES];
  constexpr int QN = C::STAGES + 1;  // queue of tile indices, one slot more than stages
  __shared__ uint32_t tile_q[QN];
  const int tid = threadIdx.x;
  const uint32_t n_full = n_traces / C::TILE_TRACES;
  const uint32_t rem = n_traces - n_full * C::TILE_TRACES;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_u32(full_bar);

  TileFeed feed(sched, n_full, C::STAGES);  // thread 0 only

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(bar_base + 8 * s, C::PAD ? C::NT : 1);
      tile_q[s] = feed.fetch_static();
    }
    fence_mbar_init();
    feed.prime();
  }
  __syncthreads();

  auto issue = [&](const uint32_t tile, const int stage) {
    const uint8_t* src = wf + (size_t)tile * C::TILE_BYTES;
    const uint32_t dst = smem_base + stage * C::STAGE_BYTES;
    const uint32_t bar = bar_base + 8 * stage;
    if constexpr (!C::PAD) {
      if (tid == 0) {
        mbar_expect_tx(bar, C::TILE_BYTES);
        tma_bulk_g2s(dst, src, C::TILE_BYTES, bar);
      }
    } else {
#pragma unroll 4
      for (int c = tid; c < C::TILE_BYTES / 16; c += C::NT) {
        const int u = c / C::NVEC;  // one extra chunk of padding per unit
        cp_async16(dst + (uint32_t)(c + u) * 16u, src + (size_t)c * 16);
      }
      cp_async_mbar_arrive(bar);
    }
  };

  // prologue: fill the ring
#pragma unroll
  for (int s = 0; s < C::STAGES; ++s) {
    const uint32_t tile = tile_q[s];
    if (tile < n_full) issue(tile, s);
  }
  // thread 0 keeps one tile index in flight: fetched while a tile is being
  // computed, published one iteration later (the atomic's latency is hidden)
  uint32_t pre = 0;
  if (tid == 0) pre = feed.fetch();

  uint32_t tile;
  for (uint32_t j = 0;; ++j) {
    tile = tile_q[j % QN];
    if (tile >= n_full) break;  // indices grow per CTA: nothing later is valid either
    const int stage = (int)(j % C::STAGES);
    const uint32_t parity = (j / C::STAGES) & 1u;
    if (tid == 0) {
      // slot (j + STAGES) % QN == (j - 1) % QN was last read before the
      // previous iteration's barrier
      tile_q[(j + C::STAGES) % QN] = pre;
      pre = feed.fetch();
    }
    mbar_wait(bar_base + 8 * stage, parity);
    const uint8_t* unit = smem + stage * C::STAGE_BYTES + tid * C::UNIT_STRIDE;
    const uint32_t g0 = tile * C::TILE_TRACES + (uint32_t)tid * C::TPT;
    compute_unit<C, MODE, C::KEYMODE>(unit, g0, C::TPT, fastmod(g0, n_pixels, pix_inv), n_pixels,
                                pedestal, gain, out_sum, out_start, out_charge, out_time,
                                vec_store != 0, ma);
    __syncthreads();  // every thread is done with this stage; tile_q slot is published
    const uint32_t next = tile_q[(j + C::STAGES) % QN];
    if (next < n_full) issue(next, stage);
  }

  // ragged tail (< one tile of traces): plain copies, by the CTA that drew index n_full
  if (rem != 0 && tile == n_full) {
    const uint8_t* src = wf + (size_t)n_full * C::TILE_BYTES;  // 16-byte aligned
    const uint32_t n_bytes = (rem * (uint32_t)C::TRACE_BITS + 7u) / 8u;
    // byte b of the tail lives at (b / UNIT_BYTES) * UNIT_STRIDE + b % UNIT_BYTES;
    // whole words first (a unit with padding is a multiple of 16 bytes), then
    // the last 0-3 bytes one by one: nothing past the caller's buffer is read
    const uint32_t n_w = n_bytes / 4u;
    for (uint32_t i = tid; i < n_w; i += C::NT) {
      uint32_t d = i;
      if constexpr (C::PAD) d += (i / (C::UNIT_BYTES / 4)) * ((C::UNIT_STRIDE - C::UNIT_BYTES) / 4);
      reinterpret_cast<uint32_t*>(smem)[d] = reinterpret_cast<const uint32_t*>(src)[i];
    }
    for (uint32_t b = 4u * n_w + tid; b < n_bytes; b += C::NT) {
      uint32_t d = b;
      if constexpr (C::PAD) d += (b / C::UNIT_BYTES) * (C::UNIT_STRIDE - C::UNIT_BYTES);
      smem[d] = src[b];
    }
    __syncthreads();
    const uint32_t first = (uint32_t)tid * C::TPT;
    if (first < rem) {
      const uint8_t* unit = smem + tid * C::UNIT_STRIDE;
      const uint32_t g0 = n_full * C::TILE_TRACES + first;
      compute_unit<C, MODE, C::KEYMODE>(unit, g0, rem - first, fastmod(g0, n_pixels, pix_inv), n_pixels,
                                  pedestal, gain, out_sum, out_start, out_charge, out_time,
                                  vec_store != 0, ma);
    }
  }

  if (tid == 0) feed.leave();
}

using RaggedTile = RtaRaggedTile;  // rta_internal.h: {src offset | n << 48, out_base, cal0}
constexpr unsigned long long kRaggedOffMask = (1ull << 48) - 1ull;

__device__ __forceinline__ void mbar_expect_tx_only(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(bytes)
               : "memory");
}

// The body of the mixed-camera tile kernel (one launch per shape class walks its tile
// table): ahead-of-time for the four BASELINE shapes (extract_ragged_kernel in
// rta_kernels.cu) and, like the uniform kernel, compiled at run time for any other shape
// whose unit fits a register copy (rta_jit.cu).
template <class C>
__device__ __forceinline__ void ragged_kernel_body(
    const uint8_t* __restrict__ wf, const RaggedTile* __restrict__ tiles, const uint32_t n_tiles,
    const int* __restrict__ pedestal, const float* __restrict__ gain, int* __restrict__ out_sum,
    int* __restrict__ out_start, float* __restrict__ out_charge, float* __restrict__ out_time,
    const int vec_store, uint32_t* __restrict__ sched) {
  static_assert(C::BITS == 16 && C::STAGES >= 2, "uint16 blocks, at least two stages");
  extern __shared__ __align__(128) uint8_t smem[];
  __shared__ __align__(8) uint64_t full_bar[C::STAGES];
  constexpr int QN = C::STAGES + 1;
  __shared__ uint32_t tile_q[QN];
  // the table entry of every queued tile, fetched by thread 0 one iteration
  // ahead together with the index: no thread waits on a dependent global load
  __shared__ RaggedTile desc_q[QN];
  const int tid = threadIdx.x;
  const uint32_t smem_base = smem_u32(smem);
  const uint32_t bar_base = smem_u32(full_bar);
  const ModeArgs ma = {};

  // tile indices: the first STAGES of a CTA are static (blockIdx.x + k * gridDim.x),
  // the rest come from the shared counter, one run of tiles per atomic
  TileFeed feed(sched, n_tiles, C::STAGES);  // thread 0 only

  const auto entry = [&](const uint32_t ti) -> RaggedTile {
    if (ti < n_tiles) return tiles[ti];
    return RaggedTile{0ull, 0u, 0u};
  };
  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < C::STAGES; ++s) {
      mbar_init(bar_base + 8 * s, C::NT);
      tile_q[s] = feed.fetch_static();
      desc_q[s] = entry(tile_q[s]);
    }
    fence_mbar_init();
    feed.prime();
  }
  __syncthreads();

  constexpr uint32_t UB = C::UNIT_BYTES, PADB = C::UNIT_STRIDE - C::UNIT_BYTES;
  constexpr uint32_t TRACE_BYTES = C::TRACE_BITS / 8;
  auto issue = [&](const int slot, const int stage) {
    const RaggedTile t = desc_q[slot];
    const uint8_t* src = wf + (size_t)(t.src & kRaggedOffMask);
    const uint32_t bytes = (uint32_t)(t.src >> 48) * TRACE_BYTES;
    uint8_t* dstp = smem + stage * C::STAGE_BYTES;
    const uint32_t dst = smem_base + stage * C::STAGE_BYTES;
    const uint32_t bar = bar_base + 8 * stage;
    const uint32_t mis = (uint32_t)(reinterpret_cast<uintptr_t>(src) & 15u);
    uint32_t done;  // bytes moved by the wide path; the rest goes halfword by halfword
    if (mis == 0) {
      if constexpr (!C::PAD) {
        done = bytes & ~15u;
        if (tid == 0 && done != 0) {
          mbar_expect_tx_only(bar, done);
          tma_bulk_g2s(dst, src, done, bar);
        }
      } else {
        done = bytes;  // a padded unit is a whole number of 16-byte chunks
        if (bytes == (uint32_t)C::TILE_BYTES) {  // full tile: compile-time trip count, as the uniform kernel
#pragma unroll 4
          for (int c = tid; c < C::TILE_BYTES / 16; c += C::NT) {
            const int u = c / C::NVEC;
            cp_async16(dst + (uint32_t)(c + u) * 16u, src + (size_t)c * 16);
          }
        } else {
          for (uint32_t c = tid; c < bytes / 16u; c += C::NT)
            cp_async16(dst + (c + c / (UB / 16u)) * 16u, src + (size_t)c * 16u);
        }
      }
    } else if ((mis & 3u) == 0) {
      done = bytes & ~3u;
      for (uint32_t c = tid; c < done / 4u; c += C::NT) {
        uint32_t d = c * 4u;
        if constexpr (C::PAD) d += (d / UB) * PADB;
        cp_async4(dst + d, src + (size_t)c * 4u);
      }
    } else {
      done = 0;
    }
    for (uint32_t b = done + 2u * tid; b < bytes; b += 2u * C::NT) {
      uint32_t d = b;
      if constexpr (C::PAD) d += (b / UB) * PADB;
      *reinterpret_cast<uint16_t*>(dstp + d) = *reinterpret_cast<const uint16_t*>(src + b);
    }
    cp_async_mbar_arrive(bar);  // counts once this thread's cp.async copies have landed
  };

#pragma unroll
  for (int s = 0; s < C::STAGES; ++s) {
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
    const int stage = (int)(j % C::STAGES);
    const uint32_t parity = (j / C::STAGES) & 1u;
    if (tid == 0) {
      tile_q[(j + C::STAGES) % QN] = pre;
      desc_q[(j + C::STAGES) % QN] = pre_d;
      pre = feed.fetch();
      pre_d = entry(pre);
    }
    const RaggedTile t = desc_q[j % QN];
    const uint32_t n = (uint32_t)(t.src >> 48);
    mbar_wait(bar_base + 8 * stage, parity);
    const uint32_t first = (uint32_t)tid * C::TPT;
    if (first < n) {
      const uint8_t* unit = smem + stage * C::STAGE_BYTES + tid * C::UNIT_STRIDE;
      // the calibration index "wraps" after the tile's last trace, so the discarded
      // second trace of an odd tile reads pedestal[0], never past the arrays
      compute_unit<C, MODE_SLIDING>(unit, t.out_base + first, n - first, t.cal0 + first,
                                    t.cal0 + n, pedestal, gain, out_sum, out_start, out_charge,
                                    out_time, vec_store != 0 && (t.out_base & 1u) == 0, ma);
    }
    __syncthreads();
    const uint32_t next = tile_q[(j + C::STAGES) % QN];
    if (next < n_tiles) issue((int)((j + C::STAGES) % QN), stage);
  }

  if (tid == 0) feed.leave();
}

template <class C, int MODE>
__global__ void __launch_bounds__(C::NT)
    extract_tile_kernel(const uint8_t* __restrict__ wf, const uint32_t n_traces,
                        const uint32_t n_pixels, const uint32_t pix_inv,
                        const int* __restrict__ pedestal, const float* __restrict__ gain,
                        int* __restrict__ out_sum, int* __restrict__ out_start,
                        float* __restrict__ out_charge, float* __restrict__ out_time,
                        const int vec_store, uint32_t* __restrict__ sched,
                        const __grid_constant__ ModeArgs ma) {
  tile_kernel_body<C, MODE>(wf, n_traces, n_pixels, pix_inv, pedestal, gain, out_sum, out_start,
                            out_charge, out_time, vec_store, sched, ma);
}

}  // namespace

#endif
