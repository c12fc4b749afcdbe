// oracle/rta_oracle_windows.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain single-threaded CPU definitions of the other members of the "several
// signal extraction algorithms [13]" family the paper says were being ported
// (§5; ref [13], is not available, so these are
// the builder's definitions: SURVEY.md §8(f) NEXT-1, DESIGN.md readings
// R22-R25). All of them share the outputs of the sliding-window extractor
// (oracle/rta_oracle.cpp) and differ only in how the window start t* is chosen
// (fixed, local peak) or in the weights of the window (FIR):
//
//   x[s] = wf[e][p][s] - pedestal[p]
//   fixed       t* = clamp(window_start[p], 0, S-W)                      (R22)
//   local peak  t* = clamp(peak - shift, 0, S-W),
//               peak = smallest s with x[s] maximal                      (R23)
//   then, for both:   out_sum = sum_{k<W} x[t*+k]
//                     num     = sum_{k<W} (t*+k) x[t*+k]
//   FIR         y(t) = sum_{k<K} c[k] x[t+k], t = 0..S-K; t* = smallest t with
//               y(t) maximal; out_sum = y(t*);
//               num = sum_{k<K} (t*+k) c[k] x[t*+k]   (W := K)            (R24)
//   always:     out_start = t*, out_charge = RN32(out_sum * gain[p]),
//               out_time = RN32(num / out_sum) if out_sum > 0 else t* + (W-1)/2
//
// Shares no code with paper_1307_6489_b200/csrc. Parity status: pinned
// (tests/test_oracle_windows_pins.py): closed forms, numpy restatements,
// reductions to the pinned sliding-window oracle (FIR with all-ones taps;
// fixed start = sliding's t*; local peak with W = 1, shift = 0).
#include <cstddef>
#include <cstdint>

namespace {

// outputs of one trace once t* and the weights are known (weights == nullptr: all ones)
void window_outputs(const uint16_t* tr, int64_t ped, float gain, int64_t tstar, int64_t W,
                    const int32_t* weights, int32_t* o_sum, int32_t* o_start, float* o_charge,
                    float* o_time) {
  int64_t sum = 0, num = 0;
  for (int64_t k = 0; k < W; ++k) {
    const int64_t c = weights ? (int64_t)weights[k] : 1;
    const int64_t x = (int64_t)tr[tstar + k] - ped;
    sum += c * x;
    num += (tstar + k) * c * x;
  }
  *o_sum = (int32_t)sum;
  *o_start = (int32_t)tstar;
  *o_charge = (float)((double)sum * (double)gain);
  *o_time = sum > 0 ? (float)((double)num / (double)sum)
                    : (float)((double)tstar + 0.5 * (double)(W - 1));
}

int64_t clamp_start(int64_t t, int64_t S, int64_t W) {
  if (t < 0) t = 0;
  if (t > S - W) t = S - W;
  return t;
}

bool bad_shape(int64_t E, int32_t P, int32_t S, int32_t W) {
  return E < 0 || P < 1 || S < 1 || W < 1 || W > S;
}

}  // namespace

extern "C" {

// Fixed window (R22): window_start[n_pixels], clamped into [0, S-W].
int rta_oracle_extract_fixed(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                             int32_t n_samples, const int32_t* pedestal, const float* gain,
                             int32_t W, const int32_t* window_start, int32_t* out_sum,
                             int32_t* out_start, float* out_charge, float* out_time) {
  if (bad_shape(n_events, n_pixels, n_samples, W)) return 1;
  for (int64_t e = 0; e < n_events; ++e)
    for (int64_t p = 0; p < n_pixels; ++p) {
      const int64_t o = e * n_pixels + p;
      const int64_t tstar = clamp_start(window_start[p], n_samples, W);
      window_outputs(wf + o * n_samples, pedestal[p], gain[p], tstar, W, nullptr, out_sum + o,
                     out_start + o, out_charge + o, out_time + o);
    }
  return 0;
}

// Local peak (R23): window placed `shift` samples before the trace's own
// largest sample (earliest on ties), clamped into [0, S-W].
int rta_oracle_extract_local_peak(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                                  int32_t n_samples, const int32_t* pedestal, const float* gain,
                                  int32_t W, int32_t shift, int32_t* out_sum, int32_t* out_start,
                                  float* out_charge, float* out_time) {
  if (bad_shape(n_events, n_pixels, n_samples, W)) return 1;
  for (int64_t e = 0; e < n_events; ++e)
    for (int64_t p = 0; p < n_pixels; ++p) {
      const int64_t o = e * n_pixels + p;
      const uint16_t* tr = wf + o * n_samples;
      const int64_t ped = pedestal[p];
      int64_t peak = 0;
      for (int64_t s = 1; s < n_samples; ++s)
        if ((int64_t)tr[s] - ped > (int64_t)tr[peak] - ped) peak = s;  // strict: earliest
      const int64_t tstar = clamp_start(peak - (int64_t)shift, n_samples, W);
      window_outputs(tr, ped, gain[p], tstar, W, nullptr, out_sum + o, out_start + o,
                     out_charge + o, out_time + o);
    }
  return 0;
}

// FIR / matched filter (R24): integer taps c[0..K-1]; the window is the
// filter's support at the position of the largest response (earliest on ties).
int rta_oracle_extract_fir(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                           int32_t n_samples, const int32_t* pedestal, const float* gain,
                           const int32_t* taps, int32_t K, int32_t* out_sum, int32_t* out_start,
                           float* out_charge, float* out_time) {
  if (bad_shape(n_events, n_pixels, n_samples, K)) return 1;
  for (int64_t e = 0; e < n_events; ++e)
    for (int64_t p = 0; p < n_pixels; ++p) {
      const int64_t o = e * n_pixels + p;
      const uint16_t* tr = wf + o * n_samples;
      const int64_t ped = pedestal[p];
      bool have = false;
      int64_t best = 0, tstar = 0;
      for (int64_t t = 0; t + K <= n_samples; ++t) {
        int64_t y = 0;
        for (int64_t k = 0; k < K; ++k) y += (int64_t)taps[k] * ((int64_t)tr[t + k] - ped);
        if (!have || y > best) {
          best = y;
          tstar = t;
          have = true;
        }
      }
      window_outputs(tr, ped, gain[p], tstar, K, taps, out_sum + o, out_start + o,
                     out_charge + o, out_time + o);
    }
  return 0;
}

}  // extern "C"
