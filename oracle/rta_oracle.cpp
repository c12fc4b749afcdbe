// oracle/rta_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, single-threaded CPU definition of the sliding-window signal
// extraction that BASELINE.json:north_star names (the paper itself only says
// "several signal extraction algorithms [13] are being currently ported to
// CUDA", §5; the definition is north_star sentence 2, expanded in
// SURVEY.md §8(c) and DESIGN.md "Readings").
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
// reference legs may call this. It shares no code, header, table or helper
// with paper_1307_6489_b200/csrc (the CUDA path) and neither includes the
// other. Parity status: every output is pinned (tests/test_oracle_pins.py):
// closed forms, hand-worked fixtures in tests/golden/, brute force against an
// independent numpy restatement, and the maximality/earliest invariants.
//
// Per trace (event e, pixel p), in the order of north_star sentence 2:
//   x[s]    = wf[e][p][s] - pedestal[p]                      (a2, reading R2/R8: signed)
//   Sum(t)  = x[t] + ... + x[t+W-1],  t = 0 .. S-W           (a3, reading R5: windows inside the trace)
//   t*      = the smallest t with Sum(t) maximal             (a4, reading R6: earliest on ties)
//   out_sum = Sum(t*), out_start = t*                        (a5)
//   charge  = RN32( Sum(t*) * gain[p] )                      (a6, reading R10)
//   time    = RN32( sum_s s*x[s] / Sum(t*) ), s in window    (a7, reading R9: absolute 0-based index)
//             and t* + (W-1)/2 when Sum(t*) <= 0             (reading R7)
// Integers are int64 inside, floats are computed in double and rounded once.

#include <cstdint>
#include <cstddef>

extern "C" {

// Returns 0 on success, 1 on a bad shape (W < 1, W > S, S < 1, P < 1, E < 0).
int rta_oracle_extract(const uint16_t* wf, int64_t n_events, int32_t n_pixels,
                       int32_t n_samples, const int32_t* pedestal,
                       const float* gain, int32_t W, int32_t* out_sum,
                       int32_t* out_start, float* out_charge, float* out_time) {
  if (n_events < 0 || n_pixels < 1 || n_samples < 1 || W < 1 || W > n_samples)
    return 1;
  const int64_t S = n_samples;
  for (int64_t e = 0; e < n_events; ++e) {
    for (int64_t p = 0; p < n_pixels; ++p) {
      const uint16_t* tr = wf + (e * n_pixels + p) * S;
      const int64_t ped = pedestal[p];
      bool have = false;
      int64_t best = 0;
      int64_t tstar = 0;
      for (int64_t t = 0; t + W <= S; ++t) {  // ascending t
        int64_t acc = 0;
        for (int64_t k = 0; k < W; ++k) acc += (int64_t)tr[t + k] - ped;
        if (!have || acc > best) {  // strict '>' keeps the earliest maximum
          best = acc;
          tstar = t;
          have = true;
        }
      }
      int64_t num = 0;
      for (int64_t k = 0; k < W; ++k)
        num += (tstar + k) * ((int64_t)tr[tstar + k] - ped);
      const int64_t o = e * n_pixels + p;
      out_sum[o] = (int32_t)best;
      out_start[o] = (int32_t)tstar;
      out_charge[o] = (float)((double)best * (double)gain[p]);
      out_time[o] = best > 0 ? (float)((double)num / (double)best)
                             : (float)((double)tstar + 0.5 * (double)(W - 1));
    }
  }
  return 0;
}

}  // extern "C"
