/* dl0gen_cpu.c — host build of the synthetic DL0 generator (see dl0gen_core.h).
 * Compile: gcc -O2 -fPIC -shared -ffp-contract=off (never -ffast-math). */
#include "dl0gen_core.h"

void dl0gen_calib(const dl0gen_params* q, int32_t* pedestal, float* gain) {
  for (int32_t p = 0; p < q->n_pixels; ++p) {
    pedestal[p] = dg_pedestal(q, p);
    gain[p] = dg_gain(q, p);
  }
}

/* wf[n_events][P][S], events first_event .. first_event+n_events-1 */
void dl0gen_events_cpu(const dl0gen_params* q, int64_t first_event,
                       int64_t n_events, uint16_t* wf) {
  const int32_t P = q->n_pixels, S = q->n_samples;
  const int32_t npairs = (S + 1) / 2;
  for (int64_t e = 0; e < n_events; ++e) {
    for (int32_t p = 0; p < P; ++p) {
      const uint64_t trace = (uint64_t)(first_event + e) * (uint64_t)P + (uint64_t)p;
      const float ped = (float)dg_pedestal(q, p);
      const dg_pulse pl = dg_trace_pulse(q, trace);
      uint16_t* out = wf + ((uint64_t)e * P + p) * (uint64_t)S;
      for (int32_t j = 0; j < npairs; ++j) {
        uint16_t a, b;
        dg_sample_pair(q, trace, ped, &pl, j, &a, &b);
        out[2 * j] = a;
        if (2 * j + 1 < S) out[2 * j + 1] = b;
      }
    }
  }
}
