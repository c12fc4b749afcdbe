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

/* P12 encoder (input preparation for the packed-ingest path; the DECODER is
 * the method's step and lives in oracle/ and in the CUDA library, not here).
 * Samples are masked to 12 bits. out holds (12 n + 7) / 8 bytes. */
void dl0gen_pack12_cpu(const uint16_t* in, int64_t n, uint8_t* out) {
  int64_t k = 0;
  for (; 2 * k + 1 < n; ++k) {
    const unsigned a = in[2 * k] & 0xFFFu, b = in[2 * k + 1] & 0xFFFu;
    out[3 * k] = (uint8_t)(a & 0xFFu);
    out[3 * k + 1] = (uint8_t)((a >> 8) | ((b & 0xFu) << 4));
    out[3 * k + 2] = (uint8_t)(b >> 4);
  }
  if (2 * k < n) {
    const unsigned a = in[2 * k] & 0xFFFu;
    out[3 * k] = (uint8_t)(a & 0xFFu);
    out[3 * k + 1] = (uint8_t)(a >> 8);
  }
}
