/* dl0gen_core.h — seeded synthetic DL0 waveform generator, arithmetic core.
 *
 * Stands in for the paper's "Prod2" simulated data (§5), which is
 * not available; recipe = BASELINE.json:configs (pedestal + Gaussian noise +
 * sparse Gaussian pulses with log-normal amplitude, 12-bit clamp), stated in
 * DESIGN.md "Input recipe". This module holds NONE of the extraction method's
 * arithmetic and is the only code shared between the oracle side and the CUDA
 * side of the tests: both read the bytes it writes.
 *
 * The same header compiles as C (dl0gen_cpu.c, gcc) and CUDA (dl0gen_cuda.cu,
 * nvcc) and produces IDENTICAL bytes on both: every floating-point step is a
 * single correctly-rounded IEEE binary32 operation (+ - * / sqrt, int<->float
 * conversion) issued through dg_* wrappers that forbid FMA contraction
 * (__fmul_rn etc. on the device, -ffp-contract=off on the host); log, exp, sin
 * and cos are short polynomials built from those operations instead of libm /
 * libdevice calls. Random numbers are counter-based (splitmix64 finaliser over
 * (seed, stream, trace, counter)), so any event range can be generated
 * independently, in any order, on either side.
 */
#ifndef DL0GEN_CORE_H
#define DL0GEN_CORE_H

#include <stdint.h>

#if defined(__CUDACC__)
#define DG_FN __host__ __device__ __forceinline__
#else
#include <math.h>
#include <string.h>
#define DG_FN static inline
#endif

typedef struct dl0gen_params {
  uint64_t seed;
  int32_t n_pixels;     /* P */
  int32_t n_samples;    /* S */
  int32_t ped_lo;       /* pedestal ~ integer U{ped_lo..ped_hi} per pixel */
  int32_t ped_hi;
  int32_t adc_max;      /* clamp to [0, adc_max] (4095 = 12 bit) */
  float gain_lo;        /* gain ~ U[gain_lo, gain_hi] per pixel */
  float gain_hi;
  float noise_sigma;    /* Gaussian noise per sample, ADC counts */
  float pulse_frac;     /* Bernoulli probability per (event, pixel) */
  float pulse_sigma;    /* pulse width, samples */
  float peak_lo;        /* pulse position ~ U[peak_lo, peak_hi], samples */
  float peak_hi;
  float amp_mu;         /* amplitude = exp(amp_mu + amp_sigma * N(0,1)), ADC */
  float amp_sigma;
} dl0gen_params;

/* ---- correctly-rounded single operations, no contraction ---------------- */
DG_FN float dg_mul(float a, float b) {
#if defined(__CUDA_ARCH__)
  return __fmul_rn(a, b);
#else
  return a * b;
#endif
}
DG_FN float dg_add(float a, float b) {
#if defined(__CUDA_ARCH__)
  return __fadd_rn(a, b);
#else
  return a + b;
#endif
}
DG_FN float dg_sub(float a, float b) {
#if defined(__CUDA_ARCH__)
  return __fsub_rn(a, b);
#else
  return a - b;
#endif
}
DG_FN float dg_div(float a, float b) {
#if defined(__CUDA_ARCH__)
  return __fdiv_rn(a, b);
#else
  return a / b;
#endif
}
DG_FN float dg_sqrt(float a) {
#if defined(__CUDA_ARCH__)
  return __fsqrt_rn(a);
#else
  return sqrtf(a);
#endif
}
DG_FN uint32_t dg_f2u(float f) {
#if defined(__CUDA_ARCH__)
  return __float_as_uint(f);
#else
  uint32_t u;
  memcpy(&u, &f, 4);
  return u;
#endif
}
DG_FN float dg_u2f(uint32_t u) {
#if defined(__CUDA_ARCH__)
  return __uint_as_float(u);
#else
  float f;
  memcpy(&f, &u, 4);
  return f;
#endif
}

/* ---- counter-based random numbers --------------------------------------- */
DG_FN uint64_t dg_mix64(uint64_t z) {
  z ^= z >> 30;
  z *= 0xBF58476D1CE4E5B9ull;
  z ^= z >> 27;
  z *= 0x94D049BB133111EBull;
  z ^= z >> 31;
  return z;
}
enum { DG_STREAM_PED = 1, DG_STREAM_GAIN = 2, DG_STREAM_PULSE = 3, DG_STREAM_NOISE = 4 };

/* key of one (seed, stream, index) triple; draws are dg_draw(key, counter) */
DG_FN uint64_t dg_key(uint64_t seed, uint32_t stream, uint64_t index) {
  uint64_t k = dg_mix64(seed + 0x9E3779B97F4A7C15ull * (uint64_t)stream);
  return dg_mix64(k ^ dg_mix64(index + 0xD1B54A32D192ED03ull));
}
DG_FN uint64_t dg_draw(uint64_t key, uint32_t counter) {
  return dg_mix64(key + 0x9E3779B97F4A7C15ull * (uint64_t)(counter + 1u));
}
/* uniform in (0,1): odd multiples of 2^-24, exactly representable */
DG_FN float dg_u01(uint64_t h) {
  uint32_t m = (uint32_t)(h >> 41) * 2u + 1u; /* 24-bit odd */
  return dg_mul((float)m, 5.9604644775390625e-08f);
}

/* ---- elementary functions from single IEEE operations ------------------- */
/* natural log, x > 0 and normal; |rel err| ~ 2e-7 */
DG_FN float dg_log(float x) {
  uint32_t b = dg_f2u(x);
  int32_t e = (int32_t)(b >> 23) - 127;
  float m = dg_u2f((b & 0x007FFFFFu) | 0x3F800000u); /* [1,2) */
  if (m > 1.41421356f) {
    m = dg_mul(m, 0.5f);
    e += 1;
  }
  float s = dg_div(dg_sub(m, 1.0f), dg_add(m, 1.0f));
  float z = dg_mul(s, s);
  float p = 0.11111111f;
  p = dg_add(dg_mul(p, z), 0.14285715f);
  p = dg_add(dg_mul(p, z), 0.2f);
  p = dg_add(dg_mul(p, z), 0.33333334f);
  p = dg_mul(p, z);
  float lm = dg_add(dg_mul(2.0f, s), dg_mul(dg_mul(2.0f, s), p));
  float ef = (float)e;
  return dg_add(dg_mul(ef, 0.693145751953125f),
                dg_add(lm, dg_mul(ef, 1.42860682030941723212e-6f)));
}
/* exp, x clamped to [-87, 88]; |rel err| ~ 2e-7 */
DG_FN float dg_exp(float x) {
  if (x < -87.0f) x = -87.0f;
  if (x > 88.0f) x = 88.0f;
  float t = dg_mul(x, 1.44269504f);
  int32_t k = (int32_t)dg_add(t, t >= 0.0f ? 0.5f : -0.5f);
  float kf = (float)k;
  float r = dg_sub(dg_sub(x, dg_mul(kf, 0.693145751953125f)),
                   dg_mul(kf, 1.42860682030941723212e-6f));
  float p = 1.98412698e-4f; /* 1/5040 */
  p = dg_add(dg_mul(p, r), 1.38888889e-3f);
  p = dg_add(dg_mul(p, r), 8.33333333e-3f);
  p = dg_add(dg_mul(p, r), 4.16666667e-2f);
  p = dg_add(dg_mul(p, r), 1.66666667e-1f);
  p = dg_add(dg_mul(p, r), 0.5f);
  p = dg_add(dg_mul(p, r), 1.0f);
  p = dg_add(dg_mul(p, r), 1.0f);
  return dg_mul(p, dg_u2f((uint32_t)(k + 127) << 23));
}
/* sin and cos of 2*pi*u, u in [0,1) */
DG_FN void dg_sincos2pi(float u, float* sn, float* cs) {
  int32_t q = (int32_t)dg_add(dg_mul(u, 4.0f), 0.5f); /* 0..4 */
  float r = dg_sub(u, dg_mul((float)q, 0.25f));       /* [-1/8, 1/8] */
  float a = dg_mul(r, 6.28318530718f);
  float z = dg_mul(a, a);
  float s = 2.75573192e-6f; /* 1/9! */
  s = dg_sub(dg_mul(s, z), 1.98412698e-4f);
  s = dg_add(dg_mul(s, z), 8.33333333e-3f);
  s = dg_sub(dg_mul(s, z), 1.66666667e-1f);
  s = dg_add(dg_mul(s, z), 1.0f);
  s = dg_mul(s, a);
  float c = -2.75573192e-7f; /* -1/10! */
  c = dg_add(dg_mul(c, z), 2.48015873e-5f);
  c = dg_sub(dg_mul(c, z), 1.38888889e-3f);
  c = dg_add(dg_mul(c, z), 4.16666667e-2f);
  c = dg_sub(dg_mul(c, z), 0.5f);
  c = dg_add(dg_mul(c, z), 1.0f);
  switch (q & 3) {
    case 0: *sn = s; *cs = c; break;
    case 1: *sn = c; *cs = -s; break;
    case 2: *sn = -s; *cs = -c; break;
    default: *sn = -c; *cs = s; break;
  }
}
/* two independent N(0,1) from two draws (Box-Muller) */
DG_FN void dg_normal2(uint64_t h1, uint64_t h2, float* n0, float* n1) {
  float r = dg_sqrt(dg_mul(-2.0f, dg_log(dg_u01(h1))));
  float sn, cs;
  dg_sincos2pi(dg_mul((float)(uint32_t)(h2 >> 40), 5.9604644775390625e-08f), &sn, &cs);
  *n0 = dg_mul(r, cs);
  *n1 = dg_mul(r, sn);
}

/* ---- calibration constants per pixel ------------------------------------ */
DG_FN int32_t dg_pedestal(const dl0gen_params* q, int32_t p) {
  uint64_t h = dg_draw(dg_key(q->seed, DG_STREAM_PED, (uint64_t)p), 0);
  uint32_t span = (uint32_t)(q->ped_hi - q->ped_lo + 1);
  return q->ped_lo + (int32_t)((h >> 33) % span);
}
DG_FN float dg_gain(const dl0gen_params* q, int32_t p) {
  uint64_t h = dg_draw(dg_key(q->seed, DG_STREAM_GAIN, (uint64_t)p), 0);
  return dg_add(q->gain_lo, dg_mul(dg_sub(q->gain_hi, q->gain_lo), dg_u01(h)));
}

/* ---- per-trace pulse parameters ------------------------------------------ */
typedef struct dg_pulse {
  int32_t on;
  float mu;   /* position, samples */
  float amp;  /* ADC counts */
} dg_pulse;

DG_FN dg_pulse dg_trace_pulse(const dl0gen_params* q, uint64_t trace) {
  dg_pulse pl;
  uint64_t key = dg_key(q->seed, DG_STREAM_PULSE, trace);
  pl.on = dg_u01(dg_draw(key, 0)) < q->pulse_frac;
  pl.mu = 0.0f;
  pl.amp = 0.0f;
  if (pl.on) {
    pl.mu = dg_add(q->peak_lo,
                   dg_mul(dg_sub(q->peak_hi, q->peak_lo), dg_u01(dg_draw(key, 1))));
    float z0, z1;
    dg_normal2(dg_draw(key, 2), dg_draw(key, 3), &z0, &z1);
    pl.amp = dg_exp(dg_add(q->amp_mu, dg_mul(q->amp_sigma, z0)));
  }
  return pl;
}

/* one sample: clamp(floor(ped + noise + pulse + 0.5), 0, adc_max) */
DG_FN uint16_t dg_quantise(const dl0gen_params* q, float ped, float noise,
                           const dg_pulse* pl, int32_t s) {
  float v = dg_add(ped, noise);
  if (pl->on) {
    float d = dg_div(dg_sub((float)s, pl->mu), q->pulse_sigma);
    float e = dg_mul(-0.5f, dg_mul(d, d));
    if (e > -40.0f) v = dg_add(v, dg_mul(pl->amp, dg_exp(e)));
  }
  float w = dg_add(v, 0.5f);
  int32_t i = (w <= 0.0f) ? 0 : (w >= 65535.0f ? 65535 : (int32_t)w);
  if (i > q->adc_max) i = q->adc_max;
  return (uint16_t)i;
}

/* samples 2j and 2j+1 of one trace (the second is ignored when 2j+1 == S) */
DG_FN void dg_sample_pair(const dl0gen_params* q, uint64_t trace, float ped,
                          const dg_pulse* pl, int32_t j, uint16_t* a, uint16_t* b) {
  uint64_t key = dg_key(q->seed, DG_STREAM_NOISE, trace);
  float n0, n1;
  dg_normal2(dg_draw(key, (uint32_t)(2 * j)), dg_draw(key, (uint32_t)(2 * j + 1)), &n0, &n1);
  *a = dg_quantise(q, ped, dg_mul(q->noise_sigma, n0), pl, 2 * j);
  *b = dg_quantise(q, ped, dg_mul(q->noise_sigma, n1), pl, 2 * j + 1);
}

#endif /* DL0GEN_CORE_H */
