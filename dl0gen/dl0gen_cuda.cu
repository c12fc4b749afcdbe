// dl0gen_cuda.cu — device build of the synthetic DL0 generator (dl0gen_core.h).
// Byte-identical to dl0gen_cpu.c by construction (tests/test_dl0gen.py checks
// it on the GPU box). Holds none of the extraction arithmetic; it only fills
// device buffers with input waveforms at bench scale (C5 is 14.84 G samples).
// Compile: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -fmad=false
#include <cuda_runtime.h>
#include "dl0gen_core.h"

__global__ void dl0gen_kernel(dl0gen_params q, long long first_event,
                              long long n_traces, unsigned short* __restrict__ wf) {
  const int S = q.n_samples;
  const int npairs = (S + 1) / 2;
  const long long total = n_traces * npairs;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
       i += (long long)gridDim.x * blockDim.x) {
    const long long lt = i / npairs;           // local trace
    const int j = (int)(i - lt * npairs);
    const unsigned long long trace =
        (unsigned long long)first_event * (unsigned long long)q.n_pixels + (unsigned long long)lt;
    const int p = (int)(trace % (unsigned long long)q.n_pixels);
    const float ped = (float)dg_pedestal(&q, p);
    const dg_pulse pl = dg_trace_pulse(&q, trace);
    uint16_t a, b;
    dg_sample_pair(&q, trace, ped, &pl, j, &a, &b);
    unsigned short* out = wf + lt * S;
    out[2 * j] = a;
    if (2 * j + 1 < S) out[2 * j + 1] = b;
  }
}

extern "C" int dl0gen_events_cuda(const dl0gen_params* q, long long first_event,
                                  long long n_events, unsigned short* wf_dev,
                                  void* stream) {
  if (n_events <= 0) return 0;
  const long long n_traces = n_events * q->n_pixels;
  const long long total = n_traces * ((q->n_samples + 1) / 2);
  long long blocks = (total + 255) / 256;
  if (blocks > 148LL * 64) blocks = 148LL * 64;
  dl0gen_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(
      *q, first_event, n_traces, wf_dev);
  return (int)cudaGetLastError();
}

// P12 encoder on the device (input preparation only; see dl0gen_cpu.c).
// One thread packs 8 samples into 3 words; n is the sample count.
__global__ void dl0gen_pack12_kernel(const unsigned short* __restrict__ in, long long n,
                                     unsigned char* __restrict__ out) {
  const long long npairs = (n + 1) / 2;
  for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < npairs;
       k += (long long)gridDim.x * blockDim.x) {
    const unsigned a = in[2 * k] & 0xFFFu;
    if (2 * k + 1 < n) {
      const unsigned b = in[2 * k + 1] & 0xFFFu;
      out[3 * k] = (unsigned char)(a & 0xFFu);
      out[3 * k + 1] = (unsigned char)((a >> 8) | ((b & 0xFu) << 4));
      out[3 * k + 2] = (unsigned char)(b >> 4);
    } else {
      out[3 * k] = (unsigned char)(a & 0xFFu);
      out[3 * k + 1] = (unsigned char)(a >> 8);
    }
  }
}

extern "C" int dl0gen_pack12_cuda(const unsigned short* in_dev, long long n,
                                  unsigned char* out_dev, void* stream) {
  if (n <= 0) return 0;
  long long blocks = ((n + 1) / 2 + 255) / 256;
  if (blocks > 148LL * 64) blocks = 148LL * 64;
  dl0gen_pack12_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(in_dev, n, out_dev);
  return (int)cudaGetLastError();
}
