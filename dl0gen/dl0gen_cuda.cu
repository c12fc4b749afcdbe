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
