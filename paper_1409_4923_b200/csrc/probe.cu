// probe.cu -- pipe-throughput probes (measurement aid for the "alu" roofline).
// Each thread runs `iters` x 64 operations of one kind on 8 independent chains so that the pipe, not latency,
// limits the rate.  The caller times the launch with CUDA events: rate = blocks*threads*iters*64 / time.
#include "dispatch.cuh"

namespace bm {

template <int OP>
__global__ void __launch_bounds__(1024) probe_kernel(int iters, float *sink) {
  const int tid = blockIdx.x * blockDim.x + threadIdx.x;
  float f[8];
  uint32_t u[8];
  double dd[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    f[i] = 1.0f + 1e-3f * (float)((tid + i) & 255);
    u[i] = 0x9E3779B9u * (uint32_t)(tid + i + 1);
    dd[i] = 1.0 + 1e-3 * (double)((tid + i) & 255);
  }
  const float ca = 0.9999f, cb = 1e-4f;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (OP == BM_PROBE_FFMA) f[i] = fmaf(f[i], ca, cb);
        if (OP == BM_PROBE_FADD) f[i] = f[i] + cb;
        if (OP == BM_PROBE_MUFU_COS) asm volatile("cos.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
        if (OP == BM_PROBE_MUFU_LG2) asm volatile("lg2.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
        if (OP == BM_PROBE_MUFU_SQRT) asm volatile("sqrt.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
        if (OP == BM_PROBE_IMAD_WIDE) {
          unsigned long long p = (unsigned long long)u[i] * 0xD2511F53u;
          u[i] = (uint32_t)(p >> 32) ^ (uint32_t)p;  // counted as 1 IMAD.WIDE + 1 LOP3
        }
        if (OP == BM_PROBE_LOP3) u[i] = (u[i] ^ u[(i + 1) & 7]) ^ 0x85EBCA6Bu;
        if (OP == BM_PROBE_DFMA) dd[i] = fma(dd[i], 0.9999, 1e-4);
        if (OP == BM_PROBE_I2F) { f[i] = (float)u[i]; u[i] += __float_as_uint(f[i]); }
        if (OP == BM_PROBE_MIX) {  // 1 MUFU + 4 FFMA + 2 integer: the rough mix of a path step
          asm volatile("cos.approx.ftz.f32 %0, %0;" : "+f"(f[i]));
          f[i] = fmaf(f[i], ca, cb); f[i] = fmaf(f[i], ca, cb); f[i] = fmaf(f[i], ca, cb); f[i] = fmaf(f[i], ca, cb);
          u[i] = (u[i] ^ u[(i + 1) & 7]) + 0x85EBCA6Bu;
        }
      }
    }
  }
  float acc = 0.f;
#pragma unroll
  for (int i = 0; i < 8; ++i) acc += f[i] + (float)u[i] + (float)dd[i];
  sink[tid] = acc;
}

cudaError_t launch_probe(int op, int iters, int blocks, int threads, float *sink, cudaStream_t st) {
  switch (op) {
#define BM_CASE(X) case X: probe_kernel<X><<<blocks, threads, 0, st>>>(iters, sink); break;
    BM_CASE(BM_PROBE_FFMA) BM_CASE(BM_PROBE_MUFU_COS) BM_CASE(BM_PROBE_MUFU_LG2) BM_CASE(BM_PROBE_MUFU_SQRT)
    BM_CASE(BM_PROBE_IMAD_WIDE) BM_CASE(BM_PROBE_LOP3) BM_CASE(BM_PROBE_DFMA) BM_CASE(BM_PROBE_I2F)
    BM_CASE(BM_PROBE_FADD) BM_CASE(BM_PROBE_MIX)
#undef BM_CASE
    default: return cudaErrorInvalidValue;
  }
  return cudaGetLastError();
}

}  // namespace bm
