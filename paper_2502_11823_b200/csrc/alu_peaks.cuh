// alu_peaks.cuh - measures the plain-ALU pipe rates that bound the SFT inner-product kernel
// (MEASURED_PEAKS.json holds only HBM copy and bf16 matmul; this path is bound by the
// FP32 / FP64 / XU pipes).  Exposed through the C ABI as sft_measure_alu_peaks; bench.py reports
// the numbers beside the roofline.  Each kernel runs ILP independent dependency chains per thread.
#pragma once
#include <cuda_runtime.h>

namespace sftk {

constexpr int PEAK_ILP = 8;
constexpr int PEAK_ITERS = 4096;

__global__ void peak_ffma_kernel(float *out, float a, float b) {
  float r[PEAK_ILP];
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) r[i] = (float)(threadIdx.x + i);
  for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(r[i]) : "f"(a), "f"(b));
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) s += r[i];
  if (s == 12345.678f) out[0] = s;
}

__global__ void peak_ffma2_kernel(float *out, float a, float b) {
  unsigned long long r[PEAK_ILP], aa, bb;
  asm("mov.b64 %0, {%1, %1};" : "=l"(aa) : "f"(a));
  asm("mov.b64 %0, {%1, %1};" : "=l"(bb) : "f"(b));
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) {
    const float v = (float)(threadIdx.x + i);
    asm("mov.b64 %0, {%1, %1};" : "=l"(r[i]) : "f"(v));
  }
  for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(r[i]) : "l"(aa), "l"(bb));
  }
  unsigned long long s = 0;
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) s ^= r[i];
  if (s == 0x123456789abcdefull) out[0] = 1.f;
}

__global__ void peak_dfma_kernel(float *out, double a, double b) {
  double r[PEAK_ILP];
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) r[i] = (double)(threadIdx.x + i);
  for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(r[i]) : "d"(a), "d"(b));
  }
  double s = 0.;
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) s += r[i];
  if (s == 12345.678) out[0] = (float)s;
}

__global__ void peak_mufu_kernel(float *out, float a) {
  float r[PEAK_ILP];
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) r[i] = a + (float)(threadIdx.x + i);
  for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i)      // the add keeps ptxas from folding rcp(rcp(x)); it runs on the 4x faster FP32 pipe
      asm volatile("rcp.approx.ftz.f32 %0, %0;\n\tadd.rn.f32 %0, %0, %1;" : "+f"(r[i]) : "f"(a));
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) s += r[i];
  if (s == 12345.678f) out[0] = s;
}

// 2 FFMA : 1 MUFU : mix, to see whether the pipes overlap
__global__ void peak_mix_kernel(float *out, float a, float b) {
  float r[PEAK_ILP], q[PEAK_ILP / 4];
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) r[i] = (float)(threadIdx.x + i);
#pragma unroll
  for (int i = 0; i < PEAK_ILP / 4; ++i) q[i] = a + (float)(threadIdx.x + i);
  for (int it = 0; it < PEAK_ITERS; ++it) {
#pragma unroll
    for (int i = 0; i < PEAK_ILP; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(r[i]) : "f"(a), "f"(b));
#pragma unroll
    for (int i = 0; i < PEAK_ILP / 4; ++i) asm volatile("rcp.approx.ftz.f32 %0, %0;" : "+f"(q[i]));
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < PEAK_ILP; ++i) s += r[i];
#pragma unroll
  for (int i = 0; i < PEAK_ILP / 4; ++i) s += q[i];
  if (s == 12345.678f) out[0] = s;
}

}  // namespace sftk
