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

// The instruction mix of one (template, SFT) pair of the moment-table kernel (ncu, profiles/r01d): per
// iteration 33 fp64, 20 packed fp32x2, 8 MUFU (+8 adds), 6 f64->f32 conversions, 80 scalar fp32 and 44 integer
// instructions = 199, spread evenly, 8 independent chains per class - i.e. with NO latency or memory stalls.
// What the schedulers sustain on it is the ceiling for this kernel's mix (B200: ~0.87 of 1 instruction/clock).
constexpr int MIXT_INSTR = 199, MIXT_ITERS = 512;
__global__ void __launch_bounds__(128) peak_mix_table_kernel(float *out, float a, float b) {
  double D[8];
  unsigned long long P[8], aa, bb;
  float M[4], S[8], Cv[4];
  int I[8];
  asm("mov.b64 %0, {%1, %1};" : "=l"(aa) : "f"(a));
  asm("mov.b64 %0, {%1, %1};" : "=l"(bb) : "f"(b));
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    D[i] = threadIdx.x + i; S[i] = (float)(threadIdx.x + i); I[i] = threadIdx.x * i;
    const float v = (float)i;
    asm("mov.b64 %0, {%1, %1};" : "=l"(P[i]) : "f"(v));
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) { M[i] = 1.5f + i; Cv[i] = 0.f; }
  const double da = a, db = b;
  constexpr int ND = 33, NP = 20, NM = 8, NC = 6, NS = 80, NI = 22;
  for (int it = 0; it < MIXT_ITERS; ++it) {
#pragma unroll
    for (int j = 0; j < 40; ++j) {
      if (j * ND / 40 != (j + 1) * ND / 40) asm volatile("fma.rn.f64 %0, %0, %1, %2;" : "+d"(D[j & 7]) : "d"(da), "d"(db));
      if (j * NP / 40 != (j + 1) * NP / 40) asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(P[j & 7]) : "l"(aa), "l"(bb));
      if (j * NM / 40 != (j + 1) * NM / 40) asm volatile("ex2.approx.ftz.f32 %0, %0;\n\tadd.rn.f32 %0, %0, %1;" : "+f"(M[j & 3]) : "f"(b));
      if (j * NC / 40 != (j + 1) * NC / 40) asm volatile("cvt.rn.f32.f64 %0, %1;" : "=f"(Cv[j & 3]) : "d"(D[(j + 3) & 7]));
#pragma unroll
      for (int r = 0; r < (NS + 39 - j) / 40; ++r) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(S[(j + r) & 7]) : "f"(a), "f"(b));
#pragma unroll
      for (int r = 0; r < (NI + 39 - j) / 40; ++r) asm volatile("add.s32 %0, %0, %1;\n\txor.b32 %0, %0, %2;" : "+r"(I[(j + r) & 7]) : "r"(it), "r"(j));
    }
  }
  float s = 0.f;
  unsigned long long x = 0;
  double d = 0.;
  int ii = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) { x ^= P[i]; s += S[i]; d += D[i]; ii ^= I[i]; }
#pragma unroll
  for (int i = 0; i < 4; ++i) s += M[i] + Cv[i];
  if (s == 1234.5f || x == 77 || d == 1234.5 || ii == 12345) out[0] = s;
}

}  // namespace sftk
