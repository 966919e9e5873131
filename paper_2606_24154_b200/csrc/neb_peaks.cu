// neb_peaks.cu — measurement aids: register-only FP64 microbenchmarks that give the
// roofline denominators MEASURED_PEAKS.json does not carry.  kind 0: independent DFMA chains (the
// plain FP64 pipe the influence kernels are bound by); kind 1: mma.sync.m8n8k4.f64 (DMMA, the
// FP64 tensor path of the LU trailing update).
#include "neb_internal.h"

namespace neb {

constexpr int kPeakThreads = 256;
constexpr int kPeakIters = 4096;
constexpr int kChains = 8;

__global__ void __launch_bounds__(kPeakThreads) dfma_peak_kernel(double* out, double a, double b) {
  double x[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) x[i] = a + i + threadIdx.x;
#pragma unroll 1
  for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < kChains; ++i) x[i] = fma(x[i], b, a);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += x[i];
  if (s == 12345.678) out[0] = s;   // never true: keeps the chains alive
}

// kind 2: the same number of independent DFMA, but every instruction reads THREE different registers (x += y z with
// per-chain y, z), as the instructions of the influence kernels do; the chain benchmark above feeds two of its three
// operands from the same two registers for all chains (operand reuse), which no real kernel can.
__global__ void __launch_bounds__(kPeakThreads) dfma3_peak_kernel(double* out, double a, double b) {
  double x[kChains], y[kChains], z[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) { x[i] = a + i + threadIdx.x; y[i] = (b + i) * 1e-3; z[i] = (a - i) * 1e-3 + threadIdx.x * 1e-9; }
#pragma unroll 1
  for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < kChains; ++i) x[i] = fma(y[(i + u) % kChains], z[(i + 2 * u + 1) % kChains], x[i]);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += x[i];
  if (s == 12345.678) out[0] = s;
}

// kind 3: as kind 2 with one multiplicand taken from the constant bank (the shape of a Horner step with a stored
// coefficient): two register sources per instruction.
__constant__ double k_peak_coef[kChains] = {1e-3, 1.1e-3, 1.2e-3, 1.3e-3, 1.4e-3, 1.5e-3, 1.6e-3, 1.7e-3};
__global__ void __launch_bounds__(kPeakThreads) dfma2c_peak_kernel(double* out, double a, double b) {
  double x[kChains], y[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) { x[i] = a + i + threadIdx.x; y[i] = (b + i) * 1e-3; }
#pragma unroll 1
  for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < kChains; ++i) x[i] = fma(y[(i + u) % kChains], k_peak_coef[(i + 2 * u + 1) % kChains], x[i]);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += x[i];
  if (s == 12345.678) out[0] = s;
}

__global__ void __launch_bounds__(kPeakThreads) dmma_peak_kernel(double* out, double a, double b) {
  double c[kChains][2];
#pragma unroll
  for (int i = 0; i < kChains; ++i) { c[i][0] = a + i; c[i][1] = b + threadIdx.x; }
  double fa = a * 1e-3, fb = b * 1e-3;
#pragma unroll 1
  for (int it = 0; it < kPeakIters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < kChains; ++i)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(fa), "d"(fb));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[0] = s;
}

neb_status fp64_peak(neb_ctx* c, int kind, double* tflops) {
  if (kind < 0 || kind > 3) return fail(c, NEB_EINVAL, "neb_fp64_peak: kind must be 0 (DFMA chains), 1 (DMMA), 2 (DFMA, three register operands) or 3 (DFMA, two register operands + constant bank)");
  NEB_TRY(ensure_scratch(c, 64));
  const int ctas = c->num_sms * 8;
  cudaEvent_t e0, e1;
  NEB_CUDA(c, cudaEventCreate(&e0));
  NEB_CUDA(c, cudaEventCreate(&e1));
  double best_ms = 1e30;
  for (int rep = 0; rep < 5; ++rep) {
    NEB_CUDA(c, cudaEventRecord(e0, c->stream));
    if (kind == 0) dfma_peak_kernel<<<ctas, kPeakThreads, 0, c->stream>>>(c->d_scratch, 1.0000001, 0.9999999);
    else if (kind == 2) dfma3_peak_kernel<<<ctas, kPeakThreads, 0, c->stream>>>(c->d_scratch, 1.0000001, 0.9999999);
    else if (kind == 3) dfma2c_peak_kernel<<<ctas, kPeakThreads, 0, c->stream>>>(c->d_scratch, 1.0000001, 0.9999999);
    else dmma_peak_kernel<<<ctas, kPeakThreads, 0, c->stream>>>(c->d_scratch, 1.0000001, 0.9999999);
    c->launches++;
    NEB_CUDA(c, cudaEventRecord(e1, c->stream));
    NEB_CUDA(c, cudaEventSynchronize(e1));
    float ms = 0.f;
    NEB_CUDA(c, cudaEventElapsedTime(&ms, e0, e1));
    if (rep > 0 && ms < best_ms) best_ms = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  double flop;
  if (kind != 1) flop = 2.0 * (double)ctas * kPeakThreads * kPeakIters * 4 * kChains;
  else flop = 2.0 * 8 * 8 * 4 * (double)ctas * (kPeakThreads / 32) * kPeakIters * 4 * kChains;
  *tflops = flop / (best_ms * 1e-3) * 1e-12;
  return NEB_OK;
}

}  // namespace neb
