// trex_probe.cu -- FP64 / FP32 FMA-pipe microbenchmark used as the roofline denominator of the |M|^2 kernels
// (MEASURED_PEAKS.json has no FP64 entry, so the peak is measured on the box in the same run).
// Every thread runs 8 independent register chains of fused multiply-adds; 2 flop per FMA.
#include "trex_ctx.h"

namespace trex {
namespace {

template <class R> __global__ void __launch_bounds__(256) k_fma_probe(R* out, int iters, R a, R b) {
  R x0 = R(threadIdx.x), x1 = x0 + R(1), x2 = x0 + R(2), x3 = x0 + R(3), x4 = x0 + R(4), x5 = x0 + R(5), x6 = x0 + R(6), x7 = x0 + R(7);
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  R s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == R(-12345.678)) out[0] = s;     // never true: keeps the chains alive
}

// the same with three REGISTER operands per FMA (the form real amplitude code has: no constant-bank operand, no operand
// reuse between consecutive instructions): what the register file can feed to the pipe
template <class R> __global__ void __launch_bounds__(256) k_fma_probe3(R* out, int iters, R a, R b) {
  R x[8], y[8], z[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) { x[k] = R(threadIdx.x + k); y[k] = a + R(1e-9) * R(threadIdx.x + 3 * k); z[k] = b + R(1e-9) * R(threadIdx.x + 5 * k); }
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int k = 0; k < 8; ++k) x[k] = fma(x[k], y[k], z[k]);
    }
  }
  R s = ((x[0] + x[1]) + (x[2] + x[3])) + ((x[4] + x[5]) + (x[6] + x[7]));
  if (s == R(-12345.678)) out[0] = s;
}

// FP64 tensor-core rate: mma.sync.m8n8k4.f64 (DMMA), 8 independent accumulator tiles per warp; 512 flop per mma.
// (tcgen05 has no f64 kind; this is the only tensor path an FP64 colour sum could take.)
__global__ void __launch_bounds__(256) k_dmma_probe(double* out, int iters, double a, double b) {
  double c[8][2];
#pragma unroll
  for (int k = 0; k < 8; ++k) { c[k][0] = threadIdx.x + k; c[k][1] = threadIdx.x - k; }
  const double fa = a + 1e-9 * threadIdx.x, fb = b + 1e-9 * threadIdx.x;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int k = 0; k < 8; ++k)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(fa), "d"(fb));
    }
  }
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < 8; ++k) s += c[k][0] + c[k][1];
  if (s == -12345.678) out[0] = s;
}

}  // namespace
}  // namespace trex

using namespace trex;

// Enqueues one probe launch on the library stream and returns the number of floating-point operations it executes
// (time it with events on that stream). fp32: 0 = FP64, 1 = FP32 (one register + two constant-bank operands per FMA);
// 2 = FP64, 3 = FP32 with three register operands per FMA; 4 = FP64 tensor cores (DMMA m8n8k4). Returns < 0 on error.
extern "C" double trex_probe_fma(int fp32, int blocks, int iters) {
  Context& c = ctx();
  if (blocks <= 0 || iters <= 0) return (double)fail(TREX_EINVAL, "trex_probe_fma: blocks and iters must be positive");
  if (!c.probe_out && cudaMalloc(&c.probe_out, 64) != cudaSuccess) return (double)fail(TREX_ENOMEM, "trex_probe_fma: cudaMalloc failed");
  if (fp32 == 4) {
    k_dmma_probe<<<blocks, 256, 0, c.stream>>>((double*)c.probe_out, iters, 0.999, 0.001);
    c.launches += 1;
    if (cudaGetLastError() != cudaSuccess) return (double)fail(TREX_ECUDA, "trex_probe_fma: launch failed");
    return 512.0 * 64.0 * (double)iters * 8.0 * (double)blocks;        // 512 flop x 64 mma per iteration x 8 warps
  }
  if (fp32 == 2) k_fma_probe3<double><<<blocks, 256, 0, c.stream>>>((double*)c.probe_out, iters, 0.999, 0.001);
  else if (fp32 == 3) k_fma_probe3<float><<<blocks, 256, 0, c.stream>>>((float*)c.probe_out, iters, 0.999f, 0.001f);
  else if (fp32) k_fma_probe<float><<<blocks, 256, 0, c.stream>>>((float*)c.probe_out, iters, 0.999f, 0.001f);
  else k_fma_probe<double><<<blocks, 256, 0, c.stream>>>((double*)c.probe_out, iters, 0.999, 0.001);
  c.launches += 1;
  if (cudaGetLastError() != cudaSuccess) return (double)fail(TREX_ECUDA, "trex_probe_fma: launch failed");
  return 2.0 * 64.0 * (double)iters * 256.0 * (double)blocks;
}
