// FP64 peak probes for the roofline denominators of bench.py: the rates the FP64 pipes of THIS device reach
// under THIS run's clocks, measured with the same instruction the hot kernels use.
//   which = 0: DMMA.8x8x4 (mma.sync.m8n8k4.f64), 8 independent accumulator chains per warp, 8 warps per SM
//   which = 1: DFMA with two loop-invariant operands (operand reuse: the friendly case), 8 chains per thread
//   which = 2: DFMA with three distinct, varying register operands per instruction (what a reflector
//              application looks like: no operand reuse) -- the register file, not the pipe, is the limit
// Nothing here is on the product path.
#include "be_common.cuh"

namespace {

__global__ void __launch_bounds__(256) k_probe_dmma(double* out, int iters) {
  double d[8][2];
#pragma unroll
  for (int i = 0; i < 8; ++i) { d[i][0] = threadIdx.x * 1e-9 + i; d[i][1] = 1.0; }
  const double a = 1.0 + 1e-12 * threadIdx.x, b = 1e-12;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int i = 0; i < 8; ++i)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                     : "+d"(d[i][0]), "+d"(d[i][1]) : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += d[i][0] + d[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_probe_dfma(double* out, int iters, double a, double b) {
  double x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = threadIdx.x + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 16; ++r)
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) k_probe_dfma3(double* out, const double* in, int iters) {
  double x[8], y[8], z[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x + i; y[i] = in[i + threadIdx.x % 3]; z[i] = in[8 + i + threadIdx.x % 5]; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 16; ++r)
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = fma(y[(i + r) & 7], z[(i + 3 * r + 1) & 7], x[i]);
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

}  // namespace

extern "C" int be_probe_fp64(be_ctx* ctx, int which, double* tflops) {
  BE_DEVICE_GUARD(ctx);
  if (!ctx || !tflops) return BE_ERR_NULL;
  if (which < 0 || which > 2) return BE_ERR_SHAPE;
  int prev = 0;
  BE_CUDA(cudaGetDevice(&prev));
  BE_CUDA(cudaSetDevice(ctx->device));
  const int blocks = ctx->sm_count * 2, threads = 256;
  double* buf = nullptr;
  BE_CUDA(cudaMalloc(&buf, ((size_t)blocks * threads + 64) * sizeof(double)));
  BE_CUDA(cudaMemsetAsync(buf, 0, ((size_t)blocks * threads + 64) * sizeof(double), ctx->stream));
  double* in = buf + (size_t)blocks * threads;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = which == 0 ? 4000 : 8000;
  double flops = 0.0;
  for (int rep = 0; rep < 2; ++rep) {   // first pass warms up
    cudaEventRecord(e0, ctx->stream);
    if (which == 0) {
      k_probe_dmma<<<blocks, threads, 0, ctx->stream>>>(buf, iters);
      flops = (double)blocks * (threads / 32) * iters * 64.0 * 512.0;          // 8 x 8 DMMAs of 2 * 8 * 8 * 4 flops
    } else if (which == 1) {
      k_probe_dfma<<<blocks, threads, 0, ctx->stream>>>(buf, iters, 1.0000001, 1e-9);
      flops = (double)blocks * threads * iters * 128.0 * 2.0;
    } else {
      k_probe_dfma3<<<blocks, threads, 0, ctx->stream>>>(buf, in, iters);
      flops = (double)blocks * threads * iters * 128.0 * 2.0;
    }
    cudaEventRecord(e1, ctx->stream);
  }
  ctx->launches += 2;
  cudaError_t e = cudaEventSynchronize(e1);
  float ms = 0.f;
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(buf);
  cudaSetDevice(prev);
  if (e != cudaSuccess) return (int)e;
  *tflops = flops / (ms * 1e-3) / 1e12;
  return BE_OK;
}
