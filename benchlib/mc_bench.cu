// mc_bench.cu -- the bench's FP64 instruments (include/mc_bench.h): DFMA peak probe and operand-bandwidth probe.
// Built into benchlib/libmc_bench.so by benchlib/build.py; NOT part of libmc.so or of the product boundary.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>

#include "../include/mc_bench.h"

namespace {

#define MC_CUDA(call)                                                                          \
  do {                                                                                         \
    cudaError_t e_ = (call);                                                                   \
    if (e_ != cudaSuccess) {                                                                   \
      fprintf(stderr, "libmc_bench: CUDA error %d: %s\n", (int)e_, cudaGetErrorString(e_));  \
      return MC_ECUDA;                                                                         \
    }                                                                                          \
  } while (0)

// ---- DFMA throughput probe -------------------------------------------------------------------------
// 16 independent FMA chains per thread, 256 threads per block, 8 blocks per SM resident.
__global__ void __launch_bounds__(256)
dfma_peak_kernel(double* sink, int iters, double a, double b) {
  double x[16];
#pragma unroll
  for (int j = 0; j < 16; ++j) x[j] = 1.0 + 1e-9 * (threadIdx.x + j);
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int rep = 0; rep < 8; ++rep) {
#pragma unroll
      for (int j = 0; j < 16; ++j) x[j] = fma(x[j], a, b);
    }
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < 16; ++j) s += x[j];
  if (s == 123.456) sink[0] = s;   // never true: keeps the chains alive
}

// Operand-bandwidth probe (mc_fp64_probe): 8 independent accumulators per thread, x_j <- fma(y_j, *, x_j).
//   KIND 0: fma(y_j, z_j, x_j) -- three distinct vector registers per instruction
//   KIND 1: fma(y_j, s,   x_j) -- two + one register shared by consecutive instructions (operand reuse cache)
//   KIND 2: fma(y_j, c[], x_j) -- two registers + a constant-bank operand
//   KIND 3: x_j * y_j          -- DMUL, two registers
__constant__ double g_probe_const[2];
template <int KIND>
__global__ void __launch_bounds__(128)
dfma_operand_probe_kernel(double* sink, int iters, double a, double b) {
  double x[8], y[8], z[8];
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    x[j] = 1.0 + 1e-9 * (threadIdx.x + j);
    y[j] = 0.9999999 + 1e-12 * (threadIdx.x + 3 * j) * a;
    z[j] = 1e-9 * (1 + j) * b + 1e-15 * threadIdx.x;
  }
  const double s = a + 1e-15 * threadIdx.x;
#pragma unroll 1
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int rep = 0; rep < 8; ++rep) {
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        if (KIND == 0) x[j] = fma(y[j], z[j], x[j]);
        else if (KIND == 1) x[j] = fma(y[j], s, x[j]);
        else if (KIND == 2) x[j] = fma(y[j], g_probe_const[1], x[j]);
        else x[j] = x[j] * y[j];
      }
    }
  }
  double t = 0.0;
#pragma unroll
  for (int j = 0; j < 8; ++j) t += x[j] + y[j] + z[j];
  if (t == 123.456) sink[0] = t + s;   // never true: keeps the chains alive
}

}  // namespace

extern "C" {

int mc_fp64_peak(int32_t device, double millis, double* out_tflops, double* out_sm_clock_mhz) {
  if (!out_tflops || !(millis > 0.0)) return MC_EINVAL;
  MC_CUDA(cudaSetDevice(device));
  cudaDeviceProp prop;
  MC_CUDA(cudaGetDeviceProperties(&prop, device));
  double* sink = nullptr;
  MC_CUDA(cudaMalloc(&sink, sizeof(double)));
  cudaEvent_t e0, e1;
  MC_CUDA(cudaEventCreate(&e0));
  MC_CUDA(cudaEventCreate(&e1));
  const int grid = prop.multiProcessorCount * 8, block = 256;
  int iters = 2000;
  double best = 0.0;
  float ms = 0.f;
  for (int pass = 0; pass < 6; ++pass) {
    MC_CUDA(cudaEventRecord(e0, 0));
    dfma_peak_kernel<<<grid, block>>>(sink, iters, 0.999999999, 1e-9);
    MC_CUDA(cudaEventRecord(e1, 0));
    MC_CUDA(cudaEventSynchronize(e1));
    MC_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    const double flops = 2.0 * 16.0 * 8.0 * (double)iters * (double)grid * block;
    const double tf = flops / (ms * 1e-3) / 1e12;
    if (pass >= 2 && tf > best) best = tf;               // passes 0-1 size the run and warm the clocks
    if (pass < 2 && ms > 0.f) iters = (int)fmin(2.0e6, fmax(100.0, iters * millis / ms));
  }
  *out_tflops = best;
  if (out_sm_clock_mhz) {
    // cycles per second implied by one DFMA per lane per clock on 64 lanes per SM
    *out_sm_clock_mhz = best * 1e12 / (2.0 * 64.0 * prop.multiProcessorCount) / 1e6;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return MC_OK;
}

int mc_fp64_probe(int32_t device, double millis, int32_t kind, double* out_cycles_per_warp_instr, double* out_tflops) {
  if (!out_cycles_per_warp_instr || !(millis > 0.0) || kind < 0 || kind > 3) return MC_EINVAL;
  MC_CUDA(cudaSetDevice(device));
  cudaDeviceProp prop;
  MC_CUDA(cudaGetDeviceProperties(&prop, device));
  const double hc[2] = {0.0, 0.999999999};
  MC_CUDA(cudaMemcpyToSymbol(g_probe_const, hc, sizeof(hc)));
  double* sink = nullptr;
  MC_CUDA(cudaMalloc(&sink, sizeof(double)));
  cudaEvent_t e0, e1;
  MC_CUDA(cudaEventCreate(&e0));
  MC_CUDA(cudaEventCreate(&e1));
  const int warps_per_smsp = 4, block = 128, grid = prop.multiProcessorCount * warps_per_smsp;   // one warp per sub-partition per block
  int iters = 2000;
  float ms = 0.f, best = 1e30f;
  for (int pass = 0; pass < 6; ++pass) {
    MC_CUDA(cudaEventRecord(e0, 0));
    switch (kind) {
      case 0: dfma_operand_probe_kernel<0><<<grid, block>>>(sink, iters, 0.999999999, 1e-9); break;
      case 1: dfma_operand_probe_kernel<1><<<grid, block>>>(sink, iters, 0.999999999, 1e-9); break;
      case 2: dfma_operand_probe_kernel<2><<<grid, block>>>(sink, iters, 0.999999999, 1e-9); break;
      default: dfma_operand_probe_kernel<3><<<grid, block>>>(sink, iters, 0.999999999, 1e-9); break;
    }
    MC_CUDA(cudaEventRecord(e1, 0));
    MC_CUDA(cudaEventSynchronize(e1));
    MC_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    if (pass >= 2 && ms < best) best = ms;
    if (pass < 2 && ms > 0.f) iters = (int)fmin(2.0e6, fmax(100.0, iters * millis / ms));
  }
  // warp instructions per sub-partition = iters * 64 * warps_per_smsp; cycles at the device's maximum SM clock
  const double inst = (double)iters * 64.0 * warps_per_smsp;
  const double clk = prop.clockRate * 1e3;
  *out_cycles_per_warp_instr = best * 1e-3 * clk / inst;
  if (out_tflops) {
    const double flop_per_inst = kind == 3 ? 1.0 : 2.0;
    *out_tflops = flop_per_inst * 32.0 * inst * 4.0 * prop.multiProcessorCount / (best * 1e-3) / 1e12;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  return MC_OK;
}

}  // extern "C"
