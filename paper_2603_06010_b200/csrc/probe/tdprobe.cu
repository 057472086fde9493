// tdprobe.cu - bench-only library (libtdprobe.so, include/tdprobe.h): register-resident throughput probes
// (SURVEY.md 7.1 step 0).  The denominators of the "alu" / fp64-tensor rooflines are measured on the box the
// bench runs on, not assumed.  Not part of the product library: nothing in libtdlike.so calls or links this.
//   kind 0: DFMA chains (vector fp64 pipe)          2 flop per lane-instruction
//   kind 1: DMMA.8x8x4 chains (fp64 tensor pipe)    512 flop per warp-instruction
//   kind 2: both in the same warps, interleaved     (do the two pipes overlap on sm_100a?)
//   kind 3: DADD chains                             1 flop per lane-instruction (the FFT's dominant op)
//   kind 4: FFMA chains (fp32 pipe)                 2 flop per lane-instruction (roofline of the fp32 evaluation mode)
#include "../../../include/tdprobe.h"

#include <cuda_runtime.h>

namespace {

constexpr int PROBE_NT = 256, PROBE_ILP = 8, PROBE_INNER = 64;

template <int KIND>
__global__ void __launch_bounds__(PROBE_NT) probe_kernel(double* sink, int iters, double seed) {
  double f[PROBE_ILP], c0[PROBE_ILP], c1[PROBE_ILP];
  float g[2 * PROBE_ILP];
  const double m = 1.0 + seed * 1e-9, a = seed * 1e-7 + (double)threadIdx.x * 1e-12;
  const float mf = (float)m, af = (float)a;
#pragma unroll
  for (int i = 0; i < PROBE_ILP; ++i) {
    f[i] = a + i; c0[i] = a * i; c1[i] = a - i;
    g[2 * i] = af + i; g[2 * i + 1] = af - i;
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PROBE_INNER; ++u) {
#pragma unroll
      for (int i = 0; i < PROBE_ILP; ++i) {
        if (KIND == 0 || KIND == 2) f[i] = fma(f[i], m, a);
        if (KIND == 3) f[i] = f[i] + a;
        if (KIND == 4) { g[2 * i] = fmaf(g[2 * i], mf, af); g[2 * i + 1] = fmaf(g[2 * i + 1], mf, af); }
        if (KIND == 1 || KIND == 2)
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                       : "+d"(c0[i]), "+d"(c1[i])
                       : "d"(m), "d"(a));
      }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < PROBE_ILP; ++i) s += f[i] + c0[i] + c1[i] + (double)g[2 * i] + (double)g[2 * i + 1];
  if (s == 12345.678) sink[0] = s;  // keeps the chains alive without a store on the timed path
}

// flops one launch performs
double probe_flops(int kind, int grid, int iters) {
  const double per_thread_steps = (double)iters * PROBE_INNER * PROBE_ILP;
  const double threads = (double)grid * PROBE_NT;
  double fl = 0.0;
  if (kind == 0 || kind == 2) fl += 2.0 * per_thread_steps * threads;
  if (kind == 3) fl += 1.0 * per_thread_steps * threads;
  if (kind == 4) fl += 4.0 * per_thread_steps * threads;
  if (kind == 1 || kind == 2) fl += 512.0 * per_thread_steps * (threads / 32.0);
  return fl;
}

}  // namespace

extern "C" int td_probe_throughput(int kind, int device, double* tflops) {
  if (kind < 0 || kind > 4 || !tflops) return 1;
  int ndev = 0, prev = -1;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return 4;
  if (device < 0 || device >= ndev) return 1;
  if (cudaGetDevice(&prev) != cudaSuccess || cudaSetDevice(device) != cudaSuccess) return 4;
  cudaDeviceProp prop;
  int rc = 0, grid = 0;
  double* sink = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  float best = 1e30f;
  const int iters = 200;
  if (cudaGetDeviceProperties(&prop, device) != cudaSuccess || cudaMalloc(&sink, sizeof(double)) != cudaSuccess) rc = 4;
  if (rc == 0) {
    grid = prop.multiProcessorCount * 8;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    for (int rep = 0; rep < 6 && rc == 0; ++rep) {
      cudaEventRecord(e0, 0);
      switch (kind) {
        case 0: probe_kernel<0><<<grid, PROBE_NT>>>(sink, iters, 1.0 + rep); break;
        case 1: probe_kernel<1><<<grid, PROBE_NT>>>(sink, iters, 1.0 + rep); break;
        case 2: probe_kernel<2><<<grid, PROBE_NT>>>(sink, iters, 1.0 + rep); break;
        case 3: probe_kernel<3><<<grid, PROBE_NT>>>(sink, iters, 1.0 + rep); break;
        default: probe_kernel<4><<<grid, PROBE_NT>>>(sink, iters, 1.0 + rep); break;
      }
      cudaEventRecord(e1, 0);
      if (cudaEventSynchronize(e1) != cudaSuccess || cudaGetLastError() != cudaSuccess) { rc = 4; break; }
      float ms = 0.f;
      cudaEventElapsedTime(&ms, e0, e1);
      if (rep > 0 && ms < best) best = ms;  // first launch is the warm-up
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
  }
  cudaFree(sink);
  cudaSetDevice(prev);
  if (rc == 0) *tflops = probe_flops(kind, grid, iters) / (best * 1e-3) / 1e12;
  return rc;
}
