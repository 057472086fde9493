// td_probe.cuh - register-resident fp64 throughput probes: the denominators
// of the "alu" / fp64-tensor rooflines are measured on the box the bench runs on, not assumed.
//   kind 0: DFMA chains (vector fp64 pipe)          2 flop per lane-instruction
//   kind 1: DMMA.8x8x4 chains (fp64 tensor pipe)    512 flop per warp-instruction
//   kind 2: both in the same warps, interleaved     (do the two pipes overlap on sm_100a?)
//   kind 3: DADD chains                             1 flop per lane-instruction (the FFT's dominant op)
#pragma once
#include <cuda_runtime.h>

namespace td {

constexpr int PROBE_NT = 256, PROBE_ILP = 8, PROBE_INNER = 64;

template <int KIND>
__global__ void __launch_bounds__(PROBE_NT) probe_kernel(double* sink, int iters, double seed) {
  double f[PROBE_ILP], c0[PROBE_ILP], c1[PROBE_ILP];
  const double m = 1.0 + seed * 1e-9, a = seed * 1e-7 + (double)threadIdx.x * 1e-12;
#pragma unroll
  for (int i = 0; i < PROBE_ILP; ++i) { f[i] = a + i; c0[i] = a * i; c1[i] = a - i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < PROBE_INNER; ++u) {
#pragma unroll
      for (int i = 0; i < PROBE_ILP; ++i) {
        if (KIND == 0 || KIND == 2) f[i] = fma(f[i], m, a);
        if (KIND == 3) f[i] = f[i] + a;
        if (KIND == 1 || KIND == 2)
          asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
                       : "+d"(c0[i]), "+d"(c1[i])
                       : "d"(m), "d"(a));
      }
    }
  }
  double s = 0.0;
#pragma unroll
  for (int i = 0; i < PROBE_ILP; ++i) s += f[i] + c0[i] + c1[i];
  if (s == 12345.678) sink[0] = s;  // keeps the chains alive without a store on the timed path
}

// flops one launch performs
inline double probe_flops(int kind, int grid, int iters) {
  const double per_thread_steps = (double)iters * PROBE_INNER * PROBE_ILP;
  const double threads = (double)grid * PROBE_NT;
  double fl = 0.0;
  if (kind == 0 || kind == 2) fl += 2.0 * per_thread_steps * threads;
  if (kind == 3) fl += 1.0 * per_thread_steps * threads;
  if (kind == 1 || kind == 2) fl += 512.0 * per_thread_steps * (threads / 32.0);
  return fl;
}

}  // namespace td
