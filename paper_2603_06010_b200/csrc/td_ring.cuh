// td_ring.cuh - damped-sinusoid ("ringdown") rows synthesised inside the first pass of the fused FFT kernels
// (second step; waveform generation, projection and placement are the
// O(N) step immediately before the hot path).  With it the template never exists in memory: 40 bytes of parameters per
// (template, segment) replace the 8 N_s-byte row, the scratch panel of td_synth.cuh and its trip through HBM.
//
//   h_i = A exp(-(t_i - t0)/tau) cos(2 pi f (t_i - t0) + phi)   for t_i = i / fs >= t0,   else 0
//       = Re z_i,   z_i = A e^{i phi} lambda^(i - t0 fs),   lambda = exp((-1/tau + 2 pi i f) / fs)
//
// A thread of the first pass needs the sample pairs (i_k, i_k + 1), i_k = i_first + k stride (k < K): it anchors z at its
// first pair that can be live (one exp, one sincospi), steps it by Lambda = lambda^stride and takes the odd sample from one
// more product with lambda.  lambda, Lambda, A e^{i phi} and the onset index are the same for every thread of an item: warp 0
// computes them for the NEXT item while the others are in the last pass (ring_prepare), hands them over through shared memory
// and the mbarrier that otherwise counts the bytes of the TMA row copy.  All of it is fp64 in both precisions (the fp32
// build rounds the residual d - h once, as with rows from memory).
#pragma once
#include <cuda_runtime.h>

namespace TD_NS {

struct RingConsts {
  double lx, ly;     // lambda
  double Lx, Ly;     // Lambda = lambda^stride
  double ax, ay;     // A e^{i phi}
  double rtf;        // 1 / (tau fs): decay per sample
  double fcyc;       // f / fs: cycles per sample
  double t0s;        // t0 fs: onset in samples (fractional)
  long long i_on;    // first live sample: the smallest i with (double)i / fs - t0 >= 0 (decided as the CPU side does)
};

// executed by ONE WARP (lanes 0..3 each compute a piece); p = the item's 5 parameters (A, f, tau, phi, t0)
__device__ __forceinline__ void ring_prepare(const double* __restrict__ p, double fs, int stride, int lane, RingConsts* out) {
  const double A = __ldg(p), f = __ldg(p + 1), tau = __ldg(p + 2), phi = __ldg(p + 3), t0 = __ldg(p + 4);
  const double rtf = 1.0 / (tau * fs), fcyc = f / fs;
  if (lane == 0) {
    double s, c;
    sincospi(2.0 * fcyc, &s, &c);
    const double m = exp(-rtf);
    out->lx = m * c; out->ly = m * s;
    out->rtf = rtf; out->fcyc = fcyc;
  } else if (lane == 1) {
    double cyc = fcyc * (double)stride, s, c;
    cyc -= rint(cyc);
    sincospi(2.0 * cyc, &s, &c);
    const double m = exp(-rtf * (double)stride);
    out->Lx = m * c; out->Ly = m * s;
  } else if (lane == 2) {
    double s, c;
    sincos(phi, &s, &c);
    out->ax = A * c; out->ay = A * s;
  } else if (lane == 3) {
    const double t0s = t0 * fs;
    long long cand = t0s > 4.0e15 ? (long long)4.0e15 : (t0s < -4.0e15 ? -(long long)4.0e15 : (long long)ceil(t0s));
    auto before = [&](long long i) { return (double)i / fs - t0 < 0.0; };
#pragma unroll 1
    for (int it = 0; it < 4 && !before(cand - 1); ++it) --cand;
#pragma unroll 1
    for (int it = 0; it < 8 && before(cand); ++it) ++cand;
    out->t0s = t0s; out->i_on = cand;
  }
}

// K pairs of samples of the item for one thread; samples at or beyond n are zero
template <int K>
__device__ __forceinline__ void ring_pairs(const RingConsts& c, int i_first, int log2_stride, int n, double2 (&h)[K]) {
  const int stride = 1 << log2_stride;
  long long ka = 0;   // first pair whose odd sample can be live
  if (c.i_on - 1 > (long long)i_first) ka = (c.i_on - 1 - i_first + stride - 1) >> log2_stride;
  if (ka >= K) {
#pragma unroll
    for (int k = 0; k < K; ++k) h[k] = make_double2(0.0, 0.0);
    return;
  }
  const int kai = (int)ka;
  const double delta = (double)(i_first + kai * stride) - c.t0s;   // >= -1 sample
  double cyc = c.fcyc * delta, s, co;
  cyc -= rint(cyc);
  sincospi(2.0 * cyc, &s, &co);
  const double m = exp(-delta * c.rtf);
  const double er = m * co, ei = m * s;
  double zr = fma(c.ax, er, -(c.ay * ei)), zi = fma(c.ax, ei, c.ay * er);
#pragma unroll
  for (int k = 0; k < K; ++k) {
    if (k > kai) {
      const double nr = fma(zr, c.Lx, -(zi * c.Ly));
      zi = fma(zr, c.Ly, zi * c.Lx);
      zr = nr;
    }
    const long long i = (long long)i_first + (long long)k * stride;
    const bool live = k >= kai;
    const double odd = fma(zr, c.lx, -(zi * c.ly));
    h[k].x = (live && i >= c.i_on && i < n) ? zr : 0.0;
    h[k].y = (live && i + 1 >= c.i_on && i + 1 < n) ? odd : 0.0;
  }
}

}  // namespace TD_NS
