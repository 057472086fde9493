// td_synth.cuh - template synthesis on the device: the step immediately before the hot
// path, waveform generation and placement in the data vector, for the analytic
// damped-sinusoid family of BASELINE.json's configs c1 / c2 / c5 / d*:
//     h_b(t_i) = A exp(-(t_i - t0)/tau) cos(2 pi f (t_i - t0) + phi)   for t_i >= t0,  0 before,   t_i = i / fs.
// A caller (a sampler) then ships 5 doubles per template instead of N: the rows are written to a scratch panel that
// is consumed by the likelihood kernels chunk by chunk while it is still L2-resident, so H never crosses PCIe and
// (for chunks that fit L2) never reaches HBM.  Thread tid owns the samples tid, tid + 256, ...: one exp and one sincos
// at its first live sample, then the complex recurrence z <- z * P, P = exp((-1/tau + i 2 pi f) 256 dt), 4 flops per
// sample; a thread takes N / 256 steps, so the recurrence's rounding stays at the 1e-15 level.
#pragma once
#include "td_common.cuh"

namespace td {

constexpr int SYN_NT = 256;

struct SynSeg { long long off; int n; int _pad; };  // a segment inside a row of H

// params: [B][n_seg][5] = (A, f, tau, phi, t0) per (template, segment / detector), time counted from the segment's first
// sample (a projected and time-shifted damped sinusoid F+ h_c + Fx h_s is again one: amplitude A hypot(F+, Fx), phase
// phi - atan2(Fx, F+), onset t0 + dt - PAPER.md:164, :209).  Block (r, s) writes segment s of row b0 + r of the batch to
// Hs[r * ldh + off_s + i], i < n_s.
__global__ void __launch_bounds__(SYN_NT) synth_ringdown_kernel(const double* __restrict__ params, long long b0, int cb,
                                                                const SynSeg* __restrict__ segs, int n_seg, double fs,
                                                                double* __restrict__ Hs, long long ldh) {
  const int r = blockIdx.x, sgi = blockIdx.y;
  if (r >= cb) return;
  const SynSeg sg = segs[sgi];
  const int n = sg.n;
  const double* p = params + ((b0 + r) * n_seg + sgi) * 5;
  const double A = p[0], f = p[1], tau = p[2], phi = p[3], t0 = p[4];
  double* row = Hs + (long long)r * ldh + sg.off;
  // thread tid owns the samples i = tid + k SYN_NT (coalesced stores); its recurrence steps SYN_NT samples at a time
  const int tid = threadIdx.x;
  if (tid >= n) return;
  const double dt = 1.0 / fs;
  int i = tid;
  for (; i < n && (double)i / fs - t0 < 0.0; i += SYN_NT) row[i] = 0.0;  // before t0 (decided exactly as the CPU side does)
  if (i >= n) return;
  const double d0 = (double)i / fs - t0;
  double s, c;
  sincos(2.0 * M_PI * f * d0 + phi, &s, &c);
  const double e0 = A * exp(-d0 / tau);
  double zr = e0 * c, zi = e0 * s;
  double rs, rc;
  sincos(2.0 * M_PI * f * (SYN_NT * dt), &rs, &rc);
  const double re = exp(-(SYN_NT * dt) / tau);
  const double pr = re * rc, pi = re * rs;
  for (; i < n; i += SYN_NT) {
    row[i] = zr;
    const double nr = fma(zr, pr, -(zi * pi));
    zi = fma(zr, pi, zi * pr);
    zr = nr;
  }
}

}  // namespace td
