// td_synth.cuh - template synthesis on the device: the step immediately before the hot
// path, waveform generation and placement in the data vector, for the analytic
// families of BASELINE.json's configs (rows of 5 parameters, t_i = i / fs from the segment's first sample):
//   0 ringdown (c1, c2, c5, d*)  (A, f, tau, phi, t0):      A exp(-(t_i - t0)/tau) cos(2 pi f (t_i - t0) + phi), t_i >= t0
//   1 sine-Gaussian (c3)         (A, f, w, phi, t0):        A exp(-((t_i - t0)/w)^2) cos(2 pi f t_i + phi)
//   2 chirp (c4)                 (A, f0, fdot, phi, alpha): A tukey_alpha(i/(n-1)) cos(2 pi (f0 t_i + fdot t_i^2 / 2) + phi)
// A caller (a sampler) then ships 5 doubles per template instead of N: the rows are written to a scratch panel that
// is consumed by the likelihood kernels chunk by chunk (about 128 MB each: through L2, spilling to HBM), so H never
// crosses PCIe.
#pragma once
#include "td_common.cuh"

namespace td {

constexpr int SYN_NT = 256;

struct SynSeg { long long off; int n; int _pad; };  // a segment inside a row of H

enum { SYN_RINGDOWN = 0, SYN_SINEGAUSS = 1, SYN_CHIRP = 2, SYN_NFAM = 3 };

// params: [B][n_seg][5], one row per (template, segment / detector), time counted from the segment's first sample (a
// projected and time-shifted damped sinusoid F+ h_c + Fx h_s is again one: amplitude A hypot(F+, Fx), phase
// phi - atan2(Fx, F+), onset t0 + dt - PAPER.md:164, :209).  Block (r, s) writes segment s of row b0 + r of the batch to
// Hs[r * ldh + off_s + i], i < n_s.  Thread tid owns the samples tid, tid + 256, ... (coalesced stores): the
// oscillation is anchored by one sincos at its first live sample and advanced by complex recurrences that step 256
// samples at a time (ringdown, sine-Gaussian: z <- z P; chirp: z <- z r, r <- r q, the phase being quadratic);
// the Gaussian envelope and the Tukey taper are evaluated directly.  A thread takes n / 256 steps, so the
// recurrences' rounding stays far below the 1e-9 parity tolerance (measured: 4e-16 ... 1e-12 on logL).
template <int FAM>
__global__ void __launch_bounds__(SYN_NT) synth_kernel(const double* __restrict__ params, long long b0, int cb,
                                                       const SynSeg* __restrict__ segs, int n_seg, double fs,
                                                       double* __restrict__ Hs, long long ldh) {
  const int r = blockIdx.x, sgi = blockIdx.y;
  if (r >= cb) return;
  const SynSeg sg = segs[sgi];
  const int n = sg.n;
  const double* p = params + ((b0 + r) * n_seg + sgi) * 5;
  const double A = p[0], p1 = p[1], p2 = p[2], phi = p[3], p4 = p[4];
  double* row = Hs + (long long)r * ldh + sg.off;
  const int tid = threadIdx.x;
  if (tid >= n) return;
  const double dt = 1.0 / fs, D = SYN_NT * dt;
  int i = tid;
  if constexpr (FAM == SYN_RINGDOWN) {
    const double f = p1, tau = p2, t0 = p4;
    for (; i < n && (double)i / fs - t0 < 0.0; i += SYN_NT) row[i] = 0.0;  // before t0 (decided exactly as the CPU side does)
    if (i >= n) return;
    const double d0 = (double)i / fs - t0;
    double s, c;
    sincos(2.0 * M_PI * f * d0 + phi, &s, &c);
    const double e0 = A * exp(-d0 / tau);
    double zr = e0 * c, zi = e0 * s;
    double rs, rc;
    sincos(2.0 * M_PI * f * D, &rs, &rc);
    const double re = exp(-D / tau);
    const double pr = re * rc, pi = re * rs;
    for (; i < n; i += SYN_NT) {
      row[i] = zr;
      const double nr = fma(zr, pr, -(zi * pi));
      zi = fma(zr, pi, zi * pr);
      zr = nr;
    }
  } else if constexpr (FAM == SYN_SINEGAUSS) {
    const double f = p1, w = p2, t0 = p4;
    double s, c;
    sincos(2.0 * M_PI * f * ((double)i / fs) + phi, &s, &c);
    double zr = c, zi = s;
    double ps, pc;
    sincos(2.0 * M_PI * f * D, &ps, &pc);
    for (; i < n; i += SYN_NT) {
      const double u = ((double)i / fs - t0) / w;
      row[i] = A * exp(-(u * u)) * zr;   // exp underflows to 0 beyond |u| ~ 27, as on the CPU side
      const double nr = fma(zr, pc, -(zi * ps));
      zi = fma(zr, ps, zi * pc);
      zr = nr;
    }
  } else {
    const double f0 = p1, fdot = p2, alpha = p4;
    const double t = (double)i / fs;
    double s, c;
    sincos(2.0 * M_PI * (f0 * t + 0.5 * fdot * t * t) + phi, &s, &c);
    double zr = c, zi = s;
    // theta(t + D) - theta(t) = 2 pi (f0 D + fdot t D + fdot D^2 / 2): rotation r(t), itself advanced by q = exp(i 2 pi fdot D^2)
    double rs, rc, qs, qc;
    sincos(2.0 * M_PI * (f0 * D + fdot * t * D + 0.5 * fdot * D * D), &rs, &rc);
    sincos(2.0 * M_PI * fdot * D * D, &qs, &qc);
    const double xn = 1.0 / (double)(n > 1 ? n - 1 : 1);
    for (; i < n; i += SYN_NT) {
      const double x = (double)i * xn;
      double win = 1.0;
      if (x < 0.5 * alpha) win = 0.5 * (1.0 + cos(2.0 * M_PI / alpha * (x - 0.5 * alpha)));
      else if (x > 1.0 - 0.5 * alpha) win = 0.5 * (1.0 + cos(2.0 * M_PI / alpha * (x - 1.0 + 0.5 * alpha)));
      row[i] = A * win * zr;
      const double nr = fma(zr, rc, -(zi * rs));
      zi = fma(zr, rs, zi * rc);
      zr = nr;
      const double mr = fma(rc, qc, -(rs * qs));
      rs = fma(rc, qs, rs * qc);
      rc = mr;
    }
  }
}

}  // namespace td
