// td_dit16.cuh - in-register radix-16 decimation-in-time butterfly whose external twiddles are
// merged into its four radix-2 stages, every twiddled butterfly in the 6-FMA form
//     X = a + w b   (4 FMA),      Y = a - w b = 2 a - X   (2 FMA).
// The plain form used by the forward (DIF) passes costs 4 ops for the twiddle product plus 4 for
// the add / subtract.  On B200 every DADD / DMUL / DFMA takes the same fp64 issue slot
// (profiles/r01_peaks.md), so instruction count is what bounds the FFT path.
//
//   dit16<INV, TW>(x, w1):   X_t = sum_s  x_s * w1^s * W^(s t),   W = exp(-+ 2 pi i / 16)  (INV: +)
//   input x[s] natural, result X_t in x[brev4(t)]  (the convention of fft_reg).
//
// With s split as 8 s3 + 4 s2 + 2 s1 + s0 and t = t0 + 2 t1 + 4 t2 + 8 t3 the four stages use the
// twiddles  w1^8;  w1^4 W^(4 t0);  w1^2 W^(2 (t0 + 2 t1));  w1 W^(t0 + 2 t1 + 4 t2):
// 1 + 1 + 2 + 4 distinct values up to factors of +-i, i.e. 25 ops of preparation (three squarings
// of a unit-modulus number, four products with constants) against 60 + 52 ops for sixteen
// separately applied powers.  Twiddled task: 192 + 25 = 217 fp64 instructions (was 254-280);
// twiddle-free task (TW = false): 148 (was 168).
#pragma once
#include "td_common.cuh"

namespace TD_NS {

// a <- a + w b,  b <- a - w b
__host__ __device__ __forceinline__ void bf6(cplx& a, cplx& b, real wr, real wi) {
  const real xr = fma(wr, b.x, fma(-wi, b.y, a.x));
  const real xi = fma(wr, b.y, fma(wi, b.x, a.y));
  b = mk(fma(real(2), a.x, -xr), fma(real(2), a.y, -xi));
  a = mk(xr, xi);
}
// a <- a + b,  b <- a - b
__host__ __device__ __forceinline__ void bf1(cplx& a, cplx& b) {
  const cplx t = mk(a.x - b.x, a.y - b.y);
  a = mk(a.x + b.x, a.y + b.y);
  b = t;
}
// a <- a + (sgn i) b,  b <- a - (sgn i) b      (SGN = +1 or -1)
template <int SGN> __host__ __device__ __forceinline__ void bfi(cplx& a, cplx& b) {
  const cplx ib = SGN > 0 ? mk(-b.y, b.x) : mk(b.y, -b.x);
  const cplx t = mk(a.x - ib.x, a.y - ib.y);
  a = mk(a.x + ib.x, a.y + ib.y);
  b = t;
}
// square of a unit-modulus number: (2x^2 - 1, 2xy), 3 ops
__host__ __device__ __forceinline__ cplx usq(cplx w) {
  const real x2 = w.x + w.x;
  return mk(fma(x2, w.x, real(-1)), x2 * w.y);
}

// butterfly with twiddle  w * (sgn i)^Q,  Q = 0 or 1
template <int Q, int SGN> __host__ __device__ __forceinline__ void bf6q(cplx& a, cplx& b, cplx w) {
  if constexpr (Q == 0) bf6(a, b, w.x, w.y);
  else if constexpr (SGN > 0) bf6(a, b, -w.y, w.x);   //  i w
  else bf6(a, b, w.y, -w.x);                           // -i w
}

template <bool INV, bool TW> __host__ __device__ __forceinline__ void dit16(cplx (&x)[16], cplx w1) {
  constexpr int SG = INV ? 1 : -1;                 // W^4 = SG * i
  constexpr real C8 = real(0.70710678118654752440);    // cos(pi/4)
  constexpr real C16 = real(0.92387953251128675613), S16 = real(0.38268343236508977173);  // cos, sin(pi/8)
  if constexpr (TW) {
    const cplx w2 = usq(w1), w4 = usq(w2), w8 = usq(w4);
    // stage A: pairs (s, s+8), twiddle w1^8
#pragma unroll
    for (int s = 0; s < 8; ++s) bf6(x[s], x[s + 8], w8.x, w8.y);
    // stage B: within half t0, pairs (s, s+4), twiddle w1^4 (SG i)^t0
#pragma unroll
    for (int s = 0; s < 4; ++s) { bf6q<0, SG>(x[s], x[s + 4], w4); bf6q<1, SG>(x[8 + s], x[12 + s], w4); }
    // stage C: group (t0, t1) at 8 t0 + 4 t1, pairs (s, s+2), twiddle w1^2 W8^(t0 + 2 t1)
    const cplx w2e = mk(C8 * (w2.x - SG * w2.y), C8 * (w2.y + SG * w2.x));  // w1^2 W8
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      bf6q<0, SG>(x[0 + s], x[2 + s], w2);     // t0 = 0, t1 = 0: exponent 0
      bf6q<1, SG>(x[4 + s], x[6 + s], w2);     // t0 = 0, t1 = 1: exponent 2
      bf6q<0, SG>(x[8 + s], x[10 + s], w2e);   // t0 = 1, t1 = 0: exponent 1
      bf6q<1, SG>(x[12 + s], x[14 + s], w2e);  // t0 = 1, t1 = 1: exponent 3
    }
    // stage D: group (t0, t1, t2) at 8 t0 + 4 t1 + 2 t2, pair (0, 1), twiddle w1 W16^(t0 + 2 t1 + 4 t2)
    const cplx v1 = mk(fma(C16, w1.x, -SG * S16 * w1.y), fma(C16, w1.y, SG * S16 * w1.x));  // w1 W16
    const cplx v2 = mk(C8 * (w1.x - SG * w1.y), C8 * (w1.y + SG * w1.x));                    // w1 W16^2
    const cplx v3 = mk(fma(S16, w1.x, -SG * C16 * w1.y), fma(S16, w1.y, SG * C16 * w1.x));  // w1 W16^3
    bf6q<0, SG>(x[0], x[1], w1);    // k = 0
    bf6q<1, SG>(x[2], x[3], w1);    // k = 4
    bf6q<0, SG>(x[4], x[5], v2);    // k = 2
    bf6q<1, SG>(x[6], x[7], v2);    // k = 6
    bf6q<0, SG>(x[8], x[9], v1);    // k = 1
    bf6q<1, SG>(x[10], x[11], v1);  // k = 5
    bf6q<0, SG>(x[12], x[13], v3);  // k = 3
    bf6q<1, SG>(x[14], x[15], v3);  // k = 7
  } else {
#pragma unroll
    for (int s = 0; s < 8; ++s) bf1(x[s], x[s + 8]);
#pragma unroll
    for (int s = 0; s < 4; ++s) { bf1(x[s], x[s + 4]); bfi<SG>(x[8 + s], x[12 + s]); }
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      bf1(x[0 + s], x[2 + s]);
      bfi<SG>(x[4 + s], x[6 + s]);
      bf6(x[8 + s], x[10 + s], C8, SG * C8);      // W8
      bf6(x[12 + s], x[14 + s], -SG * SG * C8, SG * C8);  // (SG i) W8 = (-C8, SG C8) for both signs
    }
    bf1(x[0], x[1]);
    bfi<SG>(x[2], x[3]);
    bf6(x[4], x[5], C8, SG * C8);          // W16^2
    bf6(x[6], x[7], -C8, SG * C8);         // W16^6
    bf6(x[8], x[9], C16, SG * S16);        // W16^1
    bf6(x[10], x[11], -S16, SG * C16);     // W16^5
    bf6(x[12], x[13], S16, SG * C16);      // W16^3
    bf6(x[14], x[15], -C16, SG * S16);     // W16^7
  }
}

}  // namespace TD_NS
