// td_fused.cuh - the fused FFT-path kernel: one CTA evaluates whole templates with every
// intermediate (residual, spectra, filtered vectors) resident in shared memory / registers.
//
// Per template b and segment s (Eqs. 14-16):
//   S1  r = d_s - h_bs                                  fused into the first pass's global loads
//   S2  R^ = FFT_2M(r zero-padded), 2M >= 2 N_s          real input: packed as u_j = r_2j + i r_2j+1 and
//                                                        transformed as two half-zero-pruned length-M/2
//                                                        complex DIF FFTs (even / odd output bins), then untangled
//   S3  Z = G .* R^,  G = conj(A^) + i conj(B^)          both generator spectra in one complex array; G is stored
//                                                        pre-permuted to the DIT input order and pre-scaled by
//                                                        1/(4M sqrt(v)) (1/2M inverse FFT, 1/2 untangle)
//   S4  z_i = IFFT_2M(Z)_i, i < N_s only                 two length-M complex DIT FFTs (even / odd input bins)
//                                                        + pruned last radix-2 stage; Re z = L(a)^T r/sqrt(v),
//                                                        Im z = L(b)^T r/sqrt(v)
//   S5  Q_s = sum_i Re(z_i)^2 - Im(z_i)^2               fused into the last inverse pass; warp-shuffle + block
//       out[b] = -1/2 sum_s Q_s                          reduction; one 8-byte store per template
#pragma once
#include "td_common.cuh"
#include "td_dit16.cuh"

namespace TD_NS {

struct SegDev {
  long long off;    // offset of this segment inside d / a row of H (elements)
  int n;            // N_s
  int _pad;         // index of the segment in the handle (the SYN kernels find the segment's parameter row with it)
  const cplx* G;    // [2][M]: even-bin then odd-bin generator spectrum, DIT input order, scaled
  cplx* zd;         // [M]: z of the data vector d (td_inner_batch only)
  double rscale;    // fp32 evaluation only: samples are multiplied by rscale = rho_s(0)^(-1/2) in fp64 before they are
                    // rounded to fp32, the generator spectrum carries the inverse factor ("appropriate normalization",
                    // PAPER.md:324); unused (1.0) in fp64
};

struct FusedParams {
  const double* d;
  const double* H;
  long long ldh;
  long long B;
  double* out0;        // loglike: out; inner: out_dh (may be null)
  double* out1;        // inner: out_hh (may be null)
  const SegDev* segs;  // device array
  int n_seg;
  int accumulate;      // add to out instead of overwriting (segments of another size class ran before)
  const cplx* T;       // T[k] = exp(-2 pi i k / (2M)), k < 2M
};

// x = (sample 2*idx, sample 2*idx+1) of the vector this MODE transforms, zero beyond n.
// (the combination is formed in fp64 in both precisions; the fp32 build scales by rs and rounds once)
__device__ __forceinline__ cplx to_cplx(double x, double y, double rs) {
  if constexpr (F32) return mk((real)(x * rs), (real)(y * rs));
  else return mk((real)x, (real)y);
}
template <int MODE>
__device__ __forceinline__ cplx load_pair(const double* __restrict__ drow, const double* __restrict__ hrow,
                                          int idx, int n, bool vec, double rs) {
  const int i0 = 2 * idx;
  double h0 = 0.0, h1 = 0.0, d0 = 0.0, d1 = 0.0;
  if (i0 + 1 < n && vec) {
    if (MODE != MODE_STOREZ) {
      const double2 hv = __ldg(reinterpret_cast<const double2*>(hrow + i0));
      h0 = hv.x; h1 = hv.y;
    }
    if (MODE != MODE_INNER) {
      const double2 dv = *reinterpret_cast<const double2*>(drow + i0);
      d0 = dv.x; d1 = dv.y;
    }
  } else {
    if (i0 < n) {
      if (MODE != MODE_STOREZ) h0 = __ldg(hrow + i0);
      if (MODE != MODE_INNER) d0 = drow[i0];
    }
    if (i0 + 1 < n) {
      if (MODE != MODE_STOREZ) h1 = __ldg(hrow + i0 + 1);
      if (MODE != MODE_INNER) d1 = drow[i0 + 1];
    }
  }
  if (MODE == MODE_LOGLIKE) return to_cplx(d0 - h0, d1 - h1, rs);
  if (MODE == MODE_INNER) return to_cplx(h0, h1, rs);
  return to_cplx(d0, d1, rs);
}

// First forward pass: reads the packed real input straight from global memory and produces
// pass 1 of BOTH pruned half-length transforms (even bins: plain; odd bins: input pre-twisted
// by w_M^j, split into a compile-time part w_{2R}^s on the inputs and w_M^j0 folded into the
// output twiddles).
template <int R, int MODE, class Arr>
__device__ __forceinline__ void first_pass_task(const Arr& UE, const Arr& UO, int nf, int g,
                                                const double* __restrict__ drow,
                                                const double* __restrict__ hrow, int n, bool vec,
                                                const cplx* __restrict__ T, double rs = 1.0) {
  const int S = nf / R;
  const int j = g;  // single block of length nf
  cplx x[R], y[R];
#pragma unroll
  for (int s = 0; s < R; ++s) x[s] = load_pair<MODE>(drow, hrow, j + s * S, n, vec, rs);
  static_for<0, R>([&](auto s) {
    constexpr int ss = decltype(s)::value;
    y[ss] = mul_w32<ss * (16 / R), false>(x[ss]);
  });
  cplx w[R];
  tw_powers<R>(T[4 * j], w);   // w_nf^j = w_2M^{4j}
  const cplx beta = T[2 * j];  // w_M^j
  fft_reg<R, false>(x);
  fft_reg<R, false>(y);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    cplx ve = x[brevR<R>(tt)], vo = y[brevR<R>(tt)];
    if (tt > 0) {
      ve = cmul(ve, w[tt]);
      vo = cmul(vo, cmul(w[tt], beta));
    } else {
      vo = cmul(vo, beta);
    }
    UE.st(j + tt * S, ve);
    UO.st(j + tt * S, vo);
  });
}

// Untangle + generator product for the bin held at position p of branch br's forward result.
// Only the canonical member of each conjugate pair does work.  Writes four spectrum bins.
template <class ArrU, class ArrZ>
__device__ __forceinline__ void untangle_task(const ArrU& U, const ArrZ& Z, const cplx* __restrict__ G,
                                              int br, int p, int nf, int M, const cplx* __restrict__ T) {
  const int kq = plan_freq(p, nf);
  int kq2, i1, i2, i3;
  if (br == 0) {
    if (kq > nf / 2) return;
    kq2 = (nf - kq) & (nf - 1);
    i1 = nf - kq; i2 = nf + kq; i3 = (M - kq) & (M - 1);
  } else {
    if (kq >= nf / 2) return;
    kq2 = nf - 1 - kq;
    i1 = nf - 1 - kq; i2 = nf + kq; i3 = M - 1 - kq;
  }
  const cplx U1 = U.ld(p), U2 = U.ld(plan_pos(kq2, nf));
  const cplx w = T[2 * kq + br];
  const cplx A = mk(U1.x + U2.x, U1.y - U2.y);        // 2 A_k  (the 1/2 lives in G's scale)
  const cplx Bv = mk(U1.y + U2.y, -(U1.x - U2.x));    // 2 B_k
  const cplx wB = cmul(w, Bv);
  const cplx Xk = cadd(A, wB), Xm = csub(A, wB);
  const int p0 = plan_pos(kq, M), p1 = plan_pos(i1, M), p2 = plan_pos(i2, M), p3 = plan_pos(i3, M);
  Z.st(p0, cmul(G[p0], Xk));
  Z.st(p1, cmul(G[p1], cconj(Xm)));
  Z.st(p2, cmul(G[p2], Xm));
  Z.st(p3, cmul(G[p3], cconj(Xk)));
}

// Last inverse pass (radix R, L = M) for both branches, pruned final radix-2 stage
// z_i = e_i + w_2M^{-i} o_i, restriction to i < n and the fused quadratic sums.
template <int R, int MODE, class Arr>
__device__ __forceinline__ void last_pass_task(const Arr& ZE, const Arr& ZO, int M, int g, int n,
                                               const cplx* __restrict__ T, cplx* __restrict__ zd,
                                               double& acc0, double& acc1) {
  const int S = M / R;
  const int j = g;
  cplx e[R], o[R], gm[R];     // z_t = e_t + gm_t o_t: the pruned last radix-2 stage
  const cplx beta = T[j];     // w_2M^j
  if constexpr (R == 16) {
    // merged-twiddle 6-FMA butterflies (td_dit16.cuh), as in last_pass_c
    const cplx w1 = cconj(T[2 * j]);  // w_M^(-j)
#pragma unroll
    for (int ss = 0; ss < R; ++ss) { e[ss] = ZE.ld(j + ss * S); o[ss] = ZO.ld(j + ss * S); }
    dit16<true, true>(e, w1);
    dit16<true, true>(o, w1);
    const cplx cb = cconj(beta);
    static_for<0, R>([&](auto t) { gm[decltype(t)::value] = mul_w32<decltype(t)::value, true>(cb); });
  } else {
    cplx w[R];
    tw_powers<R>(T[2 * j], w);  // w_M^j
    static_for<0, R>([&](auto s) {
      constexpr int ss = decltype(s)::value;
      cplx ve = ZE.ld(j + ss * S), vo = ZO.ld(j + ss * S);
      if (ss > 0) {
        ve = cmulc(ve, w[ss]);
        vo = cmulc(vo, cmul(w[ss], beta));
      } else {
        vo = cmulc(vo, beta);
      }
      e[ss] = ve;
      o[ss] = vo;
    });
    fft_reg<R, true>(e);
    fft_reg<R, true>(o);
    static_for<0, R>([&](auto t) {
      constexpr int tt = decltype(t)::value;
      gm[tt] = mk(cos32(tt * (16 / R)), sin32(tt * (16 / R)));
    });
  }
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    const cplx ev = e[brevR<R>(tt)], ov = o[brevR<R>(tt)];
    const cplx z = mk(fma(gm[tt].x, ov.x, fma(-gm[tt].y, ov.y, ev.x)), fma(gm[tt].x, ov.y, fma(gm[tt].y, ov.x, ev.y)));
    const int i = j + tt * S;
    if (MODE == MODE_STOREZ) {
      zd[i] = z;
    } else if (i < n) {
      if (MODE == MODE_INNER) {
        const cplx q = zd[i];
        acc0 += (double)fma(z.x, q.x, -z.y * q.y);
      }
      acc1 += (double)fma(z.x, z.x, -z.y * z.y);
    }
  });
}

// ---------------------------------------------------------------------------------------------
// Fused kernel proper: every shape is a compile-time constant, twiddle bases come from a small
// shared-memory table (tw[k] = w_2M^k, k < TWS) and conjugate pairs are enumerated directly.
// ---------------------------------------------------------------------------------------------
template <int LOG2M> struct FusedShape {
  static constexpr int M = 1 << LOG2M, NF = M / 2;
  static constexpr int RF1 = plan_r1(NF), NPF = plan_np(NF);
  static constexpr int RI1 = plan_r1(M), NPI = plan_np(M);
  static constexpr int RMIN = RF1 < RI1 ? RF1 : RI1;
  static constexpr int TWS = 2 * M / RMIN;  // largest base-twiddle index used + 1 (<= this)
  static constexpr size_t smem_bytes(int nt) {
    return sizeof(cplx) * (2 * (size_t)SmemArr::padded(NF) + 2 * (size_t)SmemArr::padded(M) + TWS + 16) +
           sizeof(double) * 2 * (nt / 32) + 16;  // + mbarrier
  }
};

template <int NT, bool FWD, int N, int L>
__device__ __forceinline__ void smem_pass16c(const SmemArr& AE, const SmemArr& AO, const cplx* __restrict__ tw,
                                             int TW, int tid) {
  constexpr int R = 16, TB = N / R, S = L / R;
  if constexpr (TB >= NT) {
#pragma unroll 1
    for (int g = tid; g < TB; g += NT) {
      cplx w[R];
      if constexpr (S > 1) tw_powers<R>(tw[(g & (S - 1)) * (TW / L)], w);
      if constexpr (FWD) { dif_task_c<R, L>(AE, g, w); dif_task_c<R, L>(AO, g, w); }
      else               { dit_task_c<R, L>(AE, g, w); dit_task_c<R, L>(AO, g, w); }
    }
  } else {
#pragma unroll 1
    for (int id = tid; id < 2 * TB; id += NT) {
      const int br = id / TB, g = id - br * TB;
      cplx w[R];
      if constexpr (S > 1) tw_powers<R>(tw[(g & (S - 1)) * (TW / L)], w);
      if constexpr (FWD) dif_task_c<R, L>(br ? AO : AE, g, w);
      else               dit_task_c<R, L>(br ? AO : AE, g, w);
    }
  }
}

// first forward pass with compile-time shapes and shared-memory twiddles
template <int R, int NF, int MODE>
__device__ __forceinline__ void first_pass_c(const SmemArr& UE, const SmemArr& UO, int j,
                                             const double* __restrict__ drow, const double* __restrict__ hrow,
                                             int n, bool vec, const cplx* __restrict__ tw, double rs = 1.0) {
  constexpr int S = NF / R;
  cplx x[R], y[R];
#pragma unroll
  for (int s = 0; s < R; ++s) x[s] = load_pair<MODE>(drow, hrow, j + s * S, n, vec, rs);
  static_for<0, R>([&](auto s) {
    constexpr int ss = decltype(s)::value;
    y[ss] = mul_w32<ss * (16 / R), false>(x[ss]);
  });
  cplx w[R];
  const cplx beta = tw[2 * j];  // w_M^j
  tw_powers<R>(tw[4 * j], w);   // w_NF^j
  fft_reg<R, false>(x);
  fft_reg<R, false>(y);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    cplx ve = x[brevR<R>(tt)], vo = y[brevR<R>(tt)];
    if constexpr (tt > 0) {
      ve = cmul(ve, w[tt]);
      vo = cmul(vo, cmul(w[tt], beta));
    } else {
      vo = cmul(vo, beta);
    }
    UE.st(j + tt * S, ve);
    UO.st(j + tt * S, vo);
  });
}

// untangle + generator product for the conjugate pair (k', partner) of branch BR.
// k' = kap + (NF/16) t: the bins of one last-pass block, so lanes t = 0..15 read 16 consecutive
// positions.  w_2M^(2k'+BR) = tw[2 kap + BR] * w_32^t.
template <int BR, int NF>
__device__ __forceinline__ void untangle_pair(const SmemArr& U, const SmemArr& Z, const cplx* __restrict__ G,
                                              int kap, int t, const cplx* __restrict__ tw,
                                              const cplx* __restrict__ c32) {
  constexpr int M = 2 * NF;
  const int kq = kap + (NF / 16) * t;
  int kq2, i1, i3;
  const int i2 = NF + kq;
  if constexpr (BR == 0) {
    kq2 = (NF - kq) & (NF - 1);
    i1 = NF - kq;
    i3 = (M - kq) & (M - 1);
  } else {
    kq2 = NF - 1 - kq;
    i1 = NF - 1 - kq;
    i3 = M - 1 - kq;
  }
  const int p0 = PlanT<M>::pos(kq), p1 = PlanT<M>::pos(i1), p2 = PlanT<M>::pos(i2), p3 = PlanT<M>::pos(i3);
  const cplx g0 = __ldg(G + p0), g1 = __ldg(G + p1), g2 = __ldg(G + p2), g3 = __ldg(G + p3);
  const cplx U1 = U.ld(PlanT<NF>::pos(kq)), U2 = U.ld(PlanT<NF>::pos(kq2));
  const cplx w = cmul(tw[2 * kap + BR], c32[t]);
  const cplx A = mk(U1.x + U2.x, U1.y - U2.y);        // 2 A_k  (the 1/2 lives in G's scale)
  const cplx Bv = mk(U1.y + U2.y, -(U1.x - U2.x));    // 2 B_k
  const cplx wB = cmul(w, Bv);
  const cplx Xk = cadd(A, wB), Xm = csub(A, wB);
  Z.st(p0, cmul(g0, Xk));
  Z.st(p1, cmul(g1, cconj(Xm)));
  Z.st(p2, cmul(g2, Xm));
  Z.st(p3, cmul(g3, cconj(Xk)));
}

template <int R, int M, int MODE>
__device__ __forceinline__ void last_pass_c(const SmemArr& ZE, const SmemArr& ZO, int j, int n,
                                            const cplx* __restrict__ tw, cplx* __restrict__ zd, double& acc0,
                                            double& acc1) {
  constexpr int S = M / R;
  cplx e[R], o[R], gm[R];      // z_t = e_t + gm_t o_t: the pruned last radix-2 stage
  const cplx beta = tw[j];     // w_2M^j
  if constexpr (R == 16) {
    // merged-twiddle 6-FMA butterflies (td_dit16.cuh); the odd branch's factor conj(beta) w_32^(-t)
    // stays outside and enters the last stage as one FMA-form product
    const cplx w1 = cconj(tw[2 * j]);  // w_M^(-j)
#pragma unroll
    for (int ss = 0; ss < R; ++ss) { e[ss] = ZE.ld(j + ss * S); o[ss] = ZO.ld(j + ss * S); }
    dit16<true, true>(e, w1);
    dit16<true, true>(o, w1);
    const cplx cb = cconj(beta);
    static_for<0, R>([&](auto t) { gm[decltype(t)::value] = mul_w32<decltype(t)::value, true>(cb); });
  } else {
    cplx w[R];
    tw_powers<R>(tw[2 * j], w);  // w_M^j
    static_for<0, R>([&](auto s) {
      constexpr int ss = decltype(s)::value;
      cplx ve = ZE.ld(j + ss * S), vo = ZO.ld(j + ss * S);
      if constexpr (ss > 0) {
        ve = cmulc(ve, w[ss]);
        vo = cmulc(vo, cmul(w[ss], beta));
      } else {
        vo = cmulc(vo, beta);
      }
      e[ss] = ve;
      o[ss] = vo;
    });
    fft_reg<R, true>(e);
    fft_reg<R, true>(o);
    static_for<0, R>([&](auto t) {
      constexpr int tt = decltype(t)::value;
      gm[tt] = mk(cos32(tt * (16 / R)), sin32(tt * (16 / R)));  // conj(w_32)^(tt 16/R), compile-time constants
    });
  }
  // four independent partial sums per output (a single chain of 2 R dependent FMAs would be latency-bound)
  real p0[4] = {real(0), real(0), real(0), real(0)}, p1[4] = {real(0), real(0), real(0), real(0)};
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    const cplx ev = e[brevR<R>(tt)], ov = o[brevR<R>(tt)];
    const cplx z = mk(fma(gm[tt].x, ov.x, fma(-gm[tt].y, ov.y, ev.x)), fma(gm[tt].x, ov.y, fma(gm[tt].y, ov.x, ev.y)));
    const int i = j + tt * S;
    if constexpr (MODE == MODE_STOREZ) {
      zd[i] = z;
    } else {
      if (i < n) {
        if constexpr (MODE == MODE_INNER) {
          const cplx q = zd[i];
          p0[tt & 1] = fma(z.x, q.x, p0[tt & 1]);
          p0[2 + (tt & 1)] = fma(-z.y, q.y, p0[2 + (tt & 1)]);
        }
        p1[tt & 1] = fma(z.x, z.x, p1[tt & 1]);
        p1[2 + (tt & 1)] = fma(-z.y, z.y, p1[2 + (tt & 1)]);
      }
    }
  });
  if constexpr (MODE == MODE_INNER) acc0 += (double)((p0[0] + p0[1]) + (p0[2] + p0[3]));
  if constexpr (MODE != MODE_STOREZ) acc1 += (double)((p1[0] + p1[1]) + (p1[2] + p1[3]));
}

// both branches of one radix-16 butterfly task interleaved (twice the independent work per thread)
template <bool FWD, int L>
__device__ __forceinline__ void pass16_pair(const SmemArr& AE, const SmemArr& AO, int g, const cplx (&w)[16]) {
  constexpr int R = 16, S = L / R, LS = ilog2(S);
  const int blk = g >> LS, j = g & (S - 1);
  const int base = blk * L + j;
  cplx x[R], y[R];
  static_for<0, R>([&](auto s) {
    constexpr int ss = decltype(s)::value;
    cplx a = AE.ld(base + ss * S), b = AO.ld(base + ss * S);
    if constexpr (!FWD && ss > 0 && (S > 1)) { a = cmulc(a, w[ss]); b = cmulc(b, w[ss]); }
    x[ss] = a; y[ss] = b;
  });
  // software pipeline: E computes while O's loads land; E's stores drain while O computes
  fft_reg<R, !FWD>(x);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    cplx a = x[brevR<R>(tt)];
    if constexpr (FWD && tt > 0 && (S > 1)) a = cmul(a, w[tt]);
    AE.st(base + tt * S, a);
  });
  fft_reg<R, !FWD>(y);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    cplx b = y[brevR<R>(tt)];
    if constexpr (FWD && tt > 0 && (S > 1)) b = cmul(b, w[tt]);
    AO.st(base + tt * S, b);
  });
}

template <int NT, bool FWD, int N, int L, bool ILV>
__device__ __forceinline__ void smem_pass16v(const SmemArr& AE, const SmemArr& AO, const cplx* __restrict__ tw,
                                             int TW, int tid) {
  constexpr int TB = N / 16, S = L / 16;
  if constexpr (ILV && TB >= NT) {
#pragma unroll 1
    for (int g = tid; g < TB; g += NT) {
      cplx w[16];
      if constexpr (S > 1) tw_powers<16>(tw[(g & (S - 1)) * (TW / L)], w);
      pass16_pair<FWD, L>(AE, AO, g, w);
    }
  } else {
    smem_pass16c<NT, FWD, N, L>(AE, AO, tw, TW, tid);
  }
}

// first pass fed from the staged (TMA-prefetched) rows in shared memory: values only
template <int R, int NF, int MODE>
__device__ __forceinline__ void first_pass_load_staged(cplx (&x)[R], int j, const double* stH, const double* stD,
                                                       int n, double rs = 1.0) {
  constexpr int S = NF / R;
#pragma unroll
  for (int s = 0; s < R; ++s) {
    const int i0 = 2 * (j + s * S);
    double2 h = make_double2(0.0, 0.0), d = make_double2(0.0, 0.0);
    if (i0 < n) {  // n even on this path: i0 + 1 < n too
      if (MODE != MODE_STOREZ) h = *reinterpret_cast<const double2*>(stH + i0);
      if (MODE != MODE_INNER) d = *reinterpret_cast<const double2*>(stD + i0);
    }
    x[s] = (MODE == MODE_LOGLIKE) ? to_cplx(d.x - h.x, d.y - h.y, rs) : (MODE == MODE_INNER ? to_cplx(h.x, h.y, rs) : to_cplx(d.x, d.y, rs));
  }
}
template <int R, int NF>
__device__ __forceinline__ void first_pass_compute(const SmemArr& UE, const SmemArr& UO, int j, cplx (&x)[R],
                                                   const cplx* __restrict__ tw) {
  constexpr int S = NF / R;
  cplx y[R];
  static_for<0, R>([&](auto s) {
    constexpr int ss = decltype(s)::value;
    y[ss] = mul_w32<ss * (16 / R), false>(x[ss]);
  });
  cplx w[R];
  const cplx beta = tw[2 * j];
  tw_powers<R>(tw[4 * j], w);
  fft_reg<R, false>(x);
  fft_reg<R, false>(y);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    cplx ve = x[brevR<R>(tt)], vo = y[brevR<R>(tt)];
    if constexpr (tt > 0) {
      ve = cmul(ve, w[tt]);
      vo = cmul(vo, cmul(w[tt], beta));
    } else {
      vo = cmul(vo, beta);
    }
    UE.st(j + tt * S, ve);
    UO.st(j + tt * S, vo);
  });
}

// untangle task id -> (branch, kap, t); E-branch ids [0, NF/2), O-branch ids [NF/2, NF).
// E: row kap = 0 is remapped: t = 0 -> the self-paired bin k' = 0 (its twin k' = NF/2 is done
// by one extra task), t = 1..7 -> kap 0, t = 8..15 -> the self-paired block kap = NF/32, t - 8.
template <int NF> struct UntangleIdx {
  int br, kap, t;
  __device__ __forceinline__ explicit UntangleIdx(int id) {
    br = id >= NF / 2;
    const int q = br ? id - NF / 2 : id;
    kap = q >> 4; t = q & 15;
    if (!br && kap == 0 && t >= 8) { kap = NF / 32; t -= 8; }
  }
};
template <int NF> struct UntanglePos {
  int pu1, pu2, p0, p1, p2, p3, twi, t;
  __device__ __forceinline__ UntanglePos(int br, int kap, int tt) {
    constexpr int M = 2 * NF;
    const int kq = kap + (NF / 16) * tt;
    int kq2, i1, i3;
    if (br == 0) { kq2 = (NF - kq) & (NF - 1); i1 = NF - kq; i3 = (M - kq) & (M - 1); }
    else         { kq2 = NF - 1 - kq; i1 = NF - 1 - kq; i3 = M - 1 - kq; }
    pu1 = PlanT<NF>::pos(kq); pu2 = PlanT<NF>::pos(kq2);
    p0 = PlanT<M>::pos(kq); p1 = PlanT<M>::pos(i1); p2 = PlanT<M>::pos(NF + kq); p3 = PlanT<M>::pos(i3);
    twi = 2 * kap + br; t = tt;
  }
};
template <int NF>
__device__ __forceinline__ void untangle_apply(const SmemArr& U, const SmemArr& Z, const UntanglePos<NF>& q,
                                               const cplx (&g)[4], const cplx* __restrict__ tw,
                                               const cplx* __restrict__ c32) {
  const cplx U1 = U.ld(q.pu1), U2 = U.ld(q.pu2);
  const cplx w = cmul(tw[q.twi], c32[q.t]);
  const cplx A = mk(U1.x + U2.x, U1.y - U2.y);        // 2 A_k  (the 1/2 lives in G's scale)
  const cplx Bv = mk(U1.y + U2.y, -(U1.x - U2.x));    // 2 B_k
  const cplx wB = cmul(w, Bv);
  const cplx Xk = cadd(A, wB), Xm = csub(A, wB);
  Z.st(q.p0, cmul(g[0], Xk));
  Z.st(q.p1, cmul(g[1], cconj(Xm)));
  Z.st(q.p2, cmul(g[2], Xm));
  Z.st(q.p3, cmul(g[3], cconj(Xk)));
}

template <int LOG2M, int NT, int MODE, bool ILV = true>
__global__ void __launch_bounds__(NT, 1) td_fused_kernel(const FusedParams P) {
  static_assert(!F32 || LOG2M < 0, "fp64 only: the two staged rows of doubles do not fit the fp32 U region");
  using Sh = FusedShape<LOG2M>;
  constexpr int M = Sh::M, NF = Sh::NF, TW = 2 * M;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sm = reinterpret_cast<cplx*>(smem_raw);
  const SmemArr UE{sm}, UO{sm + SmemArr::padded(NF)};
  const SmemArr ZE{sm + 2 * SmemArr::padded(NF)}, ZO{sm + 2 * SmemArr::padded(NF) + SmemArr::padded(M)};
  cplx* tw = sm + 2 * SmemArr::padded(NF) + 2 * SmemArr::padded(M);
  cplx* c32 = tw + Sh::TWS;
  double* red = reinterpret_cast<double*>(c32 + 16);
  const uint32_t mbar = smem_u32(red + 2 * (NT / 32));
  // staging for the prefetched rows lives in the U region (dead between untangle and the next first pass)
  double* stH = reinterpret_cast<double*>(sm);
  double* stD = stH + M;
  const int tid = threadIdx.x;

  for (int k = tid; k < Sh::TWS; k += NT) tw[k] = P.T[k];
  if (tid < 16) c32[tid] = P.T[tid * (TW / 32)];
  if (tid == 0) mbar_init(mbar, 1);
  __syncthreads();

  // rows of item (b, s); staged (TMA) only when 16-byte aligned and N_s even
  auto rows = [&](long long b, int s, const double*& drow, const double*& hrow, int& n) -> bool {
    const SegDev sg = P.segs[s];
    drow = P.d + sg.off;
    hrow = (MODE == MODE_STOREZ) ? drow : P.H + b * P.ldh + sg.off;
    n = sg.n;
    return (((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0) && ((n & 1) == 0);
  };
  auto prefetch = [&](long long b, int s) -> bool {
    const double *drow, *hrow; int n;
    const bool ok = rows(b, s, drow, hrow, n);
    if (ok && tid == 0) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      const uint32_t bytes = (uint32_t)n * 8u;
      const int ncopies = (MODE == MODE_LOGLIKE) ? 2 : 1;
      mbar_expect_tx(mbar, bytes * ncopies);
      if (MODE != MODE_STOREZ) bulk_g2s(smem_u32(stH), hrow, bytes, mbar);
      if (MODE != MODE_INNER) bulk_g2s(smem_u32(stD), drow, bytes, mbar);
    }
    return ok;
  };

  long long b = blockIdx.x;
  int s = 0;
  bool have = b < P.B;
  uint32_t parity = 0;
  bool staged = have ? prefetch(b, s) : false;
  double tot0 = 0.0, tot1 = 0.0;
  while (have) {
    long long nb = b; int ns = s + 1;
    if (ns == P.n_seg) { ns = 0; nb = b + gridDim.x; }
    const bool have_next = (MODE != MODE_STOREZ || nb == b) && nb < P.B;
    const SegDev sg = P.segs[s];
    // ---- S1+S2: forward, pass 1
    if (staged) {
      mbar_wait(mbar, parity);
      parity ^= 1;
      constexpr int NTASK = NF / Sh::RF1;
      static_assert(NTASK <= NT || NTASK % NT == 0, "first pass tiling");
      constexpr int IT = (NTASK + NT - 1) / NT;
      cplx xs[IT][Sh::RF1];
#pragma unroll
      for (int it = 0; it < IT; ++it)
        if (tid + it * NT < NTASK) first_pass_load_staged<Sh::RF1, NF, MODE>(xs[it], tid + it * NT, stH, stD, sg.n, sg.rscale);
      __syncthreads();  // staging consumed: the U region may now be overwritten
#pragma unroll
      for (int it = 0; it < IT; ++it)
        if (tid + it * NT < NTASK) first_pass_compute<Sh::RF1, NF>(UE, UO, tid + it * NT, xs[it], tw);
    } else {
      const double *drow, *hrow; int n;
      rows(b, s, drow, hrow, n);
      const bool vec = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
#pragma unroll 1
      for (int g = tid; g < NF / Sh::RF1; g += NT)
        first_pass_c<Sh::RF1, NF, MODE>(UE, UO, g, drow, hrow, n, vec, tw, sg.rscale);
    }
    __syncthreads();
    // ---- forward passes 2..NPF (radix 16)
    static_for<1, Sh::NPF>([&](auto q) {
      constexpr int L = (NF / Sh::RF1) >> (4 * (decltype(q)::value - 1));
      smem_pass16v<NT, true, NF, L, ILV>(UE, UO, tw, TW, tid);
      __syncthreads();
    });
    // ---- untangle + S3 generator product (G loads hoisted ahead of the shared-memory work)
    {
      constexpr int IT = (NF + NT - 1) / NT;
      cplx g[IT][4];
#pragma unroll
      for (int it = 0; it < IT; ++it) {
        const int id = tid + it * NT;
        if (id < NF) {
          const UntangleIdx<NF> ix(id);
          const UntanglePos<NF> q(ix.br, ix.kap, ix.t);
          const cplx* G = sg.G + ix.br * M;
          g[it][0] = __ldg(G + q.p0); g[it][1] = __ldg(G + q.p1); g[it][2] = __ldg(G + q.p2); g[it][3] = __ldg(G + q.p3);
        }
      }
#pragma unroll
      for (int it = 0; it < IT; ++it) {
        const int id = tid + it * NT;
        if (id < NF) {
          const UntangleIdx<NF> ix(id);
          const UntanglePos<NF> q(ix.br, ix.kap, ix.t);
          untangle_apply<NF>(ix.br ? UO : UE, ix.br ? ZO : ZE, q, g[it], tw, c32);
        }
      }
      if (tid == NT - 1) {  // twin self-paired bin k' = NF/2 of the even branch (kap = 0, t = 8)
        const UntanglePos<NF> q(0, 0, 8);
        cplx gg[4] = {__ldg(sg.G + q.p0), __ldg(sg.G + q.p1), __ldg(sg.G + q.p2), __ldg(sg.G + q.p3)};
        untangle_apply<NF>(UE, ZE, q, gg, tw, c32);
      }
    }
    __syncthreads();
    // ---- the U region is dead: prefetch the next item's rows into it while the inverse runs
    const bool staged_next = have_next ? prefetch(nb, ns) : false;
    // ---- S4: inverse passes (radix 16), smallest sub-transform first
    static_for<1, Sh::NPI>([&](auto q) {
      constexpr int L = 16 << (4 * (decltype(q)::value - 1));
      smem_pass16v<NT, false, M, L, ILV>(ZE, ZO, tw, TW, tid);
      __syncthreads();
    });
    // ---- last inverse pass + pruned radix-2 stage + S5
    double acc0 = 0.0, acc1 = 0.0;
#pragma unroll 1
    for (int g = tid; g < M / Sh::RI1; g += NT)
      last_pass_c<Sh::RI1, M, MODE>(ZE, ZO, g, sg.n, tw, sg.zd, acc0, acc1);
    if (MODE != MODE_STOREZ) {
      acc0 = warp_sum(acc0);
      acc1 = warp_sum(acc1);
      if ((tid & 31) == 0) { red[2 * (tid >> 5)] = acc0; red[2 * (tid >> 5) + 1] = acc1; }
    }
    __syncthreads();
    if (MODE != MODE_STOREZ && tid == 0) {
#pragma unroll
      for (int wq = 0; wq < NT / 32; ++wq) { tot0 += red[2 * wq]; tot1 += red[2 * wq + 1]; }
      if (s == P.n_seg - 1) {
        if (MODE == MODE_LOGLIKE) {
          const double v = -0.5 * tot1;
          P.out0[b] = P.accumulate ? P.out0[b] + v : v;
        } else {
          if (P.out0) P.out0[b] = P.accumulate ? P.out0[b] + tot0 : tot0;
          if (P.out1) P.out1[b] = P.accumulate ? P.out1[b] + tot1 : tot1;
        }
        tot0 = 0.0; tot1 = 0.0;
      }
    }
    b = nb; s = ns; have = have_next; staged = staged_next;
  }
}

}  // namespace TD_NS
