// td_staged.cuh - the same FFT path as td_fused.cuh with the per-template spectra staged in a
// global-memory workspace (kept L2-resident by chunking the batch) instead of shared memory.
// It serves segments whose transforms do not fit one SM's shared memory (2M > 8192 here) and
// the one-time generator transform of td_create.  Pass structure, twiddles, untangle and the
// fused last pass are the functions of td_fused.cuh / td_common.cuh called on global arrays.
#pragma once
#include "td_fused.cuh"

namespace TD_NS {

constexpr int LG_NT = 128;

// workspace of template slot c: U = [2][nf], Z = [2][M]
struct StagedParams {
  const double* d;
  const double* H;   // already offset to the first template of this chunk
  long long ldh;
  int CB;            // templates in this chunk
  SegDev seg;
  int M;             // power of two, nf = M/2
  cplx* U;           // [CB][2][nf]
  cplx* Z;           // [CB][2][M]
  const cplx* T;     // exp(-2 pi i k / (2M)), k < 2M
  double* partial;   // [CB][nblk][2]
  int nblk;
};

template <int R, int MODE>
__global__ void __launch_bounds__(LG_NT) lg_first_kernel(const StagedParams P) {
  const int nf = P.M / 2;
  const int g = blockIdx.x * LG_NT + threadIdx.x;
  const int c = blockIdx.y;
  if (g >= nf / R) return;
  const double* drow = P.d + P.seg.off;
  const double* hrow = (MODE == MODE_STOREZ) ? drow : P.H + (long long)c * P.ldh + P.seg.off;
  const bool vec = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
  const GmemArr UE{P.U + ((size_t)c * 2 + 0) * nf}, UO{P.U + ((size_t)c * 2 + 1) * nf};
  first_pass_task<R, MODE>(UE, UO, nf, g, drow, hrow, P.seg.n, vec, P.T, P.seg.rscale);
}

// generic pass over `narr` independent arrays of length n laid out back to back
template <int R, bool FWD>
__global__ void __launch_bounds__(LG_NT) lg_pass_kernel(cplx* base, int n, int L, const cplx* __restrict__ T,
                                                       int TW) {
  const int g = blockIdx.x * LG_NT + threadIdx.x;
  if (g >= n / R) return;
  const GmemArr A{base + (size_t)blockIdx.y * n};
  const int S = L / R;
  const bool tw = S > 1;
  cplx w[R];
  if (tw) tw_powers<R>(T[(size_t)(g % S) * (TW / L)], w);
  if (FWD) dif_task<R>(A, L, g, w, tw);
  else dit_task<R>(A, L, g, w, tw);
}

// Three radix-16 passes of one contiguous 4096-element block in shared memory: the forward (DIF)
// passes L = 4096, 256, 16 that end every plan, or the inverse (DIT) passes L = 16, 256, 4096 that
// start it.  One read and one write of the workspace instead of three of each: the staged path is
// bound by L2 traffic (profiles/r01_c4_staged.md), so this is where its time goes.
constexpr int LGB_NT = 256, LGB_N = 4096;
constexpr size_t LGB_SMEM = sizeof(cplx) * SmemArr::padded(LGB_N);

// the inverse (DIT) passes L = 16, 256, 4096 of one 4096-element block in shared memory (LGB_NT threads)
__device__ __forceinline__ void block_inverse3(const SmemArr& A, int tid, const cplx* __restrict__ T, int TW) {
  static_for<0, 3>([&](auto pp) {
    constexpr int L = 16 << (4 * decltype(pp)::value), S = L / 16;
    const int blk = tid / S, j = tid & (S - 1), b0 = blk * L + j;
    cplx x[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = A.ld(b0 + q * S);
    if constexpr (S > 1) dit16<true, true>(x, cconj(T[(size_t)j * (TW / L)]));
    else dit16<true, false>(x, mk(real(1), real(0)));
    static_for<0, 16>([&](auto t) { A.st(b0 + decltype(t)::value * S, x[brevR<16>(decltype(t)::value)]); });
    __syncthreads();
  });
}

template <bool FWD>
__global__ void __launch_bounds__(LGB_NT, 2) lg_block_kernel(cplx* base, int n, const cplx* __restrict__ T, int TW) {
  extern __shared__ __align__(16) unsigned char lgb_raw[];
  const SmemArr A{reinterpret_cast<cplx*>(lgb_raw)};
  cplx* g = base + (size_t)blockIdx.y * n + (size_t)blockIdx.x * LGB_N;
  const int tid = threadIdx.x;
#pragma unroll
  for (int q = 0; q < LGB_N / LGB_NT; ++q) A.st(tid + q * LGB_NT, g[tid + q * LGB_NT]);
  __syncthreads();
  if (FWD) {
    static_for<0, 3>([&](auto pp) {
      constexpr int L = LGB_N >> (4 * decltype(pp)::value), S = L / 16;
      cplx w[16];
      if constexpr (S > 1) tw_powers<16>(T[(size_t)(tid & (S - 1)) * (TW / L)], w);
      dif_task_c<16, L>(A, tid, w);
      __syncthreads();
    });
  } else {
    block_inverse3(A, tid, T, TW);
  }
#pragma unroll
  for (int q = 0; q < LGB_N / LGB_NT; ++q) g[tid + q * LGB_NT] = A.ld(tid + q * LGB_NT);
}

// Untangle + generator product for LG_UCPT templates of the chunk per thread: the pair's positions, its twiddle and its four
// generator values are computed / loaded once and reused (the generator spectrum is 2 x 16 M bytes that every template of the
// chunk would otherwise read again from L2: 2 of the 12.5 MB per template this path moved).
constexpr int LG_UCPT = 4;
__global__ void __launch_bounds__(LG_NT) lg_untangle_kernel(const StagedParams P) {
  const int nf = P.M / 2, M = P.M;
  const int p = blockIdx.x * LG_NT + threadIdx.x;
  const int br = blockIdx.y;
  if (p >= nf) return;
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
  const int pu2 = plan_pos(kq2, nf);
  const int p0 = plan_pos(kq, M), p1 = plan_pos(i1, M), p2 = plan_pos(i2, M), p3 = plan_pos(i3, M);
  const cplx* __restrict__ G = P.seg.G + (size_t)br * M;
  const cplx g0 = __ldg(G + p0), g1 = __ldg(G + p1), g2 = __ldg(G + p2), g3 = __ldg(G + p3);
  const cplx w = __ldg(P.T + 2 * kq + br);
  const int c0 = blockIdx.z * LG_UCPT, c1 = min(P.CB, c0 + LG_UCPT);
#pragma unroll LG_UCPT
  for (int c = c0; c < c1; ++c) {
    const cplx* __restrict__ U = P.U + ((size_t)c * 2 + br) * nf;
    cplx* __restrict__ Z = P.Z + ((size_t)c * 2 + br) * M;
    const cplx U1 = U[p], U2 = U[pu2];
    const cplx A = mk(U1.x + U2.x, U1.y - U2.y);        // 2 A_k  (the 1/2 lives in G's scale)
    const cplx Bv = mk(U1.y + U2.y, -(U1.x - U2.x));    // 2 B_k
    const cplx wB = cmul(w, Bv);
    const cplx Xk = cadd(A, wB), Xm = csub(A, wB);
    Z[p0] = cmul(g0, Xk);
    Z[p1] = cmul(g1, cconj(Xm));
    Z[p2] = cmul(g2, Xm);
    Z[p3] = cmul(g3, cconj(Xk));
  }
}

template <int R, int MODE>
__global__ void __launch_bounds__(LG_NT) lg_last_kernel(const StagedParams P) {
  __shared__ double red[2 * (LG_NT / 32)];
  const int g = blockIdx.x * LG_NT + threadIdx.x;
  const int c = blockIdx.y;
  const GmemArr ZE{P.Z + ((size_t)c * 2 + 0) * P.M}, ZO{P.Z + ((size_t)c * 2 + 1) * P.M};
  double acc0 = 0.0, acc1 = 0.0;
  if (g < P.M / R) last_pass_task<R, MODE>(ZE, ZO, P.M, g, P.seg.n, P.T, P.seg.zd, acc0, acc1);
  if (MODE == MODE_STOREZ) return;
  acc0 = warp_sum(acc0);
  acc1 = warp_sum(acc1);
  const int tid = threadIdx.x;
  if ((tid & 31) == 0) { red[2 * (tid >> 5)] = acc0; red[2 * (tid >> 5) + 1] = acc1; }
  __syncthreads();
  if (tid == 0) {
    double t0 = 0.0, t1 = 0.0;
#pragma unroll
    for (int w = 0; w < LG_NT / 32; ++w) { t0 += red[2 * w]; t1 += red[2 * w + 1]; }
    double* dst = P.partial + ((size_t)c * P.nblk + blockIdx.x) * 2;
    dst[0] = (MODE == MODE_LOGLIKE) ? t1 : t0;  // loglike: slot 0 carries the quadratic sum
    dst[1] = t1;
  }
}

// out[b] (+)= scale * sum_blk partial[c][blk][which]   (fixed summation order: deterministic)
__global__ void lg_finish_kernel(const double* __restrict__ partial, int nblk, int CB, double* out0, double* out1,
                                 double scale0, double scale1, int accumulate) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= CB) return;
  double t0 = 0.0, t1 = 0.0;
  for (int k = 0; k < nblk; ++k) {
    t0 += partial[((size_t)c * nblk + k) * 2];
    t1 += partial[((size_t)c * nblk + k) * 2 + 1];
  }
  if (out0) out0[c] = (accumulate ? out0[c] : 0.0) + scale0 * t0;
  if (out1) out1[c] = (accumulate ? out1[c] : 0.0) + scale1 * t1;
}

}  // namespace TD_NS
