// td_dense.cuh - dense Toeplitz-by-matrix path on the FP64 tensor pipe (SURVEY.md 8a rows S2'-S4').
//
// For short segments the two Gohberg-Semencul products of Eq. 14
//     Y1 = L(a)^T X / sqrt(v),   Y2 = L(b)^T X / sqrt(v),      X = [r_0 r_1 ... r_{B-1}]  (N x B)
// are cheaper as a dense upper-triangular-Toeplitz (N x N) by panel (N x B) contraction than as
// FFT convolutions: this is the batched form of the paper's GEMV evaluation,
// with the N x N operator never materialised.  sm_100a exposes the fp64 tensor pipe only as
// mma.sync.m8n8k4 (DMMA.8x8x4; tcgen05 has no f64 kind), so the kernel is built from that shape:
//
//   D[i][b] += sum_k T[i][k] X[k][b],   T[i][k] = g[k - i]  (g = a or b, zero for negative index)
//   A fragment (8 x 4, row i, col k):  lane holds g[(k0 - i0) + (lane & 3) - (lane >> 2)]
//   B fragment (4 x 8, row k, col b):  lane holds X[k0 + (lane & 3)][b0 + (lane >> 2)]
//
// A Toeplitz tile depends on k0 - i0 only.  A warp owns 4 row tiles (32 rows) x 2 column tiles
// (16 templates); stepping k by 4, the fragment of row tile m at step u is the fragment row tile 0
// had at step u - 2m, so ONE new fragment per generator per step feeds all 4 row tiles from a ring
// of 8 registers: per step 2 + 2 shared-memory loads against 16 DMMAs.  Tiles entirely below the
// diagonal are skipped at compile time.  X sits in shared memory template-major with row stride
// = 4 (mod 16) doubles, which makes the B-fragment loads bank-conflict free.
//
// S5 is fused: after the k loop of a 32-row group the accumulators are squared and summed per
// template (y1^2 - y2^2; for td_inner_batch also y . z_d), Y is never stored.  Warps of a CTA are
// arranged NWR (row groups, paired g / NG-1-g so the triangle is balanced) x NWC (template tiles).
#pragma once
#include "td_common.cuh"

namespace td {

constexpr int DENSE_NT = 256, DENSE_NW = 8;
constexpr int DENSE_OFFG = 8;       // zeros in front of the generators (negative lags of the diagonal tiles)
constexpr int DENSE_MAX_N = 1024;   // longest segment the dense path accepts

struct DenseSeg {
  long long off;     // offset of the segment inside d / a row of H
  int n;             // N_s
  int npad;          // N_s rounded up to a multiple of 32
  const double* a;   // device [n] prediction-error filter (a_0 = 1)
  double rsv;        // 1 / sqrt(v)
  const cplx* zd;    // z of the data vector (td_inner_batch only): (L(a)^T d, L(b)^T d) / sqrt(v)
};

struct DenseParams {
  const double* d;
  const double* H;
  long long ldh;
  long long B;
  double* out0;          // loglike: out; inner: <d,h> (may be null)
  double* out1;          // inner: <h,h> (may be null)
  const DenseSeg* segs;  // device array
  int n_seg;
  int accumulate;
  int max_npad;          // over the segments of this launch
  int nwr;               // row-group warps (1, 2, 4 or 8); NWC = 8 / nwr; templates per CTA = 16 NWC
};

struct DenseState {
  int max_n = 0;             // longest segment the dense path accepts (0: unavailable)
  int auto_n = 0;            // AUTO takes the dense path for size classes whose segments are all <= auto_n
  DenseSeg* d_all = nullptr;   // every segment (forced dense path), null if some segment is too long
  DenseSeg* d_auto = nullptr;  // the segments AUTO sends to the dense path
  int n_all = 0, n_auto = 0, npad_all = 0, npad_auto = 0;
};
inline void dense_free(DenseState& s) { cudaFree(s.d_all); cudaFree(s.d_auto); s.d_all = s.d_auto = nullptr; }

__host__ __device__ inline int dense_nwr(int max_npad) {
  int p = max_npad / 64;
  return p < 1 ? 1 : (p > 8 ? 8 : (p >= 8 ? 8 : (p >= 4 ? 4 : (p >= 2 ? 2 : 1))));
}
__host__ __device__ inline int dense_ldx(int max_npad) { return max_npad + 4; }
inline size_t dense_smem_bytes(int max_npad) {
  const int nwr = dense_nwr(max_npad), bt = 16 * (DENSE_NW / nwr);
  return sizeof(double) * (2 * (size_t)(max_npad + 16) + (size_t)bt * dense_ldx(max_npad) + 2 * (size_t)nwr * bt);
}

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}

// 8 k-steps (32 samples) of one 32-row group.  FIRST: the chunk that starts on the diagonal
// (row tile m only becomes non-zero at step 2m).
template <bool FIRST>
__device__ __forceinline__ void dense_chunk(const double* __restrict__ gaT, const double* __restrict__ gbT,
                                            const double* __restrict__ xk, int ldx8, double (&ra)[8], double (&rb)[8],
                                            double (&acc1)[4][2][2], double (&acc2)[4][2][2]) {
  static_for<0, 8>([&](auto ss) {
    constexpr int s = decltype(ss)::value;
    ra[s] = gaT[4 * s];
    rb[s] = gbT[4 * s];
    const double x0 = xk[4 * s], x1 = xk[4 * s + ldx8];
    static_for<0, 4>([&](auto mm) {
      constexpr int m = decltype(mm)::value;
      if constexpr (!FIRST || s - 2 * m >= 0) {
        constexpr int idx = (s - 2 * m) & 7;
        dmma884(acc1[m][0], ra[idx], x0);
        dmma884(acc1[m][1], ra[idx], x1);
        dmma884(acc2[m][0], rb[idx], x0);
        dmma884(acc2[m][1], rb[idx], x1);
      }
    });
  });
}

template <int MODE>
__global__ void __launch_bounds__(DENSE_NT, 2) td_dense_kernel(const DenseParams P) {
  extern __shared__ __align__(16) double smd[];
  const int glen = P.max_npad + 16, ldx = dense_ldx(P.max_npad);
  const int nwr = P.nwr, nwc = DENSE_NW / nwr, bt = 16 * nwc;
  double* ga = smd;
  double* gb = ga + glen;
  double* Xs = gb + glen;
  double* red = Xs + (size_t)bt * ldx;  // [2][nwr][bt]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r = lane >> 2, c = lane & 3;
  const int wr = warp % nwr, wc = warp / nwr;
  const long long bt0 = (long long)blockIdx.x * bt;

  double q0[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, q1[2][2] = {{0.0, 0.0}, {0.0, 0.0}};  // [column tile][e]
  for (int s = 0; s < P.n_seg; ++s) {
    const DenseSeg sg = P.segs[s];
    const int n = sg.n, npad = sg.npad;
    if (s > 0) __syncthreads();  // the previous segment's tiles are consumed
    // ---- generators (scaled by 1/sqrt(v)), zero-padded on both sides: b_j = a_{n-j}, b_0 = 0
    for (int j = tid; j < npad + 16; j += DENSE_NT) {
      const int jj = j - DENSE_OFFG;
      ga[j] = (jj >= 0 && jj < n) ? __ldg(sg.a + jj) * sg.rsv : 0.0;
      gb[j] = (jj >= 1 && jj < n) ? __ldg(sg.a + n - jj) * sg.rsv : 0.0;
    }
    // ---- S1: residual panel, template-major; rows beyond B and samples beyond n are zero
    {
      const double* __restrict__ drow = P.d + sg.off;
      for (int bl = warp; bl < bt; bl += DENSE_NW) {
        const long long b = bt0 + bl;
        const double* __restrict__ hrow = P.H + b * P.ldh + sg.off;
        double* xr = Xs + (size_t)bl * ldx;
        for (int k = lane; k < npad; k += 32) {
          double v = 0.0;
          if (b < P.B && k < n) {
            const double hv = __ldg(hrow + k);
            v = (MODE == MODE_LOGLIKE) ? drow[k] - hv : hv;
          }
          xr[k] = v;
        }
      }
    }
    __syncthreads();
    // ---- S2'-S4' + S5: this warp's 16 templates against its row groups
    const int NG = npad >> 5;
    const double* xb = Xs + (size_t)(wc * 16 + r) * ldx + c;
    const int ldx8 = 8 * ldx;
    for (int p = wr; 2 * p < NG; p += nwr) {
#pragma unroll 1
      for (int side = 0; side < 2; ++side) {
        const int g = side ? NG - 1 - p : p;
        if (side && g == p) break;  // middle group of an odd count: once
        const int i0 = 32 * g, nchunk = NG - g;
        double acc1[4][2][2], acc2[4][2][2], ra[8], rb[8];
#pragma unroll
        for (int m = 0; m < 4; ++m)
#pragma unroll
          for (int j = 0; j < 2; ++j) { acc1[m][j][0] = acc1[m][j][1] = 0.0; acc2[m][j][0] = acc2[m][j][1] = 0.0; }
        const double* gaT = ga + DENSE_OFFG + c - r;
        const double* gbT = gb + DENSE_OFFG + c - r;
        const double* xk = xb + i0;
        dense_chunk<true>(gaT, gbT, xk, ldx8, ra, rb, acc1, acc2);
#pragma unroll 1
        for (int qq = 1; qq < nchunk; ++qq) {
          gaT += 32; gbT += 32; xk += 32;
          dense_chunk<false>(gaT, gbT, xk, ldx8, ra, rb, acc1, acc2);
        }
        // fused S5 for rows i0 + 8m + r, columns 8j + 2c + e
#pragma unroll
        for (int m = 0; m < 4; ++m) {
          cplx zv = mk(0.0, 0.0);
          if (MODE == MODE_INNER) { const int i = i0 + 8 * m + r; if (i < n) zv = sg.zd[i]; }
#pragma unroll
          for (int j = 0; j < 2; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) {
              const double y1 = acc1[m][j][e], y2 = acc2[m][j][e];
              q1[j][e] = fma(y1, y1, fma(-y2, y2, q1[j][e]));
              if (MODE == MODE_INNER) q0[j][e] = fma(y1, zv.x, fma(-y2, zv.y, q0[j][e]));
            }
        }
      }
    }
  }
  // ---- reduce over the 8 rows a lane quad-group holds, then over the row-group warps (fixed order)
#pragma unroll
  for (int j = 0; j < 2; ++j)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
#pragma unroll
      for (int o = 4; o < 32; o <<= 1) {
        q1[j][e] += __shfl_xor_sync(0xffffffffu, q1[j][e], o);
        if (MODE == MODE_INNER) q0[j][e] += __shfl_xor_sync(0xffffffffu, q0[j][e], o);
      }
      if (r == 0) {
        const int col = wc * 16 + 8 * j + 2 * c + e;
        red[wr * bt + col] = q1[j][e];
        red[(nwr + wr) * bt + col] = q0[j][e];
      }
    }
  __syncthreads();
  if (tid < bt) {
    const long long b = bt0 + tid;
    if (b < P.B) {
      double t1 = 0.0, t0 = 0.0;
      for (int w = 0; w < nwr; ++w) { t1 += red[w * bt + tid]; t0 += red[(nwr + w) * bt + tid]; }
      if (MODE == MODE_LOGLIKE) {
        const double v = -0.5 * t1;
        P.out0[b] = P.accumulate ? P.out0[b] + v : v;
      } else {
        if (P.out0) P.out0[b] = P.accumulate ? P.out0[b] + t0 : t0;
        if (P.out1) P.out1[b] = P.accumulate ? P.out1[b] + t1 : t1;
      }
    }
  }
}

}  // namespace td
