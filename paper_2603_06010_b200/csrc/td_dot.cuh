// td_dot.cuh - the cross term <d, h_b> of Eq. 13 as a plain batched dot product.
//
// <d, h_b> = d^T C^{-1} h_b = u . h_b  with  u = C^{-1} d  computed once per call: the paper's CDO idea of caching
// the whitened data carried one step further - with u cached, the
// cross term needs no transform at all, one pass over H, 2 flop per 8 bytes: the one HBM-bound kernel of this
// library.  u comes from the Gohberg-Semencul form (Eq. 14) applied to the filtered data vector that
// td_inner_batch already computes, z_d = (L(a)^T d + i L(b)^T d) / sqrt(v):
//     u = C^{-1} d = ( L(a) Re z_d - L(b) Im z_d ) / sqrt(v),     (L(c) x)_i = sum_{j<=i} c_{i-j} x_j,
// b = (0, a_{N-1}, ..., a_1).  That is an O(N^2) lower-triangular Toeplitz product per segment, done directly
// (128 x 128 tiles through shared memory, one CTA per tile, then a fixed-order sum over the tiles of a row):
// N = 4096 is 17 M multiply-adds, a few microseconds, once per call.
#pragma once
#include "td_common.cuh"

namespace td {

constexpr int DOTW_NT = 128;     // outputs per CTA of the weight kernel (= threads)
constexpr int DOT_NT = 256;      // threads per CTA of the dot kernel
constexpr int DOT_MAX_N = 16384; // longest segment for which the O(N^2) weight kernel is used

// Tile (it, jt), jt <= it, of the triangular product: part[jt][i] = sum_{j in tile jt} ( a[i-j] Re zd[j] - b[i-j] Im zd[j] ),
// b[k] = a[n-k] (k >= 1), b[0] = 0.  One CTA per tile so that the N^2 / 2 multiply-adds spread over the whole GPU
// (one CTA per row tile walking its j tiles serially took 85 us at N = 4096: 32 CTAs).  blockIdx.x enumerates the
// lower-triangular tile pairs row by row.
__global__ void __launch_bounds__(DOTW_NT) dot_weight_tile_kernel(const double* __restrict__ a, const cplx* __restrict__ zd,
                                                                  int n, double* __restrict__ part, int ntile) {
  __shared__ double sa[2 * DOTW_NT];   // a at lags i0 - j0 - (NT-1) .. i0 - j0 + NT-1, zero outside [0, n)
  __shared__ double sb[2 * DOTW_NT];   // the same window of b
  __shared__ cplx sz[DOTW_NT];
  // tile pair from the linear index: it = largest t with t (t + 1) / 2 <= idx
  const int idx = blockIdx.x;
  int it = (int)((sqrt(8.0 * idx + 1.0) - 1.0) * 0.5);
  while ((it + 1) * (it + 2) / 2 <= idx) ++it;
  while (it * (it + 1) / 2 > idx) --it;
  const int jt = idx - it * (it + 1) / 2;
  const int tid = threadIdx.x, i0 = it * DOTW_NT, j0 = jt * DOTW_NT, i = i0 + tid;
  const int lag0 = i0 - j0 - (DOTW_NT - 1);  // lag held at window slot 0
  for (int k = tid; k < 2 * DOTW_NT - 1; k += DOTW_NT) {
    const int lag = lag0 + k;
    sa[k] = (lag >= 0 && lag < n) ? a[lag] : 0.0;
    sb[k] = (lag >= 1 && lag < n) ? a[n - lag] : 0.0;
  }
  sz[tid] = (j0 + tid < n) ? zd[j0 + tid] : mk(0.0, 0.0);
  __syncthreads();
  // lag of (i, j0 + jj) = i - j0 - jj  ->  slot tid + (NT-1) - jj; negative lags read the zeros of the window
  double acc0 = 0.0, acc1 = 0.0;
#pragma unroll 8
  for (int jj = 0; jj < DOTW_NT; ++jj) {
    const int k = tid + (DOTW_NT - 1) - jj;
    acc0 = fma(sa[k], sz[jj].x, acc0);
    acc1 = fma(sb[k], sz[jj].y, acc1);
  }
  if (i < n) part[(size_t)jt * ((size_t)ntile * DOTW_NT) + i] = acc0 - acc1;
}

// u[i] = rsv * sum_{jt <= i / NT} part[jt][i]   (fixed order)
__global__ void dot_weight_sum_kernel(const double* __restrict__ part, int n, int ntile, double rsv, double* __restrict__ u) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  double s = 0.0;
  const int last = i / DOTW_NT;
  for (int jt = 0; jt <= last; ++jt) s += part[(size_t)jt * ((size_t)ntile * DOTW_NT) + i];
  u[i] = rsv * s;
}

// out[b] = sum_{i < n_tot} u[i] * H[b][i].  A CTA takes two rows per pass (every weight fetched from L1 serves two
// elements of H), its warps split the columns; 16-byte streaming loads of H (evict-first, so the weights stay cached),
// four independent accumulators per thread and row, fixed summation order (bitwise repeatable).  The grid is the
// number of CTAs resident at once and row pairs are dealt round-robin: with one row pair per WARP a batch of 4096
// pairs was 1.15 waves of resident warps, i.e. the tail ran at half occupancy (ncu: 57 % of DRAM peak).
template <bool VEC>
__global__ void __launch_bounds__(DOT_NT) dot_rows_kernel(const double* __restrict__ u, const double* __restrict__ H,
                                                          long long ldh, long long B, int n_tot, double* __restrict__ out,
                                                          int accumulate) {
  __shared__ double red[2][DOT_NT / 32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (long long b = 2ll * blockIdx.x; b < B; b += 2ll * gridDim.x) {
    const bool two = b + 1 < B;
    const double* __restrict__ row0 = H + b * ldh;
    const double* __restrict__ row1 = two ? row0 + ldh : row0;
    double acc0[4] = {0.0, 0.0, 0.0, 0.0}, acc1[4] = {0.0, 0.0, 0.0, 0.0};
    if (VEC) {
      const double2* __restrict__ r0 = reinterpret_cast<const double2*>(row0);
      const double2* __restrict__ r1 = reinterpret_cast<const double2*>(row1);
      const double2* __restrict__ u2 = reinterpret_cast<const double2*>(u);
      const int n2 = n_tot >> 1;
      int k = tid;
      for (; k + 3 * DOT_NT < n2; k += 4 * DOT_NT) {
        double2 h0[4], h1[4];
#pragma unroll
        for (int q = 0; q < 4; ++q) { h0[q] = __ldcs(r0 + k + DOT_NT * q); h1[q] = __ldcs(r1 + k + DOT_NT * q); }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const double2 uv = __ldg(u2 + k + DOT_NT * q);
          acc0[q] = fma(h0[q].x, uv.x, fma(h0[q].y, uv.y, acc0[q]));
          acc1[q] = fma(h1[q].x, uv.x, fma(h1[q].y, uv.y, acc1[q]));
        }
      }
      double t0 = 0.0, t1 = 0.0;
      for (; k < n2; k += DOT_NT) {
        const double2 a0 = __ldcs(r0 + k), a1 = __ldcs(r1 + k), uv = __ldg(u2 + k);
        t0 = fma(a0.x, uv.x, fma(a0.y, uv.y, t0));
        t1 = fma(a1.x, uv.x, fma(a1.y, uv.y, t1));
      }
      if ((n_tot & 1) && tid == 0) { t0 = fma(row0[n_tot - 1], u[n_tot - 1], t0); t1 = fma(row1[n_tot - 1], u[n_tot - 1], t1); }
      acc0[0] += t0; acc1[0] += t1;
    } else {
      int k = tid;
      for (; k + 3 * DOT_NT < n_tot; k += 4 * DOT_NT) {
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const double uv = __ldg(u + k + DOT_NT * q);
          acc0[q] = fma(__ldcs(row0 + k + DOT_NT * q), uv, acc0[q]);
          acc1[q] = fma(__ldcs(row1 + k + DOT_NT * q), uv, acc1[q]);
        }
      }
      double t0 = 0.0, t1 = 0.0;
      for (; k < n_tot; k += DOT_NT) { const double uv = __ldg(u + k); t0 = fma(__ldcs(row0 + k), uv, t0); t1 = fma(__ldcs(row1 + k), uv, t1); }
      acc0[0] += t0; acc1[0] += t1;
    }
    double s0 = (acc0[0] + acc0[1]) + (acc0[2] + acc0[3]), s1 = (acc1[0] + acc1[1]) + (acc1[2] + acc1[3]);
    s0 = warp_sum(s0);
    s1 = warp_sum(s1);
    if (lane == 0) { red[0][warp] = s0; red[1][warp] = s1; }
    __syncthreads();
    if (tid < 2 && (tid == 0 || two)) {
      double s = 0.0;
#pragma unroll
      for (int w = 0; w < DOT_NT / 32; ++w) s += red[tid][w];
      out[b + tid] = accumulate ? out[b + tid] + s : s;
    }
    __syncthreads();
  }
}

}  // namespace td
