// td_cdo.cuh - the paper's "CDO" evaluation as a batched triangular contraction (second half;
// PAPER.md:215-227, III.A.2: Cholesky C = L L^T "done once and cached", whitening operator W = L^{-1} cached, per
// template r-bar = W r and lnL = -1/2 r-bar . r-bar - the GEMV of :225 for a whole batch at once).
//
//   Y = W X,   W = L^{-1} (N x N, lower-triangular),   X = [r_0 .. r_{B-1}] (N x B),   Q_b = sum_i Y[i][b]^2
//
// N^2 B flop: half of the Gohberg-Semencul dense path (td_dense.cuh, two triangular Toeplitz products), but the operator
// is N^2/2 distinct numbers instead of N, so it cannot be generated on the fly: every group of templates streams W from
// L2.  The kernel keeps that stream per template as small as shared memory allows and measures the trade
// (profiles/r02_cdo.md): panels of 8 NC templates (NC = 2 or 4 column tiles) per warp group, A fragments loaded straight
// from L2 into registers one 32-column chunk ahead (no shared-memory staging of W), B fragments from the template panel in
// shared memory, fp64 tensor pipe (mma.sync.m8n8k4.f64).
//
// W comes out of the Levinson-Durbin recursion as a by-product: row i of L^{-1} is the order-i prediction-error filter
// divided by sqrt(E_i), (L^{-1} x)_i = (x_i + sum_{j=1..i} a^(i)_j x_{i-j}) / sqrt(E_i) (the innovations form of Eq. 8-10,
// PAPER.md:134-142).  It is stored in FRAGMENT ORDER: within each 32-column chunk, column k0 + c + 4 s sits at position
// k0 + 8 c + s, so that the eight A-fragment values a lane needs for the eight k-steps of a chunk are 64 contiguous bytes.
#pragma once
#include "td_dense.cuh"

namespace td {

constexpr int CDO_MAX_N = 1024;   // longest segment of the CDO path (W is npad^2 doubles: 8 MB)
constexpr int CDO_NT = 1024;

// one CTA per segment: Levinson-Durbin with the filter in shared memory, row i of W written after order i
struct CdoSeg {
  const double* rho;  // device [n]
  double* W;          // device [npad][npad], fragment order, zero above the diagonal and beyond n
  int n, npad;
};
__device__ __forceinline__ int cdo_frag_col(int k) { return (k & ~31) + 8 * (k & 3) + ((k & 31) >> 2); }

__global__ void __launch_bounds__(CDO_NT) cdo_whitener_kernel(const CdoSeg* __restrict__ segs) {
  __shared__ double a[CDO_MAX_N];
  __shared__ double red[CDO_NT / 32];
  __shared__ double bc;
  const CdoSeg sg = segs[blockIdx.x];
  const double* __restrict__ rho = sg.rho;
  const int n = sg.n, npad = sg.npad, tid = threadIdx.x;
  for (size_t j = tid; j < (size_t)npad * npad; j += CDO_NT) sg.W[j] = 0.0;
  for (int j = tid; j < n; j += CDO_NT) a[j] = (j == 0) ? 1.0 : 0.0;
  double E = rho[0];
  __syncthreads();
  if (tid == 0) sg.W[cdo_frag_col(0)] = rsqrt(E);
  for (int k = 1; k < n; ++k) {   // (td_create has already accepted this ACF: no SPD test here)
    double acc = 0.0;
    for (int j = tid; j < k; j += CDO_NT) acc = fma(a[j], rho[k - j], acc);
    acc = warp_sum(acc);
    if ((tid & 31) == 0) red[tid >> 5] = acc;
    __syncthreads();
    if (tid < 32) {
      double v = red[tid];
      v = warp_sum(v);
      if (tid == 0) bc = v;
    }
    __syncthreads();
    const double kk = -bc / E;
    double aj = 0.0, ak = 0.0;
    const int j = 1 + tid;
    const bool act = 2 * j < k;
    if (act) { aj = a[j]; ak = a[k - j]; }
    __syncthreads();
    if (act) { a[j] = fma(kk, ak, aj); a[k - j] = fma(kk, aj, ak); }
    if (tid == 0) {
      if ((k & 1) == 0) { const double am = a[k / 2]; a[k / 2] = fma(kk, am, am); }
      a[k] = kk;
    }
    E *= (1.0 - kk * kk);
    __syncthreads();
    const double rs = 1.0 / sqrt(E);
    for (int jj = tid; jj <= k; jj += CDO_NT) sg.W[(size_t)k * npad + cdo_frag_col(k - jj)] = a[jj] * rs;
  }
}

struct CdoParams {
  const double* d;
  const double* H;
  long long ldh;
  long long B;
  double* out;
  long long off;       // offset of the segment inside d / a row of H
  int n, npad;
  const double* W;     // [npad][npad], fragment order
  int accumulate;
  int nbuf;            // panel buffers per group
  int vec_ok;
  long long ntiles;    // ceil(B / (8 NC))
};

template <int NC> inline size_t cdo_smem_bytes(int npad, int nbuf) {
  const int nwr = dense_nwr(npad), nwc = DENSE_NW / nwr;
  return sizeof(double) * ((size_t)npad + (size_t)nwc * nbuf * 8 * NC * dense_ldx(npad) + (size_t)nwc * nwr * 8 * NC);
}

// the A fragments of one 32-column chunk for this lane's 4 row tiles: 8 contiguous doubles each
__device__ __forceinline__ void cdo_load_a(const double* __restrict__ wp, size_t row8, double (&a)[4][8]) {
#pragma unroll
  for (int m = 0; m < 4; ++m)
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const double2 v = __ldg(reinterpret_cast<const double2*>(wp + m * row8) + q);
      a[m][2 * q] = v.x; a[m][2 * q + 1] = v.y;
    }
}

template <int NC>
__global__ void __launch_bounds__(DENSE_NT, 1) td_cdo_kernel(const CdoParams P) {
  extern __shared__ __align__(16) double smd[];
  constexpr int TB = 8 * NC;
  const int n = P.n, npad = P.npad, ldx = dense_ldx(npad);
  const int nwr = dense_nwr(npad), nwc = DENSE_NW / nwr, nbuf = P.nbuf;
  const size_t psz = (size_t)TB * ldx;
  double* dS = smd;
  double* Xs = dS + npad;
  double* red = Xs + (size_t)nwc * nbuf * psz;  // [nwc][nwr][TB]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r = lane >> 2, c = lane & 3;
  const int wr = warp % nwr, wc = warp / nwr;
  const bool vec = P.vec_ok != 0;
  for (int j = tid; j < npad; j += DENSE_NT) dS[j] = j < n ? P.d[P.off + j] : 0.0;
  double* Xg = Xs + (size_t)wc * nbuf * psz;
  double* redg = red + (size_t)wc * nwr * TB;
  const long long ldh = P.ldh, Btot = P.B, ntiles = P.ntiles;
  const long long gstride = (long long)gridDim.x * nwc;
  const long long t0 = (long long)blockIdx.x * nwc + wc;
  auto group_sync = [&]() {
    if (nwr == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + wc), "r"(32 * nwr) : "memory");
  };
  auto issue = [&](long long t, int buf) {
    if (t < ntiles) {
      const long long b0 = t * TB;
      const int rows = (int)(Btot - b0 < TB ? Btot - b0 : TB);
      const double* src = P.H + (b0 + wr) * ldh + P.off;
      const long long sstep = nwr * ldh;
      const uint32_t dst = smem_u32(Xg + (size_t)buf * psz + (size_t)wr * ldx);
      const uint32_t dstep = (uint32_t)(nwr * ldx * 8);
      const int nq = TB / nwr;
      if (vec) {
        const int nj = npad >> 1, nv = n >> 1;
        for (int j = lane; j < nj; j += 32) {
          const bool inj = j < nv;
          for (int q = 0; q < nq; ++q) {
            const bool in = inj && (wr + q * nwr < rows);
            cp_async16(dst + q * dstep + 16u * j, in ? src + q * sstep + 2 * j : P.H, in ? 16u : 0u);
          }
        }
      } else {
        for (int j = lane; j < npad; j += 32) {
          const bool inj = j < n;
          for (int q = 0; q < nq; ++q) {
            const bool in = inj && (wr + q * nwr < rows);
            cp_async8(dst + q * dstep + 8u * j, in ? src + q * sstep + j : P.H, in ? 8u : 0u);
          }
        }
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  for (int k = 0; k < nbuf; ++k) issue(t0 + k * gstride, k);
  __syncthreads();  // data segment visible

  const int NG = npad >> 5, ldx8 = 8 * ldx;
  const size_t row8 = (size_t)8 * npad;
  int buf = 0;
  for (long long t = t0; t < ntiles; t += gstride) {
    if (nbuf == 2) asm volatile("cp.async.wait_group 1;" ::: "memory");
    else asm volatile("cp.async.wait_group 0;" ::: "memory");
    group_sync();
    // single-buffered panels (the large tiles): the rows of this group's NEXT tile start their way from HBM into L2 now, so the
    // copy that is issued after this tile's contraction - and waited for - finds them there
    if (nbuf == 1 && vec && wr == 0) {
      const long long tn = t + gstride;
      if (tn < ntiles && lane < TB) {
        const long long bn = tn * TB + lane;
        if (bn < Btot)
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(P.H + bn * ldh + P.off), "r"((uint32_t)(n * 8)) : "memory");
      }
    }
    const double* xb = Xg + (size_t)buf * psz + (size_t)r * ldx + c;
    double q1[NC][2];
#pragma unroll
    for (int j = 0; j < NC; ++j) q1[j][0] = q1[j][1] = 0.0;
    for (int p = wr; 2 * p < NG; p += nwr) {
#pragma unroll 1
      for (int side = 0; side < 2; ++side) {
        const int g = side ? NG - 1 - p : p;
        if (side && g == p) break;
        const int i0 = 32 * g;
        double acc[4][NC][2], a0[4][8], a1[4][8];
#pragma unroll
        for (int m = 0; m < 4; ++m)
#pragma unroll
          for (int j = 0; j < NC; ++j) acc[m][j][0] = acc[m][j][1] = 0.0;
        // row i0 + 8 m + r of W, columns of chunk q at 32 q + 8 c: the lower triangle, chunks 0 .. g
        const double* wp = P.W + (size_t)(i0 + r) * npad + 8 * c;
        cdo_load_a(wp, row8, a0);
        auto chunk = [&](const double (&a)[4][8], int k0) {
          const double* xk = xb + k0;
          const double* dk = dS + k0 + c;
          static_for<0, 8>([&](auto ss) {
            constexpr int s = decltype(ss)::value;
            const double dv = dk[4 * s];
            double x[NC];
#pragma unroll
            for (int j = 0; j < NC; ++j) x[j] = dv - xk[4 * s + j * ldx8];   // S1 fused into the fragment load
#pragma unroll
            for (int m = 0; m < 4; ++m)
#pragma unroll
              for (int j = 0; j < NC; ++j) dmma884(acc[m][j], a[m][s], x[j]);
          });
        };
        int q = 0;
#pragma unroll 1
        for (; q + 1 <= g; q += 2) {          // two chunks per trip: the register buffers alternate without copies
          cdo_load_a(wp + 32 * (q + 1), row8, a1);
          chunk(a0, 32 * q);
          if (q + 2 <= g) cdo_load_a(wp + 32 * (q + 2), row8, a0);
          chunk(a1, 32 * (q + 1));
        }
        if (q <= g) chunk(a0, 32 * q);
        // fused S5
#pragma unroll
        for (int m = 0; m < 4; ++m)
#pragma unroll
          for (int j = 0; j < NC; ++j)
#pragma unroll
            for (int e = 0; e < 2; ++e) q1[j][e] = fma(acc[m][j][e], acc[m][j][e], q1[j][e]);
      }
    }
#pragma unroll
    for (int j = 0; j < NC; ++j)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
#pragma unroll
        for (int o = 4; o < 32; o <<= 1) q1[j][e] += __shfl_xor_sync(0xffffffffu, q1[j][e], o);
        if (r == 0) redg[wr * TB + 8 * j + 2 * c + e] = q1[j][e];
      }
    group_sync();
    issue(t + nbuf * gstride, buf);
    if (wr == 0 && lane < TB) {
      const long long b = t * TB + lane;
      if (b < Btot) {
        double t1 = 0.0;
        for (int w = 0; w < nwr; ++w) t1 += redg[w * TB + lane];
        const double v = -0.5 * t1;
        P.out[b] = P.accumulate ? P.out[b] + v : v;
      }
    }
    if (nbuf == 2) buf ^= 1;
  }
}

}  // namespace td
