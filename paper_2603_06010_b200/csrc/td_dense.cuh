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
  DenseSeg seg;          // ONE segment per launch (segments accumulate into out in launch order)
  int accumulate;
  int nwr;               // row-group warps (1, 2, 4 or 8) that share a group's 16 templates; NWC = 8 / nwr groups per CTA
  int nbuf;              // panel buffers per group (2: the next tile's rows are in flight while this one computes)
  int vec_ok;            // every row start is 16-byte aligned and N_s is even: 16-byte async copies (else 8-byte)
  long long ntiles;      // ceil(B / 16): tiles of 16 templates, dealt round-robin to the groups of all CTAs
  int stagger_cycles;    // start-up delay of the second half of a CTA's groups (see the kernel)
};

}  // namespace td
#include <vector>
namespace td {
struct DenseState {
  int max_n = 0;             // longest segment the dense path accepts (0: unavailable)
  int auto_n = 0;            // AUTO takes the dense path for size classes whose segments are all <= auto_n
  std::vector<DenseSeg> all;   // every segment (forced dense path); empty if some segment is too long
  std::vector<DenseSeg> aut;   // the segments AUTO sends to the dense paths
  std::vector<DenseSeg> aut_gs;  // of those, the ones whose log-likelihood stays on this kernel (the rest: td_cdo.cuh)
};

__host__ __device__ inline int dense_nwr(int max_npad) {
  int p = max_npad / 64;
  return p < 1 ? 1 : (p >= 8 ? 8 : (p >= 4 ? 4 : (p >= 2 ? 2 : 1)));
}
__host__ __device__ inline int dense_ldx(int max_npad) { return max_npad + 4; }
// shared memory: ga, gb (zero-padded generators), the data segment, per group nbuf panels of 16
// templates, the per-group reduction scratch
inline size_t dense_smem_bytes(int npad, int nbuf) {
  const int nwr = dense_nwr(npad), nwc = DENSE_NW / nwr;
  return sizeof(double) * (2 * (size_t)(npad + 16) + (size_t)npad +
                           (size_t)nwc * nbuf * 16 * dense_ldx(npad) + (size_t)nwc * 2 * nwr * 16);
}
inline int dense_nbuf(int npad) { return dense_smem_bytes(npad, 2) <= 200 * 1024 ? 2 : 1; }

__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(uint32_t dst, const void* src, uint32_t src_bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}

// 8 k-steps (32 samples) of one 32-row group.  FIRST: the chunk that starts on the diagonal
// (row tile m only becomes non-zero at step 2m).  SUB: the B fragment is the residual d - h
// (S1 fused into the fragment load), otherwise h itself.
template <bool FIRST, bool SUB>
__device__ __forceinline__ void dense_chunk(const double* __restrict__ gaT, const double* __restrict__ gbT,
                                            const double* __restrict__ xk, const double* __restrict__ dk, int ldx8,
                                            double (&ra)[8], double (&rb)[8], double (&acc1)[4][2][2],
                                            double (&acc2)[4][2][2]) {
  static_for<0, 8>([&](auto ss) {
    constexpr int s = decltype(ss)::value;
    ra[s] = gaT[4 * s];
    rb[s] = gbT[4 * s];
    double x0 = xk[4 * s], x1 = xk[4 * s + ldx8];
    if constexpr (SUB) { const double dv = dk[4 * s]; x0 = dv - x0; x1 = dv - x1; }
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

// Persistent kernel, one CTA per SM, built from INDEPENDENT warp groups: a group = the nwr warps
// that share 16 templates (nwr = 1 for N <= 127: a single warp).  A group owns its panel buffers,
// copies its own rows global -> shared with cp.async (one 16-template tile ahead of the DMMA work),
// synchronises only within itself (__syncwarp or a named barrier) and writes its own outputs:
// there is no CTA-wide barrier in the loop.  profiles/r01_dense_ncu.md: with CTA-wide barriers every
// warp is in the same phase, so the tensor pipe idles during each copy-issue / reduction phase
// (41 % DMMA-active at N = 64).  The two warps that share an SM sub-partition belong to different
// groups; the second half of the groups starts `stagger_cycles` late, and because a group alone
// runs the pipe at full rate the lag persists: one group's bookkeeping overlaps the other's DMMAs.
template <int MODE, int NWR>
__global__ void __launch_bounds__(DENSE_NT, 1) td_dense_kernel(const DenseParams P) {
  extern __shared__ __align__(16) double smd[];
  const DenseSeg sg = P.seg;
  const int n = sg.n, npad = sg.npad;
  const int glen = npad + 16, ldx = dense_ldx(npad);
  constexpr int nwr = NWR, nwc = DENSE_NW / nwr;
  const int nbuf = P.nbuf;
  const size_t psz = (size_t)16 * ldx;  // one panel: 16 templates
  double* ga = smd;
  double* gb = ga + glen;
  double* dS = gb + glen;
  double* Xs = dS + npad;
  double* red = Xs + (size_t)nwc * nbuf * psz;  // [nwc][2][nwr][16]
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int r = lane >> 2, c = lane & 3;
  const int wr = warp % nwr, wc = warp / nwr;
  const bool vec = P.vec_ok != 0;

  // generators (scaled by 1/sqrt(v)), zero-padded on both sides: b_j = a_{n-j}, b_0 = 0; data segment
  for (int j = tid; j < glen; j += DENSE_NT) {
    const int jj = j - DENSE_OFFG;
    ga[j] = (jj >= 0 && jj < n) ? __ldg(sg.a + jj) * sg.rsv : 0.0;
    gb[j] = (jj >= 1 && jj < n) ? __ldg(sg.a + n - jj) * sg.rsv : 0.0;
  }
  if (MODE == MODE_LOGLIKE)
    for (int j = tid; j < npad; j += DENSE_NT) dS[j] = j < n ? P.d[sg.off + j] : 0.0;

  double* Xg = Xs + (size_t)wc * nbuf * psz;          // this group's panels
  double* redg = red + (size_t)wc * 2 * nwr * 16;     // this group's reduction scratch
  const double* const Hg = P.H;
  const long long ldh = P.ldh, Btot = P.B, ntiles = P.ntiles;
  const long long gstride = (long long)gridDim.x * nwc;
  const long long t0 = (long long)blockIdx.x * nwc + wc;
  auto group_sync = [&]() {
    if (nwr == 1) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + wc), "r"(32 * nwr) : "memory");
  };
  // rows of tile t -> panel `buf`: 16 / nwr rows per warp, zero-filled beyond N_s and beyond the
  // last template; exactly one commit group per call keeps the group counts uniform
  auto issue = [&](long long t, int buf) {
    if (t < ntiles) {
      const long long b0 = t * 16;
      const int rows = (int)(Btot - b0 < 16 ? Btot - b0 : 16);
      const double* src = Hg + (b0 + wr) * ldh + sg.off;
      const long long sstep = nwr * ldh;
      const uint32_t dst = smem_u32(Xg + (size_t)buf * psz + (size_t)wr * ldx);
      const uint32_t dstep = (uint32_t)(nwr * ldx * 8);
      if (vec) {
        const int nj = npad >> 1, nv = n >> 1;  // 16-byte chunks per row: all / holding samples
        for (int j = lane; j < nj; j += 32) {
          const bool inj = j < nv;
#pragma unroll
          for (int q = 0; q < 16 / nwr; ++q) {
            const bool in = inj && (wr + q * nwr < rows);
            cp_async16(dst + q * dstep + 16u * j, in ? src + q * sstep + 2 * j : Hg, in ? 16u : 0u);
          }
        }
      } else {
        for (int j = lane; j < npad; j += 32) {
          const bool inj = j < n;
#pragma unroll
          for (int q = 0; q < 16 / nwr; ++q) {
            const bool in = inj && (wr + q * nwr < rows);
            cp_async8(dst + q * dstep + 8u * j, in ? src + q * sstep + j : Hg, in ? 8u : 0u);
          }
        }
      }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  for (int k = 0; k < nbuf; ++k) issue(t0 + k * gstride, k);
  __syncthreads();  // generators and data segment visible (the only CTA-wide barrier)
  if (wc >= (nwc + 1) / 2 && nwc > 1) {
    const long long c0 = clock64();
    while (clock64() - c0 < P.stagger_cycles) {}
  }

  const int NG = npad >> 5, ldx8 = 8 * ldx;
  int buf = 0;
  for (long long t = t0; t < ntiles; t += gstride) {
    if (nbuf == 2) asm volatile("cp.async.wait_group 1;" ::: "memory");
    else asm volatile("cp.async.wait_group 0;" ::: "memory");
    group_sync();  // every warp's rows of this panel have landed
    // ---- S2'-S4' + S5: the group's 16 templates against this warp's row groups
    const double* xb = Xg + (size_t)buf * psz + (size_t)r * ldx + c;
    double q0[2][2] = {{0.0, 0.0}, {0.0, 0.0}}, q1[2][2] = {{0.0, 0.0}, {0.0, 0.0}};  // [column tile][e]
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
        const double* dk = dS + i0 + c;
        constexpr bool SUB = (MODE == MODE_LOGLIKE);
        dense_chunk<true, SUB>(gaT, gbT, xk, dk, ldx8, ra, rb, acc1, acc2);
#pragma unroll 1
        for (int qq = 1; qq < nchunk; ++qq) {
          gaT += 32; gbT += 32; xk += 32; dk += 32;
          dense_chunk<false, SUB>(gaT, gbT, xk, dk, ldx8, ra, rb, acc1, acc2);
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
    // ---- reduce over the 8 rows a lane quad-group holds, then over the group's warps (fixed order)
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
          const int col = 8 * j + 2 * c + e;
          redg[wr * 16 + col] = q1[j][e];
          redg[(nwr + wr) * 16 + col] = q0[j][e];
        }
      }
    group_sync();  // partial sums visible; every warp of the group is done with panel `buf`
    issue(t + nbuf * gstride, buf);
    if (wr == 0 && lane < 16) {
      const long long b = t * 16 + lane;
      if (b < Btot) {
        double t1 = 0.0, tz = 0.0;
        for (int w = 0; w < nwr; ++w) { t1 += redg[w * 16 + lane]; tz += redg[(nwr + w) * 16 + lane]; }
        if (MODE == MODE_LOGLIKE) {
          const double v = -0.5 * t1;
          P.out0[b] = P.accumulate ? P.out0[b] + v : v;
        } else {
          if (P.out0) P.out0[b] = P.accumulate ? P.out0[b] + tz : tz;
          if (P.out1) P.out1[b] = P.accumulate ? P.out1[b] + t1 : t1;
        }
      }
    }
    if (nbuf == 2) buf ^= 1;
  }
}

}  // namespace td
