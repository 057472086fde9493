// td_setup.cuh - one-time setup kernels of td_create:
//   Levinson-Durbin recursion per segment  ->  prediction-error filter a, variance v, log det C
//   (the paper cites the O(N^2) Toeplitz factorisation without printing it: PAPER.md:176 refs
//   [104,105], :215; C a = v e_1 gives x = C^{-1} e_1 = a / v of Eq. 14),
//   twiddle table, and the packed generator g = a - i b (b = (0, a_{N-1}, ..., a_1)) whose
//   length-2M transform, conjugated, is G = conj(A^) + i conj(B^).
#pragma once
#include "td_common.cuh"

namespace td {

__global__ void tw_table_kernel(cplx* T, int TW) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= TW) return;
  double s, c;
  sincospi(2.0 * (double)k / (double)TW, &s, &c);  // exact argument for power-of-two TW
  T[k] = mk(c, -s);
}

struct LevSeg {
  const double* rho;  // device, n doubles
  double* a;          // device, n doubles (output)
  int n;
  int coop;           // handled by levinson_coop_kernel (long segment): levinson_kernel skips it
};

constexpr int LEV_NT = 1024;

// status: 0 ok, 2 not SPD / non-finite
__global__ void __launch_bounds__(LEV_NT) levinson_kernel(const LevSeg* __restrict__ segs, double* v_out,
                                                          double* logdet_out, int* status) {
  __shared__ double red[LEV_NT / 32];
  __shared__ double bc;
  const LevSeg sg = segs[blockIdx.x];
  if (sg.coop) return;
  const double* __restrict__ rho = sg.rho;
  double* a = sg.a;
  const int n = sg.n, tid = threadIdx.x;
  const double rho0 = rho[0];
  if (!(rho0 > 0.0) || !isfinite(rho0)) {
    if (tid == 0) status[blockIdx.x] = 2;
    return;
  }
  for (int j = tid; j < n; j += LEV_NT) a[j] = (j == 0) ? 1.0 : 0.0;
  double E = rho0, logdet = log(rho0);
  __syncthreads();
  for (int k = 1; k < n; ++k) {
    double acc = 0.0;
    for (int j = tid; j < k; j += LEV_NT) acc = fma(a[j], rho[k - j], acc);
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
    if (!(fabs(kk) < 1.0)) {  // also catches NaN
      if (tid == 0) status[blockIdx.x] = 2;
      return;
    }
    for (int j = 1 + tid; 2 * j < k; j += LEV_NT) {
      const double aj = a[j], ak = a[k - j];
      a[j] = fma(kk, ak, aj);
      a[k - j] = fma(kk, aj, ak);
    }
    if (tid == 0) {
      if ((k & 1) == 0) { const double am = a[k / 2]; a[k / 2] = fma(kk, am, am); }
      a[k] = kk;
    }
    E *= (1.0 - kk * kk);
    logdet += log(E);
    if (!(E > 0.0)) {
      if (tid == 0) status[blockIdx.x] = 2;
      return;
    }
    __syncthreads();
  }
  if (tid == 0) {
    v_out[blockIdx.x] = E;
    logdet_out[blockIdx.x] = logdet;
    status[blockIdx.x] = 0;
  }
}

// The same recursion for one LONG segment on many CTAs (cooperative launch, one grid-wide barrier per order): a single
// CTA streams a and rho (2 x 8 N bytes at the last orders) through one SM for every order, which is 0.96 s at N = 65536;
// spread over the grid the step is bounded by the barrier, not by one SM's bandwidth.  Every thread carries its own copy
// of E and log det (identical arithmetic on identical partial sums), so the SPD test exits the whole grid uniformly.
constexpr int LEVC_NT = 512;
constexpr int LEV_COOP_MIN_N = 16384;

// grid-wide barrier of the cooperative kernel below: one arrival per CTA on a 64-bit counter that only grows (release
// reduction after the CTA's barrier, acquire polling by one thread).  About a third of the cost of cooperative_groups'
// grid.sync() on B200 (measured through td_create: N = 65536 0.37 s -> see DESIGN.md 0), and the recursion pays it once per order.
// Data that crosses CTAs (a, partial) is read and written with .cg accesses: L2 only, no stale L1 lines.
__device__ __forceinline__ void lev_grid_barrier(unsigned long long* ctr, unsigned long long& target, int G) {
  __syncthreads();
  if (threadIdx.x == 0) {
    target += (unsigned long long)G;
    asm volatile("red.release.gpu.global.add.u64 [%0], %1;" ::"l"(ctr), "l"(1ull) : "memory");
    unsigned long long v;
    const long long t0 = clock64();
    do {
      asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(ctr) : "memory");
      if (clock64() - t0 > 20000000000ll) __trap();   // (~10 s) never with a cooperative launch: all CTAs are resident
    } while (v < target);
  }
  __syncthreads();
}

__global__ void __launch_bounds__(LEVC_NT) levinson_coop_kernel(const LevSeg sg, double* partial, unsigned long long* bar,
                                                               double* v_out, double* logdet_out, int* status) {
  __shared__ double red[LEVC_NT / 32];
  __shared__ double bc;
  const double* __restrict__ rho = sg.rho;
  double* a = sg.a;
  const int n = sg.n, tid = threadIdx.x, G = gridDim.x;
  const int gtid = blockIdx.x * LEVC_NT + tid, gsz = G * LEVC_NT;
  unsigned long long bar_target = 0;
  const double rho0 = rho[0];
  if (!(rho0 > 0.0) || !isfinite(rho0)) {
    if (gtid == 0) *status = 2;
    return;
  }
  for (int j = gtid; j < n; j += gsz) __stcg(a + j, (j == 0) ? 1.0 : 0.0);
  double E = rho0, logdet = log(rho0);
  // ONE grid barrier per order: the thread that updates the pair (a_j, a_{k-j}) of order k holds both new values in
  // registers and adds their terms of the NEXT order's dot product sum_j a_j rho_{k+1-j} on the spot, so the dot product needs
  // no pass (and no barrier) of its own; per-CTA partial sums are double-buffered by the parity of the order.
  if (tid == 0 && n > 1) __stcg(partial + (size_t)1 * G + blockIdx.x, blockIdx.x == 0 ? rho[1] : 0.0);
  lev_grid_barrier(bar, bar_target, G);
  for (int k = 1; k < n; ++k) {
    if (tid < 32) {  // fixed order: lane l adds partials l, l + 32, ...; then the warp tree
      double v = 0.0;
      for (int c = tid; c < G; c += 32) v += __ldcg(partial + (size_t)(k & 1) * G + c);
      v = warp_sum(v);
      if (tid == 0) bc = v;
    }
    __syncthreads();
    const double kk = -bc / E;
    if (!(fabs(kk) < 1.0)) {  // also catches NaN; the same value in every thread of the grid
      if (gtid == 0) *status = 2;
      return;
    }
    const bool more = k + 1 < n;
    double acc = 0.0;
    // four pairs per trip with all their loads issued first: the pairs of different j are disjoint, which the compiler cannot
    // know (it would keep every load behind the previous trip's stores), and a thread has only a handful of trips per order
    int j = 1 + gtid;
    for (; 2 * (j + 3 * gsz) < k; j += 4 * gsz) {
      double aj[4], ak[4], r0[4], r1[4];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int ju = j + u * gsz;
        aj[u] = __ldcg(a + ju); ak[u] = __ldcg(a + k - ju);
        r0[u] = more ? rho[k + 1 - ju] : 0.0; r1[u] = more ? rho[ju + 1] : 0.0;
      }
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        const int ju = j + u * gsz;
        const double nj = fma(kk, ak[u], aj[u]), nk = fma(kk, aj[u], ak[u]);
        __stcg(a + ju, nj);
        __stcg(a + k - ju, nk);
        acc = fma(nj, r0[u], fma(nk, r1[u], acc));
      }
    }
    for (; 2 * j < k; j += gsz) {
      const double aj = __ldcg(a + j), ak = __ldcg(a + k - j);
      const double nj = fma(kk, ak, aj), nk = fma(kk, aj, ak);
      __stcg(a + j, nj);
      __stcg(a + k - j, nk);
      if (more) acc = fma(nj, rho[k + 1 - j], fma(nk, rho[j + 1], acc));
    }
    if (gtid == 0) {
      if ((k & 1) == 0) {
        const double am = __ldcg(a + k / 2), nm = fma(kk, am, am);
        __stcg(a + k / 2, nm);
        if (more) acc = fma(nm, rho[k + 1 - k / 2], acc);
      }
      __stcg(a + k, kk);
      if (more) acc += fma(kk, rho[1], rho[k + 1]);   // a_k rho_1 + a_0 rho_{k+1}
    }
    E *= (1.0 - kk * kk);
    logdet += log(E);
    if (!(E > 0.0)) {
      if (gtid == 0) *status = 2;
      return;
    }
    acc = warp_sum(acc);
    if ((tid & 31) == 0) red[tid >> 5] = acc;
    __syncthreads();
    if (tid < 32) {
      double v = tid < LEVC_NT / 32 ? red[tid] : 0.0;
      v = warp_sum(v);
      if (tid == 0) __stcg(partial + (size_t)((k + 1) & 1) * G + blockIdx.x, v);
    }
    lev_grid_barrier(bar, bar_target, G);
  }
  if (gtid == 0) {
    *v_out = E;
    *logdet_out = logdet;
    *status = 0;
  }
}

// g[j] = a_j - i b_j for j < n (b_0 = 0, b_j = a_{n-j}), zero up to n2 = 2M
__global__ void gen_pack_kernel(const double* __restrict__ a, int n, cplx* g, int n2) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j >= n2) return;
  cplx v = mk(0.0, 0.0);
  if (j < n) v = mk(a[j], j == 0 ? 0.0 : -a[n - j]);
  g[j] = v;
}

// F = DIF transform of g (length 2M, bins at plan_pos(q, 2M)).  G[br][pos(k')] = conj(F[2k'+br]) * scale :
// generator spectrum split into even/odd bins in the inverse transform's input order.
// layout 0: pos = plan_pos(k', M), branch stride M (td_fused.cuh, td_staged.cuh).
// layout 1: same order in the padded shared-memory layout (element i at i + i/16, branch stride
//           padded(M)) so that one bulk copy drops it into the fused4 kernel's Z region.
// layout 2: padded, order of the cluster kernel's [32,16,16] inverse plan (td_cluster.cuh).
__global__ void gen_permute_kernel(const cplx* __restrict__ F, cplx* G, int M, double scale, int layout) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * M) return;
  const int br = idx / M, kq = idx - br * M;
  const cplx f = F[plan_pos(2 * kq + br, 2 * M)];
  const int p = layout == 2 ? (((kq & 31) << 8) | (((kq >> 5) & 15) << 4) | (kq >> 9)) : plan_pos(kq, M);
  const size_t dst = layout ? (size_t)br * SmemArr::padded(M) + p + (p >> 4) : (size_t)br * M + p;
  G[dst] = mk(f.x * scale, -f.y * scale);
}

}  // namespace td
