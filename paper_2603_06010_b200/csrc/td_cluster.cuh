// td_cluster.cuh - the fused FFT-path kernel for M = 8192 (segments of 4097..8192 samples, transform
// length 2M = 16384; configs c3 and c5), where one template-segment needs 48 M bytes = 384 KiB of
// spectra and no longer fits one SM's shared memory.
//
// A thread-block CLUSTER of two CTAs evaluates one (template, segment) item:
//   * the length-M forward transform of the packed, half-zero input splits into an even-bin and an
//     odd-bin length-NF transform, and the pruned length-2M inverse into an even-input and an odd-input
//     length-M transform (td_fused.cuh header); the two branches never touch each other's data between
//     the first forward pass and the last inverse pass.  CTA rank 0 owns the even branch, rank 1 the
//     odd branch: per CTA  U = NF complex (64 KiB), Z = M complex (128 KiB), twiddle table 16 KiB.
//   * plans NF = [16,16,16], M = [32,16,16]; forward passes 2-3, "mid" (untangle x generator + first
//     inverse pass in registers) and inverse pass 2 are the warp-local pieces of td_fused4.cuh.
//   * the last pass (radix 32 in registers) ends with z_i = e_i + w_2M^{-i} o_i, which needs both
//     branches: each CTA keeps the half of its outputs that falls in its own half of the index range
//     (rank 0: i < M/2, rank 1: i >= M/2) and stores the other half into the partner's shared memory
//     through distributed shared memory (st.shared::cluster), between two cluster barriers; then each
//     CTA reduces its half of S5.  Rank 1's partial sum travels to rank 0 the same way.
//   * the template row is TMA-bulk-prefetched into the (dead) U region, the branch's generator spectrum
//     into the Z region; d is subtracted on load straight from global memory (L2-resident).
// Only H is read from HBM; nothing but out[b] is written.
#pragma once
#include "td_fused4.cuh"

namespace td {

// ---- cos/sin(2 pi k / 64): the odd branch's output twist w_2M^{-256 t} = conj(w_64)^t -------------
__host__ __device__ constexpr double cos64q(int k) {  // k in [0, 16]
  return k == 0 ? 1.0
       : k == 1 ? 0.99518472667219688624483695310947992
       : k == 2 ? 0.98078528040323044912618223613423904
       : k == 3 ? 0.95694033573220886493579788698026997
       : k == 4 ? 0.92387953251128675612818318939678829
       : k == 5 ? 0.88192126434835502971275686366038835
       : k == 6 ? 0.83146961230254523707878837761790576
       : k == 7 ? 0.7730104533627369608109066097584698
       : k == 8 ? 0.70710678118654752440084436210484904
       : k == 9 ? 0.63439328416364549821517161322549337
       : k == 10 ? 0.55557023301960222474283081394853287
       : k == 11 ? 0.47139673682599764855638762590525438
       : k == 12 ? 0.38268343236508977172845998403039887
       : k == 13 ? 0.29028467725446236763619237581739527
       : k == 14 ? 0.19509032201612826784828486847702224
       : k == 15 ? 0.098017140329560601994195563888641846
                 : 0.0;
}
__host__ __device__ constexpr double cos64(int k) {
  k &= 63;
  return k <= 16 ? cos64q(k) : k <= 32 ? -cos64q(32 - k) : k <= 48 ? -cos64q(k - 32) : cos64q(64 - k);
}
__host__ __device__ constexpr double sin64(int k) { return cos64(k - 16); }
// a * conj(w_64)^K,  w_64 = exp(-2 pi i / 64)
template <int K> __device__ __forceinline__ cplx mul_w64_inv(cplx a) {
  constexpr int k = K & 63;
  if constexpr (k == 0) return a;
  else if constexpr (k == 16) return mk(-a.y, a.x);
  else if constexpr (k == 32) return mk(-a.x, -a.y);
  else if constexpr (k == 48) return mk(a.y, -a.x);
  else {
    constexpr double c = cos64(k), s = sin64(k);
    return mk(fma(a.x, c, -(a.y * s)), fma(a.y, c, a.x * s));
  }
}

// ---- cluster primitives -------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t map_to_cta(uint32_t smem_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void st_cluster(uint32_t addr, cplx v) {
  asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}
// asynchronous remote store that also counts its 16 bytes on the destination CTA's mbarrier: the receiver waits on a
// LOCAL mbarrier for the bytes instead of a cluster-wide barrier round trip
__device__ __forceinline__ void st_async_cluster(uint32_t addr, cplx v, uint32_t mbar) {
  asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(addr), "d"(v.x),
               "d"(v.y), "r"(mbar)
               : "memory");
}

struct ClusterShape {
  static constexpr int LOG2M = 13, M = 1 << LOG2M, NF = M / 2, TW = 2 * M;
  static constexpr int RF1 = 16, RI1 = 32, NT = 256, NW = 8;
  static constexpr int TWS = 2 * M / RF1;  // 1024 base twiddles w_2M^k
  static constexpr int PADM = SmemArr::padded(M), PADNF = SmemArr::padded(NF);
  static constexpr size_t smem_bytes() {
    return sizeof(cplx) * ((size_t)PADNF + (size_t)PADM + TWS) + sizeof(double) * (2 * NW + 2) + 48 + F4_SEGCACHE * sizeof(SegDev);
  }
  // position of bin k in the inverse transform's input order (plan [32,16,16])
  __host__ __device__ static constexpr int pos(int k) { return ((k & 31) << 8) | (((k >> 5) & 15) << 4) | (k >> 9); }
};

template <int MODE>
__global__ void __launch_bounds__(ClusterShape::NT, 1) td_cluster_kernel(const Fused4Params P4) {
  using Sh = ClusterShape;
  constexpr int M = Sh::M, NF = Sh::NF, TW = Sh::TW, NT = Sh::NT, NW = Sh::NW;
  const FusedParams& P = P4.base;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sm = reinterpret_cast<cplx*>(smem_raw);
  const SmemArr U{sm}, Z{sm + Sh::PADNF};
  cplx* tw = sm + Sh::PADNF + Sh::PADM;
  double* red = reinterpret_cast<double*>(tw + Sh::TWS);   // [2 NW] block reduction
  double* xsum = red + 2 * NW;                             // [2] rank 1's partial sums, written remotely (rank 0 only)
  const uint32_t mbar_rows = smem_u32(xsum + 2);
  const uint32_t mbar_g = mbar_rows + 8;
  int* mid_count = reinterpret_cast<int*>(xsum + 4);
  SegDev* segS = reinterpret_cast<SegDev*>(xsum + 6);
  const SegDev* segs = P.n_seg <= F4_SEGCACHE ? segS : P.segs;
  const uint32_t mbar_x = smem_u32(xsum + 5);              // half-results of the partner have landed in xbuf (tx bytes)
  double* stH = reinterpret_cast<double*>(sm);             // staged row (<= M doubles) in the U region
  cplx* xbuf = Z.p;                                        // exchange buffer [16][256] in the Z region
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int br = (int)cluster_ctarank();                   // branch: 0 even bins, 1 odd bins
  const F4Own own = f4_own<Sh::RF1, true>(br, (int)(threadIdx.x >> 5));
  const uint32_t xbuf_remote = map_to_cta(smem_u32(xbuf), (uint32_t)(br ^ 1));
  const uint32_t xsum_remote = map_to_cta(smem_u32(xsum), 0u);
  const uint32_t mbar_x_remote = map_to_cta(mbar_x, (uint32_t)(br ^ 1));
  const long long ncl = gridDim.x >> 1;

  for (int k = tid; k < Sh::TWS; k += NT) tw[k] = P.T[k];
  if (tid < P.n_seg && tid < F4_SEGCACHE) segS[tid] = P.segs[tid];
  if (tid == 0) { mbar_init(mbar_rows, 1); mbar_init(mbar_g, 1); mbar_init(mbar_x, 1); *mid_count = 0; }
  __syncthreads();

  // rows of item (b, s): hrow is the row that gets staged (the template; d itself for STOREZ)
  auto rows = [&](long long b, int s, const double*& drow, const double*& hrow, int& n) -> bool {
    const SegDev sg = segs[s];
    drow = P.d + sg.off;
    hrow = (MODE == MODE_STOREZ) ? drow : P.H + b * P.ldh + sg.off;
    n = sg.n;
    return ((reinterpret_cast<uintptr_t>(hrow) & 15) == 0) && ((n & 1) == 0);
  };
  auto prefetch_rows = [&](long long b, int s) {  // ONE thread
    const double *drow, *hrow; int n;
    if (rows(b, s, drow, hrow, n)) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      const uint32_t bytes = (uint32_t)n * 8u;
      mbar_expect_tx(mbar_rows, bytes);
      bulk_g2s(smem_u32(stH), hrow, bytes, mbar_rows);
    }
  };
  auto prefetch_g = [&](int s) {  // ONE thread
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    constexpr uint32_t bytes = (uint32_t)(Sh::PADM * sizeof(cplx));
    mbar_expect_tx(mbar_g, bytes);
    bulk_g2s(smem_u32(Z.p), P4.Gp[s] + (size_t)br * Sh::PADM, bytes, mbar_g);
  };

  long long b = blockIdx.x >> 1;
  int s = 0;
  bool have = b < P.B;
  uint32_t par_rows = 0, par_g = 0, par_x = 0;
  bool staged = false;
  if (have) {
    const double *dr, *hr; int nn;
    staged = rows(b, s, dr, hr, nn);
    if (tid == 0) { prefetch_rows(b, s); prefetch_g(s); }
  }
  // rank 0, thread 0: running totals of the current template and the item whose partner sum is in flight
  double tot0 = 0.0, tot1 = 0.0, pend0 = 0.0, pend1 = 0.0;
  long long pend_b = 0;
  bool pend = false, pend_last = false;
  auto settle = [&]() {  // rank 0 / thread 0, after a cluster barrier that follows rank 1's remote store
    if (MODE != MODE_STOREZ && pend) {
      tot0 += pend0 + xsum[0];
      tot1 += pend1 + xsum[1];
      if (pend_last) {
        if (MODE == MODE_LOGLIKE) {
          const double v = -0.5 * tot1;
          P.out0[pend_b] = P.accumulate ? P.out0[pend_b] + v : v;
        } else {
          if (P.out0) P.out0[pend_b] = P.accumulate ? P.out0[pend_b] + tot0 : tot0;
          if (P.out1) P.out1[pend_b] = P.accumulate ? P.out1[pend_b] + tot1 : tot1;
        }
        tot0 = 0.0; tot1 = 0.0;
      }
      pend = false;
    }
  };

  while (have) {
    long long nb = b; int ns = s + 1;
    if (ns == P.n_seg) { ns = 0; nb = b + ncl; }
    const bool have_next = (MODE != MODE_STOREZ || nb == b) && nb < P.B;
    const SegDev sg = segs[s];
    // ---------------- forward pass 1 (radix 16, stride 256) of THIS CTA's branch; task j = tid
    {
      const int j = tid;
      const double *drow, *hrow; int n;
      rows(b, s, drow, hrow, n);
      cplx x[16];
      if (staged) {
        double2 dv[16];
        if (MODE == MODE_LOGLIKE) {
          const bool dvec = (reinterpret_cast<uintptr_t>(drow) & 15) == 0;
#pragma unroll
          for (int q = 0; q < 16; ++q) {
            const int i0 = 2 * (j + 256 * q);
            dv[q] = mk(0.0, 0.0);
            if (i0 < n) {  // n even on this path
              if (dvec) dv[q] = __ldg(reinterpret_cast<const double2*>(drow + i0));
              else dv[q] = mk(__ldg(drow + i0), __ldg(drow + i0 + 1));
            }
          }
        }
        mbar_wait(mbar_rows, par_rows);
        par_rows ^= 1;
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          const int i0 = 2 * (j + 256 * q);
          double2 h = mk(0.0, 0.0);
          if (i0 < n) h = *reinterpret_cast<const double2*>(stH + i0);
          x[q] = (MODE == MODE_LOGLIKE) ? mk(dv[q].x - h.x, dv[q].y - h.y) : h;
        }
        __syncthreads();  // staging consumed: the U region may now be overwritten
      } else {
        const bool vec = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
#pragma unroll
        for (int q = 0; q < 16; ++q) x[q] = load_pair<MODE>(drow, hrow, j + 256 * q, n, vec);
      }
      cplx w[16];
      tw_powers<16>(tw[4 * j], w);  // w_NF^j
      if (br) {
        const cplx beta = tw[2 * j];  // w_M^j
        static_for<0, 16>([&](auto q) { x[decltype(q)::value] = mul_w32<decltype(q)::value, false>(x[decltype(q)::value]); });
        static_for<0, 16>([&](auto t) { w[decltype(t)::value] = cmul(w[decltype(t)::value], beta); });
      }
      fft_reg<16, false>(x);
      static_for<0, 16>([&](auto t) {
        constexpr int tt = decltype(t)::value;
        cplx v = x[brevR<16>(tt)];
        if (tt > 0 || br) v = cmul(v, w[tt]);
        U.st(j + 256 * tt, v);
      });
    }
    __syncthreads();
    // ---------------- forward passes 2 and 3, warp-local
    f4_forward23<TW>(U, own, lane, tw);
    __syncwarp();  // mirror-closed ownership (f4_own): mid reads only this warp's U blocks
    // ---------------- mid: untangle x generator (in place in Z) -> first inverse pass
    mbar_wait(mbar_g, par_g);
    par_g ^= 1;
    f4_mid<NF, Sh::RF1>(U, Z, br, own, lane, tw);
    __syncwarp();
    if (lane == 0) {
      const int old = atomicAdd(mid_count, 1);
      if (old == NW - 1) {
        *mid_count = 0;
        if (have_next) prefetch_rows(nb, ns);
      }
    }
    bool staged_next = false;
    if (have_next) { const double *dr, *hr; int nn; staged_next = rows(nb, ns, dr, hr, nn); }
    // ---------------- inverse pass 2 (L = 256), warp-local
    f4_inverse2<TW>(Z, own, lane, tw);
    __syncthreads();
    // ---------------- last inverse pass: radix 32 on this branch, exchange halves, fused S5
    double acc0 = 0.0, acc1 = 0.0;
    {
      const int j = tid;
      cplx x[32];
#pragma unroll
      for (int q = 0; q < 32; ++q) x[q] = Z.ld(j + 256 * q);
      // arm the exchange mbarrier for this item's 16 x 256 complex from the partner, then
      if (tid == 0) mbar_expect_tx(mbar_x, (uint32_t)(16 * NT * sizeof(cplx)));
      cluster_arrive();  // (A) my Z region is free: the partner may write its half-results into it
      {
        // x_q *= conj(w_M^{j q}) (and conj(w_2M^j) on the odd branch); powers as w^{4 hi} * w^{lo}
        cplx lo[4], hi[8];
        tw_powers<4>(tw[2 * j], lo);
        hi[0] = mk(1.0, 0.0);
        hi[1] = csq(lo[2]);
        static_for<2, 8>([&](auto q) {
          constexpr int qq = decltype(q)::value;
          if constexpr ((qq & 1) == 0) hi[qq] = csq(hi[qq / 2]);
          else hi[qq] = cmul(hi[qq - 1], hi[1]);
        });
        if (br) {
          const cplx beta = tw[j];
          static_for<0, 4>([&](auto r) { lo[decltype(r)::value] = cmul(lo[decltype(r)::value], beta); });
        }
        static_for<0, 32>([&](auto q) {
          constexpr int qq = decltype(q)::value;
          if constexpr (qq < 4) {
            if (qq > 0 || br) x[qq] = cmulc(x[qq], lo[qq]);
          } else {
            x[qq] = cmulc(x[qq], cmul(hi[qq >> 2], lo[qq & 3]));
          }
        });
      }
      fft_reg<32, true>(x);
      if (br) static_for<1, 32>([&](auto t) {
        constexpr int tt = decltype(t)::value;
        x[brevR<32>(tt)] = mul_w64_inv<tt>(x[brevR<32>(tt)]);
      });
      cluster_wait();    // (A) done on both sides
      if (br == 0 && tid == 0) settle();  // rank 1's sums of the previous item arrived before its (A)
      // output t -> index i = j + 256 t; t < 16 belongs to rank 0's half, t >= 16 to rank 1's
      if (br == 0) {
        static_for<16, 32>([&](auto t) {
          constexpr int tt = decltype(t)::value;
          st_async_cluster(xbuf_remote + (uint32_t)(((tt - 16) * 256 + j) * sizeof(cplx)), x[brevR<32>(tt)], mbar_x_remote);
        });
      } else {
        static_for<0, 16>([&](auto t) {
          constexpr int tt = decltype(t)::value;
          st_async_cluster(xbuf_remote + (uint32_t)((tt * 256 + j) * sizeof(cplx)), x[brevR<32>(tt)], mbar_x_remote);
        });
      }
      mbar_wait(mbar_x, par_x);  // (B) the partner's half-results have landed (local mbarrier: no cluster barrier)
      par_x ^= 1;
      static_for<0, 16>([&](auto t) {
        constexpr int tt = decltype(t)::value;
        const cplx mine = br ? x[brevR<32>(tt + 16)] : x[brevR<32>(tt)];
        const cplx z = cadd(mine, xbuf[tt * 256 + j]);
        const int i = j + 256 * tt + br * (M / 2);
        if constexpr (MODE == MODE_STOREZ) {
          sg.zd[i] = z;
        } else {
          if (i < sg.n) {
            if constexpr (MODE == MODE_INNER) {
              const cplx q = sg.zd[i];
              acc0 = fma(z.x, q.x, fma(-z.y, q.y, acc0));
            }
            acc1 = fma(z.x, z.x, fma(-z.y, z.y, acc1));
          }
        }
      });
    }
    if (MODE != MODE_STOREZ) {
      acc0 = warp_sum(acc0);
      acc1 = warp_sum(acc1);
      if (lane == 0) { red[2 * warp] = acc0; red[2 * warp + 1] = acc1; }
    }
    __syncthreads();  // exchange buffer (Z region) fully consumed
    if (tid == 0) {
      if (have_next) prefetch_g(ns);
      if (MODE != MODE_STOREZ) {
        double p0 = 0.0, p1 = 0.0;
#pragma unroll
        for (int wq = 0; wq < NW; ++wq) { p0 += red[2 * wq]; p1 += red[2 * wq + 1]; }
        if (br) {
          asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(xsum_remote), "d"(p0), "d"(p1) : "memory");
        } else {
          pend = true; pend0 = p0; pend1 = p1; pend_b = b; pend_last = (s == P.n_seg - 1);
        }
      }
    }
    b = nb; s = ns; have = have_next; staged = staged_next;
  }
  // rank 1's last partial sums become visible with this barrier; no CTA exits while its partner may
  // still store into its shared memory
  cluster_arrive();
  cluster_wait();
  if (br == 0 && tid == 0) settle();
}

}  // namespace td
