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
//   * generator values, data samples and pass-2 twiddles of every thread live in tensor memory (td_fused4.cuh), so the
//     Z region carries nothing between the last pass of one item and mid of the next.  That makes the exchange of the
//     last pass ASYNCHRONOUS: z_i = e_i + w_2M^{-i} o_i needs both branches, each CTA keeps the outputs of its own half
//     of the index range (rank 0: i < M/2, rank 1: i >= M/2).  A thread writes its own half into its warp's Z blocks,
//     sends the other half into the partner warp's Z blocks with st.async (distributed shared memory, bytes counted
//     on the receiver's mbarrier) and goes straight on to the next item's forward passes; the sum of squares of the
//     previous item (S5) is taken just before mid overwrites those blocks - by then the partner's half has long arrived
//     (r01: a quarter of the warp samples sat in this exchange).  The layout is warp-closed: a warp reads back only the
//     blocks it overwrites itself, so the deferred S5 needs no CTA barrier.
//   * the template row is TMA-bulk-prefetched into the (dead) U region.
// Only H is read from HBM; nothing but out[b] is written.
#pragma once
#include "td_fused4.cuh"

namespace TD_NS {

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
    constexpr real c = (real)cos64(k), s = (real)sin64(k);
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
__device__ __forceinline__ void cluster_arrive_relaxed() { asm volatile("barrier.cluster.arrive.relaxed.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }
__device__ __forceinline__ uint32_t map_to_cta(uint32_t smem_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void st_cluster(uint32_t addr, cplx v) {
#ifdef TD_F32
  asm volatile("st.shared::cluster.v2.f32 [%0], {%1, %2};" ::"r"(addr), "f"(v.x), "f"(v.y) : "memory");
#else
  asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
#endif
}
// asynchronous remote store that also counts its 16 bytes on the destination CTA's mbarrier: the receiver waits on a
// LOCAL mbarrier for the bytes instead of a cluster-wide barrier round trip
__device__ __forceinline__ void st_async_cluster(uint32_t addr, cplx v, uint32_t mbar) {
#ifdef TD_F32
  asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];" ::"r"(addr), "f"(v.x),
               "f"(v.y), "r"(mbar)
               : "memory");
#else
  asm volatile("st.async.shared::cluster.mbarrier::complete_tx::bytes.v2.f64 [%0], {%1, %2}, [%3];" ::"r"(addr), "d"(v.x),
               "d"(v.y), "r"(mbar)
               : "memory");
#endif
}

struct ClusterShape {
  static constexpr int LOG2M = 13, M = 1 << LOG2M, NF = M / 2, TW = 2 * M;
  static constexpr int RF1 = 16, RI1 = 32, NT = 256, NW = 8;
  static constexpr int TWS = 2 * M / RF1;  // 1024 base twiddles w_2M^k
  using Cols = F4Cols<16>;                 // TMEM window of a thread (256 columns in both precisions)
  static constexpr int TMEM_COLS = 2 * Cols::WINDOW;
  static constexpr int PADM = SmemArr::padded(M), PADNF = SmemArr::padded(NF);
  // the staged template row (<= M doubles) lands in the dead U region in fp64; the fp32 U region (8-byte elements) is too
  // small for a row of doubles, so the fp32 build has a staging region of its own
  static constexpr size_t STAGE_BYTES = F32 ? sizeof(double) * M : 0;
  static constexpr size_t smem_bytes() {
    return sizeof(cplx) * ((size_t)PADNF + (size_t)PADM + TWS) + STAGE_BYTES + sizeof(double) * (4 * NW + 2) + 48 + 64 +
           F4_SEGCACHE * sizeof(SegDev);
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
  double* stage = reinterpret_cast<double*>(tw + Sh::TWS);  // fp32 build only (STAGE_BYTES)
  double* red = stage + Sh::STAGE_BYTES / sizeof(double);   // [2][2 NW] per-warp partial sums, double-buffered by item parity
  double* xsum = red + 4 * NW;                             // [2] rank 1's partial sums, written remotely (rank 0 only)
  const uint32_t mbar_rows = smem_u32(xsum + 2);
  const uint32_t mbar_x = mbar_rows + 8;                   // the partner's half-results have landed (tx bytes)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(xsum + 4);
  // thread 0's bookkeeping of the deferred reduction lives in shared memory (registers are what this kernel is short of)
  struct Book { double pend0, pend1; long long pend_b, prev_b; int pend_add, prev_add; };
  Book* bk = reinterpret_cast<Book*>(xsum + 6);
  SegDev* segS = reinterpret_cast<SegDev*>(xsum + 14);
  const SegDev* segs = P.n_seg <= F4_SEGCACHE ? segS : P.segs;
  double* stH = F32 ? stage : reinterpret_cast<double*>(sm);  // staged row (<= M doubles): the U region in fp64
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int br = (int)cluster_ctarank();                   // branch: 0 even bins, 1 odd bins
  const F4Own own = f4_own<Sh::RF1, true>(br, warp);
  const F4Own pown = f4_own<Sh::RF1, true>(br ^ 1, warp);  // the partner warp's blocks (same warp index, other CTA)
  const uint32_t z_remote = map_to_cta(smem_u32(Z.p), (uint32_t)(br ^ 1));
  const uint32_t xsum_remote = map_to_cta(smem_u32(xsum), 0u);
  const uint32_t mbar_x_remote = map_to_cta(mbar_x, (uint32_t)(br ^ 1));
  const long long ncl = gridDim.x >> 1, cl = blockIdx.x >> 1;
  // half-result t (0..15) of this lane: element (t & 7) * 32 + lane of the warp's block [t >> 3]
  auto hslot = [&](int blk, int t) { const int i = blk * 256 + (t & 7) * 32 + lane; return i + (i >> 4); };

  for (int k = tid; k < Sh::TWS; k += NT) tw[k] = P.T[k];
  if (tid < P.n_seg && tid < F4_SEGCACHE) segS[tid] = P.segs[tid];
  if (tid == 0) { mbar_init(mbar_rows, 1); mbar_init(mbar_x, 1); bk->pend_b = -1; bk->prev_b = -1; }
  if (warp == 0) tmem_alloc<Sh::TMEM_COLS>(smem_u32(tmem_slot));
  tmem_fence_before();
  __syncthreads();
  tmem_fence_after();
  const uint32_t tcol = *tmem_slot + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * Sh::Cols::WINDOW);
  f4_store_twiddles<TW>(lane, tw, tcol + Sh::Cols::TW);

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

  const long long Bs = (MODE == MODE_STOREZ) ? 1 : P.B;
  const bool active = cl < Bs;   // (always: the grid is min(B, clusters); an idle cluster still takes part in the barriers below)
  uint32_t par_rows = 0, par_x = 0;
  bool staged = false;
  if (active) {
    const double *dr, *hr; int nn;
    staged = rows(cl, 0, dr, hr, nn);
    if (tid == 0) prefetch_rows(cl, 0);
  }
  // bookkeeping of the deferred reduction: `prev_*` = the item whose half-results sit in Z; rank 0 / thread 0 also keeps
  // the item whose CTA sums are complete but whose partner sums are still on their way (`pend_*`)
  int item = 0, prev_n = 0;
  cplx* prev_zd = nullptr;
  // S5 of the previous item: this half of z = e + w o from the warp's own Z blocks, squares summed per warp
  auto s5_deferred = [&]() {
    mbar_wait(mbar_x, par_x);
    par_x ^= 1;
    real p0[2] = {real(0), real(0)}, p1[2] = {real(0), real(0)};
    static_for<0, 16>([&](auto t) {
      constexpr int tt = decltype(t)::value;
      const cplx a = Z.p[hslot(tt < 8 ? own.z0 : own.z1, tt)], bq = Z.p[hslot(tt < 8 ? own.z2 : own.z3, tt)];
      const cplx z = cadd(a, bq);
      const int i = tid + 256 * tt + br * (M / 2);
      if constexpr (MODE == MODE_STOREZ) {
        prev_zd[i] = z;
      } else {
        if (i < prev_n) {
          if constexpr (MODE == MODE_INNER) {
            const cplx q = prev_zd[i];
            p0[tt & 1] = fma(z.x, q.x, fma(-z.y, q.y, p0[tt & 1]));
          }
          p1[tt & 1] = fma(z.x, z.x, fma(-z.y, z.y, p1[tt & 1]));
        }
      }
    });
    if (MODE != MODE_STOREZ) {
      double acc0 = 0.0, acc1 = warp_sum((double)(p1[0] + p1[1]));
      if (MODE == MODE_INNER) acc0 = warp_sum((double)(p0[0] + p0[1]));
      if (lane == 0) { double* r = red + 2 * NW * ((item & 1) ^ 1); r[2 * warp] = acc0; r[2 * warp + 1] = acc1; }
    }
  };
  // thread 0, after a CTA barrier that follows s5_deferred: this CTA's sums of the previous item, fixed order over the warps
  auto cta_sums = [&]() {
    if (MODE == MODE_STOREZ || bk->prev_b < 0) return;
    const double* r = red + 2 * NW * ((item & 1) ^ 1);
    double p0 = 0.0, p1 = 0.0;
#pragma unroll
    for (int wq = 0; wq < NW; ++wq) { p0 += r[2 * wq]; p1 += r[2 * wq + 1]; }
    if (br) {
      asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(xsum_remote), "d"(p0), "d"(p1) : "memory");
      asm volatile("fence.acq_rel.cluster;" ::: "memory");   // releases the sums ahead of this thread's relaxed arrive (A)
    } else {
      bk->pend0 = p0; bk->pend1 = p1; bk->pend_b = bk->prev_b; bk->pend_add = bk->prev_add;
    }
    bk->prev_b = -1;
  };
  auto settle = [&]() {  // rank 0 / thread 0, after a cluster barrier that follows rank 1's remote store
    if (MODE != MODE_STOREZ && bk->pend_b >= 0) {
      const double t0 = bk->pend0 + xsum[0], t1 = bk->pend1 + xsum[1];
      const long long pend_b = bk->pend_b;
      const int pend_add = bk->pend_add;
      if (MODE == MODE_LOGLIKE) {
        const double v = -0.5 * t1;
        P.out0[pend_b] = pend_add ? P.out0[pend_b] + v : v;
      } else {
        if (P.out0) P.out0[pend_b] = pend_add ? P.out0[pend_b] + t0 : t0;
        if (P.out1) P.out1[pend_b] = pend_add ? P.out1[pend_b] + t1 : t1;
      }
      bk->pend_b = -1;
    }
  };

  for (int s = 0; active && s < P.n_seg; ++s) {
    const SegDev sg = segs[s];
    // ---------------- per-segment constants into this thread's TMEM columns
    f4_store_generator(P4.Gp[s] + (size_t)br * Sh::PADM, own, lane, tcol + F4_TC_G);
    if (MODE == MODE_LOGLIKE) {
      const double* drow = P.d + sg.off;
      double2 dvs[16];   // loads first, (volatile) TMEM stores after: the latencies overlap
#pragma unroll
      for (int q = 0; q < 16; ++q) {
        const int i0 = 2 * (tid + 256 * q);
        dvs[q] = make_double2(i0 < sg.n ? __ldg(drow + i0) : 0.0, i0 + 1 < sg.n ? __ldg(drow + i0 + 1) : 0.0);
      }
#pragma unroll
      for (int q = 0; q < 16; ++q) tmem_st_c64(tcol + F4_TC_D + 4 * q, dvs[q]);
    }
    tmem_wait_st();
    for (long long b = cl; b < Bs; b += ncl) {
      long long nb = b + ncl; int ns = s;
      if (nb >= Bs) { nb = cl; ns = s + 1; }
      const bool have_next = ns < P.n_seg;
      // ---------------- forward pass 1 (radix 16, stride 256) of THIS CTA's branch; task j = tid
      {
        const int j = tid;
        cplx x[16];
        if (staged) {
          int dr[4][16];
          if (MODE == MODE_LOGLIKE) {
#pragma unroll
            for (int g = 0; g < 4; ++g) tmem_ld16(tcol + F4_TC_D + 16 * g, dr[g]);
          }
          mbar_wait(mbar_rows, par_rows);
          par_rows ^= 1;
          double2 hs[16];   // the staged samples, fp64 in both precisions
#pragma unroll
          for (int q = 0; q < 16; ++q) {
            const int i0 = 2 * (j + 256 * q);
            double2 h = make_double2(0.0, 0.0);
            if (i0 < sg.n) h = *reinterpret_cast<const double2*>(stH + i0);  // n even on this path
            hs[q] = h;
          }
          if (MODE == MODE_LOGLIKE) {
            tmem_wait_ld();
#pragma unroll
            for (int g = 0; g < 4; ++g) tmem_use16(dr[g]);
#pragma unroll
            for (int q = 0; q < 16; ++q) {
              const double2 dv = tmem_c64(dr[q >> 2], q & 3);
              // S1: r = d - h in fp64 (the fp32 build scales by rscale and rounds once; h = d stays exactly 0)
              x[q] = to_cplx(dv.x - hs[q].x, dv.y - hs[q].y, sg.rscale);
            }
          } else {
#pragma unroll
            for (int q = 0; q < 16; ++q) x[q] = to_cplx(hs[q].x, hs[q].y, sg.rscale);
          }
          __syncthreads();  // staging consumed: the U region may now be overwritten
        } else {
          const double *drow, *hrow; int n;
          rows(b, s, drow, hrow, n);
          const bool vec = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
#pragma unroll
          for (int q = 0; q < 16; ++q) x[q] = load_pair<MODE>(drow, hrow, j + 256 * q, n, vec, sg.rscale);
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
      f4_forward23<TW, true>(U, own, lane, tw, tcol + Sh::Cols::TW);
      __syncwarp();  // mirror-closed ownership (f4_own): mid reads only this warp's U blocks
      // ---------------- S5 of the PREVIOUS item, from the Z blocks this warp is about to overwrite
      if (item > 0) s5_deferred();
      __syncwarp();
      // ---------------- mid: untangle x generator (TMEM) -> first inverse pass -> Z
      f4_mid<NF, Sh::RF1, true>(U, Z, br, own, lane, tw, tcol + F4_TC_G);
      __syncwarp();
      bool staged_next = false;
      if (have_next) { const double *dr, *hr; int nn; staged_next = rows(nb, ns, dr, hr, nn); }
      // ---------------- inverse pass 2 (L = 256), warp-local
      f4_inverse2<TW>(Z, own, lane, tw);
      __syncthreads();
      if (tid == 0) {
        if (have_next) prefetch_rows(nb, ns);  // every warp is past mid: the U region is dead
        cta_sums();                            // every warp is past the previous item's S5
      }
      // ---------------- last inverse pass: radix 32 on this branch; halves to their owners
      {
        const int j = tid;
        cplx x[32];
#pragma unroll
        for (int q = 0; q < 32; ++q) x[q] = Z.ld(j + 256 * q);
        // arm the exchange mbarrier for this item's 16 x 256 complex from the partner, then
        if (tid == 0) mbar_expect_tx(mbar_x, (uint32_t)(16 * NT * sizeof(cplx)));
        {
          // x_q *= conj(w_M^{j q}) (and conj(w_2M^j) on the odd branch); powers as w^{4 hi} * w^{lo}
          cplx lo[4], hi[8];
          tw_powers<4>(tw[2 * j], lo);
          hi[0] = mk(real(1), real(0));
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
              x[qq] = cmulc(x[qq], lo[qq]);   // (also q = 0 on the even branch, a product with 1: every loaded value is consumed here)
            } else {
              x[qq] = cmulc(x[qq], cmul(hi[qq >> 2], lo[qq & 3]));
            }
          });
        }
        // (A) "this CTA has read its Z values: the region may be overwritten".  Placed after the twiddle products: every value
        // read from Z has been consumed by an instruction issued before the arrive (in-order issue), so a RELAXED arrive is enough
        // for this write-after-read hazard; the one datum that crosses with the barrier, rank 1's partial sums, is released by a
        // fence of the thread that stored it (cta_sums).  r02: barrier.cluster.arrive.release made every warp execute a
        // cluster-scope membar per item - 4.3 % of the warp samples, 13 % of the kernel time (c5 1.95 -> 2.20 M evals/s).
        cluster_arrive_relaxed();
        fft_reg<32, true>(x);
        if (br) static_for<1, 32>([&](auto t) {
          constexpr int tt = decltype(t)::value;
          x[brevR<32>(tt)] = mul_w64_inv<tt>(x[brevR<32>(tt)]);
        });
        cluster_wait();    // (A) on both sides
        if (br == 0 && tid == 0) settle();  // rank 1 stored the sums of the item before the previous one ahead of its (A)
        // output t -> index i = j + 256 t; t < 16 belongs to rank 0's half, t >= 16 to rank 1's.  Own half: this warp's
        // blocks z0, z1; the other half: the partner warp's blocks z2, z3 (asynchronous, counted on its mbarrier).
        static_for<0, 16>([&](auto t) {
          constexpr int tt = decltype(t)::value;
          const cplx mine = br ? x[brevR<32>(tt + 16)] : x[brevR<32>(tt)];
          const cplx theirs = br ? x[brevR<32>(tt)] : x[brevR<32>(tt + 16)];
          Z.p[hslot(tt < 8 ? own.z0 : own.z1, tt)] = mine;
          st_async_cluster(z_remote + (uint32_t)(hslot(tt < 8 ? pown.z2 : pown.z3, tt) * sizeof(cplx)), theirs, mbar_x_remote);
        });
      }
      prev_n = sg.n; prev_zd = sg.zd;
      if (tid == 0) { bk->prev_b = b; bk->prev_add = (P.accumulate || s > 0) ? 1 : 0; }
      ++item;
      staged = staged_next;
    }
  }
  // ---------------- the last item's S5, then the sums travel: CTA -> rank 0 -> out
  if (item > 0) s5_deferred();
  __syncthreads();
  if (tid == 0) {
    // rank 0 may still hold an item whose partner sums arrived with the last (A): there is none - settle() ran after it
    cta_sums();
  }
  // rank 1's last partial sums become visible with this barrier; no CTA exits while its partner may
  // still store into its shared memory
  cluster_arrive();
  cluster_wait();
  if (br == 0 && tid == 0) settle();
  __syncthreads();
  if (warp == 0) tmem_dealloc<Sh::TMEM_COLS>(*tmem_slot);
}

}  // namespace TD_NS
