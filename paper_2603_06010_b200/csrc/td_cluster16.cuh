// td_cluster16.cuh - the fused FFT path for M = 65536 (segments of 32769..65536 samples, transform length 2M = 131072;
// config c4) kept ON CHIP: a thread-block cluster of 16 CTAs evaluates one (template, segment) item with its 3 MB of
// spectra in distributed shared memory (north_star (3a): the residual is never written back).  The
// staged kernels (td_staged.cuh) move 12.5 MB per template through L2 and run at its bandwidth; here only H is read.
//
// Decomposition (plans NF = M/2 = 32768 = [16 | 8,16,16], M = [16 | 16,16,16], the leading radix-16 pass is the one that
// crosses CTAs):
//   F0  first forward pass, radix 16, stride 2048: CTA c computes it for the inputs j in [128 c, 128 c + 128) of both
//       branches (even / odd bins, td_fused.cuh header) straight from global memory (S1 fused: r = d - h) and scatters
//       output t of branch g to the CTA that owns sub-transform (g, t), with st.async into that CTA's U arrays (bytes
//       counted on the owner's mbarrier).
//   ..  a CTA owns TWO length-2048 sub-transforms of ONE branch, chosen mirror-closed: the untangle of the real-input
//       transform pairs bin k with -k (even branch) or -1-k (odd branch), bins k = t (mod 16) live in sub-transform t,
//       so {E_t, E_16-t} (CTA t, t = 1..7), {E_0, E_8} (CTA 0) and {O_t, O_15-t} (CTA 8 + t) are closed: the local
//       forward passes [8,16,16], "mid" (untangle x generator + first inverse pass, generator values in tensor memory)
//       and the local inverse passes [16,16,16] never leave the CTA; they are the warp-local pieces of td_fused4.cuh on
//       the two arrays seen as one (A || B: the padded layouts concatenate exactly).
//   L0  last inverse pass, radix 16, stride 4096, joined with the pruned radix-2 stage of the two branches and S5: CTA c
//       reduces the outputs i = j + 4096 t for j in [256 c, 256 c + 256).  Every CTA loads its two length-4096 arrays into
//       registers (32 values per thread), a cluster barrier makes all Z regions free, and the values go to their reducers
//       with st.async (Z doubles as the receive buffer: 32 sub-transforms x 256).  The butterflies and the sums of squares of
//       an item are DEFERRED until just before `mid` of the next item overwrites Z, so the exchange overlaps the next
//       item's forward passes.
// Per-CTA partial sums go to a global scratch [B][16][2]; lg_finish_kernel (td_staged.cuh) adds them in rank order.
#pragma once
#include "td_cluster.cuh"

namespace TD_NS {

struct Cluster16Shape {
  static constexpr int CS = 16;                         // CTAs per cluster
  static constexpr int LOG2M = 16, M = 1 << LOG2M, NF = M / 2, TWG = 2 * M;   // global transform, twiddle table T[k] = w_2M^k
  static constexpr int ML = M / CS, NFL = NF / CS;      // local arrays: 4096 (inverse), 2048 (forward)
  static constexpr int TWL = 2 * ML;                    // local twiddles tw[k] = w_8192^k = T[16 k]
  static constexpr int NT = 256, NW = 8, RF1 = 8;       // the local machinery is the one of Fused4Shape<12>
  static constexpr int TWS = TWL / RF1;                 // 1024 local base twiddles
  static constexpr int PADU = SmemArr::padded(2 * NFL), PADZ = SmemArr::padded(2 * ML);   // A || B
  using Cols = F4Cols<16>;                              // TMEM: generator values, 16 data samples, pass-2 twiddles
  static constexpr int TMEM_COLS = 2 * Cols::WINDOW;
  static constexpr size_t smem_bytes() { return sizeof(cplx) * ((size_t)PADU + PADZ + TWS) + 256; }   // + sums, mbarriers, TMEM slot
  static_assert(SmemArr::padded(NFL) * 2 == PADU && SmemArr::padded(ML) * 2 == PADZ, "the padded layouts of A and B concatenate");
};

struct Cluster16Params {
  FusedParams base;       // base.T: the class table w_2M^k (global memory); base.segs[s].zd: z of the data vector [M]
  const cplx* Gp;         // the segment's generator values per CTA: [16][A || B in the padded Z layout] (gen_permute_c16_kernel)
  double* partial;        // [B][16][2] per-CTA partial sums of the launch (slot 0: the quadratic / cross sum, slot 1: <h,h>)
};

// which sub-transforms CTA `c` owns (t of slot A, t of slot B) and its branch
__host__ __device__ inline int c16_branch(int c) { return c >= 8; }
__host__ __device__ inline int c16_sub(int c, int slot) {
  if (c == 0) return slot ? 8 : 0;
  if (c < 8) return slot ? 16 - c : c;
  return slot ? 15 - (c - 8) : c - 8;
}
// owner of sub-transform t of branch g: CTA and slot
__device__ __forceinline__ void c16_owner(int g, int t, int& cta, int& slot) {
  if (g == 0) {
    if (t == 0) { cta = 0; slot = 0; }
    else if (t == 8) { cta = 0; slot = 1; }
    else if (t < 8) { cta = t; slot = 0; }
    else { cta = 16 - t; slot = 1; }
  } else {
    if (t < 8) { cta = 8 + t; slot = 0; }
    else { cta = 8 + (15 - t); slot = 1; }
  }
}

// F = DIF transform of the packed generator (length 2M, bins at plan_pos(q, 2M), td_setup.cuh).  Gc[c][pad(slot * 4096 + p)] =
// conj(F[2 kb + g]) * scale for CTA c (branch g), kb = t_slot + 16 kl the branch bin that sits at position p = pos(kl) of the
// local [16,16,16] inverse plan of sub-transform t_slot.
__global__ void gen_permute_c16_kernel(const cplx* __restrict__ F, cplx* Gc, double scale) {
  constexpr int ML = Cluster16Shape::ML, M = Cluster16Shape::M;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * M) return;
  const int c = idx / (2 * ML), r = idx - c * 2 * ML, slot = r / ML, kl = r - slot * ML;
  const int kb = c16_sub(c, slot) + 16 * kl;
  const cplx f = F[plan_pos(2 * kb + c16_branch(c), 2 * M)];
  const int p = slot * ML + plan_pos(kl, ML);
  Gc[(size_t)c * Cluster16Shape::PADZ + p + (p >> 4)] = mk(f.x * scale, -f.y * scale);
}

// Blocks of 256 elements a warp owns, in the combined arrays U = A || B (blocks 0..7 | 8..15) and Z = ZA || ZB (0..15 | 16..31).
// CTA 0 holds the two self-mirrored sub-transforms (E_0: k <-> -k, E_8: k <-> -1-k): exactly the (even, odd) pair of the
// one-CTA kernel.  Every other CTA holds a cross-mirrored pair: bin k' of A <-> bin 2047 - k' of B.
struct C16Own { F4Own o; int mtype; bool cross; };
__device__ __forceinline__ C16Own c16_own(int cta, int warp) {
  C16Own r;
  if (cta == 0) {
    const int br = warp >> 2, wb = warp & 3;
    const F4Own f = f4_own<8, true>(br, wb);
    const int ub = 8 * br, zb = 16 * br;
    r.o = F4Own{f.u0 + ub, f.u1 + ub, f.z0 + zb, f.z1 + zb, f.z2 + zb, f.z3 + zb};
    r.mtype = br; r.cross = false;
  } else {
    r.o = F4Own{warp, 8 + (7 - warp), warp, 16 + (7 - warp), warp + 8, 16 + (15 - warp)};
    r.mtype = 1; r.cross = true;
  }
  return r;
}

// mid on the combined arrays (f4_mid of td_fused4.cuh with the mirror partner possibly in the other array, the untangle
// twiddle from the global table and the quarter's branch-local block index split from its array)
__device__ __forceinline__ void c16_mid(const SmemArr& U, const SmemArr& Z, const C16Own& own, int lane, cplx basew, uint32_t tg) {
  constexpr int NFL = Cluster16Shape::NFL, RF1 = 8, RI1 = 16;
  const int q4 = lane >> 3;
  const int s1c = q4 == 0 ? own.o.z0 : q4 == 1 ? own.o.z2 : q4 == 2 ? own.o.z1 : own.o.z3, s2 = lane & 7;
  const int side = s1c >> 4, s1 = s1c & 15;
  const int kap = s1 + RI1 * s2;
  int kap2;
  bool selfzero = false;
  if (own.mtype == 0) { kap2 = (NFL / 16 - kap) & (NFL / 16 - 1); selfzero = (kap == 0); }
  else                { kap2 = NFL / 16 - 1 - kap; }
  auto slot = [](int k) { const int a = k & (RF1 - 1), c = k / RF1; return (a * 16 + (c >> 1) + 8 * (c & 1)) * 16; };
  const int mside = own.cross ? side ^ 1 : side;
  const int fb = side * NFL + slot(kap), fb2 = mside * NFL + slot(kap2);
  const int zb0 = (s1c * 16 + s2) * 16;
  cplx ua[8], ub[8], e[16];
  TmemC16 gr;
  auto load_u = [&](auto par) {
    constexpr int pp = decltype(par)::value;
    static_for<0, 8>([&](auto hh) {
      constexpr int t = 2 * decltype(hh)::value + pp;
      ua[decltype(hh)::value] = U.ld(fb + t);
      ub[decltype(hh)::value] = U.ld(fb2 + (selfzero ? ((16 - t) & 15) : (15 - t)));
    });
  };
  auto untangle = [&](auto par) {
    constexpr int pp = decltype(par)::value;
    tmem_wait_ld();
    gr.use();
#pragma unroll
    for (int q = 0; q < 16; ++q) e[q] = gr.get(q);
    static_for<0, 8>([&](auto hh) {
      constexpr int h8 = decltype(hh)::value, t = 2 * h8 + pp;
      const cplx U1 = ua[h8], U2 = ub[h8];
      const cplx A = mk(U1.x + U2.x, U1.y - U2.y);
      const cplx Bv = mk(U1.y + U2.y, -(U1.x - U2.x));
      const cplx wB = cmul(basew, mul_w32<t, false>(Bv));
      e[h8] = cmul(e[h8], cadd(A, wB));
      e[8 + h8] = cmul(e[8 + h8], csub(A, wB));
    });
  };
  auto store_e = [&](auto par) {
    constexpr int pp = decltype(par)::value;
    static_for<0, 16>([&](auto t) { Z.st(zb0 + pp * 8 * 16 + decltype(t)::value, e[brevR<16>(decltype(t)::value)]); });
  };
  gr.ld(tg);
  load_u(IC<0>{});
  untangle(IC<0>{});
  gr.ld(tg + 16 * TM_CPC);
  load_u(IC<1>{});
  dit16<true, false>(e, mk(real(1), real(0)));
  store_e(IC<0>{});
  untangle(IC<1>{});
  dit16<true, false>(e, mk(real(1), real(0)));
  store_e(IC<1>{});
}


// the untangle twiddle w_2M^(2 kq + g) of this lane's first bin kq = t_sub + 16 kap (the other 15 bins of the lane are
// 2048 t further: a factor w_32^t)
__device__ __forceinline__ cplx c16_basew(const C16Own& own, int lane, const cplx* __restrict__ T, int tsubA, int tsubB, int brG) {
  const int q4 = lane >> 3;
  const int s1c = q4 == 0 ? own.o.z0 : q4 == 1 ? own.o.z2 : q4 == 2 ? own.o.z1 : own.o.z3, s2 = lane & 7;
  const int kap = (s1c & 15) + 16 * s2;
  const int tsub = (s1c >> 4) ? tsubB : tsubA;
  return __ldg(T + 2 * (tsub + 16 * kap) + brG);
}

// L0 for output column jl of this CTA (j = 256 rank + jl): radix-16 DIT over the 16 sub-transforms of each branch (received
// in Z: E_s at s * 256 + jl, O_s at 4096 + s * 256 + jl), the pruned radix-2 join and the fused sums (last_pass_c of
// td_fused.cuh with the strides of the distributed layout and the twiddles of the global table)
template <int MODE>
__device__ __forceinline__ void c16_last_regs(cplx (&e)[16], cplx (&o)[16], int j, int n, cplx beta /* w_2M^j */,
                                              cplx w1 /* w_M^(-j) */, cplx* __restrict__ zd, double& acc0, double& acc1) {
  constexpr int ML = Cluster16Shape::ML;
  cplx gm[16];
  dit16<true, true>(e, w1);
  dit16<true, true>(o, w1);
  const cplx cb = cconj(beta);
  static_for<0, 16>([&](auto t) { gm[decltype(t)::value] = mul_w32<decltype(t)::value, true>(cb); });
  real p0[4] = {real(0), real(0), real(0), real(0)}, p1[4] = {real(0), real(0), real(0), real(0)};
  static_for<0, 16>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    const cplx ev = e[brevR<16>(tt)], ov = o[brevR<16>(tt)];
    const cplx z = mk(fma(gm[tt].x, ov.x, fma(-gm[tt].y, ov.y, ev.x)), fma(gm[tt].x, ov.y, fma(gm[tt].y, ov.x, ev.y)));
    const int i = j + tt * ML;
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
template <int MODE>
__device__ __forceinline__ void c16_last(const SmemArr& Z, int jl, int j, int n, cplx beta, cplx w1, cplx* __restrict__ zd,
                                         double& acc0, double& acc1) {
  constexpr int ML = Cluster16Shape::ML;
  cplx e[16], o[16];
#pragma unroll
  for (int ss = 0; ss < 16; ++ss) { e[ss] = Z.ld(ss * 256 + jl); o[ss] = Z.ld(ML + ss * 256 + jl); }
  c16_last_regs<MODE>(e, o, j, n, beta, w1, zd, acc0, acc1);
}


// One segment per launch (P.segs[0]); grid = 16 x (clusters), cluster c takes templates c, c + clusters, ...
template <int MODE>
__global__ void __launch_bounds__(Cluster16Shape::NT, 1) td_cluster16_kernel(const Cluster16Params PC) {
  using Sh = Cluster16Shape;
  constexpr int NT = Sh::NT, NFL = Sh::NFL, ML = Sh::ML, TWL = Sh::TWL;
  const FusedParams& P = PC.base;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sm = reinterpret_cast<cplx*>(smem_raw);
  const SmemArr U{sm}, Z{sm + Sh::PADU};          // U = A || B (2 x 2048), Z = ZA || ZB (2 x 4096)
  cplx* tw = sm + Sh::PADU + Sh::PADZ;             // w_8192^k, k < 1024
  double* red = reinterpret_cast<double*>(tw + Sh::TWS);   // [2 NW] per-warp partial sums
  const uint32_t mbar_u = smem_u32(red + 2 * Sh::NW);      // the scattered first-pass outputs of an item have landed
  const uint32_t mbar_z = mbar_u + 8;                      // the sub-transform columns this CTA reduces have landed
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(red + 2 * Sh::NW + 2);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int rank = (int)cluster_ctarank();
  const int brG = c16_branch(rank), tsubA = c16_sub(rank, 0), tsubB = c16_sub(rank, 1);
  const C16Own own = c16_own(rank, warp);
  const long long ncl = gridDim.x / Sh::CS, cl = blockIdx.x / Sh::CS;
  const cplx* __restrict__ T = P.T;
  const SegDev sg = P.segs[0];

  for (int k = tid; k < Sh::TWS; k += NT) tw[k] = T[16 * k];
  if (tid == 0) { mbar_init(mbar_u, 1); mbar_init(mbar_z, 1); }
  if (warp == 0) tmem_alloc<Sh::TMEM_COLS>(smem_u32(tmem_slot));
  tmem_fence_before();
  __syncthreads();
  tmem_fence_after();
  const uint32_t tcol = *tmem_slot + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * Sh::Cols::WINDOW);
  f4_store_twiddles<TWL>(lane, tw, tcol + Sh::Cols::TW);
  f4_store_generator(PC.Gp + (size_t)rank * Sh::PADZ, own.o, lane, tcol + F4_TC_G);
  tmem_wait_st();
  const cplx basew = c16_basew(own, lane, T, tsubA, tsubB, brG);
  // per-thread constants of the two cross passes (the thread's input column j0 of F0 and output column jr of L0 never change)
  const int g0 = tid >> 7, j0 = 128 * rank + (tid & 127), jr = 256 * rank + tid;
  const cplx f0_w1 = __ldg(T + 4 * j0);            // w_NF^j0
  const cplx f0_beta = __ldg(T + 2 * j0);          // w_M^j0: the odd branch's input twist (its 2048 q part is w_32^q)
  const cplx l0_beta = __ldg(T + jr);              // w_2M^jr
  const cplx l0_w1 = cconj(__ldg(T + 2 * jr));     // w_M^(-jr)
  if (MODE == MODE_LOGLIKE) {                      // this thread's 16 sample pairs of the data vector, once per launch
    const double* drow = P.d + sg.off;
    double2 dvs[16];
#pragma unroll
    for (int q = 0; q < 16; ++q) {
      const int i0 = 2 * (j0 + NFL * q);
      dvs[q] = make_double2(i0 < sg.n ? __ldg(drow + i0) : 0.0, i0 + 1 < sg.n ? __ldg(drow + i0 + 1) : 0.0);
    }
#pragma unroll
    for (int q = 0; q < 16; ++q) tmem_st_c64(tcol + F4_TC_D + 4 * q, dvs[q]);
    tmem_wait_st();
  }
  const uint32_t u_base = smem_u32(U.p), z_base = smem_u32(Z.p);
  // every CTA's mbarriers exist before any partner's st.async can name them
  cluster_arrive();
  cluster_wait();

  const long long Bs = (MODE == MODE_STOREZ) ? 1 : P.B;
  uint32_t par_u = 0, par_z = 0;
  long long prev_b = -1;
  // S5 of the previous item: this CTA's 256 output columns, then its partial sums to the global scratch
  auto reduce_prev = [&]() {
    mbar_wait(mbar_z, par_z);
    par_z ^= 1;
    double acc0 = 0.0, acc1 = 0.0;
    c16_last<MODE>(Z, tid, jr, sg.n, l0_beta, l0_w1, sg.zd, acc0, acc1);
    if (MODE != MODE_STOREZ) {
      if (MODE == MODE_INNER) acc0 = warp_sum(acc0);
      acc1 = warp_sum(acc1);
      if (lane == 0) { red[2 * warp] = acc0; red[2 * warp + 1] = acc1; }
    }
    __syncthreads();   // Z is free for mid; the per-warp sums are visible
    if (MODE != MODE_STOREZ && tid == 0) {
      double t0 = 0.0, t1 = 0.0;
#pragma unroll
      for (int w = 0; w < Sh::NW; ++w) { t0 += red[2 * w]; t1 += red[2 * w + 1]; }
      double* dst = PC.partial + ((size_t)prev_b * Sh::CS + rank) * 2;
      dst[0] = (MODE == MODE_LOGLIKE) ? t1 : t0;
      dst[1] = t1;
    }
  };

  if (tid == 0 && cl < Bs) mbar_expect_tx(mbar_u, (uint32_t)(2 * NFL * sizeof(cplx)));
  for (long long b = cl; b < Bs; b += ncl) {
    // ---------------- F0: first forward pass (radix 16, stride 2048) for input column j0, branch g0
    {
      const double* drow = P.d + sg.off;
      const double* hrow = (MODE == MODE_STOREZ) ? drow : P.H + b * P.ldh + sg.off;
      const bool vec = ((reinterpret_cast<uintptr_t>(hrow) & 15) == 0) && ((sg.n & 1) == 0);
      cplx x[16], w[16];
      if (vec) {
        int dr[4][16];
        if (MODE == MODE_LOGLIKE) {
#pragma unroll
          for (int g = 0; g < 4; ++g) tmem_ld16(tcol + F4_TC_D + 16 * g, dr[g]);
        }
        double2 hs[16];   // all 16 loads in flight together (n even, rows 16-byte aligned: a pair is in or out as a whole)
#pragma unroll
        for (int q = 0; q < 16; ++q) {
          const int i0 = 2 * (j0 + NFL * q);
          hs[q] = i0 < sg.n ? __ldg(reinterpret_cast<const double2*>(hrow + i0)) : make_double2(0.0, 0.0);
        }
        if (MODE == MODE_LOGLIKE) {
          tmem_wait_ld();
#pragma unroll
          for (int g = 0; g < 4; ++g) tmem_use16(dr[g]);
#pragma unroll
          for (int q = 0; q < 16; ++q) {
            const double2 dv = tmem_c64(dr[q >> 2], q & 3);
            x[q] = to_cplx(dv.x - hs[q].x, dv.y - hs[q].y, sg.rscale);   // S1: r = d - h
          }
        } else {
#pragma unroll
          for (int q = 0; q < 16; ++q) x[q] = to_cplx(hs[q].x, hs[q].y, sg.rscale);
        }
      } else {
        const bool v2 = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
#pragma unroll
        for (int q = 0; q < 16; ++q) x[q] = load_pair<MODE>(drow, hrow, j0 + NFL * q, sg.n, v2, sg.rscale);
      }
      // the next item's row pieces on their way into L2 while this item computes
      if (b + ncl < Bs && MODE != MODE_STOREZ && (tid & 127) == 0 && g0 == 0) {
        const double* nrow = P.H + (b + ncl) * P.ldh + sg.off;
#pragma unroll 1
        for (int q = 0; q < 16; ++q) {
          const long long i0 = 2ll * (128 * rank + NFL * q);
          if (i0 < sg.n) {
            const long long nbytes = (sg.n - i0 < 256 ? sg.n - i0 : 256) * 8;
            const double* src = nrow + i0;
            if ((reinterpret_cast<uintptr_t>(src) & 15) == 0 && (nbytes & 15) == 0)
              asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"((uint32_t)nbytes) : "memory");
          }
        }
      }
      tw_powers<16>(f0_w1, w);
      if (g0) {
        static_for<0, 16>([&](auto q) { x[decltype(q)::value] = mul_w32<decltype(q)::value, false>(x[decltype(q)::value]); });
        static_for<0, 16>([&](auto t) { w[decltype(t)::value] = cmul(w[decltype(t)::value], f0_beta); });
      }
      fft_reg<16, false>(x);
      static_for<0, 16>([&](auto t) {
        constexpr int tt = decltype(t)::value;
        cplx v = x[brevR<16>(tt)];
        if (tt > 0 || g0) v = cmul(v, w[tt]);
        int cta, slot;
        c16_owner(g0, tt, cta, slot);
        const int i = slot * NFL + j0;
        st_async_cluster(map_to_cta(u_base, (uint32_t)cta) + (uint32_t)((i + (i >> 4)) * sizeof(cplx)), v,
                         map_to_cta(mbar_u, (uint32_t)cta));
      });
    }
    // S5 of the previous item while this item's first-pass outputs travel (it reads Z only; its barrier also orders it
    // before mid writes Z)
    if (prev_b >= 0) reduce_prev();
    mbar_wait(mbar_u, par_u);
    par_u ^= 1;
    // ---------------- local forward passes [8,16,16] on A and B
#pragma unroll 1
    for (int g = tid; g < 2 * NFL / 8; g += NT) {
      cplx w8[8];
      tw_powers<8>(tw[4 * (g & 255)], w8);   // w_2048^j
      dif_task_c<8, NFL>(U, g, w8);
    }
    __syncthreads();
    f4_forward23<TWL, true>(U, own.o, lane, tw, tcol + Sh::Cols::TW);
    __syncwarp();
    // ---------------- mid, inverse pass 2 (warp-local), inverse pass 3 (L = 4096, CTA-wide)
    c16_mid(U, Z, own, lane, basew, tcol + F4_TC_G);
    __syncwarp();
    f4_inverse2<TWL>(Z, own.o, lane, tw);
    __syncthreads();
#pragma unroll 1
    for (int g = tid; g < 2 * ML / 16; g += NT) {
      cplx x[16];
      const int blk = g >> 8, jj = g & 255, base = blk * ML + jj;
#pragma unroll
      for (int q = 0; q < 16; ++q) x[q] = Z.ld(base + 256 * q);
      dit16<true, true>(x, cconj(tw[2 * jj]));   // w_4096^(-jj)
      static_for<0, 16>([&](auto t) { Z.st(base + 256 * decltype(t)::value, x[brevR<16>(decltype(t)::value)]); });
    }
    __syncthreads();
    // ---------------- L0, first half: this CTA's two arrays to the 16 reducers
    {
      cplx xa[16], xb[16];
#pragma unroll
      for (int c = 0; c < 16; ++c) { xa[c] = Z.ld(tid + 256 * c); xb[c] = Z.ld(ML + tid + 256 * c); }
      if (tid == 0) {
        mbar_expect_tx(mbar_z, (uint32_t)(2 * ML * sizeof(cplx)));
        if (b + ncl < Bs) mbar_expect_tx(mbar_u, (uint32_t)(2 * NFL * sizeof(cplx)));
      }
      // (A) every CTA of the cluster has read its Z into registers and is past mid: all Z and U regions are free.  A relaxed
      // arrive suffices for this write-after-read hazard once the loads have returned: a register move per value makes the
      // warp wait for them (the release form costs a cluster-scope membar in every warp, td_cluster.cuh)
#pragma unroll
      for (int c = 0; c < 16; ++c) {
        asm volatile("mov.b64 %0, %0;" : "+d"(xa[c].x));
        asm volatile("mov.b64 %0, %0;" : "+d"(xb[c].x));
      }
      cluster_arrive_relaxed();
      cluster_wait();
      const int ia = (16 * brG + tsubA) * 256 + tid, ib = (16 * brG + tsubB) * 256 + tid;
      const uint32_t offa = (uint32_t)((ia + (ia >> 4)) * sizeof(cplx)), offb = (uint32_t)((ib + (ib >> 4)) * sizeof(cplx));
#pragma unroll
      for (int c = 0; c < 16; ++c) {
        const uint32_t zc = map_to_cta(z_base, (uint32_t)c), mc = map_to_cta(mbar_z, (uint32_t)c);
        st_async_cluster(zc + offa, xa[c], mc);
        st_async_cluster(zc + offb, xb[c], mc);
      }
    }
    prev_b = b;
  }
  if (prev_b >= 0) reduce_prev();
  // no CTA exits while a partner may still address its shared memory
  cluster_arrive();
  cluster_wait();
  __syncthreads();
  if (warp == 0) tmem_dealloc<Sh::TMEM_COLS>(*tmem_slot);
}

}  // namespace TD_NS
