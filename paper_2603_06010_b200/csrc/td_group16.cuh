// td_group16.cuh - the fused FFT path for M = 16384, 32768, 65536 (segments of 8193..65536 samples; config c4 is the last) as ONE
// persistent kernel whose CTAs work in groups of CS = M / 4096 = 4, 8 or 16 and exchange through L2.  The decomposition, the
// mirror-closed ownership of sub-transforms and every CTA-local pass are those of td_cluster16.cuh (written there for CS = 16);
// what differs is how the two cross passes travel, and that the cross radix is CS.
//
//   td_cluster16_kernel  F0 / L0 outputs go to the owner / reducer CTA with st.async into distributed shared memory: 16 bytes
//                        per cycle and SM, producer pays, and a 16-CTA cluster is co-resident 7 times (112 of 148 SMs).
//   td_group_kernel      F0 writes its outputs to a global exchange buffer U[group][parity] (plain coalesced 16-byte stores),
//                        the owner's first local pass (radix 8, L = 2048) reads its inputs from there instead of shared
//                        memory; the last local pass (radix 16, L = 4096) writes its outputs to Z[group][parity], and L0 reads
//                        its 32 values per thread from there.  groups x 2 parities x 48 M bytes = 54 MB, written and read once
//                        per item: it stays in the 126 MB L2.  No cluster: 37 / 18 / 9 groups = 148 / 144 / 144 of 148 SMs, and
//                        the two barriers of an item are arrival counters in global memory (CS arrivals each), the second one
//                        waited for only after the NEXT item's first pass (S5 of an item is deferred as in the cluster kernel).
//
// Plans: NF = M/2 = [CS | 8,16,16], M = [CS | 16,16,16]; the leading radix-CS pass of each direction crosses CTAs.  CTA c of a
// group owns two length-2048 (forward) / length-4096 (inverse) sub-transforms of one branch: {E_0, E_CS/2} (c = 0),
// {E_c, E_CS-c} (0 < c < CS/2), {O_t, O_CS-1-t} (c = CS/2 + t): closed under the untangle's k <-> -k / k <-> -1-k pairing.
// A thread does 16 / CS radix-CS butterflies in each cross pass (16 values in, 16 out, whatever CS).
//
// The staged kernels (td_staged.cuh) move ~12 MB per template through L2 at M = 65536 in 5 kernels per chunk; this kernel moves
// 6.5 MB in one launch per segment, with generator values, data samples and twiddles in tensor memory.
// The launch is cooperative (all CTAs co-resident, or the launch fails); a wait that does not end within ~10 s traps.
#pragma once
#include "td_cluster16.cuh"

namespace TD_NS {

template <int CS_>
struct GroupShape {
  static constexpr int CS = CS_, TPT = 16 / CS;                 // CTAs per group; cross-pass butterflies per thread
  static constexpr int ML = Cluster16Shape::ML, NFL = Cluster16Shape::NFL;   // local arrays: 4096 (inverse), 2048 (forward)
  static constexpr int M = ML * CS, NF = NFL * CS, LOG2M = ilog2(M);
  static_assert(CS == 4 || CS == 8 || CS == 16, "groups of 4, 8 or 16 CTAs");
};
// CTAs per group of a size class (0: the class is not served by this kernel)
__host__ __device__ constexpr int group_cs(int log2M) { return log2M >= 14 && log2M <= 16 ? 1 << (log2M - 12) : 0; }

// which sub-transforms CTA `c` of a group of `cs` owns (slot 0: array A, slot 1: array B) and its branch
__host__ __device__ inline int grp_branch(int cs, int c) { return c >= cs / 2; }
__host__ __device__ inline int grp_sub(int cs, int c, int slot) {
  if (c == 0) return slot ? cs / 2 : 0;
  if (c < cs / 2) return slot ? cs - c : c;
  return slot ? cs - 1 - (c - cs / 2) : c - cs / 2;
}

// gen_permute_c16_kernel for any group size: Gc[c][pad(slot * 4096 + p)] = conj(F[2 kb + g]) * scale, kb = t_slot + cs kl the
// branch bin at position p = pos(kl) of the local [16,16,16] inverse plan of sub-transform t_slot of CTA c (branch g)
__global__ void gen_permute_group_kernel(const cplx* __restrict__ F, cplx* Gc, double scale, int cs) {
  constexpr int ML = Cluster16Shape::ML;
  const int M = ML * cs;
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= 2 * M) return;
  const int c = idx / (2 * ML), r = idx - c * 2 * ML, slot = r / ML, kl = r - slot * ML;
  const int kb = grp_sub(cs, c, slot) + cs * kl;
  const cplx f = F[plan_pos(2 * kb + grp_branch(cs, c), 2 * M)];
  const int p = slot * ML + plan_pos(kl, ML);
  Gc[(size_t)c * Cluster16Shape::PADZ + p + (p >> 4)] = mk(f.x * scale, -f.y * scale);
}

// L0 for one output column j of the reducer: radix-CS DIT over the CS sub-transforms of each branch, the pruned radix-2 join
// and the fused sums (c16_last_regs of td_cluster16.cuh for CS = 16; here with explicit twiddle powers)
template <int CS, int MODE>
__device__ __forceinline__ void grp_last_regs(cplx (&e)[CS], cplx (&o)[CS], int j, int n, cplx beta /* w_2M^j */,
                                              cplx w1 /* w_M^(-j) */, cplx* __restrict__ zd, double& acc0, double& acc1) {
  constexpr int ML = Cluster16Shape::ML;
  cplx wp[CS], gm[CS];
  tw_powers<CS>(w1, wp);
  static_for<1, CS>([&](auto s) { e[decltype(s)::value] = cmul(e[decltype(s)::value], wp[decltype(s)::value]);
                                  o[decltype(s)::value] = cmul(o[decltype(s)::value], wp[decltype(s)::value]); });
  fft_reg<CS, true>(e);
  fft_reg<CS, true>(o);
  const cplx cb = cconj(beta);
  static_for<0, CS>([&](auto t) { gm[decltype(t)::value] = mul_w32<decltype(t)::value * (16 / CS), true>(cb); });
  real p0[4] = {real(0), real(0), real(0), real(0)}, p1[4] = {real(0), real(0), real(0), real(0)};
  static_for<0, CS>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    const cplx ev = e[brevR<CS>(tt)], ov = o[brevR<CS>(tt)];
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

struct GroupParams {
  FusedParams base;       // base.T: the class table w_2M^k; base.segs[0]: the segment
  const cplx* Gp;         // [CS][A || B in the padded Z layout] (gen_permute_group_kernel)
  double* partial;        // [B][CS][2] per-CTA partial sums
  cplx* wsU;              // [groups][2][2 NF]: first-pass outputs, [branch][sub-transform t][2048]
  cplx* wsZ;              // [groups][2][2 M]: inverse sub-transforms, [branch][sub-transform t][4096]
  unsigned* bar;          // [groups][2] arrival counters, zero at launch
};

// one thread, after the CTA's barrier: the CTA's stores are visible device-wide before the count moves
__device__ __forceinline__ void grp_arrive(unsigned* ctr) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(ctr), "r"(1u) : "memory");
}
__device__ __forceinline__ void grp_wait(const unsigned* ctr, unsigned target) {
  const long long t0 = clock64();
  for (;;) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
    if (v >= target) return;
    __nanosleep(32);
    if (clock64() - t0 > 20000000000ll) __trap();   // (~10 s) a partner that never arrives must not hang the device
  }
}

template <int CS, int MODE>
__global__ void __launch_bounds__(Cluster16Shape::NT, 1) td_group_kernel(const GroupParams PG) {
  using Sh = Cluster16Shape;   // the CTA-local machinery: arrays of 2 x 2048 / 2 x 4096, 256 threads, tensor-memory windows
  using Gs = GroupShape<CS>;
  constexpr int NT = Sh::NT, NFL = Sh::NFL, ML = Sh::ML, TWL = Sh::TWL, NF = Gs::NF, M = Gs::M, TPT = Gs::TPT;
  constexpr int LOGCS = ilog2(CS);
  const FusedParams& P = PG.base;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sm = reinterpret_cast<cplx*>(smem_raw);
  const SmemArr U{sm}, Z{sm + Sh::PADU};          // U = A || B (2 x 2048), Z = ZA || ZB (2 x 4096)
  cplx* tw = sm + Sh::PADU + Sh::PADZ;             // w_8192^k, k < 1024
  double* red = reinterpret_cast<double*>(tw + Sh::TWS);   // [2 NW] per-warp partial sums
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(red + 2 * Sh::NW + 2);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int rank = blockIdx.x & (CS - 1);
  const int grp = blockIdx.x >> LOGCS, ngrp = gridDim.x >> LOGCS;
  const int brG = grp_branch(CS, rank), tsubA = grp_sub(CS, rank, 0), tsubB = grp_sub(CS, rank, 1);
  const C16Own own = c16_own(rank, warp);
  const cplx* __restrict__ T = P.T;
  const SegDev sg = P.segs[0];
  cplx* const Ug = PG.wsU + (size_t)grp * 2 * (2 * NF);
  cplx* const Zg = PG.wsZ + (size_t)grp * 2 * (2 * M);
  unsigned* const bar_u = PG.bar + 2 * grp;        // item's first-pass outputs are in U
  unsigned* const bar_z = bar_u + 1;               // item's inverse sub-transforms are in Z

  for (int k = tid; k < Sh::TWS; k += NT) tw[k] = T[CS * k];   // w_2M^(CS k) = w_8192^k
  if (warp == 0) tmem_alloc<Sh::TMEM_COLS>(smem_u32(tmem_slot));
  tmem_fence_before();
  __syncthreads();
  tmem_fence_after();
  const uint32_t tcol = *tmem_slot + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * Sh::Cols::WINDOW);
  f4_store_twiddles<TWL>(lane, tw, tcol + Sh::Cols::TW);
  f4_store_generator(PG.Gp + (size_t)rank * Sh::PADZ, own.o, lane, tcol + F4_TC_G);
  tmem_wait_st();
  cplx basew;   // the untangle twiddle w_2M^(2 kq + g) of this lane's first bin kq = t_sub + CS kap (c16_basew for any CS)
  {
    const int q4 = lane >> 3;
    const int s1c = q4 == 0 ? own.o.z0 : q4 == 1 ? own.o.z2 : q4 == 2 ? own.o.z1 : own.o.z3, s2 = lane & 7;
    const int kap = (s1c & 15) + 16 * s2;
    basew = __ldg(T + 2 * (((s1c >> 4) ? tsubB : tsubA) + CS * kap) + brG);
  }
  // cross passes: this thread's butterfly u (< TPT) of F0 works on input column jF(u) of branch g0, of L0 on output column jL(u)
  const int g0 = tid >> 7;
  auto jF = [&](int u) { return (NFL / CS) * rank + (tid & 127) + 128 * u; };
  auto jL = [&](int u) { return (ML / CS) * rank + tid + 256 * u; };
  if (MODE == MODE_LOGLIKE) {                      // this thread's 16 sample pairs of the data vector, once per launch
    const double* drow = P.d + sg.off;
    double2 dvs[16];
#pragma unroll
    for (int p = 0; p < 16; ++p) {
      const int i0 = 2 * (jF(p / CS) + NFL * (p % CS));
      dvs[p] = make_double2(i0 < sg.n ? __ldg(drow + i0) : 0.0, i0 + 1 < sg.n ? __ldg(drow + i0 + 1) : 0.0);
    }
#pragma unroll
    for (int p = 0; p < 16; ++p) tmem_st_c64(tcol + F4_TC_D + 4 * p, dvs[p]);
    tmem_wait_st();
  }

  const long long Bs = (MODE == MODE_STOREZ) ? 1 : P.B;
  long long prev_b = -1;
  unsigned it = 0;   // items this group has started
  // S5 of the previous item: this CTA's 4096 / CS output columns from the 2 CS sub-transforms in Z[parity of that item]
  auto reduce_prev = [&](const cplx* __restrict__ Zb, unsigned target) {
    if (lane == 0) grp_wait(bar_z, target);   // every warp polls for itself: no CTA barrier behind the wait
    __syncwarp();
    double acc0 = 0.0, acc1 = 0.0;
    if constexpr (CS == 16) {
      const int jr = jL(0);
      cplx e[16], o[16];
#pragma unroll
      for (int ss = 0; ss < 16; ++ss) { e[ss] = __ldcg(Zb + ss * ML + jr); o[ss] = __ldcg(Zb + M + ss * ML + jr); }
      c16_last_regs<MODE>(e, o, jr, sg.n, __ldg(T + jr) /* w_2M^jr */, cconj(__ldg(T + 2 * jr)) /* w_M^(-jr) */, sg.zd, acc0, acc1);
    } else {
      cplx e[TPT][CS], o[TPT][CS];   // all 32 loads in flight
#pragma unroll
      for (int u = 0; u < TPT; ++u)
#pragma unroll
        for (int ss = 0; ss < CS; ++ss) { e[u][ss] = __ldcg(Zb + ss * ML + jL(u)); o[u][ss] = __ldcg(Zb + M + ss * ML + jL(u)); }
      static_for<0, TPT>([&](auto uu) {
        constexpr int u = decltype(uu)::value;
        const int jr = jL(u);
        grp_last_regs<CS, MODE>(e[u], o[u], jr, sg.n, __ldg(T + jr), cconj(__ldg(T + 2 * jr)), sg.zd, acc0, acc1);
      });
    }
    if (MODE != MODE_STOREZ) {
      if (MODE == MODE_INNER) acc0 = warp_sum(acc0);
      acc1 = warp_sum(acc1);
      if (lane == 0) { red[2 * warp] = acc0; red[2 * warp + 1] = acc1; }
      __syncthreads();
      if (tid == 0) {
        double t0 = 0.0, t1 = 0.0;
#pragma unroll
        for (int w = 0; w < Sh::NW; ++w) { t0 += red[2 * w]; t1 += red[2 * w + 1]; }
        double* dst = PG.partial + ((size_t)prev_b * CS + rank) * 2;
        dst[0] = (MODE == MODE_LOGLIKE) ? t1 : t0;
        dst[1] = t1;
      }
    }
  };

  for (long long b = grp; b < Bs; b += ngrp, ++it) {
    cplx* const Ub = Ug + (size_t)(it & 1) * (2 * NF);
    cplx* const Zb = Zg + (size_t)(it & 1) * (2 * M);
    // ---------------- F0: first forward pass (radix CS, stride 2048): TPT butterflies per thread, branch g0
    {
      const double* drow = P.d + sg.off;
      const double* hrow = (MODE == MODE_STOREZ) ? drow : P.H + b * P.ldh + sg.off;
      const bool vec = ((reinterpret_cast<uintptr_t>(hrow) & 15) == 0) && ((sg.n & 1) == 0);
      cplx x[16];   // x[u CS + q]: input q of butterfly u
      if (vec) {
        int dr[4][16];
        if (MODE == MODE_LOGLIKE) {
#pragma unroll
          for (int g = 0; g < 4; ++g) tmem_ld16(tcol + F4_TC_D + 16 * g, dr[g]);
        }
        double2 hs[16];   // all 16 loads in flight together (n even, rows 16-byte aligned: a pair is in or out as a whole)
#pragma unroll
        for (int p = 0; p < 16; ++p) {
          const int i0 = 2 * (jF(p / CS) + NFL * (p % CS));
          hs[p] = i0 < sg.n ? __ldg(reinterpret_cast<const double2*>(hrow + i0)) : make_double2(0.0, 0.0);
        }
        if (MODE == MODE_LOGLIKE) {
          tmem_wait_ld();
#pragma unroll
          for (int g = 0; g < 4; ++g) tmem_use16(dr[g]);
#pragma unroll
          for (int p = 0; p < 16; ++p) {
            const double2 dv = tmem_c64(dr[p >> 2], p & 3);
            x[p] = to_cplx(dv.x - hs[p].x, dv.y - hs[p].y, sg.rscale);   // S1: r = d - h
          }
        } else {
#pragma unroll
          for (int p = 0; p < 16; ++p) x[p] = to_cplx(hs[p].x, hs[p].y, sg.rscale);
        }
      } else {
        const bool v2 = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
#pragma unroll
        for (int p = 0; p < 16; ++p) x[p] = load_pair<MODE>(drow, hrow, jF(p / CS) + NFL * (p % CS), sg.n, v2, sg.rscale);
      }
      // the next item's row pieces on their way into L2 while this item computes
      if (b + ngrp < Bs && MODE != MODE_STOREZ && (tid & 127) == 0 && g0 == 0) {
        const double* nrow = P.H + (b + ngrp) * P.ldh + sg.off;
        constexpr long long piece = 2ll * (NFL / CS);   // doubles of this CTA's columns in one stride
#pragma unroll 1
        for (int q = 0; q < CS; ++q) {
          const long long i0 = 2ll * ((NFL / CS) * rank + NFL * q);
          if (i0 < sg.n) {
            const long long nbytes = (sg.n - i0 < piece ? sg.n - i0 : piece) * 8;
            const double* src = nrow + i0;
            if ((reinterpret_cast<uintptr_t>(src) & 15) == 0 && (nbytes & 15) == 0)
              asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"((uint32_t)nbytes) : "memory");
          }
        }
      }
      static_for<0, TPT>([&](auto uu) {
        constexpr int u = decltype(uu)::value;
        const int j0 = jF(u);
        // (the per-thread constants of the two cross passes are re-read per item, L1 hits: registers are what this kernel lacks)
        cplx y[CS], w[CS];
#pragma unroll
        for (int q = 0; q < CS; ++q) y[q] = x[u * CS + q];
        tw_powers<CS>(__ldg(T + 4 * j0), w);             // powers of w_NF^j0
        if (g0) {                                        // odd-bin branch: input twist w_M^(j0 + 2048 q) = w_M^j0 w_2CS^q
          const cplx f0_beta = __ldg(T + 2 * j0);
          static_for<0, CS>([&](auto q) { y[decltype(q)::value] = mul_w32<decltype(q)::value * (16 / CS), false>(y[decltype(q)::value]); });
          static_for<0, CS>([&](auto t) { w[decltype(t)::value] = cmul(w[decltype(t)::value], f0_beta); });
        }
        fft_reg<CS, false>(y);
        cplx* dst = Ub + (size_t)g0 * NF + j0;
        static_for<0, CS>([&](auto t) {
          constexpr int tt = decltype(t)::value;
          cplx v = y[brevR<CS>(tt)];
          if (tt > 0 || g0) v = cmul(v, w[tt]);
          __stcg(dst + tt * NFL, v);
        });
      });
    }
    __syncthreads();
    if (tid == 32) grp_arrive(bar_u);   // (not the thread that polls next: its fence would delay the poll)
    // S5 of the previous item while the partners finish their first pass
    if (prev_b >= 0) reduce_prev(Zg + (size_t)((it & 1) ^ 1) * (2 * M), (unsigned)CS * it);
    if (lane == 0) grp_wait(bar_u, (unsigned)CS * (it + 1));
    __syncwarp();
    // ---------------- first local forward pass (radix 8, L = 2048) of A and B: inputs from the exchange buffer
    {
      const cplx* __restrict__ sa = Ub + (size_t)brG * NF + (size_t)tsubA * NFL + tid;
      const cplx* __restrict__ sb = Ub + (size_t)brG * NF + (size_t)tsubB * NFL + tid;
      cplx xa[8], xb[8], w8[8];
#pragma unroll
      for (int q = 0; q < 8; ++q) { xa[q] = __ldcg(sa + 256 * q); xb[q] = __ldcg(sb + 256 * q); }
      tw_powers<8>(tw[4 * tid], w8);   // w_2048^j
      fft_reg<8, false>(xa);
      fft_reg<8, false>(xb);
      static_for<0, 8>([&](auto t) {
        constexpr int tt = decltype(t)::value;
        cplx va = xa[brevR<8>(tt)], vb = xb[brevR<8>(tt)];
        if constexpr (tt > 0) { va = cmul(va, w8[tt]); vb = cmul(vb, w8[tt]); }
        U.st(tid + 256 * tt, va);
        U.st(NFL + tid + 256 * tt, vb);
      });
    }
    __syncthreads();
    f4_forward23<TWL, true>(U, own.o, lane, tw, tcol + Sh::Cols::TW);
    __syncwarp();
    // ---------------- mid, inverse pass 2 (warp-local), inverse pass 3 (L = 4096, CTA-wide, outputs to the exchange buffer)
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
      cplx* dst = Zb + (size_t)brG * M + (size_t)(blk ? tsubB : tsubA) * ML + jj;
      static_for<0, 16>([&](auto t) { __stcg(dst + 256 * decltype(t)::value, x[brevR<16>(decltype(t)::value)]); });
    }
    __syncthreads();   // also: every warp is past mid and the last pass, U and Z (shared) are free for the next item
    if (tid == 32) grp_arrive(bar_z);
    prev_b = b;
  }
  if (prev_b >= 0) reduce_prev(Zg + (size_t)((it & 1) ^ 1) * (2 * M), (unsigned)CS * it);
  __syncthreads();
  if (warp == 0) tmem_dealloc<Sh::TMEM_COLS>(*tmem_slot);
}

}  // namespace TD_NS
