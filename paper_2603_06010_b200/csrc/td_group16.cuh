// td_group16.cuh - the fused FFT path for M = 65536 (config c4) as ONE persistent kernel whose CTAs work in groups of 16 and
// exchange through L2: the decomposition, the mirror-closed ownership of sub-transforms and every CTA-local pass are those of
// td_cluster16.cuh; what differs is how the two cross passes travel.
//
//   td_cluster16_kernel  F0 / L0 outputs go to the owner / reducer CTA with st.async into distributed shared memory: 16 bytes
//                        per cycle and SM, producer pays, and a 16-CTA cluster is co-resident 7 times (112 of 148 SMs).
//   td_group16_kernel    F0 writes its outputs to a global exchange buffer U[group][parity] (plain coalesced 16-byte stores),
//                        the owner's first local pass (radix 8, L = 2048) reads its inputs from there instead of shared
//                        memory; the last local pass (radix 16, L = 4096) writes its outputs to Z[group][parity], and L0 reads
//                        its 32 values per thread from there.  9 groups x 2 parities x 3 MB = 54 MB, written and read once per
//                        item: it never leaves the 126 MB L2.  No cluster: 9 groups = 144 of 148 SMs, and the two barriers of
//                        an item are arrival counters in global memory (16 arrivals each), the second one waited for only
//                        after the NEXT item's first pass (S5 of an item is deferred as in the cluster kernel).
//
// The staged kernels (td_staged.cuh) move ~12 MB per template through L2 in 5 kernels per chunk; this kernel moves 6.5 MB
// (0.5 H + 1 + 1 + 2 + 2) in one launch per segment, with generator values, data samples and twiddles in tensor memory.
// The launch is cooperative (all CTAs co-resident, or the launch fails); a wait that does not end within ~2 s traps.
#pragma once
#include "td_cluster16.cuh"

namespace TD_NS {

struct Group16Params {
  FusedParams base;       // base.T: the class table w_2M^k; base.segs[0]: the segment
  const cplx* Gp;         // [16][A || B in the padded Z layout] (gen_permute_c16_kernel)
  double* partial;        // [B][16][2] per-CTA partial sums
  cplx* wsU;              // [groups][2][2 NF]: first-pass outputs, [branch][sub-transform t][2048]
  cplx* wsZ;              // [groups][2][2 M]: inverse sub-transforms, [branch][sub-transform t][4096]
  unsigned* bar;          // [groups][2] arrival counters, zero at launch
};

// one thread, after the CTA's barrier: the CTA's stores are visible device-wide before the count moves
__device__ __forceinline__ void g16_arrive(unsigned* ctr) {
  asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(ctr), "r"(1u) : "memory");
}
__device__ __forceinline__ void g16_wait(const unsigned* ctr, unsigned target) {
  const long long t0 = clock64();
  for (;;) {
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
    if (v >= target) return;
    __nanosleep(32);
    if (clock64() - t0 > 4000000000ll) __trap();   // a partner that never arrives must not hang the device
  }
}

template <int MODE>
__global__ void __launch_bounds__(Cluster16Shape::NT, 1) td_group16_kernel(const Group16Params PG) {
  using Sh = Cluster16Shape;
  constexpr int NT = Sh::NT, NF = Sh::NF, M = Sh::M, NFL = Sh::NFL, ML = Sh::ML, TWL = Sh::TWL;
  const FusedParams& P = PG.base;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sm = reinterpret_cast<cplx*>(smem_raw);
  const SmemArr U{sm}, Z{sm + Sh::PADU};          // U = A || B (2 x 2048), Z = ZA || ZB (2 x 4096)
  cplx* tw = sm + Sh::PADU + Sh::PADZ;             // w_8192^k, k < 1024
  double* red = reinterpret_cast<double*>(tw + Sh::TWS);   // [2 NW] per-warp partial sums
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(red + 2 * Sh::NW + 2);
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int rank = blockIdx.x & 15;
  const int grp = blockIdx.x >> 4, ngrp = gridDim.x >> 4;
  const int brG = c16_branch(rank), tsubA = c16_sub(rank, 0), tsubB = c16_sub(rank, 1);
  const C16Own own = c16_own(rank, warp);
  const cplx* __restrict__ T = P.T;
  const SegDev sg = P.segs[0];
  cplx* const Ug = PG.wsU + (size_t)grp * 2 * (2 * NF);
  cplx* const Zg = PG.wsZ + (size_t)grp * 2 * (2 * M);
  unsigned* const bar_u = PG.bar + 2 * grp;        // item's first-pass outputs are in U
  unsigned* const bar_z = bar_u + 1;               // item's inverse sub-transforms are in Z

  for (int k = tid; k < Sh::TWS; k += NT) tw[k] = T[16 * k];
  if (warp == 0) tmem_alloc<Sh::TMEM_COLS>(smem_u32(tmem_slot));
  tmem_fence_before();
  __syncthreads();
  tmem_fence_after();
  const uint32_t tcol = *tmem_slot + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)((warp >> 2) * Sh::Cols::WINDOW);
  f4_store_twiddles<TWL>(lane, tw, tcol + Sh::Cols::TW);
  f4_store_generator(PG.Gp + (size_t)rank * Sh::PADZ, own.o, lane, tcol + F4_TC_G);
  tmem_wait_st();
  const cplx basew = c16_basew(own, lane, T, tsubA, tsubB, brG);
  const int g0 = tid >> 7, j0 = 128 * rank + (tid & 127), jr = 256 * rank + tid;
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

  const long long Bs = (MODE == MODE_STOREZ) ? 1 : P.B;
  long long prev_b = -1;
  unsigned it = 0;   // items this group has started
  // S5 of the previous item: this CTA's 256 output columns from the 32 sub-transforms in Z[parity of that item]
  auto reduce_prev = [&](const cplx* __restrict__ Zb, unsigned target) {
    if (tid == 0) g16_wait(bar_z, target);
    __syncthreads();
    cplx e[16], o[16];
#pragma unroll
    for (int ss = 0; ss < 16; ++ss) { e[ss] = __ldcg(Zb + ss * ML + jr); o[ss] = __ldcg(Zb + M + ss * ML + jr); }
    double acc0 = 0.0, acc1 = 0.0;
    c16_last_regs<MODE>(e, o, jr, sg.n, __ldg(T + jr) /* w_2M^jr */, cconj(__ldg(T + 2 * jr)) /* w_M^(-jr) */, sg.zd, acc0, acc1);
    if (MODE != MODE_STOREZ) {
      if (MODE == MODE_INNER) acc0 = warp_sum(acc0);
      acc1 = warp_sum(acc1);
      if (lane == 0) { red[2 * warp] = acc0; red[2 * warp + 1] = acc1; }
      __syncthreads();
      if (tid == 0) {
        double t0 = 0.0, t1 = 0.0;
#pragma unroll
        for (int w = 0; w < Sh::NW; ++w) { t0 += red[2 * w]; t1 += red[2 * w + 1]; }
        double* dst = PG.partial + ((size_t)prev_b * Sh::CS + rank) * 2;
        dst[0] = (MODE == MODE_LOGLIKE) ? t1 : t0;
        dst[1] = t1;
      }
    }
  };

  for (long long b = grp; b < Bs; b += ngrp, ++it) {
    cplx* const Ub = Ug + (size_t)(it & 1) * (2 * NF);
    cplx* const Zb = Zg + (size_t)(it & 1) * (2 * M);
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
        double2 hs[16];
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
      if (b + ngrp < Bs && MODE != MODE_STOREZ && (tid & 127) == 0 && g0 == 0) {
        const double* nrow = P.H + (b + ngrp) * P.ldh + sg.off;
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
      // (the per-thread constants of the two cross passes are re-read per item, L1 hits: registers are what this kernel lacks)
      const cplx f0_beta = __ldg(T + 2 * j0);          // w_M^j0
      tw_powers<16>(__ldg(T + 4 * j0), w);             // powers of w_NF^j0
      if (g0) {
        static_for<0, 16>([&](auto q) { x[decltype(q)::value] = mul_w32<decltype(q)::value, false>(x[decltype(q)::value]); });
        static_for<0, 16>([&](auto t) { w[decltype(t)::value] = cmul(w[decltype(t)::value], f0_beta); });
      }
      fft_reg<16, false>(x);
      cplx* dst = Ub + (size_t)g0 * NF + j0;
      static_for<0, 16>([&](auto t) {
        constexpr int tt = decltype(t)::value;
        cplx v = x[brevR<16>(tt)];
        if (tt > 0 || g0) v = cmul(v, w[tt]);
        __stcg(dst + tt * NFL, v);
      });
    }
    __syncthreads();
    if (tid == 0) g16_arrive(bar_u);
    // S5 of the previous item while the partners finish their first pass
    if (prev_b >= 0) reduce_prev(Zg + (size_t)((it & 1) ^ 1) * (2 * M), 16u * it);
    if (tid == 0) g16_wait(bar_u, 16u * (it + 1));
    __syncthreads();
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
    if (tid == 0) g16_arrive(bar_z);
    prev_b = b;
  }
  if (prev_b >= 0) reduce_prev(Zg + (size_t)((it & 1) ^ 1) * (2 * M), 16u * it);
  __syncthreads();
  if (warp == 0) tmem_dealloc<Sh::TMEM_COLS>(*tmem_slot);
}

}  // namespace TD_NS
