// td_fused4.cuh - the fused FFT-path kernel for M = 1024 / 2048 / 4096 (transform lengths
// 2M = 2048 / 4096 / 8192), restructured around the two things the first fused kernel lost
// time on (profiles/r01_fused_v3_regions.md): CTA-wide barriers that put every warp in the
// same load -> compute -> store phase, and the stand-alone untangle pass.
//
//  * plans  NF = M/2 = [RF1,16,16],  M = [RI1,16,16],  RI1 = 2 RF1;  NT = 32 RF1 = M/16 threads;
//    warps [0, NW/2) own the even-bin branch, warps [NW/2, NW) the odd-bin branch.
//  * forward passes 2 and 3 touch only the 2 x 256 elements a warp owns: one __syncwarp between them.
//  * "mid": forward bins are untangled IN REGISTERS from the two mirror blocks, multiplied by the
//    generator spectrum and pushed through the first inverse radix-16 pass before they are stored.
//    The generator spectrum of the segment is TMA-prefetched into the Z region (dead during the
//    forward half) in the padded Z layout, so mid reads G[p] and writes Z[p] in place.
//  * inverse pass 2 is again warp-local; only the last pass (which joins the two branches and
//    carries the fused quadratic reduction) needs the whole CTA.
//  * the next item's rows are TMA-prefetched into the U region by whichever warp finishes mid last.
// CTA barriers per (template, segment): 5 (was 9).
#pragma once
#include "td_fused.cuh"
#include "td_dit16.cuh"

namespace td {

constexpr int F4_SEGCACHE = 8;  // segment records cached in shared memory (more segments: read from global per item)

template <int LOG2M> struct Fused4Shape {
  static constexpr int M = 1 << LOG2M, NF = M / 2;
  static constexpr int RF1 = plan_r1(NF), RI1 = plan_r1(M);
  static_assert(plan_np(NF) == 3 && plan_np(M) == 3 && RI1 == 2 * RF1, "fused4 needs [R,16,16] plans");
  static constexpr int NT = 32 * RF1, NW = RF1, NWB = RF1 / 2;
  static constexpr int TWS = 2 * M / RF1;
  static constexpr int PADM = SmemArr::padded(M), PADNF = SmemArr::padded(NF);
  static constexpr size_t smem_bytes() {
    return sizeof(cplx) * (2 * (size_t)PADNF + 2 * (size_t)PADM + TWS) + sizeof(double) * 2 * NW + 48 + F4_SEGCACHE * sizeof(SegDev);
  }
};

struct Fused4Params {
  FusedParams base;
  const cplx* const* Gp;  // device array [n_seg]: generator spectrum in the PADDED Z layout [2][padded(M)]
};

// ---- pieces shared by the one-CTA kernel below and the 2-CTA cluster kernel (td_cluster.cuh) -------
// All three work on ONE branch (U, Z of that branch); wb = index of the warp within the branch,
// TW = 2M, RF1 = first forward radix (forward blocks of 256: RF1 per branch), RI1 = 2 RF1.

// Which 256-element blocks a warp owns.  Plain: U blocks {2wb, 2wb+1}, Z blocks {4wb .. 4wb+3}.  Mirror-closed (MC): the
// forward bins of U block r are k = r (mod RF1) and the untangle pairs k with -k (even branch) or -1-k (odd branch), so a
// warp that owns {r, mirror(r)} reads only its own blocks in mid, and the Z blocks it fills there, {r, r+RF1, m, m+RF1},
// are the ones it transforms in inverse pass 2: forward passes 2-3, mid and inverse pass 2 form ONE warp-local stretch
// with no CTA or branch barrier inside (profiles/r01_peaks.md, phase probe: barrier-free groups overlap loads, butterflies
// and stores of different warps; a barrier per pass costs ~25 %).
struct F4Own { int u0, u1, z0, z1, z2, z3; };
template <int RF1, bool MC> __device__ __forceinline__ F4Own f4_own(int br, int wb) {
  if constexpr (!MC) return F4Own{2 * wb, 2 * wb + 1, 4 * wb, 4 * wb + 1, 4 * wb + 2, 4 * wb + 3};
  else {
    const int r = wb;
    const int m = br ? RF1 - 1 - wb : (wb == 0 ? RF1 / 2 : RF1 - wb);
    return F4Own{r, m, r, m, r + RF1, m + RF1};
  }
}

// forward passes 2 and 3, warp-local (this warp owns U blocks o.u0, o.u1 of its branch)
template <int TW>
__device__ __forceinline__ void f4_forward23(const SmemArr& U, const F4Own& o, int lane, const cplx* __restrict__ tw) {
  cplx x[16], w[16];
  {
    const int s1 = (lane >> 4) ? o.u1 : o.u0, j = lane & 15;
    const int base = s1 * 256 + j;
    tw_powers<16>(tw[j * (TW / 256)], w);
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = U.ld(base + 16 * q);
    fft_reg<16, false>(x);
    static_for<0, 16>([&](auto t) {
      constexpr int tt = decltype(t)::value;
      cplx v = x[brevR<16>(tt)];
      if constexpr (tt > 0) v = cmul(v, w[tt]);
      U.st(base + 16 * tt, v);
    });
  }
  __syncwarp();
  {
    // pass 3 (L = 16).  Lane -> block (s1', s2') with s2' = (l & 15) ^ ((l & 1) << 3): both the
    // loads (block s1'*16 + s2') and the stores are bank-conflict free.  The result block is
    // stored at the warp-owned slot s1'*16 + (s2' >> 1) + 8 (s2' & 1) ("mid layout": the 8 blocks
    // one quarter-warp of mid reads are consecutive), hence all loads precede all stores.
    const int s1p = (lane >> 4) ? o.u1 : o.u0;
    const int s2p = (lane & 15) ^ ((lane & 1) << 3);
    const int src = (s1p * 16 + s2p) * 16;
    const int dst = (s1p * 16 + (s2p >> 1) + 8 * (s2p & 1)) * 16;
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = U.ld(src + q);
    __syncwarp();
    fft_reg<16, false>(x);
    static_for<0, 16>([&](auto t) { U.st(dst + decltype(t)::value, x[brevR<16>(decltype(t)::value)]); });
  }
}

// mid: untangle (registers) x generator (in place in Z) -> first inverse pass
template <int NF, int RF1>
__device__ __forceinline__ void f4_mid(const SmemArr& U, const SmemArr& Z, int br, const F4Own& o, int lane,
                                       const cplx* __restrict__ tw) {
  constexpr int RI1 = 2 * RF1;
  const int q4 = lane >> 3;
  const int s1 = q4 == 0 ? o.z0 : q4 == 1 ? o.z1 : q4 == 2 ? o.z2 : o.z3, s2 = lane & 7;
  const int kap = s1 + RI1 * s2;  // forward low-part kappa = inverse block index tau
  int kap2;
  bool selfzero = false;
  if (br == 0) { kap2 = (NF / 16 - kap) & (NF / 16 - 1); selfzero = (kap == 0); }
  else         { kap2 = NF / 16 - 1 - kap; }
  // U blocks in the "mid layout" written by forward pass 3
  auto slot = [](int k) { const int a = k & (RF1 - 1), c = k / RF1; return (a * 16 + (c >> 1) + 8 * (c & 1)) * 16; };
  const int fb = slot(kap), fb2 = slot(kap2);
  const cplx basew = tw[2 * kap + br];  // w_2M^(2 kap + br)
  const int zb0 = (s1 * 16 + s2) * 16;
  static_for<0, 2>([&](auto par) {
    constexpr int pp = decltype(par)::value;  // 0: even t -> inverse block tau; 1: odd t -> block tau + M/32
    const int zb = zb0 + pp * 8 * 16;
    cplx ua[8], ub[8], e[16];
    static_for<0, 8>([&](auto hh) {
      constexpr int t = 2 * decltype(hh)::value + pp;
      ua[decltype(hh)::value] = U.ld(fb + t);
      ub[decltype(hh)::value] = U.ld(fb2 + (selfzero ? ((16 - t) & 15) : (15 - t)));
    });
#pragma unroll
    for (int q = 0; q < 16; ++q) e[q] = Z.ld(zb + q);  // generator spectrum sits in Z
    static_for<0, 8>([&](auto hh) {
      constexpr int h8 = decltype(hh)::value, t = 2 * h8 + pp;
      const cplx U1 = ua[h8], U2 = ub[h8];
      const cplx A = mk(U1.x + U2.x, U1.y - U2.y);
      const cplx Bv = mk(U1.y + U2.y, -(U1.x - U2.x));
      const cplx wB = cmul(basew, mul_w32<t, false>(Bv));
      e[h8] = cmul(e[h8], cadd(A, wB));          // G * 2 X_{kq},      entry s = t/2
      e[8 + h8] = cmul(e[8 + h8], csub(A, wB));  // G * 2 X_{NF + kq}, entry s = 8 + t/2
    });
    dit16<true, false>(e, mk(1.0, 0.0));
    static_for<0, 16>([&](auto t) { Z.st(zb + decltype(t)::value, e[brevR<16>(decltype(t)::value)]); });
  });
}

// inverse pass 2 (L = 256), warp-local: blocks s1 = 4wb .. 4wb+3
template <int TW>
__device__ __forceinline__ void f4_inverse2(const SmemArr& Z, const F4Own& o, int lane, const cplx* __restrict__ tw) {
  cplx x[16], y[16];
  const int j = lane & 15;
  const cplx w1 = cconj(tw[j * (TW / 256)]);  // the inverse transform's w_256^(-j); its powers are built inside dit16
  const int base0 = ((lane >> 4) ? o.z1 : o.z0) * 256 + j, base1 = ((lane >> 4) ? o.z3 : o.z2) * 256 + j;
#pragma unroll
  for (int q = 0; q < 16; ++q) { x[q] = Z.ld(base0 + 16 * q); y[q] = Z.ld(base1 + 16 * q); }
  dit16<true, true>(x, w1);
  static_for<0, 16>([&](auto t) { Z.st(base0 + 16 * decltype(t)::value, x[brevR<16>(decltype(t)::value)]); });
  dit16<true, true>(y, w1);
  static_for<0, 16>([&](auto t) { Z.st(base1 + 16 * decltype(t)::value, y[brevR<16>(decltype(t)::value)]); });
}

template <int LOG2M, int MODE>
__global__ void __launch_bounds__(Fused4Shape<LOG2M>::NT, 1) td_fused4_kernel(const Fused4Params P4) {
  using Sh = Fused4Shape<LOG2M>;
  constexpr int M = Sh::M, NF = Sh::NF, TW = 2 * M, NT = Sh::NT, NW = Sh::NW, NWB = Sh::NWB;
  constexpr int RF1 = Sh::RF1, RI1 = Sh::RI1;
  const FusedParams& P = P4.base;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  cplx* sm = reinterpret_cast<cplx*>(smem_raw);
  const SmemArr UE{sm}, UO{sm + Sh::PADNF};
  const SmemArr ZE{sm + 2 * Sh::PADNF}, ZO{sm + 2 * Sh::PADNF + Sh::PADM};
  cplx* tw = sm + 2 * Sh::PADNF + 2 * Sh::PADM;
  double* red = reinterpret_cast<double*>(tw + Sh::TWS);
  const uint32_t mbar_rows = smem_u32(red + 2 * NW);
  const uint32_t mbar_g = mbar_rows + 8;
  int* mid_count = reinterpret_cast<int*>(red + 2 * NW + 2);
  int* last_count = mid_count + 1;
  double* totS = red + 2 * NW + 3;  // running sums of the current template over its segments
  SegDev* segS = reinterpret_cast<SegDev*>(red + 2 * NW + 6);
  const SegDev* segs = P.n_seg <= F4_SEGCACHE ? segS : P.segs;
  double* stH = reinterpret_cast<double*>(sm);
  double* stD = stH + M;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int br = warp / NWB, wb = warp - br * NWB;  // branch (0 even bins, 1 odd bins), warp within branch
  const SmemArr U = br ? UO : UE, Z = br ? ZO : ZE;
  const F4Own own = f4_own<RF1, true>(br, wb);

  for (int k = tid; k < Sh::TWS; k += NT) tw[k] = P.T[k];
  if (tid < P.n_seg && tid < F4_SEGCACHE) segS[tid] = P.segs[tid];
  if (tid == 0) { mbar_init(mbar_rows, 1); mbar_init(mbar_g, 1); *mid_count = 0; *last_count = 0; totS[0] = 0.0; totS[1] = 0.0; }
  __syncthreads();

  auto rows = [&](long long b, int s, const double*& drow, const double*& hrow, int& n) -> bool {
    const SegDev sg = segs[s];
    drow = P.d + sg.off;
    hrow = (MODE == MODE_STOREZ) ? drow : P.H + b * P.ldh + sg.off;
    n = sg.n;
    return (((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0) && ((n & 1) == 0);
  };
  // issued by ONE thread
  auto prefetch_rows = [&](long long b, int s) {
    const double *drow, *hrow; int n;
    if (rows(b, s, drow, hrow, n)) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      const uint32_t bytes = (uint32_t)n * 8u;
      mbar_expect_tx(mbar_rows, bytes * ((MODE == MODE_LOGLIKE) ? 2 : 1));
      if (MODE != MODE_STOREZ) bulk_g2s(smem_u32(stH), hrow, bytes, mbar_rows);
      if (MODE != MODE_INNER) bulk_g2s(smem_u32(stD), drow, bytes, mbar_rows);
    }
  };
  auto prefetch_g = [&](int s) {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    constexpr uint32_t bytes = (uint32_t)(Sh::PADM * sizeof(cplx));
    mbar_expect_tx(mbar_g, 2 * bytes);
    const cplx* g = P4.Gp[s];
    bulk_g2s(smem_u32(ZE.p), g, bytes, mbar_g);
    bulk_g2s(smem_u32(ZO.p), g + Sh::PADM, bytes, mbar_g);
  };

  long long b = blockIdx.x;
  int s = 0;
  bool have = b < P.B;
  uint32_t par_rows = 0, par_g = 0;
  bool staged = false;
  if (have) {
    const double *dr, *hr; int nn;
    staged = rows(b, s, dr, hr, nn);
    if (tid == 0) { prefetch_rows(b, s); prefetch_g(s); }
  }
  while (have) {
    long long nb = b; int ns = s + 1;
    if (ns == P.n_seg) { ns = 0; nb = b + gridDim.x; }
    const bool have_next = (MODE != MODE_STOREZ || nb == b) && nb < P.B;
    const SegDev sg = segs[s];
    // ---------------- forward pass 1 (radix RF1, stride 256): both branches from one set of inputs
    {
      constexpr int NTASK = NF / RF1;  // 256
      constexpr int IT = NTASK / NT;
      static_assert(NTASK % NT == 0, "first pass tiling");
      if (staged) {
        mbar_wait(mbar_rows, par_rows);
        par_rows ^= 1;
        cplx xs[IT][RF1];
#pragma unroll
        for (int it = 0; it < IT; ++it) first_pass_load_staged<RF1, NF, MODE>(xs[it], tid + it * NT, stH, stD, sg.n);
        __syncthreads();  // staging consumed: the U region may now be overwritten
#pragma unroll
        for (int it = 0; it < IT; ++it) first_pass_compute<RF1, NF>(UE, UO, tid + it * NT, xs[it], tw);
      } else {
        const double *drow, *hrow; int n;
        rows(b, s, drow, hrow, n);
        const bool vec = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
#pragma unroll 1
        for (int g = tid; g < NTASK; g += NT) first_pass_c<RF1, NF, MODE>(UE, UO, g, drow, hrow, n, vec, tw);
      }
    }
    __syncthreads();
    // ---------------- forward passes 2 and 3, warp-local
    f4_forward23<TW>(U, own, lane, tw);
    __syncwarp();  // mirror-closed ownership: mid reads only this warp's U blocks
    // ---------------- mid: untangle (registers) x generator (in place in Z) -> first inverse pass
    mbar_wait(mbar_g, par_g);
    par_g ^= 1;
    f4_mid<NF, RF1>(U, Z, br, own, lane, tw);
    // the warp finishing mid last knows the U region is dead: it prefetches the next item's rows
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
    // ---------------- last inverse pass (radix RI1, joins the branches) + pruned radix-2 stage + S5
    double acc0 = 0.0, acc1 = 0.0;
#pragma unroll 1
    for (int g = tid; g < M / RI1; g += NT) last_pass_c<RI1, M, MODE>(ZE, ZO, g, sg.n, tw, sg.zd, acc0, acc1);
    if (MODE != MODE_STOREZ) {
      acc0 = warp_sum(acc0);
      acc1 = warp_sum(acc1);
    }
    // No CTA barrier at the end of an item: the warp that finishes the last pass last (a counter, as for mid) knows
    // that Z is consumed and every partial sum is in place; it prefetches the next generator spectrum into Z and
    // finishes the reduction (fixed order over the warps), while the other warps are already loading the next item's
    // staged rows.  `red` is rewritten only after the next item's barriers, which this warp has to pass as well.
    __syncwarp();
    if (lane == 0) {
      if (MODE != MODE_STOREZ) { red[2 * warp] = acc0; red[2 * warp + 1] = acc1; }
      __threadfence_block();
      const int old = atomicAdd(last_count, 1);
      if (old == NW - 1) {
        *last_count = 0;
        __threadfence_block();
        if (have_next) prefetch_g(ns);
        if (MODE != MODE_STOREZ) {
          double tot0 = totS[0], tot1 = totS[1];
#pragma unroll
          for (int wq = 0; wq < NW; ++wq) { tot0 += red[2 * wq]; tot1 += red[2 * wq + 1]; }
          if (s == P.n_seg - 1) {
            if (MODE == MODE_LOGLIKE) {
              const double v = -0.5 * tot1;
              P.out0[b] = P.accumulate ? P.out0[b] + v : v;
            } else {
              if (P.out0) P.out0[b] = P.accumulate ? P.out0[b] + tot0 : tot0;
              if (P.out1) P.out1[b] = P.accumulate ? P.out1[b] + tot1 : tot1;
            }
            tot0 = 0.0; tot1 = 0.0;
          }
          totS[0] = tot0; totS[1] = tot1;
        }
      }
    }
    b = nb; s = ns; have = have_next; staged = staged_next;
  }
}

}  // namespace td
