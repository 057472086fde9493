// td_fused4.cuh - the fused FFT-path kernel for M = 1024 / 2048 / 4096 (transform lengths
// 2M = 2048 / 4096 / 8192), built around two measurements (profiles/r02_c2_fused4_ncu.md, profiles/r01_peaks.md): CTA-wide barriers put every
// warp in the same load -> compute -> store phase, and whatever a thread needs again for every template costs
// shared-memory bandwidth each time unless it lives somewhere else.
//
//  * plans  NF = M/2 = [RF1,16,16],  M = [RI1,16,16],  RI1 = 2 RF1;  NT = 32 RF1 = M/16 threads;
//    warps [0, NW/2) own the even-bin branch, warps [NW/2, NW) the odd-bin branch.
//  * forward passes 2 and 3 touch only the 2 x 256 elements a warp owns: one __syncwarp between them.
//  * "mid": forward bins are untangled IN REGISTERS from the two mirror blocks, multiplied by the
//    generator spectrum and pushed through the first inverse radix-16 pass before they are stored.
//  * inverse pass 2 is again warp-local; only the last pass (which joins the two branches and
//    carries the fused quadratic reduction) needs the whole CTA.
//  * TENSOR MEMORY AS A CONSTANT CACHE: a thread multiplies the same 32 generator values, subtracts the same 16 data
//    samples and uses the same 15 twiddle powers for every template.  They are written once per (CTA, segment) into the
//    thread's private columns of the SM's 256 KB tensor memory (tcgen05.st) and read back with tcgen05.ld, a datapath
//    that shares nothing with shared memory or the fp64 pipe.  This replaces, per template, a 128 KB + 32 KB bulk copy
//    from L2, 160 KB of shared-memory reads and 80 fp64 instructions per thread.  Segments are the OUTER loop
//    (out[b] accumulates over them) so that the constants change n_seg times per kernel, not per item.
//  * the next item's template row is TMA-prefetched into the U region by whichever warp finishes mid last.
// CTA barriers per (template, segment): 4 (staging consumed, after pass 1, before the last pass; end of item is a counter).
#pragma once
#include "td_fused.cuh"
#include "td_dit16.cuh"
#include "td_ring.cuh"

namespace TD_NS {

constexpr int F4_SEGCACHE = 8;  // segment records cached in shared memory (more segments: read from global per item)

// TMEM columns of a thread, relative to its warp's column base (a complex number = TM_CPC columns: 4 in fp64, 2 in fp32;
// warps w and w + 4 share a lane quarter and take columns [0, 256) and [256, 512))
constexpr int F4_TC_G = 0;                  // 32 complex: the 2 x 16 generator values of mid
constexpr int F4_TC_D = 32 * TM_CPC;        // ND complex fp64 samples of the data vector (first forward pass; fp64 in both
                                            // precisions: the residual d - h is formed before rounding), 4 columns each
// ND = 8 (one-CTA kernel) or 16 (cluster kernel) data samples per thread; then 16 complex: twiddle powers of forward pass 2
template <int ND> struct F4Cols {
  static constexpr int TW = F4_TC_D + 4 * ND;
  static constexpr int USED = TW + 16 * TM_CPC;
  static constexpr int WINDOW = USED <= 128 ? 128 : 256;   // a thread's window: a power of two (allocation granularity)
  static_assert(USED <= 256, "a thread's TMEM window is at most 256 columns");
};

template <int LOG2M> struct Fused4Shape {
  static constexpr int M = 1 << LOG2M, NF = M / 2;
  static constexpr int RF1 = plan_r1(NF), RI1 = plan_r1(M);
  static_assert(plan_np(NF) == 3 && plan_np(M) == 3 && RI1 == 2 * RF1, "fused4 needs [R,16,16] plans");
  static constexpr int NT = 32 * RF1, NW = RF1, NWB = RF1 / 2;
  static constexpr int TWS = 2 * M / RF1;
  static constexpr int PADM = SmemArr::padded(M), PADNF = SmemArr::padded(NF);
  using Cols = F4Cols<8>;
  // Cols::WINDOW columns per thread (256 in fp64, 128 in fp32); warps w, w + 4, w + 8, .. of a CTA share a lane quarter
  static constexpr int tmem_cols(int ngrp) { return ((NW * ngrp + 3) / 4) * Cols::WINDOW; }
  static constexpr int TMEM_COLS = tmem_cols(1);
  // bytes of one item pipeline (NGRP > 1: several independent pipelines share a CTA, see the kernel), 16-byte granular
  static constexpr size_t group_bytes() { return (smem_bytes() + 15) & ~(size_t)15; }
  // layout of a CTA with NGRP pipelines: [U, Z of every pipeline] [ONE base-twiddle table] [sums, mbarriers, segment cache of
  // every pipeline]; with one pipeline this is the layout smem_bytes() describes
  static constexpr size_t uz_bytes() { return sizeof(cplx) * (2 * (size_t)PADNF + 2 * (size_t)PADM); }
  static constexpr size_t tw_bytes() { return sizeof(cplx) * (size_t)TWS; }
  static constexpr size_t tail_bytes() { return group_bytes() - uz_bytes() - tw_bytes(); }
  static constexpr size_t total_bytes(int ngrp) { return ngrp * (uz_bytes() + tail_bytes()) + tw_bytes(); }
  static constexpr size_t smem_bytes() {
    return sizeof(cplx) * (2 * (size_t)PADNF + 2 * (size_t)PADM + TWS) + sizeof(double) * 4 * NW + 48 + F4_SEGCACHE * sizeof(SegDev) +
           96   // RingConsts of the item in flight (SYN kernels)
#ifdef TD_PHASE_CLOCKS
           + 16 * 16 * sizeof(long long)
#endif
        ;
  }
};

struct Fused4Params {
  FusedParams base;
  const cplx* const* Gp;  // device array [n_seg]: generator spectrum in the PADDED Z layout [2][padded(M)]
  double fs;              // SYN kernels: sampling rate; base.H then holds the parameter rows [B][ldh], ldh = 5 x (segments of the
                          // handle), the row of segment record sg at 5 sg._pad (td_ring.cuh)
#ifdef TD_DEBUG_KNOBS
  int skew;               // debug builds: cycles the odd-bin warps wait after the barrier that follows pass 1
#endif
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

// forward passes 2 and 3, warp-local (this warp owns U blocks o.u0, o.u1 of its branch).
// TWT: the sixteen twiddle powers of pass 2 come from the thread's TMEM columns at `ttw` (64 columns, written once per
// kernel by f4_store_twiddles) instead of being rebuilt for every item.
template <int TW, bool TWT = false>
__device__ __forceinline__ void f4_forward23(const SmemArr& U, const F4Own& o, int lane, const cplx* __restrict__ tw,
                                             uint32_t ttw = 0) {
  cplx x[16];
  {
    const int s1 = (lane >> 4) ? o.u1 : o.u0, j = lane & 15;
    const int base = s1 * 256 + j;
    cplx w[16];
    TmemC16 wr;
    if constexpr (TWT) {
      wr.ld(ttw);
    } else {
      tw_powers<16>(tw[j * (TW / 256)], w);
    }
#pragma unroll
    for (int q = 0; q < 16; ++q) x[q] = U.ld(base + 16 * q);
    if constexpr (TWT) {
      tmem_wait_ld();
      wr.use();
#pragma unroll
      for (int q = 0; q < 16; ++q) w[q] = wr.get(q);
    }
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
// the powers w_256^(j t), t = 0..15, j = lane & 15, of forward pass 2 into 64 TMEM columns at ttw (once per kernel)
template <int TW>
__device__ __forceinline__ void f4_store_twiddles(int lane, const cplx* __restrict__ tw, uint32_t ttw) {
  cplx w[16];
  tw_powers<16>(tw[(lane & 15) * (TW / 256)], w);
#pragma unroll
  for (int q = 0; q < 16; ++q) tmem_st_c(ttw + TM_CPC * q, w[q]);
}

// this lane's 2 x 16 generator values (g = one branch of the segment's spectrum in the padded Z layout, global memory)
// into 128 TMEM columns at tg: once per (CTA, segment) instead of a 128 KB bulk copy and 128 KB of shared-memory reads
// per item.  The element order is the one f4_mid multiplies in.
__device__ __forceinline__ void f4_store_generator(const cplx* __restrict__ g, const F4Own& o, int lane, uint32_t tg) {
  const int q4 = lane >> 3;
  const int s1 = q4 == 0 ? o.z0 : q4 == 1 ? o.z2 : q4 == 2 ? o.z1 : o.z3, s2 = lane & 7;  // (half-warps: {z0, z2}, {z1, z3})
  // all 32 loads are issued before the first (volatile) TMEM store, so their latencies overlap
  cplx v[2][16];
#pragma unroll
  for (int par = 0; par < 2; ++par) {
    const int zb = (s1 * 16 + s2) * 16 + par * 8 * 16;
#pragma unroll
    for (int q = 0; q < 16; ++q) {
      const int i = zb + q;
      v[par][q] = __ldg(g + i + (i >> 4));
    }
  }
#pragma unroll
  for (int par = 0; par < 2; ++par)
#pragma unroll
    for (int q = 0; q < 16; ++q) tmem_st_c(tg + TM_CPC * (16 * par + q), v[par][q]);
}

// mid: untangle (registers) x generator -> first inverse pass.  GT: the generator values come from TMEM (tg, see
// f4_store_generator); otherwise they sit in Z (bulk-copied there in the padded layout) and are multiplied in place.
// Quarter-warp q4 works on Z block z0, z2, z1, z3 (in that order): z0 and z2 = z0 + RF1 read the two halves of the same
// forward block pair, so with 8-byte elements (fp32 build, half-warp wavefronts) the 16 lanes of a half-warp fall on 16
// different bank pairs; with 16-byte elements a wavefront is a quarter-warp and either order is conflict-free.
template <int NF, int RF1, bool GT = false>
__device__ __forceinline__ void f4_mid(const SmemArr& U, const SmemArr& Z, int br, const F4Own& o, int lane,
                                       const cplx* __restrict__ tw, uint32_t tg = 0) {
  constexpr int RI1 = 2 * RF1;
  const int q4 = lane >> 3;
  const int s1 = q4 == 0 ? o.z0 : q4 == 1 ? o.z2 : q4 == 2 ? o.z1 : o.z3, s2 = lane & 7;  // (half-warps: {z0, z2}, {z1, z3})
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
  // Two halves (even t -> inverse block tau, odd t -> block tau + M/32), software-pipelined: the U loads of half 1 are in
  // flight while half 0 runs its radix-16 butterfly, and half 0's stores drain while half 1 computes.
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
  auto load_g = [&](auto par) {
    constexpr int pp = decltype(par)::value;
    if constexpr (GT) {
      gr.ld(tg + 16 * TM_CPC * pp);
    } else {
#pragma unroll
      for (int q = 0; q < 16; ++q) e[q] = Z.ld(zb0 + pp * 8 * 16 + q);  // generator spectrum sits in Z
    }
  };
  auto untangle = [&](auto par) {  // ua, ub, generator -> e
    constexpr int pp = decltype(par)::value;
    if constexpr (GT) {
      tmem_wait_ld();
      gr.use();
#pragma unroll
      for (int q = 0; q < 16; ++q) e[q] = gr.get(q);
    }
    static_for<0, 8>([&](auto hh) {
      constexpr int h8 = decltype(hh)::value, t = 2 * h8 + pp;
      const cplx U1 = ua[h8], U2 = ub[h8];
      const cplx A = mk(U1.x + U2.x, U1.y - U2.y);
      const cplx Bv = mk(U1.y + U2.y, -(U1.x - U2.x));
      const cplx wB = cmul(basew, mul_w32<t, false>(Bv));
      e[h8] = cmul(e[h8], cadd(A, wB));          // G * 2 X_{kq},      entry s = t/2
      e[8 + h8] = cmul(e[8 + h8], csub(A, wB));  // G * 2 X_{NF + kq}, entry s = 8 + t/2
    });
  };
  auto store_e = [&](auto par) {
    constexpr int pp = decltype(par)::value;
    static_for<0, 16>([&](auto t) { Z.st(zb0 + pp * 8 * 16 + decltype(t)::value, e[brevR<16>(decltype(t)::value)]); });
  };
  load_g(IC<0>{});
  load_u(IC<0>{});
  untangle(IC<0>{});
  if constexpr (GT) {
    load_g(IC<1>{});
    load_u(IC<1>{});   // in flight during the butterfly below
  }
  dit16<true, false>(e, mk(real(1), real(0)));
  store_e(IC<0>{});
  if constexpr (!GT) {
    load_g(IC<1>{});   // e is the landing area of the generator values on this path: only now free
    load_u(IC<1>{});
  }
  untangle(IC<1>{});
  dit16<true, false>(e, mk(real(1), real(0)));
  store_e(IC<1>{});
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

#ifdef TD_PHASE_CLOCKS
// debug builds only (_work probes): per-warp cycle counts of every phase of the item loop
__device__ long long g_phase_clk[148 * 16 * 16];
#define TDCLK(k) do { if (lane == 0) { const long long t_ = clock64(); clk_s[warp * 16 + (k)] += t_ - tlast; tlast = t_; } } while (0)
#else
#define TDCLK(k) do { } while (0)
#endif

// NGRP > 1: the CTA holds NGRP independent item pipelines ("groups" of NT threads, each with its own shared-memory regions,
// mbarrier, named barrier and TMEM windows) that work on different templates.  A kernel that uses tensor memory is limited
// to one CTA per SM (profiles/r02_c2_fused4_ncu.md), so this is how the fp32 build - whose working set and register need
// are half the fp64 ones - puts two items on an SM: their load / butterfly / store phases interleave instead of adding up.
// SYN = 1: the template rows are damped sinusoids synthesised from 5 parameters per (template, segment) inside the first
// pass (td_ring.cuh) - no row in memory, no TMA copy; MODE_LOGLIKE only.
template <int LOG2M, int MODE, int NGRP = 1, int SYN = 0>
__global__ void __launch_bounds__(Fused4Shape<LOG2M>::NT * NGRP, 1) td_fused4_kernel(const Fused4Params P4) {
  static_assert(SYN == 0 || MODE == MODE_LOGLIKE, "synthesis is wired into the log-likelihood mode only");
  using Sh = Fused4Shape<LOG2M>;
  constexpr int M = Sh::M, NF = Sh::NF, TW = 2 * M, NT = Sh::NT, NW = Sh::NW, NWB = Sh::NWB;
  constexpr int TMEM_COLS = Sh::tmem_cols(NGRP);
  static_assert(TMEM_COLS <= 512 && (TMEM_COLS & (TMEM_COLS - 1)) == 0, "tensor memory: 512 columns, power-of-two allocations");
  constexpr int RF1 = Sh::RF1, RI1 = Sh::RI1;
  constexpr int NTASK = NF / RF1, IT = NTASK / NT, S1 = NF / RF1;  // first pass: IT tasks of radix RF1 per thread
  static_assert(NTASK % NT == 0 && IT * RF1 == 8, "first pass tiling: 8 complex inputs per thread");
  const FusedParams& P = P4.base;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int grp = NGRP == 1 ? 0 : (int)threadIdx.x / NT;              // item pipeline of this thread
  // pipelines are what items are dealt to, pipeline 0 of every CTA first: a small batch spreads over the SMs before it stacks up on them
  const int vblock = grp * (int)gridDim.x + (int)blockIdx.x, vgrid = (int)gridDim.x * NGRP;
  auto group_sync = [&]() {
    if constexpr (NGRP == 1) __syncthreads();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + grp), "r"(NT) : "memory");
  };
  cplx* sm = reinterpret_cast<cplx*>(smem_raw + (size_t)grp * Sh::uz_bytes());
  const SmemArr UE{sm}, UO{sm + Sh::PADNF};
  const SmemArr ZE{sm + 2 * Sh::PADNF}, ZO{sm + 2 * Sh::PADNF + Sh::PADM};
  cplx* tw = reinterpret_cast<cplx*>(smem_raw + (size_t)NGRP * Sh::uz_bytes());   // ONE base-twiddle table for all pipelines
  unsigned char* tail0 = smem_raw + (size_t)NGRP * Sh::uz_bytes() + Sh::tw_bytes();
  double* red = reinterpret_cast<double*>(tail0 + (size_t)grp * Sh::tail_bytes());  // [2][2 NW]: per-warp partial sums, double-buffered by item parity
  const uint32_t mbar_rows = smem_u32(red + 4 * NW);
  // (one allocation for the CTA: every group reads group 0's slot)
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(reinterpret_cast<double*>(tail0) + 4 * NW + 1);
  SegDev* segS = reinterpret_cast<SegDev*>(red + 4 * NW + 3);
  const SegDev* segs = P.n_seg <= F4_SEGCACHE ? segS : P.segs;
  RingConsts* rcs = reinterpret_cast<RingConsts*>(segS + F4_SEGCACHE);
  double* stH = reinterpret_cast<double*>(sm);  // the staged template row lives in the U region (dead after mid)
  const int tid = (int)threadIdx.x - grp * NT, warp = tid >> 5, lane = tid & 31;   // within the group
  const int cwarp = (int)threadIdx.x >> 5;                                        // within the CTA (TMEM lane quarter, window)
  const int br = warp / NWB, wb = warp - br * NWB;  // branch (0 even bins, 1 odd bins), warp within branch
  const SmemArr U = br ? UO : UE, Z = br ? ZO : ZE;
  const F4Own own = f4_own<RF1, true>(br, wb);

  // the base-twiddle table arrives by one bulk copy (it was NT-strided global loads: the longest piece of the prologue, which is
  // most of a launch when a CTA has a single item, as on c1)
  const uint32_t mbar_tw = smem_u32(reinterpret_cast<double*>(tail0) + 4 * NW) + 16;   // pipeline 0's: it fetches the table for all
  if (tid < P.n_seg && tid < F4_SEGCACHE) segS[tid] = P.segs[tid];
  if (tid == 0) {
    mbar_init(mbar_rows, 1);
    if (grp == 0) {
      mbar_init(mbar_tw, 1);
      mbar_expect_tx(mbar_tw, (uint32_t)(Sh::TWS * sizeof(cplx)));
      bulk_g2s(smem_u32(tw), P.T, (uint32_t)(Sh::TWS * sizeof(cplx)), mbar_tw);
    }
  }
  if (cwarp == 0) tmem_alloc<TMEM_COLS>(smem_u32(tmem_slot));
#ifdef TD_PHASE_CLOCKS
  long long* clk_s = reinterpret_cast<long long*>(reinterpret_cast<unsigned char*>(segS + F4_SEGCACHE) + 96);
  if (tid < 16 * NW) clk_s[tid] = 0;
  long long tlast = clock64();
#endif
  tmem_fence_before();
  __syncthreads();
  tmem_fence_after();
  // this thread's TMEM window: lane 32 (warp % 4) + lane, Cols::WINDOW columns
  const uint32_t tcol = *tmem_slot + ((uint32_t)(32 * (cwarp & 3)) << 16) + (uint32_t)((cwarp >> 2) * Sh::Cols::WINDOW);
  mbar_wait(mbar_tw, 0);
  f4_store_twiddles<TW>(lane, tw, tcol + Sh::Cols::TW);

  // rows of item (b, s); the template row is staged by TMA when it is 16-byte aligned and N_s is even
  auto rows = [&](long long b, int s, const double*& drow, const double*& hrow, int& n) -> bool {
    const SegDev sg = segs[s];
    drow = P.d + sg.off;
    hrow = (MODE == MODE_STOREZ) ? drow : P.H + b * P.ldh + sg.off;
    n = sg.n;
    if constexpr (SYN) return true;   // nothing to stage: the "row" is 5 parameters
    return ((reinterpret_cast<uintptr_t>(hrow) & 15) == 0) && ((n & 1) == 0);
  };
  // SYN: warp 0 computes the constants of item (b, s) into shared memory and completes the phase of the mbarrier that the
  // first pass waits on (the hand-over a TMA row copy makes with its byte count)
  auto prepare_consts = [&](long long b, int s) {  // executed by WARP 0
    const SegDev sg2 = segs[s];
    ring_prepare(P.H + b * P.ldh + 5 * sg2._pad, P4.fs, 2 * NT, lane, rcs);
    __syncwarp();
    if (lane == 0) mbar_arrive(mbar_rows);
  };
  auto prefetch_rows = [&](long long b, int s) {  // issued by ONE thread
    const double *drow, *hrow; int n;
    if (rows(b, s, drow, hrow, n)) {
      asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
      const uint32_t bytes = (uint32_t)n * 8u;
      mbar_expect_tx(mbar_rows, bytes);
      bulk_g2s(smem_u32(stH), hrow, bytes, mbar_rows);
    }
  };

  const long long Bs = (MODE == MODE_STOREZ) ? 1 : P.B;  // STOREZ transforms the data vector itself, once per segment
  const bool active = (long long)vblock < Bs;             // (a pipeline without items still takes part in the CTA barriers)
  // The partial sums of an item are combined (fixed order over the warps) by thread 0 after the first CTA barrier of the
  // NEXT item: no atomics, no fences, no barrier at the end of an item.  Segments accumulate into out[b].
  long long pend_b = -1;
  int pend_add = 0, item = 0;
  auto finalize = [&]() {  // thread 0 only
    if (MODE != MODE_STOREZ && pend_b >= 0) {
      const double* r = red + 2 * NW * ((item & 1) ^ 1);   // the previous item's buffer
      double tot0 = 0.0, tot1 = 0.0;
#pragma unroll
      for (int wq = 0; wq < NW; ++wq) { tot0 += r[2 * wq]; tot1 += r[2 * wq + 1]; }
      if (MODE == MODE_LOGLIKE) {
        const double v = -0.5 * tot1;
        P.out0[pend_b] = pend_add ? P.out0[pend_b] + v : v;
      } else {
        if (P.out0) P.out0[pend_b] = pend_add ? P.out0[pend_b] + tot0 : tot0;
        if (P.out1) P.out1[pend_b] = pend_add ? P.out1[pend_b] + tot1 : tot1;
      }
      pend_b = -1;
    }
  };
  uint32_t par_rows = 0;
  bool staged;
  {
    const double *dr, *hr; int nn;
    staged = rows(vblock, 0, dr, hr, nn);
    if constexpr (SYN) { if (warp == 0 && active) prepare_consts(vblock, 0); }
    else if (tid == 0 && active) prefetch_rows(vblock, 0);
  }
  for (int s = 0; active && s < P.n_seg; ++s) {
    const SegDev sg = segs[s];
    // ---------------- per-segment constants into this thread's TMEM columns: generator values, data samples
    f4_store_generator(P4.Gp[s] + (size_t)br * Sh::PADM, own, lane, tcol + F4_TC_G);
    if (MODE == MODE_LOGLIKE) {
      const double* drow = P.d + sg.off;
      double2 dvs[IT * RF1];   // loads first, (volatile) TMEM stores after: the latencies overlap
#pragma unroll
      for (int it = 0; it < IT; ++it)
#pragma unroll
        for (int ss = 0; ss < RF1; ++ss) {
          const int i0 = 2 * (tid + it * NT + ss * S1);
          dvs[it * RF1 + ss] = make_double2(i0 < sg.n ? __ldg(drow + i0) : 0.0, i0 + 1 < sg.n ? __ldg(drow + i0 + 1) : 0.0);
        }
#pragma unroll
      for (int q = 0; q < IT * RF1; ++q) tmem_st_c64(tcol + F4_TC_D + 4 * q, dvs[q]);
    }
    tmem_wait_st();
    for (long long b = vblock; b < Bs; b += vgrid) {
      long long nb = b + vgrid; int ns = s;
      if (nb >= Bs) { nb = vblock; ns = s + 1; }
      const bool have_next = ns < P.n_seg;
      // ---------------- forward pass 1 (radix RF1, stride 256): both branches from one set of inputs
      if (staged) {
        int dr[2][16];
        if (MODE == MODE_LOGLIKE) { tmem_ld16(tcol + F4_TC_D, dr[0]); tmem_ld16(tcol + F4_TC_D + 16, dr[1]); }
        TDCLK(0);
        mbar_wait(mbar_rows, par_rows);
        par_rows ^= 1;
        TDCLK(1);
        cplx xs[IT][RF1];
        double2 hs[IT][RF1];   // the staged samples, fp64 in both precisions
        if constexpr (SYN) {
          // this thread's pairs are 2 tid + 2 NT k, k = it + IT ss (2 NT IT = 2 S1): synthesised, never read
          static_assert(2 * NT * IT == 2 * S1, "pair indices of a thread form one arithmetic progression");
          const RingConsts rc = *rcs;
          double2 hf[IT * RF1];
          ring_pairs<IT * RF1>(rc, 2 * tid, ilog2(2 * NT), sg.n, hf);
#pragma unroll
          for (int it = 0; it < IT; ++it)
#pragma unroll
            for (int ss = 0; ss < RF1; ++ss) hs[it][ss] = hf[it + IT * ss];
        } else {
#pragma unroll
        for (int it = 0; it < IT; ++it)
#pragma unroll
          for (int ss = 0; ss < RF1; ++ss) {
            const int i0 = 2 * (tid + it * NT + ss * S1);
            double2 hv = make_double2(0.0, 0.0);
            if (i0 < sg.n) hv = *reinterpret_cast<const double2*>(stH + i0);  // n even on this path: i0 + 1 < n too
            hs[it][ss] = hv;
          }
        }
        if (MODE == MODE_LOGLIKE) {
          tmem_wait_ld();
          tmem_use16(dr[0]); tmem_use16(dr[1]);
#pragma unroll
          for (int it = 0; it < IT; ++it)
#pragma unroll
            for (int ss = 0; ss < RF1; ++ss) {
              const double2 dv = tmem_c64(dr[(it * RF1 + ss) >> 2], (it * RF1 + ss) & 3);
              const double2 hv = hs[it][ss];
              // S1: r = d - h, formed in fp64 (the fp32 build scales by rscale and rounds once; h = d stays exactly 0)
              xs[it][ss] = to_cplx(dv.x - hv.x, dv.y - hv.y, sg.rscale);
            }
        } else {
#pragma unroll
          for (int it = 0; it < IT; ++it)
#pragma unroll
            for (int ss = 0; ss < RF1; ++ss) xs[it][ss] = to_cplx(hs[it][ss].x, hs[it][ss].y, sg.rscale);
        }
        TDCLK(2);
        group_sync();  // staging consumed: the U region may now be overwritten
        TDCLK(3);
#pragma unroll
        for (int it = 0; it < IT; ++it) first_pass_compute<RF1, NF>(UE, UO, tid + it * NT, xs[it], tw);
        TDCLK(4);
      } else {
        const double *drow, *hrow; int n;
        rows(b, s, drow, hrow, n);
        const bool vec = ((reinterpret_cast<uintptr_t>(drow) | reinterpret_cast<uintptr_t>(hrow)) & 15) == 0;
#pragma unroll 1
        for (int g = tid; g < NTASK; g += NT) first_pass_c<RF1, NF, MODE>(UE, UO, g, drow, hrow, n, vec, tw, sg.rscale);
      }
      group_sync();
      if (tid == 0) finalize();  // the previous item's sums: every warp has passed its last pass
#ifdef TD_DEBUG_KNOBS
      if (br && P4.skew > 0) { const long long t_ = clock64(); while (clock64() - t_ < P4.skew) { } }
#endif
      TDCLK(5);
      // ---------------- forward passes 2 and 3, warp-local
      f4_forward23<TW, true>(U, own, lane, tw, tcol + Sh::Cols::TW);
      __syncwarp();  // mirror-closed ownership: mid reads only this warp's U blocks
      TDCLK(6);
      // ---------------- mid: untangle (registers) x generator (TMEM) -> first inverse pass -> Z
      f4_mid<NF, RF1, true>(U, Z, br, own, lane, tw, tcol + F4_TC_G);
      TDCLK(8);
      bool staged_next = false;
      if (have_next) { const double *dr, *hr; int nn; staged_next = rows(nb, ns, dr, hr, nn); }
      TDCLK(9);
      // ---------------- inverse pass 2 (L = 256), warp-local
      f4_inverse2<TW>(Z, own, lane, tw);
      TDCLK(10);
      group_sync();
      // every warp is past mid: the U region is dead and takes the next item's template row
      if constexpr (SYN) { if (warp == 0 && have_next) prepare_consts(nb, ns); }
      else if (tid == 0 && have_next) prefetch_rows(nb, ns);
      TDCLK(11);
      // ---------------- last inverse pass (radix RI1, joins the branches) + pruned radix-2 stage + S5
      double acc0 = 0.0, acc1 = 0.0;
#pragma unroll 1
      for (int g = tid; g < M / RI1; g += NT) last_pass_c<RI1, M, MODE>(ZE, ZO, g, sg.n, tw, sg.zd, acc0, acc1);
      if (MODE == MODE_INNER) acc0 = warp_sum(acc0);
      if (MODE != MODE_STOREZ) acc1 = warp_sum(acc1);
      TDCLK(12);
      if (MODE != MODE_STOREZ && lane == 0) {
        double* r = red + 2 * NW * (item & 1);
        r[2 * warp] = acc0; r[2 * warp + 1] = acc1;
      }
      if (tid == 0) { pend_b = b; pend_add = (P.accumulate || s > 0) ? 1 : 0; }
      ++item;
      staged = staged_next;
    }
  }
  group_sync();
  if (tid == 0 && active) finalize();
  if constexpr (NGRP > 1) __syncthreads();   // every pipeline is done with its TMEM windows
  if (cwarp == 0) tmem_dealloc<TMEM_COLS>(*tmem_slot);
#ifdef TD_PHASE_CLOCKS
  if (tid < 16 * NW && blockIdx.x < 148) g_phase_clk[blockIdx.x * 256 + tid] = clk_s[tid];
#endif
}

}  // namespace TD_NS
