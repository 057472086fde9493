// td_common.cuh - complex helpers, in-register radix-R FFT butterflies, twiddle chains and
// mixed-radix index maps shared by the fused (shared-memory) and staged (global-memory) FFT
// kernels of the Gohberg-Semencul / circulant-embedding path (Eqs. 14-16).
// The scalar type is a compile-time choice of the translation unit: fp64 (namespace td, tdlike.cu) or, with TD_F32
// defined, fp32 (namespace td32, tdlike_f32.cu: the FP32 evaluation mode of PAPER.md:322-324, III.C.3 - operators
// precomputed in fp64, rounded once, evaluation in fp32).  Both see the same source; `real` / `cplx` are the only types
// that differ, every literal that enters arithmetic is typed `real`.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#ifdef TD_F32
#define TD_NS td32
#else
#define TD_NS td
#endif

namespace TD_NS {

#ifdef TD_F32
typedef float real;
typedef float2 cplx;
constexpr bool F32 = true;
#else
typedef double real;
typedef double2 cplx;
constexpr bool F32 = false;
#endif

// what a batch kernel accumulates: -1/2 <d-h, d-h> | (<d,h>, <h,h>) | nothing (stores z of the data vector)
enum { MODE_LOGLIKE = 0, MODE_INNER = 1, MODE_STOREZ = 2 };

__host__ __device__ __forceinline__ cplx mk(real x, real y) { cplx c; c.x = x; c.y = y; return c; }
__device__ __forceinline__ cplx cadd(cplx a, cplx b) { return mk(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ cplx csub(cplx a, cplx b) { return mk(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ cplx cconj(cplx a) { return mk(a.x, -a.y); }
// a * b
__device__ __forceinline__ cplx cmul(cplx a, cplx b) {
  return mk(fma(a.x, b.x, -(a.y * b.y)), fma(a.x, b.y, a.y * b.x));
}
// a * conj(b)
__device__ __forceinline__ cplx cmulc(cplx a, cplx b) {
  return mk(fma(a.x, b.x, a.y * b.y), fma(a.y, b.x, -(a.x * b.y)));
}
__device__ __forceinline__ cplx csq(cplx a) { return mk(fma(a.x, a.x, -(a.y * a.y)), real(2) * a.x * a.y); }

// ---- compile-time loops ---------------------------------------------------------------
template <int I> struct IC { static constexpr int value = I; };
template <int B, int E, class F> __device__ __forceinline__ void static_for(F&& f) {
  if constexpr (B < E) {
    f(IC<B>{});
    static_for<B + 1, E>(f);
  }
}
__host__ __device__ constexpr int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n >> 1); }
__host__ __device__ constexpr int brev_bits(int k, int bits) {
  int r = 0;
  for (int i = 0; i < bits; ++i) r |= ((k >> i) & 1) << (bits - 1 - i);
  return r;
}

// ---- constants cos/sin(2 pi k / 32) ------------------------------------------------------
__host__ __device__ constexpr double cos32q(int k) {  // k in [0, 8]
  return k == 0 ? 1.0
       : k == 1 ? 0.98078528040323044912618223613424
       : k == 2 ? 0.92387953251128675612818318939679
       : k == 3 ? 0.83146961230254523707878837761791
       : k == 4 ? 0.70710678118654752440084436210485
       : k == 5 ? 0.55557023301960222474283081394853
       : k == 6 ? 0.38268343236508977172845998403040
       : k == 7 ? 0.19509032201612826784828486847702
                : 0.0;
}
__host__ __device__ constexpr double cos32(int k) {
  k &= 31;
  return k <= 8 ? cos32q(k) : k <= 16 ? -cos32q(16 - k) : k <= 24 ? -cos32q(k - 16) : cos32q(32 - k);
}
__host__ __device__ constexpr double sin32(int k) { return cos32(k - 8); }

// a * w32^K (forward: w32 = exp(-2 pi i / 32)) or a * conj(w32)^K (INV)
template <int K, bool INV> __device__ __forceinline__ cplx mul_w32(cplx a) {
  constexpr int k = K & 31;
  if constexpr (k == 0) return a;
  else if constexpr (k == 16) return mk(-a.x, -a.y);
  else if constexpr (k == 8) return INV ? mk(-a.y, a.x) : mk(a.y, -a.x);
  else if constexpr (k == 24) return INV ? mk(a.y, -a.x) : mk(-a.y, a.x);
  else {
    constexpr real c = (real)cos32(k), s = (real)sin32(k);
    if constexpr (!INV) return mk(fma(a.x, c, a.y * s), fma(a.y, c, -(a.x * s)));
    else return mk(fma(a.x, c, -(a.y * s)), fma(a.y, c, a.x * s));
  }
}

// In-register radix-R DFT (R = 2,4,8,16) by radix-2 DIF stages.  On return X_k (k natural)
// is held in x[brev(k)].  Forward kernel exp(-2 pi i s k / R); INV uses the conjugate.
template <int R, bool INV> __device__ __forceinline__ void fft_reg(cplx (&x)[R]) {
  constexpr int LG = ilog2(R);
  static_for<0, LG>([&](auto st) {
    constexpr int half = R >> (decltype(st)::value + 1);
    static_for<0, R / 2>([&](auto q) {
      constexpr int blk = (decltype(q)::value / half) * 2 * half;
      constexpr int j = decltype(q)::value % half;
      cplx a = x[blk + j], b = x[blk + j + half];
      x[blk + j] = cadd(a, b);
      x[blk + j + half] = mul_w32<j * (16 / half), INV>(csub(a, b));
    });
  });
}
template <int R> __host__ __device__ constexpr int brevR(int k) { return brev_bits(k, ilog2(R)); }

// w[t] = w1^t, t = 1..R-1 (w[0] unused), by a squaring/multiply tree of depth <= log2(R)+2.
template <int R> __device__ __forceinline__ void tw_powers(cplx w1, cplx (&w)[R]) {
  w[0] = mk(real(1), real(0));
  if constexpr (R > 1) w[1] = w1;
  static_for<2, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    if constexpr ((tt & 1) == 0) w[tt] = csq(w[tt / 2]);
    else w[tt] = cmul(w[tt - 1], w1);
  });
}

// ---- mixed-radix plan [R1, 16, 16, ...] ----------------------------------------------------
// n = R1 * 16^(np-1), R1 in {2,4,8,16}.  A DIF forward transform with this plan leaves X_k at
// position pos(k); the DIT inverse with the mirrored pass order consumes that same order.
__host__ __device__ constexpr int plan_np(int n) { return (ilog2(n) + 3) / 4; }
__host__ __device__ constexpr int plan_r1(int n) { return n >> (4 * (plan_np(n) - 1)); }

__host__ __device__ __forceinline__ int ilog2_rt(int n) {
#ifdef __CUDA_ARCH__
  return 31 - __clz(n);
#else
  return ilog2(n);
#endif
}
__host__ __device__ __forceinline__ int plan_pos(int k, int n) {
  // n is a power of two: shifts and masks only (this runs per element in the staged untangle kernel)
  const int logn = ilog2_rt(n), np = (logn + 3) >> 2, lr1 = logn - 4 * (np - 1);
  int sh = logn - lr1;
  int p = (k & ((1 << lr1) - 1)) << sh;
  k >>= lr1;
  while (sh > 0) {
    sh -= 4;
    p += (k & 15) << sh;
    k >>= 4;
  }
  return p;
}
// inverse map: frequency index held at position p
__host__ __device__ __forceinline__ int plan_freq(int p, int n) {
  const int logn = ilog2_rt(n), np = (logn + 3) >> 2, lr1 = logn - 4 * (np - 1);
  int sh = logn - lr1;
  int k = p >> sh;
  int mul = lr1;
  while (sh > 0) {
    sh -= 4;
    k += ((p >> sh) & 15) << mul;
    mul += 4;
  }
  return k;
}

// compile-time version of the same maps (all shifts and masks)
template <int N> struct PlanT {
  static constexpr int LOGN = ilog2(N), NP = plan_np(N), R1 = plan_r1(N), LR1 = ilog2(R1);
  __device__ static __forceinline__ int pos(int k) {
    int p = (k & (R1 - 1)) << (LOGN - LR1);
    k >>= LR1;
#pragma unroll
    for (int q = 1; q < NP; ++q) {
      p += (k & 15) << (LOGN - LR1 - 4 * q);
      k >>= 4;
    }
    return p;
  }
  __device__ static __forceinline__ int freq(int p) {
    int k = p >> (LOGN - LR1);
#pragma unroll
    for (int q = 1; q < NP; ++q) k += ((p >> (LOGN - LR1 - 4 * q)) & 15) << (LR1 + 4 * (q - 1));
    return k;
  }
};

// ---- array accessors --------------------------------------------------------------------
// shared memory, padded one element per 16 so that stride-16 (last-pass) and contiguous
// (other passes) accesses are both bank-conflict free for 16-byte elements.
struct SmemArr {
  cplx* p;
  __device__ __forceinline__ cplx ld(int i) const { return p[i + (i >> 4)]; }
  __device__ __forceinline__ void st(int i, cplx v) const { p[i + (i >> 4)] = v; }
  __host__ __device__ static constexpr int padded(int n) { return n + (n >> 4); }
};
struct GmemArr {
  cplx* p;
  __device__ __forceinline__ cplx ld(int i) const { return p[i]; }
  __device__ __forceinline__ void st(int i, cplx v) const { p[i] = v; }
};

// ---- one butterfly task of a pass ---------------------------------------------------------
// DIF (forward): sub-transform length L, radix R, stride S = L/R, butterfly g:
//   x_s = A[base + s S];  X = DFT_R(x);  A[base + t S] = X_t * w[t]   (w[t] = w_L^{j t}; skipped if !tw)
template <int R, class Arr>
__device__ __forceinline__ void dif_task(const Arr& A, int L, int g, const cplx (&w)[R], bool tw) {
  const int S = L / R;
  const int blk = g / S, j = g - blk * S;
  const int base = blk * L + j;
  cplx x[R];
#pragma unroll
  for (int s = 0; s < R; ++s) x[s] = A.ld(base + s * S);
  fft_reg<R, false>(x);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    cplx v = x[brevR<R>(tt)];
    if (tt > 0 && tw) v = cmul(v, w[tt]);
    A.st(base + tt * S, v);
  });
}
// DIT (inverse): x_s = A[base + s S] * conj(w[s]);  X = conj-DFT_R(x);  A[base + t S] = X_t
template <int R, class Arr>
__device__ __forceinline__ void dit_task(const Arr& A, int L, int g, const cplx (&w)[R], bool tw) {
  const int S = L / R;
  const int blk = g / S, j = g - blk * S;
  const int base = blk * L + j;
  cplx x[R];
  static_for<0, R>([&](auto s) {
    constexpr int ss = decltype(s)::value;
    cplx v = A.ld(base + ss * S);
    if (ss > 0 && tw) v = cmulc(v, w[ss]);
    x[ss] = v;
  });
  fft_reg<R, true>(x);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    A.st(base + tt * S, x[brevR<R>(tt)]);
  });
}

// compile-time-shape variants (S, masks and shifts fold to constants)
template <int R, int L, class Arr>
__device__ __forceinline__ void dif_task_c(const Arr& A, int g, const cplx (&w)[R]) {
  constexpr int S = L / R, LS = ilog2(S);
  const int blk = g >> LS, j = g & (S - 1);
  const int base = blk * L + j;
  cplx x[R];
#pragma unroll
  for (int s = 0; s < R; ++s) x[s] = A.ld(base + s * S);
  fft_reg<R, false>(x);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    cplx v = x[brevR<R>(tt)];
    if constexpr (tt > 0 && (S > 1)) v = cmul(v, w[tt]);
    A.st(base + tt * S, v);
  });
}
template <int R, int L, class Arr>
__device__ __forceinline__ void dit_task_c(const Arr& A, int g, const cplx (&w)[R]) {
  constexpr int S = L / R, LS = ilog2(S);
  const int blk = g >> LS, j = g & (S - 1);
  const int base = blk * L + j;
  cplx x[R];
  static_for<0, R>([&](auto s) {
    constexpr int ss = decltype(s)::value;
    cplx v = A.ld(base + ss * S);
    if constexpr (ss > 0 && (S > 1)) v = cmulc(v, w[ss]);
    x[ss] = v;
  });
  fft_reg<R, true>(x);
  static_for<0, R>([&](auto t) {
    constexpr int tt = decltype(t)::value;
    A.st(base + tt * S, x[brevR<R>(tt)]);
  });
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- async bulk copy (TMA, 1-D) + mbarrier helpers -------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t mbar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbar), "r"(count) : "memory");
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t mbar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t mbar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(mbar)
               : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t mbar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t mbar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile("{ .reg .pred p; mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2; selp.u32 %0, 1, 0, p; }"
                 : "=r"(ok)
                 : "r"(mbar), "r"(parity)
                 : "memory");
  } while (!ok);
}

// ---- tensor memory (TMEM) as a per-thread constant cache ---------------------------------------------------
// sm_100a gives every SM 256 KB of tensor memory (512 columns x 128 lanes x 32 bit) next to the 227 KB of shared memory.
// The fp64 FFT path has no use for tcgen05.mma (no f64 kind), but tcgen05.st / tcgen05.ld move registers to and from TMEM
// on a datapath of their own (measured on B200: 228 B/cycle/SM with eight warps, _work probe; shared memory: 128 B/cycle).
// With the .32x32b shape a thread reaches exactly one TMEM lane (32 (warp % 4) + lane) and any column, so TMEM is private
// per-thread storage: 2 KB per lane, shared by the warps w and w + 4 of a CTA.  The fused kernels keep there what a
// thread needs again for every template and never changes: its 32 values of the generator spectrum, its samples of the
// data vector and its twiddle powers.  None of this touches shared memory or L2 after the first item.
// Cost, measured in r02: a kernel that executes tcgen05.alloc gets ONE resident CTA per SM from the driver's occupancy accounting
// (cudaOccupancyMaxActiveBlocksPerMultiprocessor returns 1 for a 30 KB / 120-register kernel once it contains the instruction),
// so kernels that want two items per SM put two item pipelines into one CTA (td_fused4.cuh, NGRP).
// NCOLS = 128, 256 or 512 columns (a power of two >= 32); executed by ONE whole warp, which also frees them.  A CTA that asks for
// more columns than are free on its SM waits inside the instruction until a co-resident CTA frees its own.
template <int NCOLS> __device__ __forceinline__ void tmem_alloc(uint32_t smem_slot) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_slot), "n"(NCOLS) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int NCOLS> __device__ __forceinline__ void tmem_dealloc(uint32_t taddr) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(NCOLS) : "memory");
}
__device__ __forceinline__ void tmem_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// columns per complex number of the kernel's scalar type: 4 (fp64) or 2 (fp32)
constexpr int TM_CPC = (int)(sizeof(cplx) / 4);
// one complex fp64 = 4 columns (the data samples are kept in fp64 in both precisions: r = d - h is formed in fp64)
__device__ __forceinline__ void tmem_st_c64(uint32_t taddr, double2 v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(__double2loint(v.x)),
               "r"(__double2hiint(v.x)), "r"(__double2loint(v.y)), "r"(__double2hiint(v.y))
               : "memory");
}
// one complex number of the kernel's scalar type = TM_CPC columns
__device__ __forceinline__ void tmem_st_c(uint32_t taddr, cplx v) {
#ifdef TD_F32
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(__float_as_int(v.x)),
               "r"(__float_as_int(v.y))
               : "memory");
#else
  tmem_st_c64(taddr, v);
#endif
}
// 16 columns.  tcgen05.ld is asynchronous: issue all loads, tmem_wait_ld(), then tmem_use16() on each register group (an
// empty asm that "rewrites" the registers, so that no use can be scheduled above the wait), then read.
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, int (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_use16(int (&r)[16]) {
  asm volatile("" : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]), "+r"(r[8]),
               "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15])
               :
               : "memory");
}
__device__ __forceinline__ double2 tmem_c64(const int (&r)[16], int q) {  // q-th complex fp64 of a group of 4
  return make_double2(__hiloint2double(r[4 * q + 1], r[4 * q]), __hiloint2double(r[4 * q + 3], r[4 * q + 2]));
}
// sixteen complex numbers of the kernel's scalar type held in 16 TM_CPC consecutive columns: NG x16 loads
struct TmemC16 {
  static constexpr int NG = TM_CPC;  // 16 * TM_CPC columns / 16 per load
  int r[NG][16];
  __device__ __forceinline__ void ld(uint32_t taddr) {
#pragma unroll
    for (int g = 0; g < NG; ++g) tmem_ld16(taddr + 16 * g, r[g]);
  }
  __device__ __forceinline__ void use() {
#pragma unroll
    for (int g = 0; g < NG; ++g) tmem_use16(r[g]);
  }
  __device__ __forceinline__ cplx get(int q) const {  // q compile-time after unrolling
#ifdef TD_F32
    return mk(__int_as_float(r[q >> 3][2 * (q & 7)]), __int_as_float(r[q >> 3][2 * (q & 7) + 1]));
#else
    return tmem_c64(r[q >> 2], q & 3);
#endif
  }
};

}  // namespace TD_NS
