// td_staged_host.cuh - host driver of the staged kernels (td_staged.cuh): launch helpers, workspace geometry and the two-lane
// chunk pipeline.  Precision-generic like the kernels: compiled in namespace td (fp64, tdlike.cu) and td32 (fp32,
// tdlike_f32.cu); the handle lends the workspace (the fp32 build uses the same bytes for twice the templates per chunk).
#pragma once
#include <algorithm>
#include <cstdint>

#include "td_host.h"
#include "td_staged.cuh"

namespace TD_NS {

using tdhost::kernel_config;
using tdhost::TD_MAX_DEV;

constexpr size_t STAGED_WS_BYTES = 96ull << 20;  // staged workspace, both lanes: inside the 126 MB L2 (measured 64: 0.91 ms, 96: 0.756, 128: 0.761, 192: 0.745, 384: 0.750 on c4)

template <bool FWD>
td_status launch_pass(int R, cplx* base, int narr, int n, int L, const cplx* T, int TW, cudaStream_t st) {
  dim3 grid((n / R + LG_NT - 1) / LG_NT, narr);
  switch (R) {
    case 2: lg_pass_kernel<2, FWD><<<grid, LG_NT, 0, st>>>(base, n, L, T, TW); break;
    case 4: lg_pass_kernel<4, FWD><<<grid, LG_NT, 0, st>>>(base, n, L, T, TW); break;
    case 8: lg_pass_kernel<8, FWD><<<grid, LG_NT, 0, st>>>(base, n, L, T, TW); break;
    case 16: lg_pass_kernel<16, FWD><<<grid, LG_NT, 0, st>>>(base, n, L, T, TW); break;
    default: return TD_EINVAL;
  }
  CK(cudaGetLastError());
  return TD_OK;
}

template <bool FWD>
td_status launch_block(int device, cplx* base, int narr, int n, const cplx* T, int TW, cudaStream_t st, bool dry = false) {
  auto kern = lg_block_kernel<FWD>;
  static int cache[TD_MAX_DEV];
  int nb = 0;
  td_status cs = kernel_config(kern, LGB_NT, LGB_SMEM, LGB_SMEM, device, cache, &nb);
  if (cs != TD_OK || dry) return cs;
  kern<<<dim3(n / LGB_N, narr), LGB_NT, LGB_SMEM, st>>>(base, n, T, TW);
  CK(cudaGetLastError());
  return TD_OK;
}

// forward DIF of `narr` arrays of length n with plan [r1,16,16,...]; the last three passes
// (L = 4096, 256, 16) run as one shared-memory block kernel when the plan has them
inline td_status staged_forward(int device, cplx* base, int narr, int n, int first_pass_done, const cplx* T, int TW,
                         cudaStream_t st, int* launches) {
  int L = n;
  const int r1 = plan_r1(n), np = plan_np(n);
  for (int q = 0; q < np; ++q) {
    const int R = q == 0 ? r1 : 16;
    if (q >= 1 && q == np - 3 && L == LGB_N) {
      td_status s = launch_block<true>(device, base, narr, n, T, TW, st);
      if (s != TD_OK) return s;
      ++*launches;
      break;
    }
    if (!(q == 0 && first_pass_done)) {
      td_status s = launch_pass<true>(R, base, narr, n, L, T, TW, st);
      if (s != TD_OK) return s;
      ++*launches;
    }
    L /= R;
  }
  return TD_OK;
}

// inverse DIT passes except the last (radix r1, L = n) one; the first three (L = 16, 256, 4096)
// as one shared-memory block kernel when the plan has them
inline td_status staged_inverse_but_last(int device, cplx* base, int narr, int n, const cplx* T, int TW, cudaStream_t st,
                                  int* launches) {
  const int np = plan_np(n);
  int L = 16, q = 1;
  if (np - 1 >= 3) {
    td_status s = launch_block<false>(device, base, narr, n, T, TW, st);
    if (s != TD_OK) return s;
    ++*launches;
    L <<= 12; q = 4;
  }
  for (; q < np; ++q) {
    td_status s = launch_pass<false>(16, base, narr, n, L, T, TW, st);
    if (s != TD_OK) return s;
    ++*launches;
    L <<= 4;
  }
  return TD_OK;
}

template <int MODE>
td_status launch_first(int R, dim3 grid, const StagedParams& P, cudaStream_t st) {
  switch (R) {
    case 2: lg_first_kernel<2, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    case 4: lg_first_kernel<4, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    case 8: lg_first_kernel<8, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    case 16: lg_first_kernel<16, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    default: return TD_EINVAL;
  }
  CK(cudaGetLastError());
  return TD_OK;
}
template <int MODE>
td_status launch_last(int R, dim3 grid, const StagedParams& P, cudaStream_t st) {
  switch (R) {
    case 2: lg_last_kernel<2, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    case 4: lg_last_kernel<4, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    case 8: lg_last_kernel<8, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    case 16: lg_last_kernel<16, MODE><<<grid, LG_NT, 0, st>>>(P); break;
    default: return TD_EINVAL;
  }
  CK(cudaGetLastError());
  return TD_OK;
}

// staged path geometry of one size class: templates per lane chunk, workspace shares
struct StagedGeom { int64_t CB; size_t uh, zh; int nblk, rI, rF; };
inline StagedGeom staged_geom(int log2M) {
  const int M = 1 << log2M, nf = M / 2;
  const size_t per_tmpl = (size_t)(2 * nf + 2 * M) * sizeof(cplx);
  StagedGeom g;
  g.CB = std::max<int64_t>(1, (int64_t)(STAGED_WS_BYTES / 2 / per_tmpl));
  g.CB = std::min<int64_t>(g.CB, 32767);  // grid.y = 2*CB arrays per pass
  g.rI = plan_r1(M); g.rF = plan_r1(nf);
  g.nblk = (M / g.rI + LG_NT - 1) / LG_NT;
  g.uh = (size_t)g.CB * 2 * nf; g.zh = (size_t)g.CB * 2 * M;
  return g;
}

// what a staged run borrows from the handle
struct StagedCtx {
  int device;
  void* wsU; size_t wsU_bytes;      // both lanes of the U workspace
  void* wsZ; size_t wsZ_bytes;
  double* wsPartial; size_t wsP_elems;
  cudaStream_t aux_stream;          // second lane
  cudaEvent_t ev_fork, ev_join;
  int* launches;                    // kernel launches are counted here
};

// One segment of a size class through the staged pipeline for templates [0, B).
template <int MODE>
td_status run_staged_sub(StagedCtx& C, int log2M, const cplx* T, const SegDev& sg, const double* d, const double* H,
                         int64_t ldh, int64_t B, double* out0, double* out1, double scale0, double scale1,
                         int accumulate, cudaStream_t st) {
  const int M = 1 << log2M, nf = M / 2, TW = 2 * M;
  // Two lanes: chunks alternate between the caller's stream and an internal one, each lane with its own half of the
  // L2-resident workspace.  No kernel of the pipeline fills the GPU on its own (a few hundred CTAs, each bound by L2
  // latency at the start and end of its life), so two chunks in flight overlap one another's ramps and tails.
  const StagedGeom g = staged_geom(log2M);
  const int64_t CB = std::min<int64_t>(g.CB, std::max<int64_t>(B, 1));
  const bool two = B > CB;
  const int rI = g.rI, rF = g.rF, nblk = g.nblk;
  const size_t uh = g.uh, zh = g.zh;  // one lane's share
  if (C.wsU_bytes < 2 * uh * sizeof(cplx) || C.wsZ_bytes < 2 * zh * sizeof(cplx)) return TD_EUNSUPPORTED;  // (never: td_create sized them)
  cplx* const wsU = static_cast<cplx*>(C.wsU);
  cplx* const wsZ = static_cast<cplx*>(C.wsZ);
  if (two) {
    CK(cudaEventRecord(C.ev_fork, st));          // everything enqueued on the caller's stream so far comes first
    CK(cudaStreamWaitEvent(C.aux_stream, C.ev_fork, 0));
  }
  int lane = 0;
  td_status s = TD_OK;
  for (int64_t b0 = 0; b0 < B && s == TD_OK; b0 += CB, lane ^= 1) {
    const int cb = (int)std::min<int64_t>(CB, B - b0);
    cudaStream_t ls = (two && lane) ? C.aux_stream : st;
    cplx* U = wsU + (two && lane ? uh : 0);
    cplx* Z = wsZ + (two && lane ? zh : 0);
    StagedParams P;
    P.d = d; P.H = H ? H + b0 * ldh : nullptr; P.ldh = ldh; P.CB = cb;
    P.seg = sg;
    P.M = M; P.U = U; P.Z = Z; P.T = T; P.partial = C.wsPartial + (size_t)b0 * nblk * 2; P.nblk = nblk;
    s = launch_first<MODE>(rF, dim3((nf / rF + LG_NT - 1) / LG_NT, cb), P, ls);
    if (s != TD_OK) break;
    ++*C.launches;
    s = staged_forward(C.device, U, 2 * cb, nf, 1, T, TW, ls, C.launches);
    if (s != TD_OK) break;
    // (fusing the untangle into the inverse block kernel - one CTA building a block, or a mirror pair of blocks, of Z in
    // shared memory straight from U and G - was measured: 50-68 us per chunk against 18 + 24 us for the two kernels; the
    // gather serialises 16 index-heavy tasks per thread, which the stand-alone kernel hides behind 1.4 M threads)
    lg_untangle_kernel<<<dim3((nf + LG_NT - 1) / LG_NT, 2, (cb + LG_UCPT - 1) / LG_UCPT), LG_NT, 0, ls>>>(P);
    if (cudaGetLastError() != cudaSuccess) { s = TD_ECUDA; break; }
    ++*C.launches;
    s = staged_inverse_but_last(C.device, Z, 2 * cb, M, T, TW, ls, C.launches);
    if (s != TD_OK) break;
    s = launch_last<MODE>(rI, dim3(nblk, cb), P, ls);
    if (s != TD_OK) break;
    ++*C.launches;
  }
  if (two) {  // the aux lane is joined on every path, also after an error
    const bool j = cudaEventRecord(C.ev_join, C.aux_stream) == cudaSuccess && cudaStreamWaitEvent(st, C.ev_join, 0) == cudaSuccess;
    if (!j && s == TD_OK) s = TD_ECUDA;
  }
  if (s != TD_OK) return s;
  if (MODE != MODE_STOREZ && B > 0) {  // one reduction of the per-block partial sums for the whole sub-batch (fixed order)
    lg_finish_kernel<<<(unsigned)((B + 127) / 128), 128, 0, st>>>(C.wsPartial, nblk, (int)B, out0, out1, scale0, scale1, accumulate);
    CK(cudaGetLastError());
    ++*C.launches;
  }
  return TD_OK;
}

// sub-batches of as many templates as the partial-sum buffer holds (td_reserve sizes it for the caller's largest batch)
template <int MODE>
td_status run_staged(StagedCtx& C, int log2M, const cplx* T, const SegDev& sg, const double* d, const double* H,
                     int64_t ldh, int64_t B, double* out0, double* out1, double scale0, double scale1,
                     int accumulate, cudaStream_t st) {
  const StagedGeom g = staged_geom(log2M);
  const int64_t SB = std::min<int64_t>(std::max<int64_t>(1, (int64_t)(C.wsP_elems / ((size_t)g.nblk * 2))), 1 << 30);
  if (C.wsP_elems < (size_t)g.nblk * 2) return TD_EUNSUPPORTED;  // (never: td_create holds at least one template)
  for (int64_t b0 = 0; b0 < std::max<int64_t>(B, 1); b0 += SB) {
    const int64_t nb = std::min<int64_t>(SB, B - b0);
    td_status s = run_staged_sub<MODE>(C, log2M, T, sg, d, H ? H + b0 * ldh : nullptr, ldh, nb, out0 ? out0 + b0 : nullptr,
                                       out1 ? out1 + b0 : nullptr, scale0, scale1, accumulate, st);
    if (s != TD_OK) return s;
  }
  return TD_OK;
}


}  // namespace TD_NS
