// tdlike_f32.cu - the fused FFT-path kernels compiled with real = float (namespace td32): the FP32 evaluation mode
// (SURVEY.md 8(f) NEXT-2; PAPER.md:268 "FP32 is sufficient ...", :322-324 III.C.3 "carry out all the analysis with FP32
// with appropriate normalization ... operators should be precomputed in FP64").  Setup (Levinson-Durbin, generator
// spectra, twiddles) stays in fp64 in tdlike.cu; this unit rounds those tables once and runs S1-S5 in fp32:
//   S1  r = (d - h) rho_0^(-1/2) is formed in fp64 from the fp64 inputs and rounded once (normalisation by rho_0);
//   S2-S4 in fp32 (the same kernels, butterflies, plans and TMEM constant cache as the fp64 build);
//   S5  per-thread sums of squares in fp32, warp / CTA / segment sums in fp64.
#define TD_F32 1
#include "td_f32.h"
#include "td_host.h"

#include <algorithm>
#include <new>
#include <vector>

#include "td_cluster.cuh"
#include "td_fused4.cuh"
#include "td_staged_host.cuh"
#include "td_group16.cuh"

using namespace td32;
using namespace tdhost;

namespace {

__global__ void cvt_cplx_kernel(const double2* __restrict__ src, float2* __restrict__ dst, size_t n, double scale) {
  const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) dst[i] = make_float2((float)(src[i].x * scale), (float)(src[i].y * scale));
}

// Several item pipelines per CTA (NGRP of td_fused4.cuh): a kernel that uses tensor memory gets one CTA per SM, so the other items
// on the SM live in the same CTA.  M = 4096: two (113 KB each); M = 2048 / 1024, whose pipelines have 128 / 64 threads: four /
// eight, i.e. sixteen warps of 128 registers in every shape.
constexpr int f32_ngrp(int log2M) { return log2M == 10 ? 8 : log2M == 11 ? 4 : 2; }
template <int LOG2M, int MODE, int SYN = 0>
td_status launch_fused4(const td32api::ClassTables& t, const FusedParams& P, int num_sms, int device, cudaStream_t st, bool dry,
                        double fs = 0.0) {
  constexpr int F32_NGRP = f32_ngrp(LOG2M);
  auto kern = td_fused4_kernel<LOG2M, MODE, F32_NGRP, SYN>;
  constexpr int NT = Fused4Shape<LOG2M>::NT * F32_NGRP;
  const size_t smem = Fused4Shape<LOG2M>::total_bytes(F32_NGRP);
  static int cache[TD_MAX_DEV];
  int nb = 0;
  td_status cs = kernel_config(kern, NT, smem, smem, device, cache, &nb);
  if (cs != TD_OK) return cs;
  if (nb < 1) return TD_EUNSUPPORTED;
  if (dry) return TD_OK;
  const long long want = MODE == MODE_STOREZ ? 1 : P.B;   // one CTA per item while SMs are free, then F32_NGRP items per CTA
  const int grid = (int)std::max<long long>(1, std::min<long long>(want, num_sms));
  Fused4Params P4;
  P4.base = P; P4.Gp = reinterpret_cast<const cplx* const*>(t.Gp_ptrs); P4.fs = fs;
  kern<<<grid, NT, smem, st>>>(P4);
  CK(cudaGetLastError());
  return TD_OK;
}

template <int MODE>
td_status launch_cluster(const td32api::ClassTables& t, const FusedParams& P, int num_sms, int device, cudaStream_t st, bool dry) {
  auto kern = td_cluster_kernel<MODE>;
  const size_t smem = ClusterShape::smem_bytes();
  static int cache[TD_MAX_DEV];  // 0 = not configured on this device yet, else 1 + clusters that can be co-resident
  if (device < 0 || device >= TD_MAX_DEV) return TD_EUNSUPPORTED;
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3(ClusterShape::NT); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if (cache[device] == 0) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cfg.gridDim = dim3(2 * (num_sms / 2));
    int n = 0;
    CK(cudaOccupancyMaxActiveClusters(&n, kern, &cfg));
    cache[device] = n + 1;
  }
  const int ncl = cache[device] - 1;
  if (ncl < 1) return TD_EUNSUPPORTED;
  if (dry) return TD_OK;
  const long long want = MODE == MODE_STOREZ ? 1 : P.B;
  cfg.gridDim = dim3(2 * (unsigned)std::max<long long>(1, std::min<long long>(want, ncl)));
  Fused4Params P4;
  P4.base = P; P4.Gp = reinterpret_cast<const cplx* const*>(t.Gp_ptrs); P4.fs = 0.0;
  CK(cudaLaunchKernelEx(&cfg, kern, P4));
  return TD_OK;
}

// ---- the group kernel (td_group16.cuh) in fp32: classes 14..16, one cooperative launch per segment
constexpr int GRP_MAX_GROUPS = 64;   // as in tdlike.cu: the counters' array holds this many groups
template <int CS, int MODE>
td_status launch_group(const GroupParams& PG, int cap, int num_sms, int device, cudaStream_t st, bool dry) {
  auto kern = td_group_kernel<CS, MODE>;
  const size_t smem = Cluster16Shape::smem_bytes();
  static int cache[TD_MAX_DEV];
  int per_sm = 0;
  td_status cs = kernel_config(kern, Cluster16Shape::NT, smem, smem, device, cache, &per_sm);
  if (cs != TD_OK || dry) return cs;
  const int ng = std::min(std::min(cap, GRP_MAX_GROUPS), per_sm * num_sms / CS);
  if (ng < 1) return TD_EUNSUPPORTED;
  const long long want = MODE == MODE_STOREZ ? 1 : PG.base.B;
  const unsigned groups = (unsigned)std::max<long long>(1, std::min<long long>(want, ng));
  CK(cudaMemsetAsync(PG.bar, 0, sizeof(unsigned) * 2 * GRP_MAX_GROUPS, st));
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative;
  attr[0].val.cooperative = 1;
  cfg.gridDim = dim3(CS * groups); cfg.blockDim = dim3(Cluster16Shape::NT);
  cfg.dynamicSmemBytes = smem; cfg.stream = st; cfg.attrs = attr; cfg.numAttrs = 1;
  const cudaError_t le = cudaLaunchKernelEx(&cfg, kern, PG);
  if (le == cudaErrorCooperativeLaunchTooLarge) { cudaGetLastError(); return TD_EUNSUPPORTED; }   // the caller falls back to the staged kernels
  CK(le);
  return TD_OK;
}
template <int CS>
td_status launch_group_mode(int mode, const GroupParams& PG, int cap, int num_sms, int device, cudaStream_t st, bool dry) {
  switch (mode) {
    case MODE_LOGLIKE: return launch_group<CS, MODE_LOGLIKE>(PG, cap, num_sms, device, st, dry);
    case MODE_INNER: return launch_group<CS, MODE_INNER>(PG, cap, num_sms, device, st, dry);
    case MODE_STOREZ: return launch_group<CS, MODE_STOREZ>(PG, cap, num_sms, device, st, dry);
    default: return TD_EINVAL;
  }
}
td_status launch_group_any(int cs, int mode, const GroupParams& PG, int cap, int num_sms, int device, cudaStream_t st, bool dry) {
  return cs == 4 ? launch_group_mode<4>(mode, PG, cap, num_sms, device, st, dry)
       : cs == 8 ? launch_group_mode<8>(mode, PG, cap, num_sms, device, st, dry)
                 : launch_group_mode<16>(mode, PG, cap, num_sms, device, st, dry);
}

template <int MODE>
td_status launch_mode(const td32api::ClassTables& t, const FusedParams& P, int num_sms, int device, cudaStream_t st, bool dry) {
  switch (t.log2M) {
    case 10: return launch_fused4<10, MODE>(t, P, num_sms, device, st, dry);
    case 11: return launch_fused4<11, MODE>(t, P, num_sms, device, st, dry);
    case 12: return launch_fused4<12, MODE>(t, P, num_sms, device, st, dry);
    case 13: return launch_cluster<MODE>(t, P, num_sms, device, st, dry);
    default: return TD_EUNSUPPORTED;
  }
}

}  // namespace

namespace td32api {

void free_class(ClassTables* t) {
  if (!t) return;
  cudaFree(t->T); cudaFree(t->segs); cudaFree(t->Gp_ptrs);
  for (int s = 0; s < t->n_seg; ++s) {
    if (t->Gp) cudaFree(t->Gp[s]);
    if (t->zd) cudaFree(t->zd[s]);
    if (t->Gc) cudaFree(t->Gc[s]);
  }
  delete[] t->Gp; delete[] t->zd; delete[] t->Gc;
  delete[] static_cast<SegDev*>(t->host_segs);
  *t = ClassTables();
}

td_status build_class(int log2M, int n_seg, const SegIn* segs, const void* T64, ClassTables* out) {
  if (!supported(log2M) || n_seg < 1 || !segs || !T64 || !out) return TD_EINVAL;
  ClassTables t;
  t.log2M = log2M; t.n_seg = n_seg;
  t.Gp = new (std::nothrow) void*[n_seg]();
  t.zd = new (std::nothrow) void*[n_seg]();
  const int gcs = group_cs(log2M);
  if (gcs) t.Gc = new (std::nothrow) void*[n_seg]();
  if (!t.Gp || !t.zd || (gcs && !t.Gc)) { free_class(&t); return TD_ENOMEM; }
  const bool staged = staged_class(log2M);
  const size_t M = (size_t)1 << log2M, TW = 2 * M, gp_elems = staged ? 2 * M : 2 * (size_t)SmemArr::padded((int)M);
  auto fail = [&](td_status s) { free_class(&t); return s; };
  if (cudaMalloc(&t.T, sizeof(float2) * TW) != cudaSuccess) return fail(TD_ENOMEM);
  cvt_cplx_kernel<<<(unsigned)((TW + 255) / 256), 256>>>(static_cast<const double2*>(T64), static_cast<float2*>(t.T), TW, 1.0);
  std::vector<SegDev> sd(n_seg);
  std::vector<const cplx*> gp(n_seg);
  for (int s = 0; s < n_seg; ++s) {
    if (!(segs[s].rho0 > 0.0)) return fail(TD_ENOTSPD);
    if (cudaMalloc(&t.Gp[s], sizeof(float2) * gp_elems) != cudaSuccess) return fail(TD_ENOMEM);
    if (cudaMalloc(&t.zd[s], sizeof(float2) * M) != cudaSuccess) return fail(TD_ENOMEM);
    const void* src = staged ? segs[s].G64 : segs[s].Gp64;
    if (!src) return fail(TD_EINVAL);
    cvt_cplx_kernel<<<(unsigned)((gp_elems + 255) / 256), 256>>>(static_cast<const double2*>(src), static_cast<float2*>(t.Gp[s]),
                                                                 gp_elems, sqrt(segs[s].rho0));
    if (gcs && segs[s].Gc64) {
      const size_t ge = (size_t)gcs * Cluster16Shape::PADZ;
      if (cudaMalloc(&t.Gc[s], sizeof(float2) * ge) != cudaSuccess) return fail(TD_ENOMEM);
      cvt_cplx_kernel<<<(unsigned)((ge + 255) / 256), 256>>>(static_cast<const double2*>(segs[s].Gc64), static_cast<float2*>(t.Gc[s]), ge,
                                                            sqrt(segs[s].rho0));
    }
    sd[s].off = segs[s].off; sd[s].n = segs[s].n; sd[s]._pad = segs[s].sid; sd[s].G = staged ? static_cast<const cplx*>(t.Gp[s]) : nullptr;
    sd[s].zd = static_cast<cplx*>(t.zd[s]); sd[s].rscale = 1.0 / sqrt(segs[s].rho0);
    gp[s] = static_cast<const cplx*>(t.Gp[s]);
  }
  if (cudaGetLastError() != cudaSuccess) return fail(TD_ECUDA);
  if (cudaMalloc(&t.segs, sizeof(SegDev) * n_seg) != cudaSuccess || cudaMalloc(&t.Gp_ptrs, sizeof(cplx*) * n_seg) != cudaSuccess)
    return fail(TD_ENOMEM);
  if (cudaMemcpy(t.segs, sd.data(), sizeof(SegDev) * n_seg, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemcpy(t.Gp_ptrs, gp.data(), sizeof(cplx*) * n_seg, cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaDeviceSynchronize() != cudaSuccess)
    return fail(TD_ECUDA);
  if (staged) {
    SegDev* hs = new (std::nothrow) SegDev[n_seg];
    if (!hs) return fail(TD_ENOMEM);
    for (int s = 0; s < n_seg; ++s) hs[s] = sd[s];
    t.host_segs = hs;
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return fail(TD_ECUDA);
    td_status a = launch_block<true>(dev, nullptr, 0, 0, nullptr, 0, nullptr, true);   // shared-memory attribute of the block kernels
    if (a == TD_OK) a = launch_block<false>(dev, nullptr, 0, 0, nullptr, 0, nullptr, true);
    if (a != TD_OK) return fail(a);
  }
  *out = t;
  return TD_OK;
}

td_status launch(const ClassTables& t, const Launch& L, int num_sms, int device, cudaStream_t st, bool dry) {
  FusedParams P;
  P.d = L.d; P.H = L.H; P.ldh = L.ldh; P.B = L.B; P.out0 = L.out0; P.out1 = L.out1;
  P.segs = static_cast<const SegDev*>(t.segs); P.n_seg = t.n_seg; P.accumulate = L.accumulate;
  P.T = static_cast<const cplx*>(t.T);
  if (staged_class(t.log2M)) {
    const int gcs = t.Gc ? group_cs(t.log2M) : 0;
    if (dry) {   // configure the group kernels of the class (attribute, occupancy cache)
      GroupParams PG = {};
      for (int m = 0; gcs && m < 3; ++m) {
        td_status r = launch_group_any(gcs, m, PG, 0, num_sms, device, st, true);
        if (r != TD_OK) return r;
      }
      return TD_OK;
    }
    if (!L.staged || !t.host_segs) return TD_EINVAL;
    if (gcs && L.staged->group_cap > 0 && L.staged->grp_bar) {   // one cooperative launch + the sum of the per-CTA partials per segment
      bool all = true;
      for (int s = 0; s < t.n_seg; ++s) all = all && t.Gc[s];
      const long long SB = std::max<long long>(1, (long long)(L.staged->wsP_elems / ((size_t)gcs * 2)));
      const double sc0 = L.mode == MODE_LOGLIKE ? -0.5 : 1.0;
      int accumulate = L.accumulate;
      for (int s = 0; all && s < t.n_seg; ++s) {
        const long long Bn = L.mode == MODE_STOREZ ? 1 : L.B;
        for (long long b0 = 0; b0 < Bn; b0 += SB) {
          const long long nb = std::min<long long>(SB, Bn - b0);
          GroupParams PG;
          PG.base = P; PG.base.H = L.H ? L.H + b0 * L.ldh : nullptr; PG.base.B = nb; PG.base.out0 = nullptr; PG.base.out1 = nullptr;
          PG.base.segs = static_cast<const SegDev*>(t.segs) + s; PG.base.n_seg = 1; PG.base.accumulate = 0;
          PG.Gp = static_cast<const cplx*>(t.Gc[s]); PG.partial = L.staged->wsPartial;
          PG.wsU = static_cast<cplx*>(L.staged->wsU); PG.wsZ = static_cast<cplx*>(L.staged->wsZ); PG.bar = L.staged->grp_bar;
          td_status r = launch_group_any(gcs, L.mode, PG, L.staged->group_cap, num_sms, device, st, false);
          if (r == TD_EUNSUPPORTED && s == 0 && b0 == 0) { all = false; break; }   // refused before anything ran: staged kernels below
          if (r != TD_OK) return r;
          ++*L.staged->launches;
          if (L.mode != MODE_STOREZ) {
            lg_finish_kernel<<<(unsigned)((nb + 127) / 128), 128, 0, st>>>(L.staged->wsPartial, gcs, (int)nb, L.out0 ? L.out0 + b0 : nullptr,
                                                                          L.out1 ? L.out1 + b0 : nullptr, sc0, 1.0, accumulate);
            CK(cudaGetLastError());
            ++*L.staged->launches;
          }
        }
        accumulate = 1;
      }
      if (all) return TD_OK;
    }
    StagedCtx C;
    C.device = device;
    C.wsU = L.staged->wsU; C.wsU_bytes = L.staged->wsU_bytes; C.wsZ = L.staged->wsZ; C.wsZ_bytes = L.staged->wsZ_bytes;
    C.wsPartial = L.staged->wsPartial; C.wsP_elems = L.staged->wsP_elems;
    C.aux_stream = L.staged->aux_stream; C.ev_fork = L.staged->ev_fork; C.ev_join = L.staged->ev_join;
    C.launches = L.staged->launches;
    const SegDev* hs = static_cast<const SegDev*>(t.host_segs);
    const double sc0 = L.mode == MODE_LOGLIKE ? -0.5 : 1.0;
    int accumulate = L.accumulate;
    for (int s = 0; s < t.n_seg; ++s) {   // one segment after the other, accumulating into the outputs
      td_status r;
      switch (L.mode) {
        case MODE_LOGLIKE: r = run_staged<MODE_LOGLIKE>(C, t.log2M, P.T, hs[s], L.d, L.H, L.ldh, L.B, L.out0, L.out1, sc0, 1.0, accumulate, st); break;
        case MODE_INNER: r = run_staged<MODE_INNER>(C, t.log2M, P.T, hs[s], L.d, L.H, L.ldh, L.B, L.out0, L.out1, sc0, 1.0, accumulate, st); break;
        case MODE_STOREZ: r = run_staged<MODE_STOREZ>(C, t.log2M, P.T, hs[s], L.d, L.H, L.ldh, L.B, L.out0, L.out1, sc0, 1.0, accumulate, st); break;
        default: return TD_EINVAL;
      }
      if (r != TD_OK) return r;
      accumulate = 1;
    }
    return TD_OK;
  }
  if (L.syn) {
    if (L.mode != MODE_LOGLIKE) return TD_EINVAL;
    switch (t.log2M) {
      case 10: return launch_fused4<10, MODE_LOGLIKE, 1>(t, P, num_sms, device, st, dry, L.fs);
      case 11: return launch_fused4<11, MODE_LOGLIKE, 1>(t, P, num_sms, device, st, dry, L.fs);
      case 12: return launch_fused4<12, MODE_LOGLIKE, 1>(t, P, num_sms, device, st, dry, L.fs);
      default: return TD_EUNSUPPORTED;
    }
  }
  switch (L.mode) {
    case MODE_LOGLIKE: return launch_mode<MODE_LOGLIKE>(t, P, num_sms, device, st, dry);
    case MODE_INNER: return launch_mode<MODE_INNER>(t, P, num_sms, device, st, dry);
    case MODE_STOREZ: return launch_mode<MODE_STOREZ>(t, P, num_sms, device, st, dry);
    default: return TD_EINVAL;
  }
}

}  // namespace td32api
