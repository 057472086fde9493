// tdlike.cu - host side of the C ABI declared in include/tdlike.h.
// Owns the handle, runs the one-time setup (td_setup.cuh) and dispatches the batch calls to
// the fused shared-memory kernel (td_fused.cuh), the staged kernels (td_staged.cuh) or the
// dense tensor-pipe kernel (td_dense.cuh).  No CPU fallback exists on any path.
#include "../../include/tdlike.h"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <new>
#include <vector>

#include "td_host.h"
#include "td_f32.h"
#include "td_dense.cuh"
#include "td_cdo.cuh"
#include "td_dot.cuh"
#include "td_fused.cuh"
#include "td_cluster.cuh"
#include "td_cluster16.cuh"
#include "td_group16.cuh"
#include "td_fused4.cuh"
#include "td_setup.cuh"
#include "td_staged_host.cuh"
#include "td_synth.cuh"

using namespace td;
using namespace tdhost;

namespace {

constexpr int FUSED_MIN_LOG2M = 8;   // M = 256
// one-CTA fused kernels: M = 256..4096 (2M = 8192-point transform, 204 KiB of shared memory at M = 4096)
constexpr int CLUSTER_LOG2M = 13;    // M = 8192: 2-CTA cluster, one branch per CTA (td_cluster.cuh)
constexpr int FUSED_NT = 256;
constexpr int DENSE_AUTO_N = 512;     // AUTO: dense paths for segments up to this length (measured crossover: profiles/r01_chooser.md)
constexpr int CDO_AUTO_MAX_N = 512;   // AUTO, log-likelihood: size classes whose segments are all at most this long take the CDO kernel
                                      // (profiles/r02_cdo.md: 768 while the M = 1024 FFT kernel ran one 64-thread pipeline per SM - 31 M evals/s
                                      // against 41 for CDO at N = 768; with four pipelines it does 80 M and wins from 513 samples up)
constexpr int CDO_AUTO_MIN_N = 65;    // AUTO, log-likelihood: cached-L^-1 contraction from this length up, the Gohberg-Semencul
                                      // dense kernel below (measured: profiles/r02_cdo.md; 0.95x at N = 64, 1.08-1.55x above)

struct SegHost {
  int64_t off = 0;
  int n = 0;
  int log2M = 0;
  double v = 0.0, logdet = 0.0;
  double rho0 = 0.0;    // rho_s(0): normalisation of the fp32 evaluation mode
  bool auto_cdo = false;  // AUTO evaluates this segment's log-likelihood with the CDO kernel
  double* a = nullptr;  // device [n]
  cplx* G = nullptr;    // device [2][M]
  cplx* Gp = nullptr;   // device [2][padded(M)], padded Z layout (fused4 classes only)
  cplx* Gc16 = nullptr; // device [CS][padded(8192)]: per-CTA generator values of the group kernel (M = 16384 ... 65536, CS = M / 4096) and of the 16-CTA cluster kernel
  cplx* zd = nullptr;   // device [M] (lazy)
};

struct ClassInfo {
  int log2M = 0;
  cplx* T = nullptr;            // device [2M]
  std::vector<int> seg_ids;
  int max_n = 0;                // longest segment of the class
  SegDev* d_segs = nullptr;     // device [seg_ids.size()]
  const cplx** d_Gp = nullptr;  // device [seg_ids.size()] (fused4 classes only)
  td32api::ClassTables t32;     // fp32 tables (td_set_precision(TD_PREC_F32); classes the fp32 kernels serve)
  bool has32 = false;
};

struct DevGuard {
  int prev = -1;
  bool ok = true;
  explicit DevGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) { ok = false; return; }
    if (prev != dev && cudaSetDevice(dev) != cudaSuccess) ok = false;
  }
  ~DevGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

}  // namespace

struct td_handle {
  int device = 0, n_seg = 0, num_sms = 0;
  size_t smem_optin = 0;  // opt-in shared memory per CTA of the device
  int64_t n_tot = 0;
  std::vector<SegHost> segs;
  std::vector<ClassInfo> classes;
  int path = TD_PATH_AUTO, fft_variant = 0, last_path = 0, last_launches = 0;
  int precision = TD_PREC_F64;
  bool any_auto_ll = false;   // some size class goes to the dense kernels for the log-likelihood under AUTO
  int group_cap[3] = {0, 0, 0};  // groups of 4 / 8 / 16 CTAs of td_group_kernel (td_group16.cuh) that are co-resident AND fit the
                                 // exchange buffers (0: not asked yet, -1: the class stays on the staged kernels)
  unsigned* grp_bar = nullptr;   // device [GRP_MAX_GROUPS][2] arrival counters of that kernel
  int cluster16_cap = 0;   // co-resident 16-CTA clusters of td_cluster16_kernel (0: M = 65536 stays on the staged kernels)
  int max_n = 0;
  // staged workspace: U / Z sized by td_create (two lanes of an L2-resident chunk), the per-block partial sums by
  // td_create / td_reserve (a batch larger than they hold is processed in sub-batches)
  cplx* wsU = nullptr; cplx* wsZ = nullptr; double* wsPartial = nullptr;
  double* wsDot = nullptr;  // per-tile partial weights of the dot path (td_dot.cuh)
  double* synH = nullptr; size_t synH_elems = 0;  // scratch panel of synthesised templates (td_synth.cuh)
  double* synP = nullptr; size_t synP_elems = 0;  // device copy of host parameters
  SynSeg* synSeg = nullptr;                       // device [n_seg]: offsets and lengths for the synthesis kernel
  double* ud = nullptr;  // [n_tot] weights u = C^{-1} d of the dot path (td_dot.cuh), lazily allocated
  size_t wsU_elems = 0, wsZ_elems = 0, wsP_elems = 0;
  // dense path state
  DenseState dense;
  // CDO path (td_cdo.cuh): device copy of the ACFs (kept for the whitening-operator setup), one W per segment (lazy)
  double* d_rho = nullptr;
  std::vector<double*> cdoW;
  // host-buffer entry point: staging (grow-only), copy stream, events
  double* hsD = nullptr; double* hsH[2] = {nullptr, nullptr}; double* hsOut = nullptr;
  size_t hsH_elems = 0, hsOut_elems = 0;
  cudaStream_t copy_stream = nullptr;
  cudaStream_t aux_stream = nullptr;              // second lane of the staged path (chunks alternate between two streams)
  cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
  cudaEvent_t ev_copied[2] = {nullptr, nullptr}, ev_done[2] = {nullptr, nullptr};
  // cross-stream ordering of calls that touch handle-owned scratch (include/tdlike.h "Streams")
  cudaEvent_t ev_last = nullptr;
  cudaStream_t last_stream = nullptr;
  bool last_valid = false, touched = false;
};

#ifdef TD_DEBUG_KNOBS
// experiment knobs of debug builds (_work probes); the product build compiles the defaults in
static int g_tune[16] = {-1, -1, -1, -1, -1, -1, -1, -1, -1, -1, -1, -1, -1, -1, -1, -1};
static inline int tune(int i, int dflt) { return g_tune[i] < 0 ? dflt : g_tune[i]; }
extern "C" void td_debug_set_tune(int i, int v) { if (i >= 0 && i < 16) g_tune[i] = v; }
#else
static inline constexpr int tune(int, int dflt) { return dflt; }
#endif

namespace {

int next_log2(int n) { int l = 0; while ((1 << l) < n) ++l; return l; }

void free_handle(td_handle* h) {
  if (!h) return;
  for (auto& s : h->segs) { cudaFree(s.a); cudaFree(s.G); cudaFree(s.Gp); cudaFree(s.Gc16); cudaFree(s.zd); }
  for (auto& c : h->classes) { cudaFree(c.T); cudaFree(c.d_segs); cudaFree(c.d_Gp); if (c.has32) td32api::free_class(&c.t32); }
  cudaFree(h->wsU); cudaFree(h->wsZ); cudaFree(h->wsPartial); cudaFree(h->grp_bar); cudaFree(h->wsDot); cudaFree(h->ud); cudaFree(h->synH); cudaFree(h->synP); cudaFree(h->synSeg);
  cudaFree(h->hsD); cudaFree(h->hsH[0]); cudaFree(h->hsH[1]); cudaFree(h->hsOut);
  cudaFree(h->d_rho);
  for (double* w : h->cdoW) cudaFree(w);
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  if (h->aux_stream) cudaStreamDestroy(h->aux_stream);
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  if (h->ev_last) cudaEventDestroy(h->ev_last);
  for (int i = 0; i < 2; ++i) { if (h->ev_copied[i]) cudaEventDestroy(h->ev_copied[i]); if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]); }
  delete h;
}

// grow-only device buffer (td_create / td_reserve; a batch call reaches the cudaMalloc only when the caller did not reserve)
template <class T> td_status grow(T*& p, size_t& have, size_t want) {
  if (want <= have) return TD_OK;
  cudaFree(p); p = nullptr; have = 0;
  CK(cudaMalloc(&p, want * sizeof(T)));
  have = want;
  return TD_OK;
}

constexpr size_t STAGED_PARTIAL_DEFAULT = 16ull << 20, STAGED_PARTIAL_MAX = 1ull << 30;  // bytes of per-block partial sums

// cross-stream ordering of the calls that use handle-owned scratch (staged workspace, z / u of the data vector, the
// synthesis panel): a call on another stream than the previous such call first waits for it.  Inside a stream capture
// nothing is recorded or waited on (the graph's own edges order the work).
td_status order_begin(td_handle* h, cudaStream_t st) {
  h->touched = false;
  if (!h->last_valid || h->last_stream == st) return TD_OK;
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  CK(cudaStreamIsCapturing(st, &cs));
  if (cs == cudaStreamCaptureStatusNone) CK(cudaStreamWaitEvent(st, h->ev_last, 0));
  return TD_OK;
}
td_status order_end(td_handle* h, cudaStream_t st) {
  if (!h->touched) return TD_OK;
  cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
  CK(cudaStreamIsCapturing(st, &cs));
  if (cs != cudaStreamCaptureStatusNone) { h->last_valid = false; return TD_OK; }
  CK(cudaEventRecord(h->ev_last, st));
  h->last_stream = st; h->last_valid = true;
  return TD_OK;
}

// the staged kernels' driver (td_staged_host.cuh) borrows workspace, second stream and events from the handle
StagedCtx staged_ctx(td_handle* h) {
  StagedCtx C;
  C.device = h->device;
  C.wsU = h->wsU; C.wsU_bytes = h->wsU_elems * sizeof(cplx);
  C.wsZ = h->wsZ; C.wsZ_bytes = h->wsZ_elems * sizeof(cplx);
  C.wsPartial = h->wsPartial; C.wsP_elems = h->wsP_elems;
  C.aux_stream = h->aux_stream; C.ev_fork = h->ev_fork; C.ev_join = h->ev_join;
  C.launches = &h->last_launches;
  return C;
}
template <int MODE>
td_status run_staged(td_handle* h, const ClassInfo& cls, const SegHost& sg, const double* d, const double* H,
                     int64_t ldh, int64_t B, double* out0, double* out1, double scale0, double scale1,
                     int accumulate, cudaStream_t st) {
  StagedCtx C = staged_ctx(h);
  SegDev sd;
  sd.off = sg.off; sd.n = sg.n; sd._pad = 0; sd.G = sg.G; sd.zd = sg.zd; sd.rscale = 1.0;
  h->touched = true;
  return td::run_staged<MODE>(C, cls.log2M, cls.T, sd, d, H, ldh, B, out0, out1, scale0, scale1, accumulate, st);
}

template <int LOG2M, int MODE, int FUSED_NT, bool ILV = true>
td_status launch_fused_nt(td_handle* h, const FusedParams& P, cudaStream_t st, bool dry) {
  auto kern = td_fused_kernel<LOG2M, FUSED_NT, MODE, ILV>;
  const size_t smem = FusedShape<LOG2M>::smem_bytes(FUSED_NT);
  static int cache[TD_MAX_DEV];
  int nb = 0;
  td_status cs = kernel_config(kern, FUSED_NT, smem, smem, h->device, cache, &nb);
  if (cs != TD_OK) return cs;
  if (nb < 1) return TD_EUNSUPPORTED;
  if (dry) return TD_OK;
  const long long maxg = (long long)nb * h->num_sms;
  const int grid = (int)std::max<long long>(1, std::min<long long>(MODE == MODE_STOREZ ? 1 : P.B, maxg));
  kern<<<grid, FUSED_NT, smem, st>>>(P);
  CK(cudaGetLastError());
  ++h->last_launches;
  return TD_OK;
}

// SYN = 1: P.H holds parameter rows (ldh = 5 n_seg), the rows are synthesised in the first pass (td_ring.cuh)
// Item pipelines per CTA (NGRP of td_fused4.cuh).  A kernel that allocates tensor memory gets ONE resident CTA per SM, and the CTA
// of the M = 1024 shape has 64 threads, that of M = 2048 has 128: four / two pipelines (independent items, one shared base-twiddle
// table; 222 KB / 221 KB of shared memory) put eight warps on the SM in every shape.  M = 4096 (256 threads, 204 KB) holds one.
constexpr int f64_ngrp(int log2M) { return log2M == 10 ? 4 : log2M == 11 ? 2 : 1; }
template <int LOG2M, int MODE, int SYN = 0>
td_status launch_fused4(td_handle* h, const FusedParams& P, const cplx* const* Gp, cudaStream_t st, bool dry, double fs = 0.0) {
  constexpr int NGRP = f64_ngrp(LOG2M);
  auto kern = td_fused4_kernel<LOG2M, MODE, NGRP, SYN>;
  constexpr int NT = Fused4Shape<LOG2M>::NT * NGRP;
  const size_t smem = Fused4Shape<LOG2M>::total_bytes(NGRP);
  static int cache[TD_MAX_DEV];
  int nb = 0;
  td_status cs = kernel_config(kern, NT, smem, smem, h->device, cache, &nb);
  if (cs != TD_OK) return cs;
  if (nb < 1) return TD_EUNSUPPORTED;
  if (dry) return TD_OK;
  nb = std::min(nb, 512 / Fused4Shape<LOG2M>::tmem_cols(NGRP));  // co-resident CTAs share the SM's 512 tensor-memory columns
  const long long maxg = (long long)nb * h->num_sms;
  const long long want = MODE == MODE_STOREZ ? 1 : P.B;   // one CTA per item while SMs are free, then NGRP items per CTA
  const int grid = (int)std::max<long long>(1, std::min<long long>(want, maxg));
  Fused4Params P4;
  P4.base = P; P4.Gp = Gp; P4.fs = fs;
#ifdef TD_DEBUG_KNOBS
  P4.skew = tune(1, 0);
#endif
  kern<<<grid, NT, smem, st>>>(P4);
  CK(cudaGetLastError());
  ++h->last_launches;
  return TD_OK;
}

template <int MODE>
td_status launch_cluster(td_handle* h, const FusedParams& P, const cplx* const* Gp, cudaStream_t st, bool dry) {
  auto kern = td_cluster_kernel<MODE>;
  const size_t smem = ClusterShape::smem_bytes();
  static int cache[TD_MAX_DEV];  // 0 = not configured on this device yet, else 1 + clusters that can be co-resident
  if (h->device < 0 || h->device >= TD_MAX_DEV) return TD_EUNSUPPORTED;
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3(ClusterShape::NT); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if (cache[h->device] == 0) {
    CK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    cfg.gridDim = dim3(2 * (h->num_sms / 2));
    int n = 0;
    CK(cudaOccupancyMaxActiveClusters(&n, kern, &cfg));
    cache[h->device] = n + 1;
  }
  const int ncl = cache[h->device] - 1;
  if (ncl < 1) return TD_EUNSUPPORTED;
  if (dry) return TD_OK;
  const long long want = MODE == MODE_STOREZ ? 1 : P.B;
  cfg.gridDim = dim3(2 * (unsigned)std::max<long long>(1, std::min<long long>(want, ncl)));
  Fused4Params P4;
  P4.base = P; P4.Gp = Gp; P4.fs = 0.0;
#ifdef TD_DEBUG_KNOBS
  P4.skew = 0;
#endif
  CK(cudaLaunchKernelEx(&cfg, kern, P4));
  ++h->last_launches;
  return TD_OK;
}

template <int LOG2M, int MODE>
td_status launch_fused_t(td_handle* h, const FusedParams& P, cudaStream_t st, bool dry) {
  return launch_fused_nt<LOG2M, MODE, FUSED_NT>(h, P, st, dry);
}

template <int MODE>
td_status launch_fused(td_handle* h, int log2M, const FusedParams& P, const cplx* const* Gp, cudaStream_t st,
                       bool dry = false) {
  if (log2M == CLUSTER_LOG2M) return Gp ? launch_cluster<MODE>(h, P, Gp, st, dry) : TD_EUNSUPPORTED;
  if (Gp) {
    switch (log2M) {
      case 10: return launch_fused4<10, MODE>(h, P, Gp, st, dry);
      case 11: return launch_fused4<11, MODE>(h, P, Gp, st, dry);
      case 12: return launch_fused4<12, MODE>(h, P, Gp, st, dry);
      default: break;
    }
  }
  switch (log2M) {
    case 8: return launch_fused_t<8, MODE>(h, P, st, dry);
    case 9: return launch_fused_t<9, MODE>(h, P, st, dry);
    default: return TD_EUNSUPPORTED;  // M >= 1024 always has the padded generator copy (Gp) of td_create
  }
}

bool class_is_fused_shape(int log2M) { return log2M >= FUSED_MIN_LOG2M && log2M <= CLUSTER_LOG2M; }
bool class_is_fused(const td_handle* h, const ClassInfo& c) {
  if (h->fft_variant == 2) return false;
  return class_is_fused_shape(c.log2M);
}


// AUTO sends a size class to the dense paths when every segment in it is short enough: up to CDO_AUTO_MAX_N samples for the
// log-likelihood (CDO kernel), up to dense.auto_n for the cross terms (Gohberg-Semencul dense kernel)
bool class_is_dense(const td_handle* h, const ClassInfo& c, int mode) {
  if (h->path == TD_PATH_DENSE || h->path == TD_PATH_CDO) return true;
  if (h->path == TD_PATH_FFT) return false;
  return c.max_n <= (mode == MODE_LOGLIKE ? CDO_AUTO_MAX_N : h->dense.auto_n);
}

// (re)builds the segment tables of the dense path from the host-side segment records
td_status dense_upload(td_handle* h) {
  DenseState& D = h->dense;
  D.all.clear(); D.aut.clear(); D.aut_gs.clear();
  for (const ClassInfo& c : h->classes)
    for (int id : c.seg_ids) {
      const SegHost& sg = h->segs[id];
      if (sg.n > DENSE_MAX_N) continue;
      DenseSeg ds;
      ds.off = sg.off; ds.n = sg.n; ds.npad = (sg.n + 31) / 32 * 32; ds.a = sg.a; ds.rsv = 1.0 / std::sqrt(sg.v); ds.zd = sg.zd;
      D.all.push_back(ds);
      if (c.max_n <= D.auto_n) D.aut.push_back(ds);
      if (c.max_n <= CDO_AUTO_MAX_N && sg.n < CDO_AUTO_MIN_N) D.aut_gs.push_back(ds);
    }
  D.max_n = DENSE_MAX_N;
  if (h->max_n > DENSE_MAX_N) D.all.clear();
  return TD_OK;
}

// one launch per segment; segments accumulate into the outputs in launch order
template <int MODE>
td_status launch_dense(td_handle* h, const std::vector<DenseSeg>& segs, const double* d, const double* H, int64_t ldh,
                       int64_t B, double* out0, double* out1, int accumulate, cudaStream_t st, bool dry = false) {
  static int cache[4][TD_MAX_DEV];  // per NWR instantiation of this MODE
  for (const DenseSeg& sg : segs) {
    DenseParams P;
    P.d = d; P.H = H; P.ldh = ldh; P.B = B; P.out0 = out0; P.out1 = out1; P.seg = sg;
    P.accumulate = accumulate; P.nwr = dense_nwr(sg.npad); P.nbuf = dense_nbuf(sg.npad);
    void (*kern)(const DenseParams) = P.nwr == 1 ? td_dense_kernel<MODE, 1> : P.nwr == 2 ? td_dense_kernel<MODE, 2>
                                    : P.nwr == 4 ? td_dense_kernel<MODE, 4> : td_dense_kernel<MODE, 8>;
    // 16-byte copies when every row start is 16-byte aligned and the length is even
    P.vec_ok = (sg.off % 2 == 0) && (sg.n % 2 == 0) && (ldh % 2 == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    P.ntiles = (B + 15) / 16;
    // DMMAs of one warp per tile x 16 cycles each: the lag that lets one group's bookkeeping hide under the other's DMMAs
    {
      const int NG = sg.npad / 32;
      long long nd = 0;
      for (int p = 0; 2 * p < NG; p += P.nwr) {  // warp wr = 0
        nd += 80 + 128ll * (NG - p - 1);
        if (NG - 1 - p != p) nd += 80 + 128ll * p;
      }
      P.stagger_cycles = (int)std::min<long long>(nd * 16, 1 << 22);
    }
    const size_t smem = dense_smem_bytes(sg.npad, P.nbuf);
    {
      // the attribute is set once to the device's opt-in maximum (the size itself varies with the segment length)
      int nb = 0;
      td_status cs = kernel_config(kern, DENSE_NT, h->smem_optin, smem, h->device,
                                   cache[P.nwr == 1 ? 0 : P.nwr == 2 ? 1 : P.nwr == 4 ? 2 : 3], &nb);
      if (cs != TD_OK) return cs;
      if (smem > h->smem_optin) return TD_EUNSUPPORTED;
    }
    if (dry) continue;
    const int nwc = DENSE_NW / P.nwr;
    const int64_t grid = std::min<int64_t>((P.ntiles + nwc - 1) / nwc, h->num_sms);
    kern<<<(unsigned)grid, DENSE_NT, smem, st>>>(P);
    CK(cudaGetLastError());
    ++h->last_launches;
    accumulate = 1;
  }
  return TD_OK;
}

// CDO path (td_cdo.cuh): W = L^{-1} per segment, built on the first use of TD_PATH_CDO
// (every segment, or the ones AUTO gives to the CDO kernel, that do not have their W yet; synchronous)
td_status cdo_setup(td_handle* h, bool all_segments) {
  if (h->cdoW.empty()) h->cdoW.assign(h->n_seg, nullptr);
  std::vector<CdoSeg> cs;
  std::vector<int> ids;
  td_status st = TD_OK;
  for (int s = 0; s < h->n_seg && st == TD_OK; ++s) {
    const SegHost& sg = h->segs[s];
    if (!(all_segments || sg.auto_cdo) || sg.n > CDO_MAX_N || h->cdoW[s]) continue;
    const int npad = (sg.n + 31) / 32 * 32;
    double* W = nullptr;
    if (cudaMalloc(&W, sizeof(double) * (size_t)npad * npad) != cudaSuccess) { st = TD_ENOMEM; break; }
    CdoSeg c;
    c.rho = h->d_rho + sg.off; c.W = W; c.n = sg.n; c.npad = npad;
    cs.push_back(c); ids.push_back(s);
  }
  CdoSeg* d_cs = nullptr;
  if (st == TD_OK && !cs.empty()) {
    if (cudaMalloc(&d_cs, sizeof(CdoSeg) * cs.size()) != cudaSuccess) st = TD_ENOMEM;
    else if (cudaMemcpy(d_cs, cs.data(), sizeof(CdoSeg) * cs.size(), cudaMemcpyHostToDevice) != cudaSuccess) st = TD_ECUDA;
    else {
      cdo_whitener_kernel<<<(unsigned)cs.size(), CDO_NT>>>(d_cs);
      if (cudaGetLastError() != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess) st = TD_ECUDA;
    }
  }
  cudaFree(d_cs);
  if (st != TD_OK) { for (const CdoSeg& c : cs) cudaFree(c.W); return st; }
  for (size_t i = 0; i < ids.size(); ++i) h->cdoW[ids[i]] = cs[i].W;
  return TD_OK;
}

template <int NC>
td_status launch_cdo_nc(td_handle* h, const CdoParams& P0, int nbuf, cudaStream_t st, bool dry) {
  auto kern = td_cdo_kernel<NC>;
  static int cache[TD_MAX_DEV];
  CdoParams P = P0;
  P.nbuf = nbuf; P.ntiles = (P.B + 8 * NC - 1) / (8 * NC);
  const size_t smem = cdo_smem_bytes<NC>(P.npad, nbuf);
  int nb = 0;
  td_status cs = kernel_config(kern, DENSE_NT, h->smem_optin, smem, h->device, cache, &nb);
  if (cs != TD_OK) return cs;
  if (smem > h->smem_optin) return TD_EUNSUPPORTED;
  if (dry) return TD_OK;
  const int nwc = DENSE_NW / dense_nwr(P.npad);
  const int64_t grid = std::min<int64_t>((P.ntiles + nwc - 1) / nwc, h->num_sms);
  kern<<<(unsigned)std::max<int64_t>(grid, 1), DENSE_NT, smem, st>>>(P);
  CK(cudaGetLastError());
  ++h->last_launches;
  return TD_OK;
}

// one launch per segment; 32-template panels (NC = 4) where one fits shared memory, else 16 (NC = 2); double-buffered
// panels where two fit
// (every segment, or the ones AUTO gives to the CDO kernel; *count receives how many ran)
td_status launch_cdo(td_handle* h, const double* d, const double* H, int64_t ldh, int64_t B, double* out, int accumulate,
                     cudaStream_t st, bool all_segments, int* count, bool dry = false) {
  if (count) *count = 0;
  for (int s = 0; s < h->n_seg; ++s) {
    const SegHost& sg = h->segs[s];
    if (!(all_segments || sg.auto_cdo)) continue;
    if (h->cdoW.empty() || !h->cdoW[s]) return TD_EUNSUPPORTED;  // (never: td_create / td_set_path built it)
    if (count) ++*count;
    CdoParams P;
    P.d = d; P.H = H; P.ldh = ldh; P.B = B; P.out = out; P.off = sg.off; P.n = sg.n; P.npad = (sg.n + 31) / 32 * 32;
    P.W = h->cdoW[s]; P.accumulate = accumulate;
    P.vec_ok = (sg.off % 2 == 0) && (sg.n % 2 == 0) && (ldh % 2 == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
    td_status r;
    if (cdo_smem_bytes<4>(P.npad, 1) <= h->smem_optin)
      r = launch_cdo_nc<4>(h, P, cdo_smem_bytes<4>(P.npad, 2) <= h->smem_optin ? 2 : 1, st, dry);
    else
      r = launch_cdo_nc<2>(h, P, cdo_smem_bytes<2>(P.npad, 2) <= h->smem_optin ? 2 : 1, st, dry);
    if (r != TD_OK) return r;
    accumulate = 1;
  }
  return TD_OK;
}

// FFT path over all size classes.  MODE_LOGLIKE: out0 = loglike.  MODE_INNER: out0 = <d,h>, out1 = <h,h>.
// Ringdown parameters straight into the fused kernels (td_ring.cuh): possible when every size class of the handle is served
// by td_fused4_kernel (segments of 513..4096 samples) and none is sent elsewhere (dense chooser, forced staged variant)
bool ring_fused_ok(const td_handle* h) {
  if (h->fft_variant != 0 || (h->path != TD_PATH_AUTO && h->path != TD_PATH_FFT)) return false;
  for (const ClassInfo& c : h->classes)
    if (c.log2M < 10 || c.log2M > 12 || !c.d_Gp) return false;
  return true;
}
td_status run_ring_fused(td_handle* h, const double* d, const double* params, int64_t B, double fs, double* out,
                         cudaStream_t st, bool dry = false) {
  int accumulate = 0;
  const bool f32 = h->precision == TD_PREC_F32;
  for (const ClassInfo& cls : h->classes) {
    if (f32 && cls.has32) {
      td32api::Launch L;
      L.d = d; L.H = params; L.ldh = 5ll * h->n_seg; L.B = B; L.out0 = out; L.out1 = nullptr; L.accumulate = accumulate;
      L.mode = MODE_LOGLIKE; L.syn = 1; L.fs = fs;
      td_status s = td32api::launch(cls.t32, L, h->num_sms, h->device, st, dry);
      if (s != TD_OK) return s;
    } else {
      FusedParams P;
      P.d = d; P.H = params; P.ldh = 5ll * h->n_seg; P.B = B; P.out0 = out; P.out1 = nullptr;
      P.segs = cls.d_segs; P.n_seg = (int)cls.seg_ids.size(); P.accumulate = accumulate; P.T = cls.T;
      td_status s = cls.log2M == 10 ? launch_fused4<10, MODE_LOGLIKE, 1>(h, P, cls.d_Gp, st, dry, fs)
                  : cls.log2M == 11 ? launch_fused4<11, MODE_LOGLIKE, 1>(h, P, cls.d_Gp, st, dry, fs)
                                    : launch_fused4<12, MODE_LOGLIKE, 1>(h, P, cls.d_Gp, st, dry, fs);
      if (s != TD_OK) return s;
    }
    if (!dry) { if (f32 && cls.has32) ++h->last_launches; accumulate = 1; }   // (launch_fused4 counts its own)
  }
  if (!dry) h->last_path = TD_PATH_FFT;
  return TD_OK;
}

// ---- M = 65536 on a 16-CTA cluster (td_cluster16.cuh): one launch per segment + the rank-ordered sum of the 16 partials
template <int MODE>
td_status launch_cluster16(td_handle* h, const Cluster16Params& PC, int* nclusters, cudaStream_t st, bool dry) {
  auto kern = td_cluster16_kernel<MODE>;
  const size_t smem = Cluster16Shape::smem_bytes();
  static int cache[TD_MAX_DEV];  // 0 = not configured on this device yet, else 1 + clusters that can be co-resident
  if (h->device < 0 || h->device >= TD_MAX_DEV) return TD_EUNSUPPORTED;
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = Cluster16Shape::CS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  cfg.blockDim = dim3(Cluster16Shape::NT); cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cfg.attrs = attr; cfg.numAttrs = 1;
  if (cache[h->device] == 0) {
    int n = 0;
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) == cudaSuccess &&
        cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
      cfg.gridDim = dim3(Cluster16Shape::CS * (h->num_sms / Cluster16Shape::CS));
      if (cudaOccupancyMaxActiveClusters(&n, kern, &cfg) != cudaSuccess) n = 0;
    }
    cudaGetLastError();   // a device that cannot host the cluster is not an error: the staged kernels serve the class
    cache[h->device] = n + 1;
  }
  *nclusters = cache[h->device] - 1;
  if (dry || *nclusters < 1) return TD_OK;
  const long long want = MODE == MODE_STOREZ ? 1 : PC.base.B;
  cfg.gridDim = dim3(Cluster16Shape::CS * (unsigned)std::max<long long>(1, std::min<long long>(want, *nclusters)));
  CK(cudaLaunchKernelEx(&cfg, kern, PC));
  ++h->last_launches;
  return TD_OK;
}

// ---- M = 16384 / 32768 / 65536 as one persistent kernel of 4- / 8- / 16-CTA groups exchanging through L2 (td_group16.cuh)
constexpr int GRP_MAX_GROUPS = 64;
inline int group_slot(int cs) { return cs == 4 ? 0 : cs == 8 ? 1 : 2; }
template <int CS, int MODE>
td_status launch_group(td_handle* h, const GroupParams& PG, int* ngroups, cudaStream_t st, bool dry) {
  auto kern = td_group_kernel<CS, MODE>;
  const size_t smem = Cluster16Shape::smem_bytes();
  static int cache[TD_MAX_DEV];
  int per_sm = 0;
  td_status cs = kernel_config(kern, Cluster16Shape::NT, smem, smem, h->device, cache, &per_sm);
  if (cs != TD_OK) return cs;
  *ngroups = std::min(GRP_MAX_GROUPS, per_sm * h->num_sms / CS);
  if (dry || *ngroups < 1) return TD_OK;
  *ngroups = std::min(*ngroups, h->group_cap[group_slot(CS)]);   // what the exchange buffers hold (group_setup)
  const long long want = MODE == MODE_STOREZ ? 1 : PG.base.B;
  const unsigned groups = (unsigned)std::max<long long>(1, std::min<long long>(want, *ngroups));
  CK(cudaMemsetAsync(PG.bar, 0, sizeof(unsigned) * 2 * GRP_MAX_GROUPS, st));
  cudaLaunchConfig_t cfg = {};
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeCooperative;   // every CTA co-resident: the groups synchronise through global counters
  attr[0].val.cooperative = 1;
  cfg.gridDim = dim3(CS * groups); cfg.blockDim = dim3(Cluster16Shape::NT);
  cfg.dynamicSmemBytes = smem; cfg.stream = st; cfg.attrs = attr; cfg.numAttrs = 1;
  const cudaError_t le = cudaLaunchKernelEx(&cfg, kern, PG);
  if (le == cudaErrorCooperativeLaunchTooLarge) {   // the device is shared (MPS, a partition): fewer CTAs fit than the occupancy
    cudaGetLastError();                             // query promised - the class goes back to the staged kernels for good
    h->group_cap[group_slot(CS)] = -1;
    return TD_EUNSUPPORTED;
  }
  CK(le);
  ++h->last_launches;
  return TD_OK;
}
template <int CS>
int group_capacity(td_handle* h) {
  GroupParams PG = {};
  int n = 0, m = 0, z = 0;
  if (launch_group<CS, MODE_LOGLIKE>(h, PG, &n, nullptr, true) != TD_OK) return 0;
  if (launch_group<CS, MODE_INNER>(h, PG, &m, nullptr, true) != TD_OK) return 0;
  if (launch_group<CS, MODE_STOREZ>(h, PG, &z, nullptr, true) != TD_OK) return 0;
  return std::min(n, std::min(m, z));
}
// the exchange buffers are the staged workspace (L2-resident by size): groups x 2 parities x (2 NF | 2 M) elements
bool group_fits(const td_handle* h, int cs, int groups) {
  const size_t M = (size_t)cs * Cluster16Shape::ML;
  return h->grp_bar && h->wsU_elems >= (size_t)groups * 2 * M && h->wsZ_elems >= (size_t)groups * 4 * M && h->wsP_elems >= (size_t)cs * 2;
}

// counters + occupancy; leaves group_cap = -1 (class stays on the staged kernels) when the device cannot host a group
td_status group_setup(td_handle* h, int cs) {
  if (!h->grp_bar && cudaMalloc(&h->grp_bar, sizeof(unsigned) * 2 * GRP_MAX_GROUPS) != cudaSuccess) { cudaGetLastError(); return TD_ENOMEM; }
  int& cap = h->group_cap[group_slot(cs)];
  int coop = 0;
  if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, h->device) != cudaSuccess || !coop) { cudaGetLastError(); cap = -1; return TD_OK; }
  cap = cs == 4 ? group_capacity<4>(h) : cs == 8 ? group_capacity<8>(h) : group_capacity<16>(h);
  while (cap > 0 && !group_fits(h, cs, cap)) --cap;
  if (cap < 1) cap = -1;   // asked and answered
  return TD_OK;
}

template <int CS, int MODE>
td_status run_group(td_handle* h, const ClassInfo& cls, int idx_in_class, const double* d, const double* H, int64_t ldh,
                    int64_t B, double* out0, double* out1, double scale0, double scale1, int accumulate, cudaStream_t st) {
  const SegHost& sg = h->segs[cls.seg_ids[idx_in_class]];
  const int64_t SB = std::max<int64_t>(1, (int64_t)(h->wsP_elems / (CS * 2)));   // templates per partial buffer
  h->touched = true;
  const int64_t Bn = (MODE == MODE_STOREZ) ? 1 : B;
  for (int64_t b0 = 0; b0 < Bn; b0 += SB) {
    const int64_t nb = std::min<int64_t>(SB, Bn - b0);
    GroupParams PG;
    PG.base.d = d; PG.base.H = H ? H + b0 * ldh : nullptr; PG.base.ldh = ldh; PG.base.B = nb;
    PG.base.out0 = nullptr; PG.base.out1 = nullptr; PG.base.segs = cls.d_segs + idx_in_class; PG.base.n_seg = 1;
    PG.base.accumulate = 0; PG.base.T = cls.T;
    PG.Gp = sg.Gc16; PG.partial = h->wsPartial;
    PG.wsU = static_cast<cplx*>(h->wsU); PG.wsZ = static_cast<cplx*>(h->wsZ); PG.bar = h->grp_bar;
    int ng = 0;
    td_status s = launch_group<CS, MODE>(h, PG, &ng, st, false);
    if (s != TD_OK) return s;
    if (ng < 1) return TD_EUNSUPPORTED;
    if (MODE != MODE_STOREZ) {
      lg_finish_kernel<<<(unsigned)((nb + 127) / 128), 128, 0, st>>>(h->wsPartial, CS, (int)nb, out0 ? out0 + b0 : nullptr,
                                                                    out1 ? out1 + b0 : nullptr, scale0, scale1, accumulate);
      CK(cudaGetLastError());
      ++h->last_launches;
    }
  }
  return TD_OK;
}

// how many 16-CTA clusters of the kernel fit the device (0: the class stays on the staged kernels)
int cluster16_capacity(td_handle* h) {
  int n = 0;
  Cluster16Params PC = {};
  if (launch_cluster16<MODE_LOGLIKE>(h, PC, &n, nullptr, true) != TD_OK) return 0;
  int m = 0;
  if (launch_cluster16<MODE_INNER>(h, PC, &m, nullptr, true) != TD_OK) return 0;
  int z = 0;
  if (launch_cluster16<MODE_STOREZ>(h, PC, &z, nullptr, true) != TD_OK) return 0;
  return std::min(n, std::min(m, z));
}

template <int MODE>
td_status run_cluster16(td_handle* h, const ClassInfo& cls, int idx_in_class, const double* d, const double* H, int64_t ldh,
                        int64_t B, double* out0, double* out1, double scale0, double scale1, int accumulate, cudaStream_t st) {
  const SegHost& sg = h->segs[cls.seg_ids[idx_in_class]];
  const int64_t SB = std::max<int64_t>(1, (int64_t)(h->wsP_elems / (Cluster16Shape::CS * 2)));   // templates per partial buffer
  h->touched = true;
  const int64_t Bn = (MODE == MODE_STOREZ) ? 1 : B;
  for (int64_t b0 = 0; b0 < Bn; b0 += SB) {
    const int64_t nb = std::min<int64_t>(SB, Bn - b0);
    Cluster16Params PC;
    PC.base.d = d; PC.base.H = H ? H + b0 * ldh : nullptr; PC.base.ldh = ldh; PC.base.B = nb;
    PC.base.out0 = nullptr; PC.base.out1 = nullptr; PC.base.segs = cls.d_segs + idx_in_class; PC.base.n_seg = 1;
    PC.base.accumulate = 0; PC.base.T = cls.T;
    PC.Gp = sg.Gc16; PC.partial = h->wsPartial;
    int ncl = 0;
    td_status s = launch_cluster16<MODE>(h, PC, &ncl, st, false);
    if (s != TD_OK) return s;
    if (ncl < 1) return TD_EUNSUPPORTED;
    if (MODE != MODE_STOREZ) {
      lg_finish_kernel<<<(unsigned)((nb + 127) / 128), 128, 0, st>>>(h->wsPartial, Cluster16Shape::CS, (int)nb, out0 ? out0 + b0 : nullptr,
                                                                    out1 ? out1 + b0 : nullptr, scale0, scale1, accumulate);
      CK(cudaGetLastError());
      ++h->last_launches;
    }
  }
  return TD_OK;
}

// `f32`: classes that have fp32 tables and are not served by the dense kernel run the fp32 build of their kernel
template <int MODE>
td_status run_fft_path(td_handle* h, const double* d, const double* H, int64_t ldh, int64_t B, double* out0,
                       double* out1, cudaStream_t st, bool skip_dense_classes = false, int accumulate = 0, bool f32 = false) {
  const double sc0 = (MODE == MODE_LOGLIKE) ? -0.5 : 1.0, sc1 = 1.0;
  for (const ClassInfo& cls : h->classes) {
    if (skip_dense_classes && class_is_dense(h, cls, MODE)) continue;
    const bool st32 = td32api::staged_class(cls.log2M);   // (a fused-shape class forced onto the staged kernels stays fp64)
    if (f32 && cls.has32 && !class_is_dense(h, cls, MODE) && (st32 || class_is_fused(h, cls)) && h->fft_variant != 3) {
      td32api::Launch L;
      L.d = d; L.H = H; L.ldh = ldh; L.B = B; L.out0 = out0; L.out1 = out1; L.accumulate = accumulate; L.mode = MODE;
      td32api::StagedBorrow sb;
      if (st32) {
        sb.wsU = h->wsU; sb.wsU_bytes = h->wsU_elems * sizeof(cplx); sb.wsZ = h->wsZ; sb.wsZ_bytes = h->wsZ_elems * sizeof(cplx);
        sb.wsPartial = h->wsPartial; sb.wsP_elems = h->wsP_elems;
        sb.aux_stream = h->aux_stream; sb.ev_fork = h->ev_fork; sb.ev_join = h->ev_join; sb.launches = &h->last_launches;
        const int gcs = group_cs(cls.log2M);   // the group kernel where the fp64 path would use it (its buffers hold twice the groups in fp32)
        sb.grp_bar = h->grp_bar;
        sb.group_cap = (gcs && h->fft_variant != 2) ? std::max(0, h->group_cap[group_slot(gcs)]) : 0;
        L.staged = &sb;
        h->touched = true;
      }
      td_status s = td32api::launch(cls.t32, L, h->num_sms, h->device, st, false);
      if (s != TD_OK) return s;
      if (!st32) ++h->last_launches;
      accumulate = 1;
      continue;
    }
    if (class_is_fused(h, cls)) {
      FusedParams P;
      P.d = d; P.H = H; P.ldh = ldh; P.B = B; P.out0 = out0; P.out1 = out1;
      P.segs = cls.d_segs; P.n_seg = (int)cls.seg_ids.size(); P.accumulate = accumulate; P.T = cls.T;
      td_status s = launch_fused<MODE>(h, cls.log2M, P, cls.d_Gp, st);
      if (s != TD_OK) return s;
      accumulate = 1;
    } else {
      // M = 16384 / 32768 / 65536: the group kernel (4 / 8 / 16 CTAs per template exchanging through L2, td_group16.cuh) when the
      // device co-hosts a group, else the staged kernels.  The 16-CTA cluster kernel only on request (variant 3): measured 0.885 ms against 0.737 ms for the staged
      // kernels on c4 - its two all-to-all exchanges run at the 16 B/cycle/SM of distributed-shared-memory stores and only 7
      // clusters (112 of 148 SMs) are co-resident (profiles/r02_c4_cluster16.md)
      const bool c16 = cls.log2M == Cluster16Shape::LOG2M && h->fft_variant == 3 && h->cluster16_cap > 0;
      const int gcs = group_cs(cls.log2M);
      const bool grp = gcs && h->fft_variant != 2 && !c16 && h->group_cap[group_slot(gcs)] > 0;
      for (size_t i = 0; i < cls.seg_ids.size(); ++i) {
        const int id = cls.seg_ids[i];
        td_status s = c16 ? run_cluster16<MODE>(h, cls, (int)i, d, H, ldh, B, out0, out1, sc0, sc1, accumulate, st)
                      : !grp ? run_staged<MODE>(h, cls, h->segs[id], d, H, ldh, B, out0, out1, sc0, sc1, accumulate, st)
                      : gcs == 4 ? run_group<4, MODE>(h, cls, (int)i, d, H, ldh, B, out0, out1, sc0, sc1, accumulate, st)
                      : gcs == 8 ? run_group<8, MODE>(h, cls, (int)i, d, H, ldh, B, out0, out1, sc0, sc1, accumulate, st)
                                 : run_group<16, MODE>(h, cls, (int)i, d, H, ldh, B, out0, out1, sc0, sc1, accumulate, st);
        if (s == TD_EUNSUPPORTED && grp && h->group_cap[group_slot(gcs)] < 0)   // the cooperative launch was refused: nothing ran
          s = run_staged<MODE>(h, cls, h->segs[id], d, H, ldh, B, out0, out1, sc0, sc1, accumulate, st);
        if (s != TD_OK) return s;
        accumulate = 1;
      }
    }
  }
  return TD_OK;
}

// One batch call: the dense kernel for the classes the chooser (or td_set_path) gives it, the FFT
// kernels for the rest, all accumulating into the same outputs.
template <int MODE>
td_status run_batch(td_handle* h, const double* d, const double* H, int64_t ldh, int64_t B, double* out0,
                    double* out1, cudaStream_t st) {
  const DenseState& D = h->dense;
  if (MODE == MODE_LOGLIKE && (h->path == TD_PATH_CDO || (h->path == TD_PATH_AUTO && h->any_auto_ll))) {
    // log-likelihood of the short segments: the triangular contraction with the cached L^{-1} (measured faster than the
    // Gohberg-Semencul dense kernel at every length up to 1024, profiles/r02_cdo.md); AUTO: the dense-class segments
    int nc = 0, ng = 0, acc = 0;
    const bool forced = h->path == TD_PATH_CDO;
    if (!forced && !D.aut_gs.empty()) {   // AUTO: the shortest segments stay on the Gohberg-Semencul dense kernel
      td_status s = launch_dense<MODE>(h, D.aut_gs, d, H, ldh, B, out0, out1, 0, st);
      if (s != TD_OK) return s;
      ng = (int)D.aut_gs.size(); acc = 1;
    }
    td_status s = launch_cdo(h, d, H, ldh, B, out0, acc, st, forced, &nc);
    if (s != TD_OK) return s;
    const bool all = nc + ng == h->n_seg;
    h->last_path = all ? (nc > 0 ? TD_PATH_CDO : TD_PATH_DENSE) : TD_PATH_FFT;
    if (all) return TD_OK;
    return run_fft_path<MODE>(h, d, H, ldh, B, out0, out1, st, true, 1, h->precision == TD_PREC_F32);
  }
  const std::vector<DenseSeg>* dsegs = nullptr;
  if (h->path == TD_PATH_DENSE || h->path == TD_PATH_CDO) dsegs = &D.all;
  else if (h->path == TD_PATH_AUTO) dsegs = &D.aut;
  const int nd = dsegs ? (int)dsegs->size() : 0;
  int accumulate = 0;
  if (nd > 0) {
    td_status s = launch_dense<MODE>(h, *dsegs, d, H, ldh, B, out0, out1, 0, st);
    if (s != TD_OK) return s;
    accumulate = 1;
  }
  h->last_path = (nd == h->n_seg) ? TD_PATH_DENSE : TD_PATH_FFT;
  if (nd == h->n_seg) return TD_OK;
  return run_fft_path<MODE>(h, d, H, ldh, B, out0, out1, st, true, accumulate, h->precision == TD_PREC_F32);
}

// <d, h_b> = u . h_b with u = C^{-1} d (td_dot.cuh); z of the data vector is already in every segment's zd
td_status run_dot(td_handle* h, const double* H, int64_t ldh, int64_t B, double* out_dh, cudaStream_t st) {
  // h->ud and the per-tile partial weights (h->wsDot) were allocated by td_create
  for (const SegHost& sg : h->segs) {
    const int nt = (int)((sg.n + DOTW_NT - 1) / DOTW_NT);
    dot_weight_tile_kernel<<<(unsigned)(nt * (nt + 1) / 2), DOTW_NT, 0, st>>>(sg.a, sg.zd, (int)sg.n, h->wsDot, nt);
    CK(cudaGetLastError());
    dot_weight_sum_kernel<<<(unsigned)((sg.n + 255) / 256), 256, 0, st>>>(h->wsDot, (int)sg.n, nt, 1.0 / std::sqrt(sg.v), h->ud + sg.off);
    CK(cudaGetLastError());
    h->last_launches += 2;
  }
  const bool vec = (ldh % 2 == 0) && ((reinterpret_cast<uintptr_t>(H) & 15) == 0);
  void (*kern)(const double*, const double*, long long, long long, int, double*, int) =
      vec ? dot_rows_kernel<true> : dot_rows_kernel<false>;
  static int cache[2][TD_MAX_DEV];
  int nb = 0;
  {
    td_status cs = kernel_config(kern, DOT_NT, 0, 0, h->device, cache[vec ? 1 : 0], &nb);
    if (cs != TD_OK) return cs;
  }
  const unsigned grid = (unsigned)std::max<int64_t>(1, std::min<int64_t>((B + 1) / 2, (int64_t)std::max(nb, 1) * h->num_sms));
  kern<<<grid, DOT_NT, 0, st>>>(h->ud, H, ldh, B, (int)h->n_tot, out_dh, 0);
  CK(cudaGetLastError());
  ++h->last_launches;
  h->last_path = TD_PATH_DOT;
  return TD_OK;
}

// workspace of the staged kernels for every class that may run through them (all classes when the staged variant is forced)
td_status staged_alloc(td_handle* h, bool all_classes) {
  for (const ClassInfo& c : h->classes) {
    if (!all_classes && class_is_fused_shape(c.log2M)) continue;
    const StagedGeom g = staged_geom(c.log2M);
    td_status a = grow(h->wsU, h->wsU_elems, 2 * g.uh);
    if (a == TD_OK) a = grow(h->wsZ, h->wsZ_elems, 2 * g.zh);
    if (a == TD_OK) a = grow(h->wsPartial, h->wsP_elems, std::max<size_t>(STAGED_PARTIAL_DEFAULT / sizeof(double), (size_t)g.nblk * 2));
    if (a != TD_OK) return a;
  }
  return TD_OK;
}

// Dry pass over every kernel the handle's size classes can reach, in all three modes: sets the shared-memory attributes
// and caches the occupancy figures (kernel_config), launches nothing.
template <int MODE> td_status warm_mode(td_handle* h) {
  FusedParams P = {};
  P.B = 1;
  for (const ClassInfo& cls : h->classes) {
    if (!class_is_fused_shape(cls.log2M)) continue;
    td_status s = launch_fused<MODE>(h, cls.log2M, P, cls.d_Gp, nullptr, true);
    if (s != TD_OK) return s;
  }
  if (!h->dense.all.empty()) {
    td_status s = launch_dense<MODE>(h, h->dense.all, nullptr, nullptr, 0, 1, nullptr, nullptr, 0, nullptr, true);
    if (s != TD_OK) return s;
  } else if (!h->dense.aut.empty()) {
    td_status s = launch_dense<MODE>(h, h->dense.aut, nullptr, nullptr, 0, 1, nullptr, nullptr, 0, nullptr, true);
    if (s != TD_OK) return s;
  }
  return TD_OK;
}
td_status warm_kernels(td_handle* h) {
  if (ring_fused_ok(h)) {
    td_status r = run_ring_fused(h, nullptr, nullptr, 1, 1.0, nullptr, nullptr, true);
    if (r != TD_OK) return r;
  }
  td_status s = warm_mode<MODE_LOGLIKE>(h);
  if (s == TD_OK) s = warm_mode<MODE_INNER>(h);
  if (s == TD_OK) s = warm_mode<MODE_STOREZ>(h);
  if (s == TD_OK) s = launch_block<true>(h->device, nullptr, 0, 0, nullptr, 0, nullptr, true);
  if (s == TD_OK) s = launch_block<false>(h->device, nullptr, 0, 0, nullptr, 0, nullptr, true);
  return s;
}

}  // namespace

// ------------------------------------------------------------------------------------------
// C ABI
// ------------------------------------------------------------------------------------------
extern "C" {

const char* td_strerror(td_status s) {
  switch (s) {
    case TD_OK: return "ok";
    case TD_EINVAL: return "invalid argument";
    case TD_ENOTSPD: return "autocorrelation is not symmetric positive definite (or not finite)";
    case TD_ENOMEM: return "out of memory";
    case TD_ECUDA: return "CUDA error";
    case TD_EUNSUPPORTED: return "unsupported request";
  }
  return "unknown status";
}

static td_status create_impl(td_handle* h, const double* acf, const int64_t* seg_lengths, int n_seg) {
  cudaDeviceProp prop;
  CK(cudaGetDeviceProperties(&prop, h->device));
  h->num_sms = prop.multiProcessorCount;
  h->smem_optin = prop.sharedMemPerBlockOptin;
  h->n_seg = n_seg;
  h->segs.resize(n_seg);
  int64_t off = 0;
  for (int s = 0; s < n_seg; ++s) {
    SegHost& sg = h->segs[s];
    sg.off = off; sg.n = (int)seg_lengths[s]; sg.rho0 = acf[off];
    sg.log2M = std::max(FUSED_MIN_LOG2M, next_log2(sg.n));
    off += sg.n;
    h->max_n = std::max(h->max_n, sg.n);
  }
  h->n_tot = off;
  // ---- device copies of the ACFs, Levinson-Durbin per segment (one CTA each)
  double* d_v = nullptr; double* d_ld = nullptr; int* d_status = nullptr; LevSeg* d_lev = nullptr;
  struct Tmp { double*& b; double*& c; int*& d; LevSeg*& e; ~Tmp() { cudaFree(b); cudaFree(c); cudaFree(d); cudaFree(e); } }
      tmp{d_v, d_ld, d_status, d_lev};
  CK(cudaMalloc(&h->d_rho, sizeof(double) * h->n_tot));   // owned by the handle (the CDO setup reads it again)
  double* const d_rho = h->d_rho;
  CK(cudaMemcpy(d_rho, acf, sizeof(double) * h->n_tot, cudaMemcpyHostToDevice));
  CK(cudaMalloc(&d_v, sizeof(double) * n_seg));
  CK(cudaMalloc(&d_ld, sizeof(double) * n_seg));
  CK(cudaMalloc(&d_status, sizeof(int) * n_seg));
  CK(cudaMemset(d_status, 0xff, sizeof(int) * n_seg));
  CK(cudaMalloc(&d_lev, sizeof(LevSeg) * n_seg));
  std::vector<LevSeg> lev(n_seg);
  for (int s = 0; s < n_seg; ++s) {
    SegHost& sg = h->segs[s];
    CK(cudaMalloc(&sg.a, sizeof(double) * sg.n));
    lev[s].rho = d_rho + sg.off; lev[s].a = sg.a; lev[s].n = sg.n; lev[s].coop = sg.n >= LEV_COOP_MIN_N ? 1 : 0;
  }
  CK(cudaMemcpy(d_lev, lev.data(), sizeof(LevSeg) * n_seg, cudaMemcpyHostToDevice));
  levinson_kernel<<<n_seg, LEV_NT>>>(d_lev, d_v, d_ld, d_status);
  CK(cudaGetLastError());
  {
    // long segments: the cooperative multi-CTA recursion, one launch each
    int coop_ok = 0, nb = 0;
    CK(cudaDeviceGetAttribute(&coop_ok, cudaDevAttrCooperativeLaunch, h->device));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&nb, levinson_coop_kernel, LEVC_NT, 0));
    // one CTA per SM (measured with the counter barrier of td_setup.cuh, td_create at N = 65536 / 2^18 / 2^20: 48 CTAs 0.24 / 1.26 /
    // 9.8 s, 148 CTAs 0.24 / 1.02 / 5.5 s, 296 CTAs 0.27 / 1.08 / 5.2 s)
    const int G = std::min(h->num_sms, std::max(1, nb) * h->num_sms);
    double* d_part = nullptr;
    for (int s = 0; s < n_seg; ++s) {
      if (!lev[s].coop) continue;
      if (!coop_ok) return TD_EUNSUPPORTED;
      if (!d_part) CK(cudaMalloc(&d_part, sizeof(double) * (2 * G + 1)));   // + the 64-bit arrival counter of the grid barrier
      unsigned long long* d_bar = reinterpret_cast<unsigned long long*>(d_part + 2 * G);
      CK(cudaMemsetAsync(d_bar, 0, sizeof(unsigned long long), 0));
      LevSeg one = lev[s];
      double* pv = d_v + s; double* pl = d_ld + s; int* ps = d_status + s;
      void* args[] = {&one, &d_part, &d_bar, &pv, &pl, &ps};
      CK(cudaLaunchCooperativeKernel((void*)levinson_coop_kernel, dim3(G), dim3(LEVC_NT), args, 0, 0));
    }
    CK(cudaDeviceSynchronize());
    cudaFree(d_part);
  }
  std::vector<int> status(n_seg);
  std::vector<double> v(n_seg), ld(n_seg);
  CK(cudaMemcpy(status.data(), d_status, sizeof(int) * n_seg, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(v.data(), d_v, sizeof(double) * n_seg, cudaMemcpyDeviceToHost));
  CK(cudaMemcpy(ld.data(), d_ld, sizeof(double) * n_seg, cudaMemcpyDeviceToHost));
  for (int s = 0; s < n_seg; ++s) {
    if (status[s] != 0 || !(v[s] > 0.0) || !std::isfinite(v[s])) return TD_ENOTSPD;
    h->segs[s].v = v[s]; h->segs[s].logdet = ld[s];
  }
  // ---- size classes, twiddle tables
  for (int s = 0; s < n_seg; ++s) {
    const int l2 = h->segs[s].log2M;
    auto it = std::find_if(h->classes.begin(), h->classes.end(), [&](const ClassInfo& c) { return c.log2M == l2; });
    if (it == h->classes.end()) { h->classes.emplace_back(); h->classes.back().log2M = l2; it = h->classes.end() - 1; }
    it->seg_ids.push_back(s);
    it->max_n = std::max(it->max_n, h->segs[s].n);
  }
  for (ClassInfo& c : h->classes) {
    const int TW = 2 << c.log2M;
    CK(cudaMalloc(&c.T, sizeof(cplx) * TW));
    tw_table_kernel<<<(TW + 255) / 256, 256>>>(c.T, TW);
    CK(cudaGetLastError());
  }
  // ---- generator spectra: G = conj(FFT_2M(a - i b)) / (4M sqrt(v)), split even/odd, DIT order
  for (ClassInfo& c : h->classes) {
    const int M = 1 << c.log2M, n2 = 2 * M;
    cplx* F = nullptr;
    CK(cudaMalloc(&F, sizeof(cplx) * n2));
    td_status st = TD_OK;
    for (int id : c.seg_ids) {
      SegHost& sg = h->segs[id];
      if (cudaMalloc(&sg.G, sizeof(cplx) * n2) != cudaSuccess) { st = TD_ENOMEM; break; }
      if (cudaMalloc(&sg.zd, sizeof(cplx) * M) != cudaSuccess) { st = TD_ENOMEM; break; }  // z of the data vector (td_inner_batch)
      gen_pack_kernel<<<(n2 + 255) / 256, 256>>>(sg.a, sg.n, F, n2);
      int launches = 0;
      st = staged_forward(h->device, F, 1, n2, 0, c.T, n2, 0, &launches);
      if (st != TD_OK) break;
      const double gscale = 0.5 / ((double)n2 * std::sqrt(sg.v));
      gen_permute_kernel<<<(n2 + 255) / 256, 256>>>(F, sg.G, M, gscale, 0);
      if (c.log2M >= 10 && c.log2M <= CLUSTER_LOG2M) {
        const size_t pb = sizeof(cplx) * 2 * SmemArr::padded(M);
        if (cudaMalloc(&sg.Gp, pb) != cudaSuccess) { st = TD_ENOMEM; break; }
        cudaMemsetAsync(sg.Gp, 0, pb, 0);
        gen_permute_kernel<<<(n2 + 255) / 256, 256>>>(F, sg.Gp, M, gscale, c.log2M == CLUSTER_LOG2M ? 2 : 1);
      }
      if (const int gcs = group_cs(c.log2M)) {   // per-CTA generator values of the group kernel (and, M = 65536, the cluster kernel)
        const size_t cb = sizeof(cplx) * gcs * Cluster16Shape::PADZ;
        if (cudaMalloc(&sg.Gc16, cb) != cudaSuccess) { st = TD_ENOMEM; break; }
        cudaMemsetAsync(sg.Gc16, 0, cb, 0);
        gen_permute_group_kernel<<<(n2 + 255) / 256, 256>>>(F, sg.Gc16, gscale, gcs);
      }
      if (cudaGetLastError() != cudaSuccess) { st = TD_ECUDA; break; }
    }
    cudaError_t e = cudaDeviceSynchronize();
    cudaFree(F);
    if (st != TD_OK) return st;
    if (e != cudaSuccess) return TD_ECUDA;
    std::vector<SegDev> sd(c.seg_ids.size());
    for (size_t i = 0; i < sd.size(); ++i) {
      const SegHost& sg = h->segs[c.seg_ids[i]];
      sd[i].off = sg.off; sd[i].n = sg.n; sd[i]._pad = c.seg_ids[i]; sd[i].G = sg.G; sd[i].zd = sg.zd; sd[i].rscale = 1.0;
    }
    CK(cudaMalloc(&c.d_segs, sizeof(SegDev) * sd.size()));
    CK(cudaMemcpy(c.d_segs, sd.data(), sizeof(SegDev) * sd.size(), cudaMemcpyHostToDevice));
    if (c.log2M >= 10 && c.log2M <= CLUSTER_LOG2M) {
      std::vector<const cplx*> gp(c.seg_ids.size());
      for (size_t i = 0; i < gp.size(); ++i) gp[i] = h->segs[c.seg_ids[i]].Gp;
      CK(cudaMalloc(&c.d_Gp, sizeof(cplx*) * gp.size()));
      CK(cudaMemcpy(c.d_Gp, gp.data(), sizeof(cplx*) * gp.size(), cudaMemcpyHostToDevice));
    }
  }
  // ---- dense path tables (the chooser's crossover is measured: DESIGN.md 6.4)
  h->dense.auto_n = DENSE_AUTO_N;
  td_status ds = dense_upload(h);
  if (ds != TD_OK) return ds;
  for (const ClassInfo& c : h->classes)   // AUTO evaluates the log-likelihood of the short classes with the cached L^{-1} (td_cdo.cuh)
    if (c.max_n <= CDO_AUTO_MAX_N) {
      h->any_auto_ll = true;
      for (int id : c.seg_ids) h->segs[id].auto_cdo = h->segs[id].n >= CDO_AUTO_MIN_N;
    }
  if (h->any_auto_ll) {
    ds = cdo_setup(h, false);
    if (ds == TD_OK) ds = launch_cdo(h, nullptr, nullptr, h->n_tot, 1, nullptr, 0, nullptr, false, nullptr, true);
    if (ds != TD_OK) return ds;
  }
  // ---- everything a batch call would otherwise create on first use: streams, events, scratch that does not grow with B
  CK(cudaStreamCreateWithFlags(&h->aux_stream, cudaStreamNonBlocking));
  CK(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  CK(cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming));
  CK(cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming));
  CK(cudaEventCreateWithFlags(&h->ev_last, cudaEventDisableTiming));
  for (int i = 0; i < 2; ++i) {
    CK(cudaEventCreateWithFlags(&h->ev_copied[i], cudaEventDisableTiming));
    CK(cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming));
  }
  CK(cudaMalloc(&h->ud, sizeof(double) * (size_t)h->n_tot));
  if (h->max_n <= DOT_MAX_N) {  // per-tile partial weights of the longest segment: ntile rows of ntile * 128 doubles
    size_t need = 0;
    for (const SegHost& sg : h->segs) { const size_t nt = (sg.n + DOTW_NT - 1) / DOTW_NT; need = std::max(need, nt * nt * DOTW_NT); }
    CK(cudaMalloc(&h->wsDot, sizeof(double) * need));
  }
  {
    std::vector<SynSeg> hs(n_seg);
    for (int s = 0; s < n_seg; ++s) { hs[s].off = h->segs[s].off; hs[s].n = (int)h->segs[s].n; hs[s]._pad = 0; }
    CK(cudaMalloc(&h->synSeg, sizeof(SynSeg) * n_seg));
    CK(cudaMemcpy(h->synSeg, hs.data(), sizeof(SynSeg) * n_seg, cudaMemcpyHostToDevice));
  }
  // staged classes: both lanes of the L2-resident workspace, partial sums for a default batch (td_reserve grows them)
  {
    td_status a = staged_alloc(h, false);
    if (a != TD_OK) return a;
  }
  // the 16384 / 32768 / 65536 classes run on the group kernel (td_group16.cuh) when the device can co-host at least one group; its
  // exchange buffers are the staged workspace
  for (const ClassInfo& c : h->classes)
    if (group_cs(c.log2M) && h->group_cap[group_slot(group_cs(c.log2M))] == 0) {
      td_status g = group_setup(h, group_cs(c.log2M));
      if (g != TD_OK) return g;
    }
  // ---- one dry pass over every kernel this handle can launch: shared-memory attributes and occupancy are cached now,
  // so that a batch call is launches only (and can be captured into a CUDA graph)
  return warm_kernels(h);
}

td_status td_create(const double* acf, const int64_t* seg_lengths, int n_seg, int device, td_handle** out) {
  if (!acf || !seg_lengths || !out || n_seg < 1) return TD_EINVAL;
  int64_t tot = 0;
  for (int s = 0; s < n_seg; ++s) {
    if (seg_lengths[s] < 1 || seg_lengths[s] > (1 << 26)) return TD_EINVAL;
    tot += seg_lengths[s];
  }
  for (int64_t i = 0; i < tot; ++i) if (!std::isfinite(acf[i])) return TD_ENOTSPD;
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) return TD_ECUDA;
  if (device < 0 || device >= ndev) return TD_EINVAL;
  DevGuard guard(device);
  if (!guard.ok) return TD_ECUDA;
  td_handle* h = new (std::nothrow) td_handle();
  if (!h) return TD_ENOMEM;
  h->device = device;
  td_status s = create_impl(h, acf, seg_lengths, n_seg);
  if (s != TD_OK) { free_handle(h); return s; }
  *out = h;
  return TD_OK;
}

td_status td_destroy(td_handle* h) {
  if (!h) return TD_OK;
  DevGuard guard(h->device);
  free_handle(h);
  return TD_OK;
}

td_status td_loglike_batch(td_handle* h, const double* d, const double* H, int64_t ldh, int64_t B, double* out,
                           void* stream) {
  if (!h || B < 0) return TD_EINVAL;
  if (B == 0) return TD_OK;
  if (!d || !H || !out || ldh < h->n_tot) return TD_EINVAL;
  DevGuard guard(h->device);
  if (!guard.ok) return TD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_launches = 0;
  td_status s = order_begin(h, st);
  if (s != TD_OK) return s;
  s = run_batch<MODE_LOGLIKE>(h, d, H, ldh, B, out, nullptr, st);
  const td_status e = order_end(h, st);
  return s != TD_OK ? s : e;
}

// rows per chunk of the host entry point: ~32 MiB of template data, at least one row
static int64_t host_chunk_rows(const td_handle* h, int64_t B) {
  return std::max<int64_t>(1, std::min<int64_t>(B, (32ll << 20) / (8 * h->n_tot)));
}
// rows per chunk of the synthesis panel: a whole number of waves of the persistent kernels, about 128 MB (measured on
// c2 / c3 / c5: 64 MB chunks, which stay in L2, give 11.1-11.9 / 1.47 / 1.61 M evals/s end to end, 136 MB chunks
// 12.2 / 1.51 / 1.64: fewer launches and tails outweigh the panel's trip through HBM, which the ALU-bound kernels hide)
static int64_t family_chunk_rows(const td_handle* h, int64_t B, int64_t ldh) {
  int64_t CH = std::max<int64_t>(1, (136ll << 20) / (8 * ldh));
  if (CH > h->num_sms) CH -= CH % h->num_sms;
  return std::min<int64_t>(CH, B);
}
// section offsets of the packed device buffer of td_loglike_family_batch_host, each rounded up to an even element count so
// that d (and out) start on a 16-byte boundary whatever the parity of 5 n_seg B (the TMA-staged first pass needs it)
static size_t even_up(size_t x) { return (x + 1) & ~(size_t)1; }

td_status td_reserve(td_handle* h, int64_t B_max) {
  if (!h || B_max < 0) return TD_EINVAL;
  if (B_max == 0) return TD_OK;
  DevGuard guard(h->device);
  if (!guard.ok) return TD_ECUDA;
  const int64_t n = h->n_tot, ldh = (n + 1) & ~1ll;
  // staged classes: per-block partial sums for B_max templates (bounded: larger batches run in sub-batches)
  for (const ClassInfo& c : h->classes) {
    if (class_is_fused(h, c)) continue;
    const StagedGeom g = staged_geom(c.log2M);
    const size_t want = std::min<size_t>((size_t)B_max * g.nblk * 2, std::max<size_t>(STAGED_PARTIAL_MAX / sizeof(double), (size_t)g.nblk * 2));
    td_status a = grow(h->wsPartial, h->wsP_elems, want);
    if (a != TD_OK) return a;
  }
  // host entry points: staging of H, d and out; parameter entry points: the synthesis panel and the packed parameter buffer
  const int64_t CH = host_chunk_rows(h, B_max);
  if ((size_t)(CH * n) > h->hsH_elems) {
    for (int i = 0; i < 2; ++i) { cudaFree(h->hsH[i]); h->hsH[i] = nullptr; }
    h->hsH_elems = 0;
    for (int i = 0; i < 2; ++i) CK(cudaMalloc(&h->hsH[i], sizeof(double) * CH * n));
    h->hsH_elems = (size_t)(CH * n);
  }
  if (!h->hsD) CK(cudaMalloc(&h->hsD, sizeof(double) * n));
  td_status a = grow(h->hsOut, h->hsOut_elems, (size_t)B_max);
  if (a == TD_OK) a = grow(h->synH, h->synH_elems, (size_t)(family_chunk_rows(h, B_max, ldh) * ldh));
  if (a == TD_OK) a = grow(h->synP, h->synP_elems, even_up((size_t)(5ll * h->n_seg * B_max)) + even_up((size_t)n) + (size_t)B_max);
  return a;
}

td_status td_loglike_batch_host(td_handle* h, const double* d, const double* H, int64_t ldh, int64_t B, double* out,
                                void* stream) {
  if (!h || B < 0) return TD_EINVAL;
  if (B == 0) return TD_OK;
  if (!d || !H || !out || ldh < h->n_tot) return TD_EINVAL;
  DevGuard guard(h->device);
  if (!guard.ok) return TD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = h->n_tot;
  const int64_t CH = host_chunk_rows(h, B);
  if ((size_t)(CH * n) > h->hsH_elems || (size_t)B > h->hsOut_elems || !h->hsD) {  // not reserved: grow now
    td_status a = td_reserve(h, B);
    if (a != TD_OK) return a;
  }
  h->touched = false;
  td_status s = order_begin(h, st);
  if (s != TD_OK) return s;
  cudaError_t ce = cudaMemcpyAsync(h->hsD, d, sizeof(double) * n, cudaMemcpyHostToDevice, st);
  int launches = 0, k = 0;
  for (int64_t b0 = 0; b0 < B && ce == cudaSuccess && s == TD_OK; b0 += CH, ++k) {
    const int buf = k & 1;
    const int64_t cb = std::min<int64_t>(CH, B - b0);
    if (k >= 2) ce = cudaStreamWaitEvent(h->copy_stream, h->ev_done[buf], 0);  // staging buffer free again
    if (ce == cudaSuccess)
      ce = cudaMemcpy2DAsync(h->hsH[buf], sizeof(double) * n, H + b0 * ldh, sizeof(double) * ldh, sizeof(double) * n,
                             (size_t)cb, cudaMemcpyHostToDevice, h->copy_stream);
    if (ce == cudaSuccess) ce = cudaEventRecord(h->ev_copied[buf], h->copy_stream);
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(st, h->ev_copied[buf], 0);
    if (ce != cudaSuccess) break;
    h->last_launches = 0;
    s = run_batch<MODE_LOGLIKE>(h, h->hsD, h->hsH[buf], n, cb, h->hsOut + b0, nullptr, st);
    launches += h->last_launches;
    if (s == TD_OK) ce = cudaEventRecord(h->ev_done[buf], st);
  }
  h->last_launches = launches;
  if (ce == cudaSuccess && s == TD_OK) ce = cudaMemcpyAsync(out, h->hsOut, sizeof(double) * B, cudaMemcpyDeviceToHost, st);
  // on every path, also after an error: no copy that touches the caller's H / out is left in flight
  const cudaError_t c1 = cudaStreamSynchronize(h->copy_stream), c2 = cudaStreamSynchronize(st);
  h->last_valid = false;  // both streams are idle: nothing to order against
  if (s != TD_OK) return s;
  if (ce != cudaSuccess || c1 != cudaSuccess || c2 != cudaSuccess) return TD_ECUDA;
  return TD_OK;
}

static td_status family_batch_impl(td_handle* h, const double* d, int family, const double* params, int64_t B, double fs,
                                   double* out, cudaStream_t st) {
  // Small batches (launch-bound): the rows are synthesised inside the first pass of the fused kernel, one launch, no panel.
  // Large batches: the separate synthesis kernel + panel is measured 3 % (fp64) to 25 % (fp32) faster on c2, because the
  // in-kernel synthesis puts its exp / sincos anchors on the pipes that already bound the FFT kernel (profiles/r02_ring_fused.md).
  // Segments of 513..1024 samples (M = 1024: four item pipelines per CTA, eight with fp32): the fused route is the faster one at
  // every batch size (B = 16384: fp64 0.271 against 0.275 ms, fp32 0.171 against 0.207 ms; at M = 2048 / 4096 the panel wins
  // by 3-14 %, profiles/r02_ring_fused.md).
  bool short_only = true;
  for (const ClassInfo& c : h->classes) short_only = short_only && c.log2M == 10;
  if (family == SYN_RINGDOWN && ring_fused_ok(h) && (short_only || B <= 2ll * h->num_sms)) {
    h->last_launches = 0;
    return run_ring_fused(h, d, params, B, fs, out, st);
  }
  const int64_t n = h->n_tot, ldh = (n + 1) & ~1ll;  // even leading dimension: 16-byte aligned rows
  const int64_t CH = family_chunk_rows(h, B, ldh);
  {
    td_status a = grow(h->synH, h->synH_elems, (size_t)(CH * ldh));  // no-op after td_reserve / the first call
    if (a != TD_OK) return a;
  }
  h->touched = true;
  int launches = 0;
  for (int64_t b0 = 0; b0 < B; b0 += CH) {
    const int64_t cb = std::min<int64_t>(CH, B - b0);
    const dim3 sgrid((unsigned)cb, (unsigned)h->n_seg);
    if (family == SYN_RINGDOWN) synth_kernel<SYN_RINGDOWN><<<sgrid, SYN_NT, 0, st>>>(params, b0, (int)cb, h->synSeg, h->n_seg, fs, h->synH, ldh);
    else if (family == SYN_SINEGAUSS) synth_kernel<SYN_SINEGAUSS><<<sgrid, SYN_NT, 0, st>>>(params, b0, (int)cb, h->synSeg, h->n_seg, fs, h->synH, ldh);
    else synth_kernel<SYN_CHIRP><<<sgrid, SYN_NT, 0, st>>>(params, b0, (int)cb, h->synSeg, h->n_seg, fs, h->synH, ldh);
    CK(cudaGetLastError());
    h->last_launches = 0;
    td_status s = run_batch<MODE_LOGLIKE>(h, d, h->synH, ldh, cb, out + b0, nullptr, st);
    if (s != TD_OK) return s;
    launches += 1 + h->last_launches;
  }
  h->last_launches = launches;
  return TD_OK;
}

td_status td_loglike_family_batch(td_handle* h, const double* d, int family, const double* params, int64_t B, double fs,
                                  double* out, void* stream) {
  if (!h || B < 0 || family < 0 || family >= SYN_NFAM) return TD_EINVAL;
  if (B == 0) return TD_OK;
  if (!d || !params || !out || !(fs > 0.0)) return TD_EINVAL;
  DevGuard guard(h->device);
  if (!guard.ok) return TD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  td_status s = order_begin(h, st);
  if (s != TD_OK) return s;
  s = family_batch_impl(h, d, family, params, B, fs, out, st);
  const td_status e = order_end(h, st);
  return s != TD_OK ? s : e;
}

td_status td_loglike_family_batch_host(td_handle* h, const double* d, int family, const double* params, int64_t B,
                                       double fs, double* out, void* stream) {
  if (!h || B < 0 || family < 0 || family >= SYN_NFAM) return TD_EINVAL;
  if (B == 0) return TD_OK;
  if (!d || !params || !out || !(fs > 0.0)) return TD_EINVAL;
  DevGuard guard(h->device);
  if (!guard.ok) return TD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t n = h->n_tot, np5 = 5ll * h->n_seg * B;
  const size_t offD = even_up((size_t)np5), offO = offD + even_up((size_t)n);  // parameters | data vector | results
  {
    td_status a = grow(h->synP, h->synP_elems, offO + (size_t)B);  // no-op after td_reserve
    if (a != TD_OK) return a;
  }
  td_status s = order_begin(h, st);
  if (s != TD_OK) return s;
  double* dP = h->synP; double* dD = dP + offD; double* dO = dP + offO;
  cudaError_t ce = cudaMemcpyAsync(dP, params, sizeof(double) * np5, cudaMemcpyHostToDevice, st);
  if (ce == cudaSuccess) ce = cudaMemcpyAsync(dD, d, sizeof(double) * n, cudaMemcpyHostToDevice, st);
  if (ce == cudaSuccess) s = family_batch_impl(h, dD, family, dP, B, fs, dO, st);
  if (ce == cudaSuccess && s == TD_OK) ce = cudaMemcpyAsync(out, dO, sizeof(double) * B, cudaMemcpyDeviceToHost, st);
  const cudaError_t c2 = cudaStreamSynchronize(st);  // on every path: no copy touching the caller's buffers stays in flight
  h->last_valid = false;
  if (s != TD_OK) return s;
  return (ce != cudaSuccess || c2 != cudaSuccess) ? TD_ECUDA : TD_OK;
}

td_status td_inner_batch(td_handle* h, const double* d, const double* H, int64_t ldh, int64_t B, double* out_dh,
                         double* out_hh, void* stream) {
  if (!h || B < 0) return TD_EINVAL;
  if (B == 0 || (!out_dh && !out_hh)) return TD_OK;
  if (!d || !H || ldh < h->n_tot) return TD_EINVAL;
  DevGuard guard(h->device);
  if (!guard.ok) return TD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_launches = 0;
  td_status s = order_begin(h, st);
  if (s != TD_OK) return s;
  h->touched = true;  // z of the data vector (and u on the dot path) live in the handle
  // z of the data vector, once per call (per segment), then the bilinear sums against it
  // only the cross term is wanted: one streaming pass over H against the cached weights u = C^{-1} d (fp64 in both
  // precisions: the pass is HBM-bound, and u needs the fp64 z of the data vector)
  const bool use_dot = out_dh && !out_hh && h->path == TD_PATH_AUTO && h->max_n <= DOT_MAX_N && h->n_tot <= 0x7fffffff;
  s = run_fft_path<MODE_STOREZ>(h, d, nullptr, h->n_tot, 1, nullptr, nullptr, st, false, 0,
                                h->precision == TD_PREC_F32 && !use_dot);
  if (s == TD_OK) {
    if (use_dot)
      s = run_dot(h, H, ldh, B, out_dh, st);
    else
      s = run_batch<MODE_INNER>(h, d, H, ldh, B, out_dh, out_hh, st);
  }
  const td_status e = order_end(h, st);
  return s != TD_OK ? s : e;
}

td_status td_set_path(td_handle* h, int path) {
  if (!h || (path != TD_PATH_AUTO && path != TD_PATH_FFT && path != TD_PATH_DENSE && path != TD_PATH_CDO)) return TD_EINVAL;
  if ((path == TD_PATH_DENSE || path == TD_PATH_CDO) && h->max_n > h->dense.max_n) return TD_EUNSUPPORTED;
  if (path == TD_PATH_CDO) {   // first use: builds W = L^{-1} per segment (synchronous), configures the kernel
    DevGuard guard(h->device);
    if (!guard.ok) return TD_ECUDA;
    td_status s = cdo_setup(h, true);
    if (s == TD_OK) s = launch_cdo(h, nullptr, nullptr, h->n_tot, 1, nullptr, 0, nullptr, true, nullptr, true);
    if (s != TD_OK) return s;
  }
  h->path = path;
  return TD_OK;
}

td_status td_set_fft_variant(td_handle* h, int variant) {
  if (!h || variant < 0 || variant > 4) return TD_EINVAL;
  if (variant == 4) {   // 4- / 8- / 16-CTA groups exchanging through L2: what variant 0 uses for the 16384 ... 65536 classes when it can
    bool any = false;
    for (const ClassInfo& c : h->classes) any = any || (group_cs(c.log2M) && h->group_cap[group_slot(group_cs(c.log2M))] > 0);
    if (!any) return TD_EUNSUPPORTED;
  }
  if (variant == 3) {   // the 16-CTA cluster kernel needs a 65536-class segment and a device that can host the cluster
    bool has16 = false;
    for (const ClassInfo& c : h->classes) has16 = has16 || c.log2M == Cluster16Shape::LOG2M;
    if (!has16) return TD_EUNSUPPORTED;
    DevGuard guard(h->device);
    if (!guard.ok) return TD_ECUDA;
    if (h->cluster16_cap < 1) h->cluster16_cap = cluster16_capacity(h);   // configures the kernels, asks how many clusters fit
    if (h->cluster16_cap < 1) return TD_EUNSUPPORTED;
  }
  if (variant == 2) {
    DevGuard guard(h->device);
    if (!guard.ok) return TD_ECUDA;
    td_status a = staged_alloc(h, true);
    if (a != TD_OK) return a;
  }
  h->fft_variant = variant;
  return TD_OK;
}

td_status td_set_precision(td_handle* h, int precision) {
  if (!h || (precision != TD_PREC_F64 && precision != TD_PREC_F32)) return TD_EINVAL;
  if (precision == TD_PREC_F32) {
    DevGuard guard(h->device);
    if (!guard.ok) return TD_ECUDA;
    bool any = false;
    for (ClassInfo& c : h->classes) {
      if (!td32api::supported(c.log2M)) continue;
      any = true;
      if (c.has32) continue;
      std::vector<td32api::SegIn> in(c.seg_ids.size());
      for (size_t i = 0; i < in.size(); ++i) {
        const SegHost& sg = h->segs[c.seg_ids[i]];
        in[i].off = sg.off; in[i].n = sg.n; in[i].sid = c.seg_ids[i]; in[i].Gp64 = sg.Gp; in[i].G64 = sg.G; in[i].rho0 = sg.rho0; in[i].Gc64 = sg.Gc16;
      }
      td_status s = td32api::build_class(c.log2M, (int)in.size(), in.data(), c.T, &c.t32);
      if (s != TD_OK) return s;
      c.has32 = true;
      for (int mode = 0; mode < 3; ++mode) {  // dry pass: attributes and occupancy of the fp32 kernels
        td32api::Launch L = {};
        L.B = 1; L.mode = mode;
        s = td32api::launch(c.t32, L, h->num_sms, h->device, nullptr, true);
        if (s != TD_OK) return s;
      }
      if (c.log2M <= 12) {   // and of the fp32 kernel that synthesises ringdown rows in its first pass
        td32api::Launch L = {};
        L.B = 1; L.mode = MODE_LOGLIKE; L.syn = 1; L.fs = 1.0;
        s = td32api::launch(c.t32, L, h->num_sms, h->device, nullptr, true);
        if (s != TD_OK) return s;
      }
    }
    if (!any) return TD_EUNSUPPORTED;  // no size class of this handle has an fp32 kernel
  }
  h->precision = precision;
  return TD_OK;
}

td_status td_get_info(const td_handle* h, int64_t* n_tot, int* n_seg, double* v, double* logdet, int* last_path) {
  if (!h) return TD_EINVAL;
  if (n_tot) *n_tot = h->n_tot;
  if (n_seg) *n_seg = h->n_seg;
  for (int s = 0; s < h->n_seg; ++s) {
    if (v) v[s] = h->segs[s].v;
    if (logdet) logdet[s] = h->segs[s].logdet;
  }
  if (last_path) *last_path = h->last_path;
  return TD_OK;
}

td_status td_get_generator(const td_handle* h, int seg, double* a) {
  if (!h || !a || seg < 0 || seg >= h->n_seg) return TD_EINVAL;
  DevGuard guard(h->device);
  if (!guard.ok) return TD_ECUDA;
  CK(cudaMemcpy(a, h->segs[seg].a, sizeof(double) * h->segs[seg].n, cudaMemcpyDeviceToHost));
  return TD_OK;
}

int td_last_launches(const td_handle* h) { return h ? h->last_launches : 0; }

#ifdef TD_PHASE_CLOCKS
int td_debug_phase_clocks(long long* host, int n) {
  return (int)cudaMemcpyFromSymbol(host, td::g_phase_clk, sizeof(long long) * n);
}
#endif

}  // extern "C"

// ------------------------------------------------------------------------------------------------------------------------
// td_loglike_batch_static - the log-likelihood through the staged kernels (td_staged.cuh) with their workspace in a file-scope
// device array instead of the handle's cudaMalloc'ed buffers: for callers that may not allocate (include/tdlike.h).
// New code only: it shares the kernels and the launch helpers of td_staged_host.cuh with the existing path and none of its
// buffers.  The array belongs to the library image: every GPU that loads libtdlike.so holds TD_STATIC_SCRATCH_BYTES of it
// until the process exits.
// ------------------------------------------------------------------------------------------------------------------------
#include <mutex>

static __device__ __align__(256) unsigned char td_static_scratch[TD_STATIC_SCRATCH_BYTES];

namespace {

// In host code `td_static_scratch` is only the host-side shadow of the symbol: its DEVICE address comes from
// cudaGetSymbolAddress, once per device, with that device current.
void* g_static_dev_ptr[TD_MAX_DEV];
std::mutex g_static_mu;
thread_local char g_static_err[256] = "";

td_status static_fail(td_status s, const char* fmt, long long a = 0, long long b = 0, long long c = 0) {
  std::snprintf(g_static_err, sizeof(g_static_err), fmt, a, b, c);
  return s;
}

// the caller holds a DevGuard on `device`
td_status static_scratch_address(int device, unsigned char** out) {
  if (device < 0 || device >= TD_MAX_DEV) return static_fail(TD_EUNSUPPORTED, "device index %lld is beyond the %lld this library tracks", device, TD_MAX_DEV);
  std::lock_guard<std::mutex> lk(g_static_mu);
  if (!g_static_dev_ptr[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, td_static_scratch);
    if (e != cudaSuccess || !p) {
      cudaGetLastError();
      return static_fail(TD_ECUDA, "cudaGetSymbolAddress(td_static_scratch) failed on device %lld (CUDA error %lld)", device, (long long)e);
    }
    g_static_dev_ptr[device] = p;
  }
  *out = static_cast<unsigned char*>(g_static_dev_ptr[device]);
  return TD_OK;
}

// bytes of scratch one template of a size class needs: U [2][M/2] + Z [2][M] complex, per-block partial sums [nblk][2]
size_t static_bytes_per_template(int log2M) {
  const StagedGeom g = staged_geom(log2M);
  return sizeof(cplx) * 3 * ((size_t)1 << log2M) + sizeof(double) * 2 * (size_t)g.nblk;
}

}  // namespace

extern "C" {

size_t td_static_scratch_bytes(void) { return TD_STATIC_SCRATCH_BYTES; }
const char* td_static_last_error(void) { return g_static_err; }

td_status td_static_setup(int device) {
  g_static_err[0] = 0;
  DevGuard guard(device);
  if (!guard.ok) return static_fail(TD_ECUDA, "cannot make device %lld current", device);
  unsigned char* p = nullptr;
  td_status s = static_scratch_address(device, &p);
  if (s != TD_OK) return s;
  // the launch configuration of the two shared-memory block kernels (attribute + occupancy, cached per device)
  s = launch_block<true>(device, nullptr, 0, 0, nullptr, 0, nullptr, true);
  if (s == TD_OK) s = launch_block<false>(device, nullptr, 0, 0, nullptr, 0, nullptr, true);
  if (s != TD_OK) return static_fail(s, "the staged block kernels cannot be configured on device %lld", device);
  return TD_OK;
}

td_status td_loglike_batch_static(td_handle* h, const double* d, const double* H, int64_t ldh, int64_t B, double* out,
                                  void* stream) {
  g_static_err[0] = 0;
  if (!h || B < 0) return static_fail(TD_EINVAL, "null handle or negative batch size");
  if (B == 0) return TD_OK;
  if (!d || !H || !out || ldh < h->n_tot) return static_fail(TD_EINVAL, "null pointer, or ldh = %lld below N_tot = %lld", ldh, h->n_tot);
  // every size class must fit at least one template into the array: refuse before anything is launched
  for (const ClassInfo& cls : h->classes) {
    const size_t need = static_bytes_per_template(cls.log2M);
    if (need > TD_STATIC_SCRATCH_BYTES)
      return static_fail(TD_EUNSUPPORTED, "a segment of up to %lld samples needs %lld bytes of scratch per template; the static array holds %lld "
                         "(segments of at most 262144 samples)", 1ll << cls.log2M, (long long)need, (long long)TD_STATIC_SCRATCH_BYTES);
  }
  DevGuard guard(h->device);
  if (!guard.ok) return static_fail(TD_ECUDA, "cannot make device %lld current", h->device);
  unsigned char* base = nullptr;
  td_status s = static_scratch_address(h->device, &base);   // (a table look-up after td_static_setup / the first call)
  if (s != TD_OK) return s;
  cudaStream_t st = (cudaStream_t)stream;
  h->last_launches = 0;
  int accumulate = 0;
  for (const ClassInfo& cls : h->classes) {
    const int log2M = cls.log2M, M = 1 << log2M, nf = M / 2, TW = 2 * M;
    const StagedGeom g = staged_geom(log2M);   // only the radices and the block count are used: the chunk size is ours
    const int64_t CB = std::min<int64_t>({(int64_t)(TD_STATIC_SCRATCH_BYTES / static_bytes_per_template(log2M)), (int64_t)32767, B});
    // one chunk's layout inside the array: U | Z | partial sums (each region a multiple of 16 bytes, the base 256-aligned)
    cplx* const U = reinterpret_cast<cplx*>(base);
    cplx* const Z = U + (size_t)CB * 2 * nf;
    double* const part = reinterpret_cast<double*>(Z + (size_t)CB * 2 * M);
    for (size_t i = 0; i < cls.seg_ids.size(); ++i) {
      const SegHost& sg = h->segs[cls.seg_ids[i]];
      SegDev sd;
      sd.off = sg.off; sd.n = sg.n; sd._pad = 0; sd.G = sg.G; sd.zd = sg.zd; sd.rscale = 1.0;
      for (int64_t b0 = 0; b0 < B; b0 += CB) {
        const int cb = (int)std::min<int64_t>(CB, B - b0);
        StagedParams P;
        P.d = d; P.H = H + b0 * ldh; P.ldh = ldh; P.CB = cb; P.seg = sd;
        P.M = M; P.U = U; P.Z = Z; P.T = cls.T; P.partial = part; P.nblk = g.nblk;
        s = launch_first<MODE_LOGLIKE>(g.rF, dim3((nf / g.rF + LG_NT - 1) / LG_NT, cb), P, st);
        if (s == TD_OK) { ++h->last_launches; s = staged_forward(h->device, U, 2 * cb, nf, 1, cls.T, TW, st, &h->last_launches); }
        if (s == TD_OK) {
          lg_untangle_kernel<<<dim3((nf + LG_NT - 1) / LG_NT, 2, (cb + LG_UCPT - 1) / LG_UCPT), LG_NT, 0, st>>>(P);
          s = cudaGetLastError() == cudaSuccess ? TD_OK : TD_ECUDA;
          ++h->last_launches;
        }
        if (s == TD_OK) s = staged_inverse_but_last(h->device, Z, 2 * cb, M, cls.T, TW, st, &h->last_launches);
        if (s == TD_OK) { s = launch_last<MODE_LOGLIKE>(g.rI, dim3(g.nblk, cb), P, st); ++h->last_launches; }
        if (s == TD_OK) {   // the chunk's partial sums, in block order, into out[b0 .. b0 + cb)
          lg_finish_kernel<<<(unsigned)((cb + 127) / 128), 128, 0, st>>>(part, g.nblk, cb, out + b0, nullptr, -0.5, 1.0, accumulate);
          s = cudaGetLastError() == cudaSuccess ? TD_OK : TD_ECUDA;
          ++h->last_launches;
        }
        if (s != TD_OK) return static_fail(s, "a kernel launch failed (segment %lld, template %lld)", cls.seg_ids[i], b0);
      }
      accumulate = 1;
    }
  }
  h->last_path = TD_PATH_FFT;
  return TD_OK;
}

}  // extern "C"
